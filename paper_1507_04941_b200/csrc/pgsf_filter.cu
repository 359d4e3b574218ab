// Tiled sm_100a filter kernels (placeholder until the fast path lands).
#include "pgsf_internal.h"
namespace pgsf {
bool fast_xy_radius(int, int *c) { *c = 0; return false; }
bool fast_z_radius(int, int *c) { *c = 0; return false; }
cudaError_t fast_filter3d(pgsf_plan *, int, const float *, float *, float *, cudaStream_t) { return cudaErrorNotSupported; }
}  // namespace pgsf
