// Tiled sm_100a local-statistics kernel (placeholder until the fast path lands).
#include "pgsf_internal.h"
namespace pgsf {
bool fast_stats_supported(const pgsf_plan *) { return false; }
cudaError_t fast_threshold(pgsf_plan *, const float *, uint8_t *, int, float *, float *, unsigned long long *, cudaStream_t) { return cudaErrorNotSupported; }
}  // namespace pgsf
