// Internal declarations shared by the translation units of libpgsf.so (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>
#include <vector>

#include "pgsf.h"

namespace pgsf {

constexpr int kMaxTaps = 2 * PGSF_MAX_RADIUS + 1;  // 193

// Voxel selection is evaluated as  n f - S1 > k sqrt(max(n S2 - S1^2, 0)).  Where the window is flat
// to fp32 precision (sd below ~3e-4 |mean|, the rounding floor of S2/n - m^2 in fp32) the sign of
// n f - S1 is rounding noise; requiring n f - S1 > kFlatGuard * n |f| keeps such regions unselected
// ("with std = 0 nothing is selected", reading C-10) and cannot change a well-conditioned decision.
constexpr float kFlatGuard = 1e-5f;

// Taps of one axis, passed BY VALUE as a kernel parameter: kernel parameters live in constant
// bank 0, so a compile-time tap index becomes a uniform-register operand of FFMA/FFMA2 (the role
// constant memory plays in the paper's kernel) without any per-module __constant__
// state shared between plans.
constexpr int kTapPad = 8;  // zero taps in front of (and behind) the z taps of the tiled kernel
struct Taps {
    float g[kMaxTaps + 2 * kTapPad + 2];  // generic path: g[o + r], o = -r..r; zero beyond
    int r;                                // tiled z pass:  g[o + r + kTapPad]
};

struct TapsXY {  // small radii only (x and y passes)
    float gx[32];
    float gy[32];
};

struct ScalePlan {
    int r[3];            // true radii ceil(truncate*sigma)
    int rxy_c;           // compiled radius used by the fast xy kernel (>= max(r[0], r[1])), 0 = none
    int rz_c;            // compiled radius used by the fast z kernel (>= r[2]), 0 = none
    Taps taps[3];        // true taps (generic path; also what pgsf_plan_get_taps reports)
    TapsXY txy;          // taps centred in a 2*rxy_c+1 window, zero padded
    Taps tz;             // taps centred in a 2*rz_c+1 window, zero padded
    TapsXY txy_box;      // all-ones taps over the true radii: the box of the filter support (Eq. 1 denominator)
    Taps tz_box;
};

struct Dims {
    int nx, ny, nz;
    long long plane;     // nx*ny
    long long cube;      // nx*ny*nz
};

// A section of the frequency march of k_zm (pgsf_find_multiscale_host): entering channels [c0, c1), multiples of
// the kernel's step; `state` = 4 planes of floats carrying the running window sums between the sections' launches.
// The cube pointers of such a launch are VIRTUAL: buffer - (first buffered plane) * plane.
struct ZmSection {
    int c0, c1;
    float *state;
    const float *t2_buf;     // the buffer behind the virtual input pointer: channels t2_base .. t2_hi - 1 (for the TMA map)
    int t2_base, t2_hi;
};

}  // namespace pgsf

namespace pgsf {
// Optional per-kernel timing (pgsf_plan_set_profiling): one cudaEvent pair around every launch, on
// the stream the kernel is launched on; durations are summed per kernel name on collect.
struct ProfRec {
    int name_id;
    cudaEvent_t a, b;
};
struct ProfAcc {
    std::string name;
    unsigned long long launches;
    double ms;
};
}  // namespace pgsf

struct pgsf_plan {
    pgsf_plan_desc desc;
    double sigmas[PGSF_MAX_SCALES * 3];
    pgsf::ScalePlan scales[PGSF_MAX_SCALES];
    pgsf::Dims dims;
    int device;
    bool dry;            // PGSF_FLAG_DRY_RUN: no device behind this plan
    int sm_count;
    bool fast_filter;    // all scales have compiled radii, nx % 4 == 0
    bool fast_stats;
    size_t ws_bytes;     // total workspace
    size_t ws_cube_bytes;
    int group;           // cubes of a batch that the fast path of pgsf_find_multiscale processes per launch
    int group_max;       // the plan's default (the workspace is sized for it); PGSF_OPT_GROUP_CUBES lowers `group`
    std::string why_filter, why_stats;   // why a stage runs the generic kernels ("" = tiled); pgsf_plan_path
    long long host_section_planes;       // PGSF_OPT_HOST_SECTION_PLANES (0 = automatic)
    long long host_budget;               // PGSF_OPT_HOST_DEVICE_BUDGET  (0 = automatic)
    int tune;                            // PGSF_OPT_TUNE bits (measurement aid; no bit changes a result)
    unsigned long long launches;
    std::string err;
    bool prof_on;
    std::vector<pgsf::ProfRec> prof_recs;      // pending (not yet collected) launches
    std::vector<cudaEvent_t> prof_free;        // recycled events
    std::vector<pgsf::ProfAcc> prof_acc;
    float *d_pivot;      // device scalar: the constant the statistics subtract from f before squaring (D-2)
    // plan-owned device staging for pgsf_find_multiscale_host
    float *h_d_in;
    float *h_d_f[PGSF_MAX_SCALES];
    uint8_t *h_d_mask;
    unsigned long long *h_d_count;
    void *h_d_ws;
    cudaStream_t h_stream;
    struct pgsf_host_stage *hs;          // streamed sections (pgsf_host.cu)
    bool tensor_z;                       // PGSF_FLAG_TENSOR_ZPASS: k_ztc for compiled z radii >= 24 (pgsf_ztc.cu)
    float *d_tc_strips[PGSF_MAX_SCALES]; // its band-matrix operands
    int tc_march[PGSF_MAX_SCALES];       // kernel of the march in progress (sections): 0 none yet, 1 k_ztc, 2 k_zm
};

namespace pgsf {

// Counts a launch and, when profiling is on, brackets it with events on `st`.
struct LaunchScope {
    pgsf_plan *p;
    cudaStream_t st;
    cudaEvent_t b;
    LaunchScope(pgsf_plan *plan, const char *name, cudaStream_t stream);
    ~LaunchScope();
};

// ---- generic kernels (pgsf_generic.cu): any shape, any radius <= PGSF_MAX_RADIUS ----------------
cudaError_t generic_filter3d(pgsf_plan *p, int scale, const float *in, float *out, float *tmp_a,
                             float *tmp_b, cudaStream_t st);
// Pivot of the statistics (D-2): *p->d_pivot = mean of a lattice of <= 10^6 samples of the central half
// of the cube at `data` (for a group of cubes: of its first cube).
// The selection n f - S1 > k sqrt(n S2 - S1^2) is invariant under f -> f - c for any constant c; taking c near the
// level of the data keeps S2/n - m^2 well conditioned in fp32 when the cube carries an offset |mean| >> sd.
// 64 CTAs reduce fixed ranges of the samples, one thread adds their partial sums in order (deterministic; exact under
// power-of-two scaling of the data).
cudaError_t compute_pivot(pgsf_plan *p, const float *data, cudaStream_t st);
// tmp: 4 cubes
cudaError_t generic_threshold(pgsf_plan *p, const float *f, uint8_t *mask, int or_into, float *mean,
                              float *sd, unsigned long long *count, float *tmp4, cudaStream_t st);

// ---- fast kernels (pgsf_filter.cu, pgsf_stats.cu): nx % 4 == 0, 16-byte aligned, compiled radii --
bool fast_xy_radius(int r, int *compiled);
bool fast_z_radius(int r, int *compiled);
// box = true: the same passes with all-ones taps (sum over the box of the filter support);
// wgt != NULL: the input is multiplied by this cube while it is staged (numerator of Eq. 1);
// ratio != NULL: the result is not written to `out` but divides the cube `ratio` in place (denominator of Eq. 1)
cudaError_t fast_filter3d(pgsf_plan *p, int scale, const float *in, float *out, float *tmp,
                          cudaStream_t st, bool box = false, const float *wgt = nullptr, float *ratio = nullptr);
// `ncubes` consecutive cubes (stride dims.cube) per call, for the entry points that take it
// nplanes > 0: a stack of that many planes instead of ncubes whole cubes (the x and y passes do not couple planes)
cudaError_t fast_xy_multi(pgsf_plan *p, const int *scales, int n, const float *in, float *const *out, int ncubes,
                          cudaStream_t st, bool box = false, const float *wgt = nullptr, int nplanes = 0);
cudaError_t fast_z(pgsf_plan *p, int scale, const float *in, float *out, cudaStream_t st, bool box = false,
                   float *ratio = nullptr);
cudaError_t fast_zm(pgsf_plan *p, int scale, const float *in, float *out, float *Z1, float *Z2, int ncubes,
                    cudaStream_t st, const ZmSection *sec = nullptr);
// channels per march step of k_zm<RZ>: 64, or 128 where the slab of 64 + 2 RZ channels would leave room for two 4-warp
// CTAs only (RZ = 96) and -- PGSF_ZM_WIDE_STEP_MAX_RZ, a build-time experiment -- for small radii
#ifndef PGSF_ZM_WIDE_STEP_MAX_RZ
#define PGSF_ZM_WIDE_STEP_MAX_RZ 0
#endif
constexpr int zm_step_rule(int rz_compiled) { return (rz_compiled >= 96 || rz_compiled <= PGSF_ZM_WIDE_STEP_MAX_RZ) ? 128 : 64; }
int zm_step_channels_of(int rz_compiled);
// the tensor-core variant of fast_zm (pgsf_ztc.cu): cudaErrorNotSupported = not for this plan / scale, run fast_zm
bool ztc_radius(int rz_compiled);
// channels per march step of the tensor-core z pass if `scale` runs on it in this plan, else 0
int ztc_step_channels(const pgsf_plan *p, int scale);
cudaError_t ztc_prepare(pgsf_plan *p);
void ztc_release(pgsf_plan *p);
cudaError_t fast_ztc(pgsf_plan *p, int scale, const float *in, float *out, float *Z1, float *Z2, int ncubes,
                     cudaStream_t st, const ZmSection *sec = nullptr);
bool fast_stats_supported(const pgsf_plan *p, std::string *why);
// frees the plan-owned staging of pgsf_find_multiscale_host (buffers, streams, events); the plan's device must be current
void host_release(pgsf_plan *p);
void host_stage_release(pgsf_plan *p);      // (pgsf_host.cu)
// the streamed form of pgsf_find_multiscale_host; *handled = false if this plan / call cannot be streamed
pgsf_status host_streamed(pgsf_plan *p, const float *h_in, float *const *h_filtered, uint8_t *h_mask,
                          unsigned long long *h_count, bool *handled);
// x/y window sums + selection from precomputed z-direction window sums Z1, Z2 (of fast_zm / k_zbox)
// mode: 0 overwrite the mask, 1 OR into it (count = all set voxels), 2 sparse OR (only with stats_sparse_or():
// touches only newly selected bytes, count += voxels that were not set before)
cudaError_t fast_threshold_xy(pgsf_plan *p, const float *f, const float *Z1, const float *Z2, uint8_t *mask,
                              int mode, float *mean, float *sd, unsigned long long *count, int ncubes,
                              cudaStream_t st);
// k_xyb (pgsf_xyb.cu): the successor of k_ymarch; same arguments
bool xyb_supported(const pgsf_plan *p);
inline bool stats_sparse_or(const pgsf_plan *p)
{
    const int hx = p->desc.box_half[0];
    const bool legacy_ok = (hx == 4 || hx == 8 || hx == 16) && p->desc.nx % (hx / 2) == 0;
    return p->fast_stats && xyb_supported(p) && (!(p->tune & 2) || !legacy_ok);
}
// nplanes > 0: the pointers address planes z_off .. z_off + nplanes - 1 of one cube (a section of the streamed cube)
cudaError_t xyb_threshold(pgsf_plan *p, const float *f, const float *Z1, const float *Z2, uint8_t *mask, int mode,
                          float *mean, float *sd, unsigned long long *count, int ncubes, cudaStream_t st,
                          int nplanes = 0, int z_off = 0);
// pivot from a list of samples already gathered in lattice order (pgsf_find_multiscale_host gathers them on the host)
void pivot_lattice(const Dims &d, int lo[3], int st[3], int cnt[3]);
cudaError_t compute_pivot_list(pgsf_plan *p, const float *d_list, int nsamp, cudaStream_t st);
// tmp2: 2 cubes (the z-direction window sums of f and f^2)
cudaError_t fast_threshold(pgsf_plan *p, const float *f, uint8_t *mask, int or_into, float *mean,
                           float *sd, unsigned long long *count, float *tmp2, cudaStream_t st);

// ---- Eq. 1, weighted convolution (pgsf_weighted.cu): one cube per call
cudaError_t weighted_mul(pgsf_plan *p, const float *d, const float *w, float *prod, cudaStream_t st);
cudaError_t weighted_boxsum(pgsf_plan *p, int scale, const float *w, float *a, float *b, cudaStream_t st);
cudaError_t weighted_div(pgsf_plan *p, float *c, const float *den, cudaStream_t st);

// ---- NEXT-4: connected components of the mask (pgsf_label.cu): the whole batch per call
cudaError_t label_objects(pgsf_plan *p, const uint8_t *mask, unsigned *labels, unsigned long long *count, cudaStream_t st);

// ---- Eq. 2 for an arbitrary filter array, direct summation (pgsf_direct.cu): one cube per call
bool direct_supported(const pgsf_plan *p, int rx, int ry, int rz, int *smem_bytes);
cudaError_t direct_filter3d(pgsf_plan *p, const float *filt, int rx, int ry, int rz, const float *in, float *out,
                            bool fp64, cudaStream_t st);

}  // namespace pgsf
