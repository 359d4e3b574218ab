// Tiled sm_100a kernels for the separable form of Eq. 2 (index ranges Eq. 3-5).
//
//   k_xym<NS,R..> : per z-plane, the x and y passes of up to four scales from one read of the input
//              (this file); result t2 to HBM.
//   k_z<RZ>, k_zm<RZ> : the frequency axis (filters are largest along z), alone or fused with the
//              z-direction window sums of the statistics (pgsf_zpass.cuh, one translation unit per radius).
//
// Both passes are plain FP32 FMAs: the inner loops are packed `fma.rn.f32x2` (SASS FFMA2) whose
// tap operand is a kernel-parameter constant, i.e. a uniform register broadcast -- the sm_100a form
// of the paper's "filter value is read from constant memory".  One FFMA2 retires two
// voxel-taps per issue slot, which leaves issue slots for the shared-memory loads.
//
// Preconditions (checked by the plan): nx % 4 == 0, 16-byte aligned cubes, radius in the compiled
// set (smaller radii run in the next larger window with exact-zero padding taps).
#include <stdio.h>

#include "pgsf_internal.h"
#include "pgsf_device.cuh"

namespace pgsf {
// per-radius entry points of the frequency-axis kernels (pgsf_z_r*.cu)
cudaError_t launch_z_r6(const float *in, float *out, float *ratio, const Dims &d, const Taps &t, cudaStream_t st, bool tma);
cudaError_t launch_zm_r6(const float *in, float *out, float *Z1, float *Z2, const Dims &d, int hz, const float *pivot, const Taps &t, int ncubes, cudaStream_t st, const ZmSection *sec, bool tma);
cudaError_t launch_z_r12(const float *in, float *out, float *ratio, const Dims &d, const Taps &t, cudaStream_t st, bool tma);
cudaError_t launch_zm_r12(const float *in, float *out, float *Z1, float *Z2, const Dims &d, int hz, const float *pivot, const Taps &t, int ncubes, cudaStream_t st, const ZmSection *sec, bool tma);
cudaError_t launch_z_r24(const float *in, float *out, float *ratio, const Dims &d, const Taps &t, cudaStream_t st, bool tma);
cudaError_t launch_zm_r24(const float *in, float *out, float *Z1, float *Z2, const Dims &d, int hz, const float *pivot, const Taps &t, int ncubes, cudaStream_t st, const ZmSection *sec, bool tma);
cudaError_t launch_z_r48(const float *in, float *out, float *ratio, const Dims &d, const Taps &t, cudaStream_t st, bool tma);
cudaError_t launch_zm_r48(const float *in, float *out, float *Z1, float *Z2, const Dims &d, int hz, const float *pivot, const Taps &t, int ncubes, cudaStream_t st, const ZmSection *sec, bool tma);
cudaError_t launch_z_r72(const float *in, float *out, float *ratio, const Dims &d, const Taps &t, cudaStream_t st, bool tma);
cudaError_t launch_zm_r72(const float *in, float *out, float *Z1, float *Z2, const Dims &d, int hz, const float *pivot, const Taps &t, int ncubes, cudaStream_t st, const ZmSection *sec, bool tma);
cudaError_t launch_z_r96(const float *in, float *out, float *ratio, const Dims &d, const Taps &t, cudaStream_t st, bool tma);
cudaError_t launch_zm_r96(const float *in, float *out, float *Z1, float *Z2, const Dims &d, int hz, const float *pivot, const Taps &t, int ncubes, cudaStream_t st, const ZmSection *sec, bool tma);

namespace {

// ------------------------------------------------------------------------------------ x/y passes
//
// k_xym<NS, RA..RD>: one CTA = one z plane, a strip of 256 columns, one chunk of rows; it marches
// down y in batches of 8 row PAIRS and evaluates the x and y passes of up to four scales from ONE
// read of the input ("several sigma scales evaluated per input read", BASELINE.json north_star).
//   x pass (Eq. 3): warp w stages row pair w of the batch (+16 columns either side, zero fill outside
//                   the cube = C-5) with the two rows interleaved, so one LDS.128 yields two columns
//                   of both rows; a lane owns 8 columns x 2 rows and gathers its taps as packed
//                   FFMA2 over the row pair.  Results u go to shared memory, one slab per scale.
//   y pass (Eq. 4): a thread owns ONE column and keeps the R + 1 unfinished output row pairs of
//                   every scale in registers.  Each new pair (u[2k], u[2k+1]) is scattered into
//                   them with FFMA2 (even taps use the pair as loaded, odd taps the pair shifted by
//                   one row), the accumulators rotate through the destination register of the
//                   FFMA2 (no moves), and the pair that has seen all its taps is stored.
// Both passes are pure FFMA2 streams with uniform-register taps; no y halo is recomputed and the
// only shared-memory traffic is the x pass' operand reads.

constexpr int XM_HALO = 16;         // staged columns either side (>= largest x radius, multiple of 4)
constexpr int XM_MAXS = 4;
// GS = columns per lane of the x pass: 8 (256-column strips, 8 warps) or 4 (128-column strips, 4 warps: cubes whose nx
// would leave most of a second 256-column strip idle, e.g. nx = 320)
template <int GS>
struct XmShape {
    static constexpr int NT = 32 * GS;          // threads = columns per CTA
    static constexpr int NB = GS;               // row pairs per batch (= warps)
    static constexpr int SW = NT + 2 * XM_HALO;
    static constexpr int GP = GS == 8 ? 10 : 6; // pitch in pairs of a GS-column group (even; spreads the banks)
    static constexpr int SIN = (SW / GS) * GP;  // pairs of one staged row pair
    static constexpr int U = (NT / GS) * GP;    // pairs of one x-filtered row pair
    static constexpr int NQ = (SW / 4 + 31) / 32;   // float4 loads per lane and staged row
};

// 128-column strips where they stage fewer columns than 256-column ones (nx = 320: 3 x 128 against 2 x 256)
inline int xm_strip_width(int nx) { return (nx + 127) / 128 * 128 < (nx + 255) / 256 * 256 ? 128 : 256; }

struct XymParams {
    Dims d;
    int ychunk;                       // output rows per CTA (multiple of 16)
    float *out[XM_MAXS];              // x/y-filtered cube of each scale
    const float *wgt;                 // Eq. 1: the input is multiplied by this cube while it is staged (NULL: Eq. 2)
    TapsXY t[XM_MAXS];
};

__device__ __forceinline__ float2 fmul2(float2 a, float g)
{
    const float2 gg = make_float2(g, g);
    unsigned long long ra = *reinterpret_cast<const unsigned long long *>(&a);
    unsigned long long rb = *reinterpret_cast<const unsigned long long *>(&gg);
    unsigned long long rd;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(rd) : "l"(ra), "l"(rb));
    return *reinterpret_cast<float2 *>(&rd);
}

// x pass of one scale for the warp's staged row pair: lane -> columns 8 lane .. 8 lane + 7
template <int R, int GS>
__device__ __forceinline__ void xm_xpass(const float2 *__restrict__ s_in, float2 *__restrict__ s_u,
                                         const float (&gx)[32], int lane)
{
    constexpr int XM_GP = XmShape<GS>::GP;
    constexpr int C0 = XM_HALO - R;     // staged column of tap -R of output column 0
    constexpr int SH = C0 & 1;          // 16-byte loads start at an even staged column
    constexpr int NL = (GS + 2 * R + SH + 1) / 2;
    float2 acc[GS];
#pragma unroll
    for (int i = 0; i < GS; ++i) acc[i] = make_float2(0.f, 0.f);
#pragma unroll
    for (int l = 0; l < NL; ++l) {
        const int sc = C0 - SH + 2 * l;                 // relative to 8 lane; compile time
        const float4 q = *reinterpret_cast<const float4 *>(s_in + (lane + sc / GS) * XM_GP + sc % GS);
        const float2 v[2] = {make_float2(q.x, q.y), make_float2(q.z, q.w)};
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            const int j = 2 * l + e - SH;               // input index relative to tap -R of output 0
#pragma unroll
            for (int i = 0; i < GS; ++i) {
                const int o = j - i;
                if (j >= 0 && o >= 0 && o <= 2 * R) acc[i] = ffma2(v[e], gx[o], acc[i]);
            }
        }
    }
    float4 *dst = reinterpret_cast<float4 *>(s_u + lane * XM_GP);
#pragma unroll
    for (int i = 0; i < GS / 2; ++i) dst[i] = make_float4(acc[2 * i].x, acc[2 * i].y, acc[2 * i + 1].x, acc[2 * i + 1].y);
}

// y pass state of one scale and one column: B[j] = unfinished output pair m = k + dmin + j
template <int R>
struct XmY {
    float2 B[R];
    float prev;     // u[2k - 1]
    __device__ __forceinline__ void init()
    {
#pragma unroll
        for (int j = 0; j < R; ++j) B[j] = make_float2(0.f, 0.f);
        prev = 0.f;
    }
    // scatter the pair U = (u[2k], u[2k+1]); returns the finished pair of rows 2m, 2m+1, m = k - ceil(R/2)
    __device__ __forceinline__ float2 step(float2 U, const float (&gy)[32])
    {
        constexpr int dmin = -((R + 1) / 2), dmax = R / 2;
        const float2 Uo = make_float2(prev, U.x);
        prev = U.y;
        float2 out = make_float2(0.f, 0.f);
#pragma unroll
        for (int d = dmin; d <= dmax; ++d) {
            const int oe = -2 * d, oo = -2 * d - 1;     // taps fed by U and by Uo
            const bool he = oe >= -R && oe <= R, ho = oo >= -R && oo <= R;
            float2 t;
            if (d < dmax) {
                t = B[d - dmin];
                if (he) t = ffma2(U, gy[oe + R], t);
                if (ho) t = ffma2(Uo, gy[oo + R], t);
            } else {                                    // newest pair: first contribution(s)
                if (he) { t = fmul2(U, gy[oe + R]); if (ho) t = ffma2(Uo, gy[oo + R], t); }
                else t = fmul2(Uo, gy[oo + R]);
            }
            if (d == dmin) out = t;
            else B[d - 1 - dmin] = t;
        }
        return out;
    }
};

template <int NS, int RA, int RB, int RC, int RD, bool WGT = false, int GS = 8>
__global__ void __launch_bounds__(XmShape<GS>::NT, GS == 8 ? 2 : 4) k_xym(const float *__restrict__ in, const __grid_constant__ XymParams P)
{
    using XS = XmShape<GS>;
    constexpr int XM_NT = XS::NT, XM_NB = XS::NB, XM_SW = XS::SW, XM_GP = XS::GP, XM_SIN = XS::SIN, XM_U = XS::U;
    extern __shared__ __align__(16) float2 xm_smem[];
    float2 *s_in = xm_smem;                        // [8 warps][XM_SIN]
    float2 *s_u = xm_smem + XM_NB * XM_SIN;        // [8 row pairs][NS][XM_U]
    const Dims &d = P.d;
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const int x0 = blockIdx.x * XM_NT, z = blockIdx.z;
    const int ya = blockIdx.y * P.ychunk, yb = min(ya + P.ychunk, d.ny);
    const int ys = ya - 16;                        // first input row of the first batch (even)
    const int nbatch = (yb + 12 - ys + 2 * XM_NB - 1) / (2 * XM_NB);
    const long long plane_off = (long long)z * d.plane;
    const int gx = x0 + tid;
    const bool col_ok = gx < d.nx;
    // running output pointers: row 2 m of scale s for the current march step k, m = k - ceil(R_s / 2)
    constexpr int RMAX = NS > 3 ? RD : NS > 2 ? RC : NS > 1 ? RB : RA;   // (the scales are sorted by radius)
    constexpr int RMIN = RA;
    const long long col0 = plane_off + (col_ok ? gx : 0);
    const int k0 = ys / 2;
    float *o0 = P.out[0] + col0 + (long long)(2 * (k0 - (RA + 1) / 2)) * d.nx;
    float *o1 = NS > 1 ? P.out[NS > 1 ? 1 : 0] + col0 + (long long)(2 * (k0 - (RB + 1) / 2)) * d.nx : nullptr;
    float *o2 = NS > 2 ? P.out[NS > 2 ? 2 : 0] + col0 + (long long)(2 * (k0 - (RC + 1) / 2)) * d.nx : nullptr;
    float *o3 = NS > 3 ? P.out[NS > 3 ? 3 : 0] + col0 + (long long)(2 * (k0 - (RD + 1) / 2)) * d.nx : nullptr;

    XmY<RA> sa; XmY<RB> sb; XmY<RC> sc; XmY<RD> sd;
    sa.init(); sb.init(); sc.init(); sd.init();

    // this warp's row pair of batch b: rows ys + 2 NB b + 2 w (+1); lane loads float4 columns lane, lane+32, ...
    float4 pf[2][XS::NQ];
    auto prefetch = [&](int b) {
        const int r0 = ys + 2 * XM_NB * b + 2 * w;
#pragma unroll
        for (int rr = 0; rr < 2; ++rr) {
            const int r = r0 + rr;
            const bool rok = r >= 0 && r < d.ny;
#pragma unroll
            for (int q = 0; q < XS::NQ; ++q) {
                const int idx = lane + 32 * q;
                const int xx = x0 - XM_HALO + 4 * idx;
                const bool ok = rok && idx < XM_SW / 4 && xx >= 0 && xx < d.nx;
                const long long o = plane_off + (long long)r * d.nx + xx;
                pf[rr][q] = ok ? __ldg(reinterpret_cast<const float4 *>(in + o)) : make_float4(0.f, 0.f, 0.f, 0.f);
                if (WGT && ok) {
                    const float4 w4 = __ldg(reinterpret_cast<const float4 *>(P.wgt + o));
                    pf[rr][q].x *= w4.x; pf[rr][q].y *= w4.y; pf[rr][q].z *= w4.z; pf[rr][q].w *= w4.w;
                }
            }
        }
    };
    prefetch(0);
    for (int b = 0; b < nbatch; ++b) {
        // ---- x phase: stage the row pair interleaved, then the x pass of every scale
        {
            float2 *sw = s_in + w * XM_SIN;
#pragma unroll
            for (int q = 0; q < XS::NQ; ++q) {
                const int idx = lane + 32 * q;
                if (idx < XM_SW / 4) {
                    float4 *dst = GS == 8 ? reinterpret_cast<float4 *>(sw + (idx >> 1) * XM_GP + (idx & 1) * 4)
                                          : reinterpret_cast<float4 *>(sw + idx * XM_GP);
                    const float4 a = pf[0][q], c = pf[1][q];
                    dst[0] = make_float4(a.x, c.x, a.y, c.y);
                    dst[1] = make_float4(a.z, c.z, a.w, c.w);
                }
            }
            __syncwarp();
            float2 *su = s_u + (w * NS) * XM_U;
            xm_xpass<RA, GS>(sw, su, P.t[0].gx, lane);
            if constexpr (NS > 1) xm_xpass<RB, GS>(sw, su + XM_U, P.t[NS > 1 ? 1 : 0].gx, lane);
            if constexpr (NS > 2) xm_xpass<RC, GS>(sw, su + 2 * XM_U, P.t[NS > 2 ? 2 : 0].gx, lane);
            if constexpr (NS > 3) xm_xpass<RD, GS>(sw, su + 3 * XM_U, P.t[NS > 3 ? 3 : 0].gx, lane);
        }
        if (b + 1 < nbatch) prefetch(b + 1);
        __syncthreads();
        // ---- y phase: 8 steps of the march
        const int kbase = ys / 2 + XM_NB * b;      // ys is even
        const int pi = (tid / GS) * XM_GP + tid % GS;
#pragma unroll 2
        for (int kk = 0; kk < XM_NB; ++kk) {
            const float2 *su = s_u + (kk * NS) * XM_U + pi;
            const int k = kbase + kk;
            const float2 va = sa.step(su[0], P.t[0].gy);
            float2 vb, vc, vd;
            if constexpr (NS > 1) vb = sb.step(su[XM_U], P.t[NS > 1 ? 1 : 0].gy);
            if constexpr (NS > 2) vc = sc.step(su[2 * XM_U], P.t[NS > 2 ? 2 : 0].gy);
            if constexpr (NS > 3) vd = sd.step(su[3 * XM_U], P.t[NS > 3 ? 3 : 0].gy);
            // rows 2 m, 2 m + 1 with m = k - ceil(R/2) per scale; the common case (all of them inside the
            // chunk) stores through the running row pointers without any test
            const bool all_in = 2 * (k - (RMAX + 1) / 2) >= ya && 2 * (k - (RMIN + 1) / 2) + 1 < yb;
            if (all_in) {
                if (col_ok) {
                    o0[0] = va.x; o0[d.nx] = va.y;
                    if constexpr (NS > 1) { o1[0] = vb.x; o1[d.nx] = vb.y; }
                    if constexpr (NS > 2) { o2[0] = vc.x; o2[d.nx] = vc.y; }
                    if constexpr (NS > 3) { o3[0] = vd.x; o3[d.nx] = vd.y; }
                }
            } else {
                auto emit = [&](float *o, float2 v, int m) {
                    const int r0 = 2 * m;
                    if (col_ok) {
                        if (r0 >= ya && r0 < yb) o[0] = v.x;
                        if (r0 + 1 >= ya && r0 + 1 < yb) o[d.nx] = v.y;
                    }
                };
                emit(o0, va, k - (RA + 1) / 2);
                if constexpr (NS > 1) emit(o1, vb, k - (RB + 1) / 2);
                if constexpr (NS > 2) emit(o2, vc, k - (RC + 1) / 2);
                if constexpr (NS > 3) emit(o3, vd, k - (RD + 1) / 2);
            }
            o0 += 2 * d.nx;
            if constexpr (NS > 1) o1 += 2 * d.nx;
            if constexpr (NS > 2) o2 += 2 * d.nx;
            if constexpr (NS > 3) o3 += 2 * d.nx;
        }
        __syncthreads();
    }
}

template <int NS, int RA, int RB, int RC, int RD, bool WGT, int GS>
cudaError_t launch_xym_g(const float *in, const XymParams &P, cudaStream_t st)
{
    using XS = XmShape<GS>;
    constexpr int SMEM = (XS::NB * XS::SIN + XS::NB * NS * XS::U) * (int)sizeof(float2);
    cudaError_t e = ensure_dynamic_smem(k_xym<NS, RA, RB, RC, RD, WGT, GS>, SMEM);
    if (e != cudaSuccess) return e;
    dim3 grid((P.d.nx + XS::NT - 1) / XS::NT, (P.d.ny + P.ychunk - 1) / P.ychunk, P.d.nz);
    k_xym<NS, RA, RB, RC, RD, WGT, GS><<<grid, XS::NT, SMEM, st>>>(in, P);
    return cudaGetLastError();
}

template <int NS, int RA, int RB, int RC, int RD, bool WGT = false>
cudaError_t launch_xym(const float *in, const XymParams &P, int sm_count, cudaStream_t st)
{
    (void)sm_count;
    if (xm_strip_width(P.d.nx) == 128) return launch_xym_g<NS, RA, RB, RC, RD, WGT, 4>(in, P, st);
    return launch_xym_g<NS, RA, RB, RC, RD, WGT, 8>(in, P, st);
}

}  // namespace

bool fast_xy_radius(int r, int *c)
{
    static const int set[] = {3, 6, 9, 12};
    for (int v : set)
        if (r <= v) { *c = v; return true; }
    *c = 0;
    return false;
}

bool fast_z_radius(int r, int *c)
{
    static const int set[] = {6, 12, 24, 48, 72, 96};
    for (int v : set)
        if (r <= v) { *c = v; return true; }
    *c = 0;
    return false;
}

// One launch of k_xym for the (already radius-sorted) scales g[0..n): true if that radius tuple is compiled.
static bool xym_dispatch(int n, const int *rc, const float *in, const XymParams &P, int sm_count, cudaStream_t st,
                         bool probe, cudaError_t *err)
{
#define XYM_CASE(NS, A, B, C, D)                                                              \
    if (n == NS && rc[0] == A && (NS < 2 || rc[1] == B) && (NS < 3 || rc[2] == C) && (NS < 4 || rc[3] == D)) { \
        if (!probe) {                                                                         \
            if (NS == 1 && P.wgt != nullptr) *err = launch_xym<1, A, 3, 3, 3, true>(in, P, sm_count, st); \
            else if (P.wgt != nullptr) *err = cudaErrorNotSupported;  /* weighted staging: single-scale launches only */ \
            else *err = launch_xym<NS, A, (NS > 1 ? B : 3), (NS > 2 ? C : 3), (NS > 3 ? D : 3)>(in, P, sm_count, st); \
        }                                                                                     \
        return true;                                                                          \
    }
    XYM_CASE(4, 3, 6, 9, 12)
    XYM_CASE(3, 3, 6, 9, 0)
    XYM_CASE(3, 3, 6, 6, 0)
    XYM_CASE(3, 6, 9, 9, 0)
    XYM_CASE(2, 3, 3, 0, 0)
    XYM_CASE(2, 3, 6, 0, 0)
    XYM_CASE(2, 3, 9, 0, 0)
    XYM_CASE(2, 3, 12, 0, 0)
    XYM_CASE(2, 6, 6, 0, 0)
    XYM_CASE(2, 6, 9, 0, 0)
    XYM_CASE(2, 6, 12, 0, 0)
    XYM_CASE(2, 9, 9, 0, 0)
    XYM_CASE(2, 9, 12, 0, 0)
    XYM_CASE(2, 12, 12, 0, 0)
    XYM_CASE(1, 3, 0, 0, 0)
    XYM_CASE(1, 6, 0, 0, 0)
    XYM_CASE(1, 9, 0, 0, 0)
    XYM_CASE(1, 12, 0, 0, 0)
#undef XYM_CASE
    return false;
}

// x and y passes of the scales `scales[0..n)` of one cube: in -> out[i] (x/y-filtered cubes).  The
// scales are sorted by compiled radius and cut into the largest groups a k_xym instance exists for;
// every group reads the input once.
cudaError_t fast_xy_multi(pgsf_plan *p, const int *scales, int n, const float *in, float *const *out, int ncubes,
                          cudaStream_t st, bool box, const float *wgt, int nplanes)
{
    // the x and y passes do not couple planes: `ncubes` consecutive cubes are one stack of ncubes * nz planes
    Dims d = p->dims;
    d.nz = nplanes > 0 ? nplanes : d.nz * ncubes;
    d.cube = d.plane * d.nz;
    if (d.nz > 65535 || n < 1 || n > PGSF_MAX_SCALES) return cudaErrorInvalidConfiguration;
    int order[PGSF_MAX_SCALES];
    for (int i = 0; i < n; ++i) order[i] = i;
    for (int i = 1; i < n; ++i)          // insertion sort by compiled radius (stable)
        for (int j = i; j > 0 && p->scales[scales[order[j]]].rxy_c < p->scales[scales[order[j - 1]]].rxy_c; --j) {
            const int t = order[j]; order[j] = order[j - 1]; order[j - 1] = t;
        }
    // rows per CTA: a few waves of CTAs; a chunk start recomputes 16 + 12 rows
    int nch = 1;
    {
        const long long base = (long long)((d.nx + xm_strip_width(d.nx) - 1) / xm_strip_width(d.nx)) * d.nz;
        const long long want = 6LL * p->sm_count * 2;
        nch = (int)((want + base - 1) / base);
        const int maxch = (d.ny + 127) / 128;
        if (nch > maxch) nch = maxch;
        if (nch < 1) nch = 1;
    }
    int ychunk = ((d.ny + nch - 1) / nch + 15) / 16 * 16;
    if ((d.ny + ychunk - 1) / ychunk > 65535) return cudaErrorInvalidConfiguration;
    int pos = 0;
    while (pos < n) {
        int take = n - pos < XM_MAXS ? n - pos : XM_MAXS;
        int rc[XM_MAXS];
        XymParams P;
        for (; take >= 1; --take) {
            for (int i = 0; i < take; ++i) rc[i] = p->scales[scales[order[pos + i]]].rxy_c;
            if (xym_dispatch(take, rc, nullptr, P, 0, st, true, nullptr)) break;
        }
        if (take < 1) return cudaErrorNotSupported;
        P.d = d;
        P.ychunk = ychunk;
        P.wgt = wgt;
        unsigned mask = 0;
        for (int i = 0; i < XM_MAXS; ++i) {
            const int j = i < take ? i : 0;
            const int sidx = scales[order[pos + j]];
            P.out[i] = out[order[pos + j]];
            P.t[i] = box ? p->scales[sidx].txy_box : p->scales[sidx].txy;
            if (i < take) mask |= 1u << sidx;
        }
        char name[32];
        snprintf(name, sizeof name, box ? "bxy_m%u" : "xy_m%u", mask);
        LaunchScope ls(p, name, st);
        cudaError_t e = cudaSuccess;
        xym_dispatch(take, rc, in, P, p->sm_count, st, false, &e);
        if (e != cudaSuccess) return e;
        pos += take;
    }
    return cudaSuccess;
}

// frequency pass of one scale: in (x/y-filtered cube) -> out
cudaError_t fast_z(pgsf_plan *p, int scale, const float *in, float *out, cudaStream_t st, bool box, float *ratio)
{
    const Dims &d = p->dims;
    const ScalePlan &sp = p->scales[scale];
    if (d.ny > 65535 || d.nz > 65535 * 64) return cudaErrorInvalidConfiguration;
    char name[32];
    snprintf(name, sizeof name, box ? "bz_s%d" : "z_s%d", scale);
    LaunchScope ls(p, name, st);
    const Taps &tz = box ? sp.tz_box : sp.tz;
    // slab by TMA up to RZ = 24; above, 128 - 256 threads issuing cp.async keep more copies in flight than one TMA
    // box of 160 - 256 rows of 256 bytes (measured at config 3, RZ = 48: 11.7 ms with TMA, 11.0 ms without).
    // PGSF_OPT_TUNE bit 2 = cp.async everywhere, bit 3 = TMA everywhere.
    const bool tma = (p->tune & 8) != 0 || ((p->tune & 4) == 0 && sp.rz_c <= 24);
    switch (sp.rz_c) {
    case 6: return launch_z_r6(in, out, ratio, d, tz, st, tma);
    case 12: return launch_z_r12(in, out, ratio, d, tz, st, tma);
    case 24: return launch_z_r24(in, out, ratio, d, tz, st, tma);
    case 48: return launch_z_r48(in, out, ratio, d, tz, st, tma);
    case 72: return launch_z_r72(in, out, ratio, d, tz, st, tma);
    case 96: return launch_z_r96(in, out, ratio, d, tz, st, tma);
    default: return cudaErrorNotSupported;
    }
}

// frequency pass of one scale fused with the z-direction window sums of the statistics:
// in (x/y-filtered cube) -> out (filtered cube), Z1, Z2
int zm_step_channels_of(int rz_compiled) { return zm_step_rule(rz_compiled); }   // = zm_step_channels<RZ>()

cudaError_t fast_zm(pgsf_plan *p, int scale, const float *in, float *out, float *Z1, float *Z2, int ncubes,
                    cudaStream_t st, const ZmSection *sec)
{
    const Dims &d = p->dims;
    const ScalePlan &sp = p->scales[scale];
    if (d.ny > 65535 || ncubes < 1 || ncubes > 65535) return cudaErrorInvalidConfiguration;
    if (p->tensor_z) {      // the optional tensor-core variant (pgsf_ztc.cu) where the plan asks for it and it applies
        const cudaError_t te = fast_ztc(p, scale, in, out, Z1, Z2, ncubes, st, sec);
        if (te != cudaErrorNotSupported) return te;
    }
    const int hz = p->desc.box_half[2];
    char name[32];
    snprintf(name, sizeof name, "zm_s%d", scale);
    LaunchScope ls(p, name, st);
    const bool tma = (p->tune & 8) != 0 || ((p->tune & 4) == 0 && sp.rz_c <= 24);     // (see fast_z)
    switch (sp.rz_c) {
    case 6: return launch_zm_r6(in, out, Z1, Z2, d, hz, p->d_pivot, sp.tz, ncubes, st, sec, tma);
    case 12: return launch_zm_r12(in, out, Z1, Z2, d, hz, p->d_pivot, sp.tz, ncubes, st, sec, tma);
    case 24: return launch_zm_r24(in, out, Z1, Z2, d, hz, p->d_pivot, sp.tz, ncubes, st, sec, tma);
    case 48: return launch_zm_r48(in, out, Z1, Z2, d, hz, p->d_pivot, sp.tz, ncubes, st, sec, tma);
    case 72: return launch_zm_r72(in, out, Z1, Z2, d, hz, p->d_pivot, sp.tz, ncubes, st, sec, tma);
    case 96: return launch_zm_r96(in, out, Z1, Z2, d, hz, p->d_pivot, sp.tz, ncubes, st, sec, tma);
    default: return cudaErrorNotSupported;
    }
}

cudaError_t fast_filter3d(pgsf_plan *p, int scale, const float *in, float *out, float *tmp,
                          cudaStream_t st, bool box, const float *wgt, float *ratio)
{
    float *outs[1] = {tmp};
    cudaError_t e = fast_xy_multi(p, &scale, 1, in, outs, 1, st, box, wgt);
    if (e != cudaSuccess) return e;
    return fast_z(p, scale, tmp, out, st, box, ratio);
}

}  // namespace pgsf
