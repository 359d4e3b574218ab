// k_xyb: x- and y-direction window sums of the local statistics + voxel selection ("three directional
// sums", P:33 / P:282 thresholds; readings C-6..C-10), the successor of k_ymarch (pgsf_stats.cu).
//
// Input: the z-direction window sums Z1 = sum f, Z2 = sum f^2 (of k_zm / k_zbox) and the filtered cube f.
// One CTA = 256 staged columns (1, 2 or 4 strips of 32 G columns, G = hx / 2, each of some z plane), one chunk of
// rows; it marches down y in batches of RB rows.  Every batch has two phases:
//
//   y phase   a thread owns ONE PAIR of adjacent columns and keeps the y-direction window sums
//             Y1 = sum_{|o|<=hy} Z1(y+o), Y2 likewise, in registers: the row entering the window is added,
//             the row leaving it subtracted (Y2 compensated, see comp_add2).  The entering row comes from
//             HBM; the leaving row was read 2 hy rows earlier by the same thread.  Only 256 columns x 3-4 CTAs
//             are resident per SM, so the 2 hy + 1 live rows of all resident CTAs (~30-40 MB) stay in L2 and
//             the leaving row never goes back to HBM -- k_ymarch kept 8 columns and ~20 registers per column
//             in every thread, i.e. 120 MB of live rows, and paid 8 B / voxel of HBM reads for them.
//             The pair (Y1, Y2) of every column goes to a shared-memory row buffer.
//   x phase   warp w takes row w of the batch; lane l owns the group of G columns l of its strip and forms the
//             prefix sums P and suffix sums Q of (Y1, Y2) over its group (packed add.f32x2).  The window of
//             2 hx + 1 = 4 G + 1 columns of output column j of group l + 2 is exactly
//                 Q_l[j] + total(l+1) + total(l+2) + total(l+3) + P_{l+4}[j],
//             so lane l collects P from lane l + 4 and three totals by warp shuffles and finishes the outputs
//             of group l + 2: every output is a plain sum of the elements of its own window (no cancellation).
//             Then m = S1 / n, var = S2 / n - m^2 and the selection f > m + k sd in the division-free form of
//             pgsf_generic.cu, halo exclusion, mask bytes, count.
// One __syncthreads per batch (the row buffer is double buffered).
//
// Mask modes: overwrite (every byte written), OR with the previous mask (read-modify-write), and the sparse OR
// pgsf_find_multiscale uses for the scales after the first: only the bytes of newly selected voxels are
// touched (a few in 10^4), and `count` receives the number of voxels that were not set before.
#include <stdio.h>

#include "pgsf_internal.h"
#include "pgsf_device.cuh"

#ifndef XYB_MINB
#define XYB_MINB 4      // CTAs per SM the register budget is set for
#endif

namespace pgsf {
namespace {

template <int G>
struct XybShape {
    static constexpr int HX = 2 * G;
    static constexpr int SWS = 32 * G;             // staged columns of one strip (one warp-row of the x phase)
    static constexpr int WMAX = SWS - 2 * HX;      // output columns of one strip
    static constexpr int NSTRIP = 256 / SWS;       // strips per CTA (G = 6: one strip of 192 columns, 32 threads without a y pair)
    static constexpr int NT = 128;                 // threads: one per pair of the 256 staged columns
    static constexpr int RB = 4;                   // rows per batch
    static constexpr int UPW = NSTRIP * RB / 4;    // (strip, row) units of the x phase per warp and batch
    static constexpr int TPS = SWS / 2;            // y-phase threads per strip
    static constexpr int CPL = G / 2;              // 16-byte chunks (column pairs) per x-phase lane
    static constexpr int VL = (G % 4 == 0) ? 4 : 2; // columns per global load / mask word of the x phase
    static constexpr int NV = G / VL;
};

struct XybParams {
    Dims d;              // one cube (or, for a section of a streamed cube: d.nz = planes of the launch)
    int z_off, nz_full;  // channel of plane 0 of the launch inside its cube, channels of the whole cube
    int hy, hz;
    int gx, gy, gz;      // halo excluded from mask and count (C-11)
    int mode;            // 0 overwrite, 1 OR (dense), 2 OR (sparse; counts newly set voxels)
    float k2;            // k^2
    int wo;              // output columns per strip (multiple of 8, <= WMAX)
    int nstrips;         // strips across nx
    long long nplanes;   // planes of the launch (all cubes)
    int ychunk;          // output rows per CTA
};

__device__ __forceinline__ float2 add2(float2 a, float2 b)
{
    unsigned long long ra = *reinterpret_cast<const unsigned long long *>(&a);
    unsigned long long rb = *reinterpret_cast<const unsigned long long *>(&b);
    unsigned long long rd;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(rd) : "l"(ra), "l"(rb));
    return *reinterpret_cast<float2 *>(&rd);
}
__device__ __forceinline__ float2 sub2(float2 a, float2 b)
{
    unsigned long long ra = *reinterpret_cast<const unsigned long long *>(&a);
    unsigned long long rb = *reinterpret_cast<const unsigned long long *>(&b);
    unsigned long long rd;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(rd) : "l"(ra), "l"(rb));
    return *reinterpret_cast<float2 *>(&rd);
}
// Compensated running sum on a pair of columns: (s, c) += v, the value is s + c.  The rounding error of s + v is
// recovered exactly (Knuth's branch-free two-sum) and gathered in c, so what the sum retains after a large addend has
// come and gone is O(eps^2) of it.  (Kahan's form, which folds the compensation into the NEXT addend, commits an
// untracked eps |v| there: a source 10^3 - 10^4 x the noise in f^2 left 2e-5 of relative error in the sum of f^2 of
// every later row of its column -- a fifth of the mask band.)
__device__ __forceinline__ void comp_add2(float2 &s, float2 &c, float2 v)
{
    const float2 t = add2(s, v);
    const float2 bp = sub2(t, s);
    const float2 da = sub2(s, sub2(t, bp));
    const float2 db = sub2(v, bp);
    c = add2(c, add2(da, db));
    s = t;
}
// (s, c) -= v
__device__ __forceinline__ void comp_sub2(float2 &s, float2 &c, float2 v)
{
    const float2 t = sub2(s, v);
    const float2 bp = sub2(t, s);          // ~ -v
    const float2 da = sub2(s, sub2(t, bp));
    const float2 nb = add2(v, bp);         // -((-v) - bp)
    c = add2(c, sub2(da, nb));
    s = t;
}

// p + i * stride as one IMAD.WIDE.U32
__device__ __forceinline__ const char *row_ptr(const char *p, unsigned stride, unsigned i)
{
    unsigned long long r;
    asm("mad.wide.u32 %0, %1, %2, %3;" : "=l"(r) : "r"(stride), "r"(i), "l"(reinterpret_cast<unsigned long long>(p)));
    return reinterpret_cast<const char *>(r);
}

__device__ __forceinline__ int xyb_clipped_len(int c, int h, int n)
{
    return min(c + h, n - 1) - max(c - h, 0) + 1;
}

// shared-memory row buffer: chunk c (16 bytes = two columns x (Y1, Y2)) of a row lives at c ^ ((c >> 3) & 3):
// conflict-free both for the y phase (thread t writes chunk t) and for the x phase (lane l reads chunks
// CPL l .. CPL l + CPL - 1)
// an LDS.128 the compiler cannot merge with an earlier load of the same address
__device__ __forceinline__ float4 lds128(const float4 *p)
{
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];"
                 : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"((unsigned)__cvta_generic_to_shared(p)));
    return v;
}

__device__ __forceinline__ int swz(int c) { return c ^ ((c >> 3) & 3); }

// MODE: 0 overwrite the mask, 1 OR (dense read-modify-write), 2 sparse OR.  STATS: also write mean / sd.
template <int G, int MODE, bool STATS>
__global__ void __launch_bounds__(128, XYB_MINB) k_xyb(const float *__restrict__ f, const float *__restrict__ Z1,
                                                const float *__restrict__ Z2, uint8_t *__restrict__ mask,
                                                float *__restrict__ mean, float *__restrict__ sd,
                                                unsigned long long *__restrict__ count, const XybParams p,
                                                const float *__restrict__ pivot, const float *__restrict__ zeros)
{
    using S = XybShape<G>;
    constexpr int HX = S::HX, NSTRIP = S::NSTRIP, RB = S::RB, UPW = S::UPW, TPS = S::TPS, CPL = S::CPL, VL = S::VL, NV = S::NV;
    __shared__ __align__(16) float4 ybuf[2][RB][128];
    __shared__ unsigned wsum[4];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nx = p.d.nx, ny = p.d.ny;
    // A CTA takes NSTRIP consecutive SLOTS; slot = (plane of the stack of cubes) * nstrips + (x strip): with several
    // strips per CTA (G < 8) the strips of a CTA may belong to different planes, so narrow cubes leave no slot idle.
    const int ya = blockIdx.y * p.ychunk, yb = min(ya + p.ychunk, ny);
    const int hy = p.hy;
    const float piv = __ldg(pivot);                    // Z1, Z2 are sums of f - c0 and (f - c0)^2 (D-2)

    // ---- y phase: this thread's column pair.  Batch b brings in rows r0 + RB b + i (i < RB) and retires rows
    //      r - 2 hy.  Interior batches (every such row inside the cube and inside this chunk's window history) read
    //      through four running pointers with no predicate; threads of columns outside the cube run the same code
    //      on a buffer of zeros with stride 0.
    const long long yslot = (long long)blockIdx.x * NSTRIP + tid / TPS;
    const int ystrip = (int)(yslot % p.nstrips);
    const long long yplane = yslot / p.nstrips;
    const int cy = ystrip * p.wo - HX + 2 * (tid % TPS);
    const bool ycol_ok = tid / TPS < NSTRIP && yplane < p.nplanes && cy >= 0 && cy + 2 <= nx;
    const int r0 = ya - hy;                            // first row entering the window of output row ya
    const int nrows = (yb - ya) + 2 * hy;              // entering rows r0 .. yb - 1 + hy
    const int nb = (nrows + RB - 1) / RB;
    const int rl_min = max(r0, 0);                     // rows before it never entered the sums
    // batches b_lo <= b < b_hi are interior
    const int b_lo = (rl_min + 2 * hy - r0 + RB - 1) / RB;         // first leaving row r0 + RB b - 2 hy >= rl_min
    const int b_hi = (ny - r0) / RB;                               // last entering row r0 + RB b + RB - 1 < ny
    const unsigned rstride = ycol_ok ? (unsigned)nx * 4u : 0u;     // bytes between rows
    const char *pe1, *pe2, *pl1, *pl2;                             // row 0 of the current batch: entering, leaving
    {
        const long long o = (ycol_ok ? yplane : 0) * p.d.plane + (ycol_ok ? cy : 0);
        pe1 = reinterpret_cast<const char *>(ycol_ok ? Z1 + o : zeros);
        pe2 = reinterpret_cast<const char *>(ycol_ok ? Z2 + o : zeros);
        const long long oe = ycol_ok ? (long long)r0 * nx * 4 : 0, ol = ycol_ok ? (long long)(r0 - 2 * hy) * nx * 4 : 0;
        pl1 = pe1 + ol; pl2 = pe2 + ol;
        pe1 += oe; pe2 += oe;
    }

    float2 e1[RB], e2[RB], l1[RB], l2[RB];             // rows entering / leaving in the current batch
    auto load_rows = [&](int b) {
        if (b >= b_lo && b < b_hi) {
#pragma unroll
            for (int i = 0; i < RB; ++i) {
                e1[i] = __ldg(reinterpret_cast<const float2 *>(i ? row_ptr(pe1, rstride, i) : pe1));
                e2[i] = __ldg(reinterpret_cast<const float2 *>(i ? row_ptr(pe2, rstride, i) : pe2));
                l1[i] = __ldg(reinterpret_cast<const float2 *>(i ? row_ptr(pl1, rstride, i) : pl1));
                l2[i] = __ldg(reinterpret_cast<const float2 *>(i ? row_ptr(pl2, rstride, i) : pl2));
            }
        } else {
#pragma unroll
            for (int i = 0; i < RB; ++i) {
                const int r = r0 + RB * b + i, rl = r - 2 * hy;
                const bool oke = r >= 0 && r < ny;
                const bool okl = rl >= rl_min && rl < ny;
                e1[i] = oke ? __ldg(reinterpret_cast<const float2 *>(pe1 + i * rstride)) : make_float2(0.f, 0.f);
                e2[i] = oke ? __ldg(reinterpret_cast<const float2 *>(pe2 + i * rstride)) : make_float2(0.f, 0.f);
                l1[i] = okl ? __ldg(reinterpret_cast<const float2 *>(pl1 + i * rstride)) : make_float2(0.f, 0.f);
                l2[i] = okl ? __ldg(reinterpret_cast<const float2 *>(pl2 + i * rstride)) : make_float2(0.f, 0.f);
            }
        }
        pe1 = row_ptr(pe1, rstride, RB); pe2 = row_ptr(pe2, rstride, RB);
        pl1 = row_ptr(pl1, rstride, RB); pl2 = row_ptr(pl2, rstride, RB);
    };

    // ---- x phase: this warp's units u = 0 .. UPW - 1: strip (of the CTA) and row (of the batch)
    //      lane l finishes the outputs of group l + 2 of the strip: columns xo .. xo + G - 1
    bool out_ok[UPW];
    float nxz[UPW][G];                                 // clipped window lengths along x times along z
    unsigned core_x[UPW];                              // bit j: column j is outside the x / z halo
    long long voff[UPW];                               // element offset of (xo, row of the current batch's unit)
    int nvq[UPW];                                      // load / store words of the group that lie inside the cube
    {
#pragma unroll
        for (int u = 0; u < UPW; ++u) {
            const int unit = warp + 4 * u;
            const long long slot = (long long)blockIdx.x * NSTRIP + unit / RB;
            const int strip = (int)(slot % p.nstrips);
            const long long zz = slot / p.nstrips;                 // plane of the stack of cubes
            const int z = (int)(zz % p.d.nz) + p.z_off;            // channel inside its cube
            const long long plane_off = (zz < p.nplanes ? zz : 0) * p.d.plane;
            const float nzc = (float)xyb_clipped_len(z, p.hz, p.nz_full);
            const bool core_z = z >= p.gz && z < p.nz_full - p.gz;
            const int xo = strip * p.wo + G * lane;
            out_ok[u] = zz < p.nplanes && G * lane < p.wo && xo < nx;
            nvq[u] = min(NV, max(0, (nx - xo) / VL));          // (the last group of a row may stick out of the cube)
            core_x[u] = 0;
#pragma unroll
            for (int j = 0; j < G; ++j) {
                const int c = min(xo + j, nx - 1);
                nxz[u][j] = (float)xyb_clipped_len(c, HX, nx) * nzc;
                if (core_z && xo + j >= p.gx && xo + j < nx - p.gx) core_x[u] |= 1u << j;
            }
            // output row of unit u in batch b: r0 + RB b + (unit % RB) - hy
            voff[u] = plane_off + (long long)(r0 + unit % RB - hy) * nx + (out_ok[u] ? xo : 0);
        }
    }
    // shared-memory slots: the y phase writes chunk tid, the x phase reads chunks CPL lane .. + CPL - 1 of its strip
    float4 *const yw = &ybuf[0][0][swz(tid)];
    int xr[UPW][CPL];
#pragma unroll
    for (int u = 0; u < UPW; ++u)
#pragma unroll
        for (int v = 0; v < CPL; ++v)
            xr[u][v] = ((warp + 4 * u) % RB) * 128 + swz(((warp + 4 * u) / RB) * TPS + CPL * lane + v);

    float2 Y1 = make_float2(0.f, 0.f), Y2 = make_float2(0.f, 0.f), E2 = make_float2(0.f, 0.f), E1 = make_float2(0.f, 0.f);
    unsigned my_count = 0;
    const float guard = kFlatGuard, k2 = p.k2;
    const float nyfull = (float)(2 * hy + 1);
    const int gy = p.gy;
    load_rows(0);
    // centre values (and previous mask bytes) of the outputs of batch b: fetched one batch ahead, so that they are in
    // flight for a whole batch (two register sets used alternately)
    auto load_centre = [&](int b, float (&fv)[UPW][G], unsigned (&mk)[UPW][NV]) {
#pragma unroll
        for (int u = 0; u < UPW; ++u) {
            const int yo = r0 - hy + RB * b + (warp + 4 * u) % RB;
            const bool okr = out_ok[u] && yo >= ya && yo < yb;
            const long long o = voff[u] + (long long)(RB * b) * nx;
#pragma unroll
            for (int q = 0; q < NV; ++q) {
                const bool ok = okr && q < nvq[u];
                if constexpr (VL == 2) {
                    const float2 t = ok ? __ldg(reinterpret_cast<const float2 *>(f + o) + q) : make_float2(0.f, 0.f);
                    fv[u][2 * q] = t.x; fv[u][2 * q + 1] = t.y;
                    mk[u][q] = (MODE == 1 && ok) ? *reinterpret_cast<const unsigned short *>(mask + o + 2 * q) : 0u;
                } else {
                    const float4 t = ok ? __ldg(reinterpret_cast<const float4 *>(f + o) + q) : make_float4(0.f, 0.f, 0.f, 0.f);
                    fv[u][4 * q] = t.x; fv[u][4 * q + 1] = t.y; fv[u][4 * q + 2] = t.z; fv[u][4 * q + 3] = t.w;
                    mk[u][q] = (MODE == 1 && ok) ? *reinterpret_cast<const unsigned *>(mask + o + 4 * q) : 0u;
                }
            }
        }
    };
    auto batch = [&](int b, float (&fv)[UPW][G], unsigned (&mk)[UPW][NV], float (&fvn)[UPW][G],
                     unsigned (&mkn)[UPW][NV]) {
        const int par = b & 1;
        const int yrow = r0 - hy + RB * b;             // output row of batch row 0
        if (b + 1 < nb) load_centre(b + 1, fvn, mkn);
        // ---- y phase
#pragma unroll
        for (int i = 0; i < RB; ++i) {
            float2 y1;
            if constexpr (STATS) { comp_add2(Y1, E1, e1[i]); y1 = add2(Y1, E1); }    // (the mean is an output: 1e-5 sd)
            else { Y1 = add2(Y1, e1[i]); y1 = Y1; }
            comp_add2(Y2, E2, e2[i]);
            const float2 y2 = add2(Y2, E2);
            yw[par * (RB * 128) + i * 128] = make_float4(y1.x, y2.x, y1.y, y2.y);
            if constexpr (STATS) comp_sub2(Y1, E1, l1[i]);
            else Y1 = sub2(Y1, l1[i]);                 // the row leaving the window after this output
            comp_sub2(Y2, E2, l2[i]);
        }
        if (b + 1 < nb) load_rows(b + 1);              // in flight during the x phase
        __syncthreads();
        // ---- x phase
        const float4 *yb4 = &ybuf[par][0][0];
#pragma unroll
        for (int u = 0; u < UPW; ++u) {
            float2 P[G], Q[G];
#pragma unroll
            for (int v = 0; v < CPL; ++v) {
                const float4 t = yb4[xr[u][v]];
                P[2 * v] = make_float2(t.x, t.y);
                P[2 * v + 1] = make_float2(t.z, t.w);
            }
#pragma unroll
            for (int v = 0; v < CPL; ++v) {            // (a second read is cheaper than G register copies)
                const float4 t = lds128(&yb4[xr[u][v]]);
                Q[2 * v] = make_float2(t.x, t.y);
                Q[2 * v + 1] = make_float2(t.z, t.w);
            }
#pragma unroll
            for (int j = 1; j < G; ++j) P[j] = add2(P[j], P[j - 1]);
#pragma unroll
            for (int j = G - 2; j >= 0; --j) Q[j] = add2(Q[j], Q[j + 1]);
            // totals of groups l+1, l+2, l+3
            const float2 tot = P[G - 1];
            float2 M, M3;
            M.x = __shfl_down_sync(0xffffffffu, tot.x, 1);
            M.y = __shfl_down_sync(0xffffffffu, tot.y, 1);
            M3.x = __shfl_down_sync(0xffffffffu, tot.x, 2);
            M3.y = __shfl_down_sync(0xffffffffu, tot.y, 2);
            M = add2(M, M3);
            M3.x = __shfl_down_sync(0xffffffffu, tot.x, 3);
            M3.y = __shfl_down_sync(0xffffffffu, tot.y, 3);
            M = add2(M, M3);
            const int yo = yrow + (warp + 4 * u) % RB;
            const bool row_ok = out_ok[u] && yo >= ya && yo < yb;
            const float nyc = (yo >= hy && yo + hy < ny) ? nyfull : (float)xyb_clipped_len(min(max(yo, 0), ny - 1), hy, ny);
            const bool core_y = yo >= gy && yo < ny - gy;
            unsigned bits = 0;
            float S1[STATS ? G : 1], S2[STATS ? G : 1];
#pragma unroll
            for (int j = 0; j < G; ++j) {
                float2 R;
                R.x = __shfl_down_sync(0xffffffffu, P[j].x, 4);
                R.y = __shfl_down_sync(0xffffffffu, P[j].y, 4);
                const float2 X = add2(add2(Q[j], R), M);
                if constexpr (STATS) { S1[j] = X.x; S2[j] = X.y; }
                // selection  n v - S1 > k sqrt(max(n S2 - S1^2, 0))  (+ the flat-window guard D-1)
                const float n = nxz[u][j] * nyc;
                const float v = fv[u][j] - piv;
                const float a = fmaf(n, v, -X.x);
                const float q = fmaxf(fmaf(n, X.y, -X.x * X.x), 0.f);
                const bool sel = (a > (guard * n) * fabsf(v)) && (a * a > k2 * q);
                if (sel) bits |= 1u << j;
            }
            bits = core_y ? (bits & core_x[u]) : 0u;
            if (!row_ok) continue;
            const long long idx = voff[u] + (long long)(RB * b) * nx;
            if constexpr (MODE == 2) {
                // sparse OR: touch only the bytes of selected voxels, count those that were not set before
                if (bits) {
#pragma unroll
                    for (int j = 0; j < G; ++j)
                        if ((bits >> j) & 1u) {
                            if (mask[idx + j] == 0) { mask[idx + j] = 1; ++my_count; }
                        }
                }
            } else {
                if constexpr (MODE == 1) {   // previous mask: any non-zero byte counts as set
#pragma unroll
                    for (int q = 0; q < NV; ++q) {
                        const unsigned old = mk[u][q];
                        if constexpr (VL == 2) {
                            bits |= (((old & 0xffu) ? 1u : 0u) | ((old & 0xff00u) ? 2u : 0u)) << (2 * q);
                        } else {
                            const unsigned nzb = ((old | ((old & 0x7f7f7f7fu) + 0x7f7f7f7fu)) >> 7) & 0x01010101u;
                            bits |= ((nzb & 1u) | ((nzb >> 7) & 2u) | ((nzb >> 14) & 4u) | ((nzb >> 21) & 8u)) << (4 * q);
                        }
                    }
                    bits = core_y ? (bits & core_x[u]) : 0u;
                }
                my_count += __popc(bits);
#pragma unroll
                for (int q = 0; q < NV; ++q) {
                    if (q >= nvq[u]) break;
                    if constexpr (VL == 2) {
                        const unsigned b2 = (bits >> (2 * q)) & 3u;
                        *reinterpret_cast<unsigned short *>(mask + idx + 2 * q) = (unsigned short)((b2 & 1u) | ((b2 & 2u) << 7));
                    } else {
                        const unsigned b4 = (bits >> (4 * q)) & 15u;
                        // bit i -> byte i: the partial products i + 7 k land on a multiple of 8 only for k = i
                        *reinterpret_cast<unsigned *>(mask + idx + 4 * q) = (b4 * 0x00204081u) & 0x01010101u;
                    }
                }
            }
            if constexpr (STATS) {
#pragma unroll
                for (int j = 0; j < G; ++j) {
                    const float n = nxz[u][j] * nyc;
                    const float m = S1[j] / n;
                    if (j >= VL * nvq[u]) break;
                    if (mean != nullptr) mean[idx + j] = m + piv;
                    if (sd != nullptr) sd[idx + j] = sqrtf(fmaxf(S2[j] / n - m * m, 0.f));
                }
            }
        }
    };
    {
        float fvA[UPW][G], fvB[UPW][G];
        unsigned mkA[UPW][NV], mkB[UPW][NV];
        load_centre(0, fvA, mkA);
        for (int b = 0; b < nb; b += 2) {
            batch(b, fvA, mkA, fvB, mkB);
            if (b + 1 < nb) batch(b + 1, fvB, mkB, fvA, mkA);
        }
    }

    if (count != nullptr) {
        unsigned c = my_count;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
        if (lane == 0) wsum[warp] = c;
        __syncthreads();
        if (tid == 0) {
            const unsigned t = wsum[0] + wsum[1] + wsum[2] + wsum[3];
            if (t) atomicAdd(count, (unsigned long long)t);
        }
    }
}

template <int G, int MODE>
cudaError_t launch_xyb_m(const float *f, const float *Z1, const float *Z2, uint8_t *mask, float *mean, float *sd,
                         unsigned long long *count, const XybParams &p, dim3 grid, const float *pivot, const float *zeros,
                         cudaStream_t st)
{
    if (mean != nullptr || sd != nullptr)
        k_xyb<G, MODE, true><<<grid, XybShape<G>::NT, 0, st>>>(f, Z1, Z2, mask, mean, sd, count, p, pivot, zeros);
    else
        k_xyb<G, MODE, false><<<grid, XybShape<G>::NT, 0, st>>>(f, Z1, Z2, mask, mean, sd, count, p, pivot, zeros);
    return cudaGetLastError();
}

template <int G>
cudaError_t launch_xyb(const pgsf_plan *pl, const float *f, const float *Z1, const float *Z2, uint8_t *mask,
                       float *mean, float *sd, unsigned long long *count, XybParams p, int ncubes, cudaStream_t st)
{
    using S = XybShape<G>;
    const Dims &d = p.d;
    (void)pl;
    // balanced strips of whole column groups
    int ns = (d.nx + S::WMAX - 1) / S::WMAX;
    constexpr int WQ = (G == 6) ? 24 : 8;          // whole groups of G columns and whole 32-byte sectors
    p.wo = ((d.nx + ns - 1) / ns + WQ - 1) / WQ * WQ;
    if (p.wo > S::WMAX) p.wo = S::WMAX;
    ns = (d.nx + p.wo - 1) / p.wo;
    p.nstrips = ns;
    p.nplanes = (long long)d.nz * ncubes;
    const long long gxl = ((long long)ns * p.nplanes + S::NSTRIP - 1) / S::NSTRIP;
    // y chunks: a function of ny alone -- the running sums of a chunk start afresh, so the rounding of a voxel's
    // statistics must not depend on how many planes a launch happens to hold (a streamed cube is launched section
    // by section and must reproduce the resident call bit for bit).  A chunk start re-reads 2 hy rows.
    int nch = (d.ny + 1535) / 2048;
    if (nch < 1) nch = 1;
    p.ychunk = (d.ny + nch - 1) / nch;
    nch = (d.ny + p.ychunk - 1) / p.ychunk;
    if (gxl > 0x7fffffffLL || nch > 65535) return cudaErrorInvalidConfiguration;
    dim3 grid((unsigned)gxl, nch, 1);
    const float *zeros = pl->d_pivot + 16;            // (the plan's constant block: 256 bytes, zero beyond the pivot)
    switch (p.mode) {
    case 0: return launch_xyb_m<G, 0>(f, Z1, Z2, mask, mean, sd, count, p, grid, pl->d_pivot, zeros, st);
    case 1: return launch_xyb_m<G, 1>(f, Z1, Z2, mask, mean, sd, count, p, grid, pl->d_pivot, zeros, st);
    default: return launch_xyb_m<G, 2>(f, Z1, Z2, mask, mean, sd, count, p, grid, pl->d_pivot, zeros, st);
    }
}

}  // namespace

bool xyb_supported(const pgsf_plan *p)
{
    const int hx = p->desc.box_half[0];
    return p->desc.nx % 4 == 0 && (hx == 4 || hx == 8 || hx == 12 || hx == 16) && p->desc.nz <= 65535;
}

cudaError_t xyb_threshold(pgsf_plan *p, const float *f, const float *Z1, const float *Z2, uint8_t *mask, int mode,
                          float *mean, float *sd, unsigned long long *count, int ncubes, cudaStream_t st, int nplanes,
                          int z_off)
{
    XybParams xp;
    xp.d = p->dims;
    xp.z_off = 0;
    xp.nz_full = p->dims.nz;
    if (nplanes > 0) {      // a section of one cube
        xp.d.nz = nplanes;
        xp.d.cube = xp.d.plane * nplanes;
        xp.z_off = z_off;
        ncubes = 1;
    }
    xp.hy = p->desc.box_half[1];
    xp.hz = p->desc.box_half[2];
    xp.gx = p->desc.halo[0];
    xp.gy = p->desc.halo[1];
    xp.gz = p->desc.halo[2];
    xp.mode = mode;
    xp.k2 = (float)(p->desc.k * p->desc.k);
    xp.wo = xp.nstrips = xp.ychunk = 0;
    LaunchScope ls(p, "stats_xybox", st);
    switch (p->desc.box_half[0]) {
    case 4: return launch_xyb<2>(p, f, Z1, Z2, mask, mean, sd, count, xp, ncubes, st);
    case 8: return launch_xyb<4>(p, f, Z1, Z2, mask, mean, sd, count, xp, ncubes, st);
    case 12: return launch_xyb<6>(p, f, Z1, Z2, mask, mean, sd, count, xp, ncubes, st);
    case 16: return launch_xyb<8>(p, f, Z1, Z2, mask, mean, sd, count, xp, ncubes, st);
    default: return cudaErrorNotSupported;
    }
}

}  // namespace pgsf
