// Local statistics + voxel selection for sm_100a ("three directional sums" of the filtered
// data and of its square, then the z-score; P:33 / P:282 threshold and voxel selection; readings
// C-6..C-10).  Two kernels per filtered cube:
//
//   k_zbox    frequency direction first.  Every thread owns four adjacent (x, y) columns and marches
//             along z with the window sums  Z1 = sum_{|o|<=hz} f(z+o),  Z2 = sum f(z+o)^2  in registers:
//             the plane entering the window is added, the plane leaving it subtracted (both read from
//             HBM; nothing is staged).  The running sums are fp64 ("sums in double"): a bright source is
//             > 10^3 x the filtered noise in f^2, and an fp32 running sum would keep the rounding error made
//             while the source was inside the window long after it has left.
//             Writes Z1, Z2 (two workspace cubes).
//   k_ymarch  per z plane: y-direction window sums marched in registers, x-direction window from the
//             prefix / suffix sums of thread-owned column groups, then m = S1/n, var = S2/n - m^2,
//             selection f > m + k sd (division-free form of pgsf_generic.cu), halo, mask write / OR, count
//             (details at the kernel).
// Inside pgsf_find_multiscale the z direction comes out of the frequency pass itself (k_zm, pgsf_zpass.cuh)
// and k_zbox is not launched.
//
// Preconditions (else the generic kernels run): fast_stats_supported() below.
#include <stdio.h>

#include "pgsf_internal.h"
#include "pgsf_device.cuh"

namespace pgsf {
namespace {

// ------------------------------------------------------------------------------------ k_zbox

constexpr int ZB_NT = 256;

struct ZboxParams {
    Dims d;
    int hz;
    int zchunk, nchunks;
    long long cols4;     // nx*ny/4 float4 columns per cube
};

__global__ void __launch_bounds__(ZB_NT) k_zbox(const float4 *__restrict__ f, float4 *__restrict__ Z1,
                                                float4 *__restrict__ Z2, ZboxParams p, const float *__restrict__ pivot)
{
    const float c0 = __ldg(pivot);     // sums of f - c0 and (f - c0)^2 (D-2); planes outside the cube contribute nothing
    const long long c = (long long)blockIdx.x * ZB_NT + threadIdx.x;
    if (c >= p.cols4) return;
    const int chunk = blockIdx.y;
    const int za = chunk * p.zchunk, zb = min(za + p.zchunk, p.d.nz);
    const long long plane4 = p.d.plane / 4;
    const int hz = p.hz, nz = p.d.nz;
    // fp64 running sums, the arithmetic of k_zm's window phase (pgsf_zpass.cuh: window_run), so that the per-scale call
    // and pgsf_find_multiscale see the same Z1 / Z2
    double s1[4] = {0.0, 0.0, 0.0, 0.0}, s2[4] = {0.0, 0.0, 0.0, 0.0};
    // planes za-hz .. za+hz-1 of the first window (clipped to the cube, C-7)
    for (int z = max(za - hz, 0); z < min(za + hz, nz); ++z) {
        const float4 v = __ldg(f + (long long)z * plane4 + c);
        const double a[4] = {(double)(v.x - c0), (double)(v.y - c0), (double)(v.z - c0), (double)(v.w - c0)};
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            s1[u] += a[u];
            s2[u] = fma(a[u], a[u], s2[u]);
        }
    }
#pragma unroll 4
    for (int zc = za; zc < zb; ++zc) {
        const int zl = zc + hz, zt = zc - hz;
        float4 l = make_float4(c0, c0, c0, c0), t = make_float4(c0, c0, c0, c0);
        if (zl < nz) l = __ldg(f + (long long)zl * plane4 + c);
        if (zt >= 0) t = __ldg(f + (long long)zt * plane4 + c);   // leaves after this output
        const double a[4] = {(double)(l.x - c0), (double)(l.y - c0), (double)(l.z - c0), (double)(l.w - c0)};
        const double b[4] = {(double)(t.x - c0), (double)(t.y - c0), (double)(t.z - c0), (double)(t.w - c0)};
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            s1[u] += a[u];
            s2[u] = fma(a[u], a[u], s2[u]);
        }
        const long long o = (long long)zc * plane4 + c;
        Z1[o] = make_float4((float)s1[0], (float)s1[1], (float)s1[2], (float)s1[3]);
        Z2[o] = make_float4((float)s2[0], (float)s2[1], (float)s2[2], (float)s2[3]);
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            s1[u] -= b[u];
            s2[u] = fma(-b[u], b[u], s2[u]);
        }
    }
}

// ------------------------------------------------------------------------------------ k_ymarch
//
// One CTA = one z plane, one x tile, one y chunk.  A thread owns G = hx/2 adjacent columns and
// marches down y with the y-direction window sums  Y1 = sum_{|o|<=hy} Z1(y+o),  Y2 likewise  in
// registers (row entering the window added, row leaving it subtracted; the leaving row was read
// 2 hy + 1 steps earlier, so it comes from L2).  Y2 is Kahan-compensated for the same reason as in
// k_zbox; Y1 only enters through the mean, whose tolerance is ~n times looser, and stays plain.
// The x-direction window of 2 hx + 1 = 4 G + 1 columns is then exactly
//      (suffix of the thread two to the left) + (the three threads in between) + (prefix of the
//      thread two to the right),
// so every thread publishes the G prefix and G suffix sums of its own columns in shared memory and
// combines five neighbours' values: ~4 additions per voxel, every output a plain sum of the elements
// of its own window (no cancellation).  One __syncthreads per row (double-buffered exchange).

constexpr int YM_MAX_NT = 256;

struct YmParams {
    Dims d;
    int hy, hz;
    int gx, gy, gz;      // halo excluded from mask and count (C-11)
    int or_into;
    float k2;            // k^2
    int wo;              // output columns per x tile (tiles overlap by 2 hx staged columns)
    int ntiles;
    int ychunk;          // rows per CTA
};

template <int G> struct VecT { using type = float4; static constexpr int L = 4; };
template <> struct VecT<2> { using type = float2; static constexpr int L = 2; };

__device__ __forceinline__ int clipped_len(int c, int h, int n)
{
    return min(c + h, n - 1) - max(c - h, 0) + 1;
}

template <int G>
__device__ __forceinline__ void ld_cols(const float *__restrict__ p, bool ok, float (&v)[G])
{
    if constexpr (G == 2) {
        const float2 t = ok ? __ldg(reinterpret_cast<const float2 *>(p)) : make_float2(0.f, 0.f);
        v[0] = t.x; v[1] = t.y;
    } else {
#pragma unroll
        for (int q = 0; q < G / 4; ++q) {
            const float4 t = ok ? __ldg(reinterpret_cast<const float4 *>(p) + q) : make_float4(0.f, 0.f, 0.f, 0.f);
            v[4 * q] = t.x; v[4 * q + 1] = t.y; v[4 * q + 2] = t.z; v[4 * q + 3] = t.w;
        }
    }
}

template <int G>
struct YmRow {          // everything one march step reads from global memory
    float l1[G], l2[G];  // row entering the window
    float t1[G], t2[G];  // row leaving it
    float fc[G];         // centre values
    unsigned mk[(G + 3) / 4];   // previous mask bytes (OR mode)
};

template <int G>
__device__ __forceinline__ void ym_load(YmRow<G> &r, const float *__restrict__ f, const float *__restrict__ Z1,
                                        const float *__restrict__ Z2, const uint8_t *__restrict__ mask,
                                        long long col_off, int y, const YmParams &p, bool col_ok)
{
    const int nx = p.d.nx, ny = p.d.ny;
    const int yl = y + p.hy, yt = y - p.hy;
    const bool okl = col_ok && yl < ny, okt = col_ok && yt >= 0, okc = col_ok && y < ny;
    const long long ol = okl ? col_off + (long long)yl * nx : 0;
    const long long ot = okt ? col_off + (long long)yt * nx : 0;
    const long long oc = okc ? col_off + (long long)y * nx : 0;
    ld_cols<G>(Z1 + ol, okl, r.l1);
    ld_cols<G>(Z2 + ol, okl, r.l2);
    ld_cols<G>(Z1 + ot, okt, r.t1);
    ld_cols<G>(Z2 + ot, okt, r.t2);
    ld_cols<G>(f + oc, okc, r.fc);
    if (p.or_into) {
        if constexpr (G == 2) r.mk[0] = okc ? *reinterpret_cast<const unsigned short *>(mask + oc) : 0u;
        else {
#pragma unroll
            for (int q = 0; q < G / 4; ++q) r.mk[q] = okc ? *reinterpret_cast<const unsigned *>(mask + oc + 4 * q) : 0u;
        }
    } else {
#pragma unroll
        for (int q = 0; q < (G + 3) / 4; ++q) r.mk[q] = 0u;
    }
}

template <int G>
__global__ void __launch_bounds__(YM_MAX_NT) k_ymarch(const float *__restrict__ f, const float *__restrict__ Z1,
                                                      const float *__restrict__ Z2, uint8_t *__restrict__ mask,
                                                      float *__restrict__ mean, float *__restrict__ sd,
                                                      unsigned long long *__restrict__ count, const YmParams p,
                                                      const float *__restrict__ pivot)
{
    const float piv = __ldg(pivot);    // Z1, Z2 are sums of f - c0 and (f - c0)^2; the centre value is shifted alike
    using V = typename VecT<G>::type;
    constexpr int VL = VecT<G>::L, NV = G / VL, HX = 2 * G;
    extern __shared__ __align__(16) unsigned char ym_smem[];
    V *sm = reinterpret_cast<V *>(ym_smem);
    const int NT = blockDim.x, SL = NT + 4, tid = threadIdx.x;
    // exchange buffers [parity][array Y1/Y2][prefix/suffix][NV][SL]; thread t lives in slot t + 2,
    // the two slots on either side stay zero (= nothing beyond the staged columns)
    auto buf = [&](int par, int arr, int kind, int v) -> V * { return sm + ((((par * 2 + arr) * 2 + kind) * NV + v) * SL); };
    for (int i = tid; i < 32 * NV; i += NT) {
        V *b = sm + (i / 4) * SL;
        const int e = i & 3;
        V z;
        if constexpr (G == 2) z = make_float2(0.f, 0.f); else z = make_float4(0.f, 0.f, 0.f, 0.f);
        b[e < 2 ? e : NT + e] = z;
    }
    const Dims &d = p.d;
    const int zz = blockIdx.z;                         // plane of the stack of cubes
    const int z = zz % d.nz;                           // channel inside its cube
    const int out_lo = (p.ntiles == 1) ? 0 : blockIdx.x * p.wo;
    const int out_hi = (p.ntiles == 1) ? d.nx : min(d.nx, out_lo + p.wo);
    const int xs = (p.ntiles == 1) ? 0 : out_lo - HX;
    const int c0 = xs + G * tid;                       // first of this thread's G columns
    const bool col_ok = c0 >= 0 && c0 + G <= d.nx;     // (extents are multiples of the vector width)
    const long long col_off = (long long)zz * d.plane + (col_ok ? c0 : 0);
    const int ya = blockIdx.y * p.ychunk, yb = min(ya + p.ychunk, d.ny);
    const bool is_out = col_ok && c0 >= out_lo && c0 < out_hi;

    float nxz[G];                                      // clipped window lengths along x times along z
    unsigned core_x = 0;                               // bit j: column j is outside the x/z halo
    {
        const float nzc = (float)clipped_len(z, p.hz, d.nz);
        const bool core_z = z >= p.gz && z < d.nz - p.gz;
#pragma unroll
        for (int j = 0; j < G; ++j) {
            const int c = min(max(c0 + j, 0), d.nx - 1);
            nxz[j] = (float)clipped_len(c, HX, d.nx) * nzc;
            if (core_z && c0 + j >= p.gx && c0 + j < d.nx - p.gx) core_x |= 1u << j;
        }
    }

    float s1[G], s2[G], e2[G];
#pragma unroll
    for (int j = 0; j < G; ++j) s1[j] = s2[j] = e2[j] = 0.f;
    // rows ya-hy .. ya+hy-1 of the first window (clipped to the cube, C-7)
    for (int r = max(ya - p.hy, 0); r < min(ya + p.hy, d.ny); ++r) {
        float a1[G], a2[G];
        ld_cols<G>(Z1 + col_off + (long long)r * d.nx, col_ok, a1);
        ld_cols<G>(Z2 + col_off + (long long)r * d.nx, col_ok, a2);
#pragma unroll
        for (int j = 0; j < G; ++j) {
            s1[j] += a1[j];
            kahan_add(s2[j], e2[j], a2[j]);
        }
    }
    __syncthreads();   // zero padding of the exchange buffers is in place

    unsigned my_count = 0;
    YmRow<G> cur, nxt;
    ym_load<G>(cur, f, Z1, Z2, mask, col_off, ya, p, col_ok);
    const float guard = kFlatGuard;
#pragma unroll 2
    for (int y = ya; y < yb; ++y) {
        if (y + 1 < yb) ym_load<G>(nxt, f, Z1, Z2, mask, col_off, y + 1, p, col_ok);
        const int par = (y - ya) & 1;
        // window sums along y of this thread's columns; prefix / suffix sums across its columns
        float P1[G], Q1[G], P2[G], Q2[G];
#pragma unroll
        for (int j = 0; j < G; ++j) {
            s1[j] += cur.l1[j];
            kahan_add(s2[j], e2[j], cur.l2[j]);
            P1[j] = Q1[j] = s1[j];
            P2[j] = Q2[j] = s2[j] - e2[j];
        }
#pragma unroll
        for (int j = 1; j < G; ++j) { P1[j] += P1[j - 1]; P2[j] += P2[j - 1]; }
#pragma unroll
        for (int j = G - 2; j >= 0; --j) { Q1[j] += Q1[j + 1]; Q2[j] += Q2[j + 1]; }
#pragma unroll
        for (int v = 0; v < NV; ++v) {
            if constexpr (G == 2) {
                buf(par, 0, 0, v)[tid + 2] = make_float2(P1[0], P1[1]);
                buf(par, 0, 1, v)[tid + 2] = make_float2(Q1[0], Q1[1]);
                buf(par, 1, 0, v)[tid + 2] = make_float2(P2[0], P2[1]);
                buf(par, 1, 1, v)[tid + 2] = make_float2(Q2[0], Q2[1]);
            } else {
                buf(par, 0, 0, v)[tid + 2] = make_float4(P1[4 * v], P1[4 * v + 1], P1[4 * v + 2], P1[4 * v + 3]);
                buf(par, 0, 1, v)[tid + 2] = make_float4(Q1[4 * v], Q1[4 * v + 1], Q1[4 * v + 2], Q1[4 * v + 3]);
                buf(par, 1, 0, v)[tid + 2] = make_float4(P2[4 * v], P2[4 * v + 1], P2[4 * v + 2], P2[4 * v + 3]);
                buf(par, 1, 1, v)[tid + 2] = make_float4(Q2[4 * v], Q2[4 * v + 1], Q2[4 * v + 2], Q2[4 * v + 3]);
            }
        }
        // the row leaving the window (after this output)
#pragma unroll
        for (int j = 0; j < G; ++j) {
            s1[j] -= cur.t1[j];
            kahan_add(s2[j], e2[j], -cur.t2[j]);
        }
        __syncthreads();
        // x-direction window: suffix(t-2) + total(t-1) + total(t) + total(t+1) + prefix(t+2)
        float S1[G], S2[G];
        {
            const float m1 = reinterpret_cast<const float *>(buf(par, 0, 1, 0) + tid + 1)[0] + P1[G - 1] +
                             reinterpret_cast<const float *>(buf(par, 0, 1, 0) + tid + 3)[0];
            const float m2 = reinterpret_cast<const float *>(buf(par, 1, 1, 0) + tid + 1)[0] + P2[G - 1] +
                             reinterpret_cast<const float *>(buf(par, 1, 1, 0) + tid + 3)[0];
#pragma unroll
            for (int v = 0; v < NV; ++v) {
                const V a1 = buf(par, 0, 1, v)[tid], b1 = buf(par, 0, 0, v)[tid + 4];
                const V a2 = buf(par, 1, 1, v)[tid], b2 = buf(par, 1, 0, v)[tid + 4];
                const float *pa1 = reinterpret_cast<const float *>(&a1), *pb1 = reinterpret_cast<const float *>(&b1);
                const float *pa2 = reinterpret_cast<const float *>(&a2), *pb2 = reinterpret_cast<const float *>(&b2);
#pragma unroll
                for (int e = 0; e < VL; ++e) {
                    S1[VL * v + e] = m1 + (pa1[e] + pb1[e]);
                    S2[VL * v + e] = m2 + (pa2[e] + pb2[e]);
                }
            }
        }
        // selection (division-free form, see pgsf_generic.cu), halo, OR, mask bytes
        const float nyc = (float)clipped_len(y, p.hy, d.ny);
        const bool core_y = y >= p.gy && y < d.ny - p.gy;
        unsigned bits = 0;
#pragma unroll
        for (int j = 0; j < G; ++j) {
            const float n = nxz[j] * nyc;
            const float v = cur.fc[j] - piv;
            const float a = fmaf(n, v, -S1[j]);
            const float q = fmaxf(fmaf(n, S2[j], -S1[j] * S1[j]), 0.f);
            const bool sel = (a > guard * n * fabsf(v)) && (a * a > p.k2 * q);
            if (sel) bits |= 1u << j;
        }
        if (p.or_into) {   // previous mask: any non-zero byte counts as set
            if constexpr (G == 2) {
                bits |= ((cur.mk[0] & 0xffu) ? 1u : 0u) | ((cur.mk[0] & 0xff00u) ? 2u : 0u);
            } else {
#pragma unroll
                for (int q4 = 0; q4 < G / 4; ++q4) {
                    const unsigned old = cur.mk[q4];
                    const unsigned nz = ((old | ((old & 0x7f7f7f7fu) + 0x7f7f7f7fu)) >> 7) & 0x01010101u;
                    bits |= ((nz & 1u) | ((nz >> 7) & 2u) | ((nz >> 14) & 4u) | ((nz >> 21) & 8u)) << (4 * q4);
                }
            }
        }
        bits = core_y ? (bits & core_x) : 0u;
        if (is_out) {
            const long long idx = col_off + (long long)y * d.nx;
            my_count += __popc(bits);
            if constexpr (G == 2) {
                *reinterpret_cast<unsigned short *>(mask + idx) = (unsigned short)((bits & 1u) | ((bits & 2u) << 7));
            } else {
#pragma unroll
                for (int q4 = 0; q4 < G / 4; ++q4) {
                    const unsigned b4 = (bits >> (4 * q4)) & 15u;
                    *reinterpret_cast<unsigned *>(mask + idx + 4 * q4) =
                        (b4 & 1u) | ((b4 & 2u) << 7) | ((b4 & 4u) << 14) | ((b4 & 8u) << 21);
                }
            }
            if (mean != nullptr || sd != nullptr) {
#pragma unroll
                for (int j = 0; j < G; ++j) {
                    const float n = nxz[j] * nyc;
                    const float m = S1[j] / n;
                    if (mean != nullptr) mean[idx + j] = m + piv;
                    if (sd != nullptr) sd[idx + j] = sqrtf(fmaxf(S2[j] / n - m * m, 0.f));
                }
            }
        }
        cur = nxt;
    }

    if (count != nullptr) {
        __shared__ unsigned wsum[YM_MAX_NT / 32];
        unsigned c = my_count;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
        if ((tid & 31) == 0) wsum[tid >> 5] = c;
        __syncthreads();
        if (tid == 0) {
            unsigned t = 0;
            for (int w = 0; w < NT / 32; ++w) t += wsum[w];
            if (t) atomicAdd(count, (unsigned long long)t);
        }
    }
}

template <int G>
cudaError_t launch_ymarch(const pgsf_plan *pl, const float *f, const float *Z1, const float *Z2, uint8_t *mask,
                          float *mean, float *sd, unsigned long long *count, YmParams p, int ncubes, cudaStream_t st)
{
    constexpr int VL = VecT<G>::L;
    const Dims &d = p.d;
    // threads: cover the whole row when it fits in one CTA, else tiles overlapping by 2 hx columns
    // (CTAs of at most 128 threads: at 152 registers four of them share an SM, one of 256 threads would be alone)
    constexpr int kPreferredNT = 128;
    int nt = ((d.nx + G - 1) / G + 31) / 32 * 32;
    if (nt <= kPreferredNT) {
        p.ntiles = 1;
        p.wo = d.nx;
    } else {
        const int wo_max = kPreferredNT * G - 4 * G;
        p.ntiles = (d.nx + wo_max - 1) / wo_max;
        p.wo = ((d.nx + p.ntiles - 1) / p.ntiles + G - 1) / G * G;      // balanced tiles, whole column groups
        nt = ((p.wo + 4 * G) / G + 31) / 32 * 32;
    }
    // y chunks: enough CTAs for a few waves; a chunk start re-reads 2 hy rows
    const long long resident = (long long)pl->sm_count * (nt <= 128 ? 4 : 2);
    const long long base = (long long)p.ntiles * d.nz * ncubes;
    int nch = (int)((4 * resident + base - 1) / base);
    const int min_rows = 8 * p.hy > 64 ? 8 * p.hy : 64;
    if (nch > (d.ny + min_rows - 1) / min_rows) nch = (d.ny + min_rows - 1) / min_rows;
    if (nch < 1) nch = 1;
    p.ychunk = (d.ny + nch - 1) / nch;
    nch = (d.ny + p.ychunk - 1) / p.ychunk;
    const int smem = 8 * (G / VL) * (nt + 4) * VL * (int)sizeof(float);
    cudaError_t ce = ensure_dynamic_smem(k_ymarch<G>, smem);
    if (ce != cudaSuccess) return ce;
    if ((long long)d.nz * ncubes > 65535) return cudaErrorInvalidConfiguration;
    dim3 grid(p.ntiles, nch, d.nz * ncubes);
    k_ymarch<G><<<grid, nt, smem, st>>>(f, Z1, Z2, mask, mean, sd, count, p, pl->d_pivot);
    return cudaGetLastError();
}

}  // namespace

bool fast_stats_supported(const pgsf_plan *p, std::string *why)
{
    const int hx = p->desc.box_half[0];
    char buf[128];
    buf[0] = 0;
    if (p->desc.nx % 4 != 0) snprintf(buf, sizeof buf, "nx %% 4 != 0");
    else if (xyb_supported(p)) { /* k_xyb: hx in {4, 8, 12, 16}, any nx that is a multiple of 4 */ }
    else if (hx != 4 && hx != 8 && hx != 12 && hx != 16) snprintf(buf, sizeof buf, "hx = %d is not one of the compiled 4, 8, 12, 16", hx);
    else if (p->desc.nz > 65535) snprintf(buf, sizeof buf, "nz above 65535");
    if (why) *why = buf;
    return buf[0] == 0;
}

cudaError_t fast_threshold(pgsf_plan *p, const float *f, uint8_t *mask, int or_into, float *mean, float *sd,
                           unsigned long long *count, float *tmp2, cudaStream_t st)
{
    const Dims &d = p->dims;
    float *Z1 = tmp2, *Z2 = tmp2 + d.cube;
    ZboxParams zp;
    zp.d = d;
    zp.hz = p->desc.box_half[2];
    zp.cols4 = d.plane / 4;
    // z chunks: enough threads to fill the machine; a chunk re-reads 2 hz planes, so keep it long
    const long long blocks = (zp.cols4 + ZB_NT - 1) / ZB_NT;
    const long long want = 2LL * p->sm_count * (2048 / ZB_NT);
    int nchunks = (int)((want + blocks - 1) / blocks);
    const int min_chunk = 8 * zp.hz > 32 ? 8 * zp.hz : 32;
    if (nchunks > (d.nz + min_chunk - 1) / min_chunk) nchunks = (d.nz + min_chunk - 1) / min_chunk;
    if (nchunks < 1) nchunks = 1;
    zp.zchunk = (d.nz + nchunks - 1) / nchunks;
    zp.nchunks = (d.nz + zp.zchunk - 1) / zp.zchunk;
    if (blocks > 0x7fffffffLL || zp.nchunks > 65535) return cudaErrorInvalidConfiguration;
    {
        LaunchScope ls(p, "stats_zbox", st);
        dim3 grid((unsigned)blocks, (unsigned)zp.nchunks);
        k_zbox<<<grid, ZB_NT, 0, st>>>(reinterpret_cast<const float4 *>(f), reinterpret_cast<float4 *>(Z1),
                                       reinterpret_cast<float4 *>(Z2), zp, p->d_pivot);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    return fast_threshold_xy(p, f, Z1, Z2, mask, or_into, mean, sd, count, 1, st);
}

cudaError_t fast_threshold_xy(pgsf_plan *p, const float *f, const float *Z1, const float *Z2, uint8_t *mask,
                              int mode, float *mean, float *sd, unsigned long long *count, int ncubes,
                              cudaStream_t st)
{
    // k_ymarch (PGSF_OPT_TUNE bit 1) exists for hx = 4, 8, 16 with nx a multiple of hx / 2 only
    const int hx0 = p->desc.box_half[0];
    const bool legacy_ok = (hx0 == 4 || hx0 == 8 || hx0 == 16) && p->desc.nx % (hx0 / 2) == 0;
    if (xyb_supported(p) && (!(p->tune & 2) || !legacy_ok)) return xyb_threshold(p, f, Z1, Z2, mask, mode, mean, sd, count, ncubes, st);
    if (mode == 2) return cudaErrorNotSupported;   // (callers ask stats_sparse_or() first)
    const int or_into = mode;
    const Dims &d = p->dims;
    YmParams yp;
    yp.d = d;
    yp.hy = p->desc.box_half[1];
    yp.hz = p->desc.box_half[2];
    yp.gx = p->desc.halo[0];
    yp.gy = p->desc.halo[1];
    yp.gz = p->desc.halo[2];
    yp.or_into = or_into;
    yp.k2 = (float)(p->desc.k * p->desc.k);
    yp.wo = yp.ntiles = yp.ychunk = 0;
    LaunchScope ls(p, "stats_xybox", st);
    switch (p->desc.box_half[0]) {
    case 4: return launch_ymarch<2>(p, f, Z1, Z2, mask, mean, sd, count, yp, ncubes, st);
    case 8: return launch_ymarch<4>(p, f, Z1, Z2, mask, mean, sd, count, yp, ncubes, st);
    case 16: return launch_ymarch<8>(p, f, Z1, Z2, mask, mean, sd, count, yp, ncubes, st);
    default: return cudaErrorNotSupported;
    }
}

}  // namespace pgsf
