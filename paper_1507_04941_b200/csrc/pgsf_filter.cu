// Tiled sm_100a kernels for the separable form of Eq. 2 (index ranges Eq. 3-5).
//
//   k_xy<R>  : per z-plane, x and y passes staged through shared memory (input tile + halo, zero
//              filled outside the cube = the zero padding of reading C-5), result t2 to HBM.
//   k_z<RZ>  : the frequency axis (filters are largest along z).  A CTA stages a slab of
//              ZB + 2 RZ planes of a 128-column strip in shared memory; every thread owns four
//              x columns and PZ consecutive channels and walks along z with its accumulators in
//              registers.
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

namespace pgsf {
namespace {

// ------------------------------------------------------------------------------------ helpers

__device__ __forceinline__ float2 ffma2(float2 a, float g, float2 c)
{
    // d = a * {g, g} + c, both halves in one instruction
    const float2 gg = make_float2(g, g);
    unsigned long long ra = *reinterpret_cast<const unsigned long long *>(&a);
    unsigned long long rb = *reinterpret_cast<const unsigned long long *>(&gg);
    unsigned long long rc = *reinterpret_cast<const unsigned long long *>(&c);
    unsigned long long rd;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(rd) : "l"(ra), "l"(rb), "l"(rc));
    return *reinterpret_cast<float2 *>(&rd);
}

__device__ __forceinline__ void cp_async16(void *smem, const void *gmem, bool valid)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    const int bytes = valid ? 16 : 0;  // src-size 0 -> 16 bytes of zeros
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(s), "l"(gmem), "r"(bytes));
}
__device__ __forceinline__ void cp_async_wait_all()
{
    asm volatile("cp.async.commit_group;\n\tcp.async.wait_group 0;" ::: "memory");
}

__host__ __device__ constexpr int round4(int v) { return (v + 3) & ~3; }

// ------------------------------------------------------------------------------------ x/y passes
//
// k_xy_multi<RMAX>: one z plane tile of 128 x 32 voxels.  The input tile + RMAX halo is staged ONCE
// (zero fill outside the cube, C-5) and the x and y passes of EVERY scale of the bank are evaluated
// from it ("several sigma scales evaluated per input read", BASELINE.json north_star): the input cube
// is read once for all scales instead of once per scale.
//   y pass (Eq. 4): thread = 4 staged columns x 4 rows; walks down the staged rows (LDS.128), packed
//                   FFMA2 over x pairs; result stored with the rows of a row PAIR interleaved,
//                   t1[(row/2)][col][row%2], so that
//   x pass (Eq. 3): thread = 2 rows x 8 columns; one LDS.128 yields two columns of both rows as two
//                   (row, row+1) register pairs, i.e. the x pass is packed FFMA2 over row pairs.

constexpr int XM_TX = 128;
constexpr int XM_TY = 32;
constexpr int XM_NT = 256;
constexpr int XM_PY = 4;        // rows per thread in the y pass
constexpr int XM_QX = 8;        // columns per thread in the x pass (times two rows)

struct XYMultiParams {
    Dims d;
    int n;                          // scales in this launch
    int rc[PGSF_MAX_SCALES];        // compiled radius of each
    float *out[PGSF_MAX_SCALES];    // x/y-filtered plane stack of each
    TapsXY t[PGSF_MAX_SCALES];
};

template <int RMAX>
struct XMShape {
    static constexpr int R4M = round4(RMAX);
    static constexpr int W = XM_TX + 2 * R4M;                    // staged columns
    static constexpr int HI = XM_TY + 2 * RMAX;                  // staged rows
    static constexpr int WT = W + ((2 - W % 16) + 16) % 16;      // t1 pitch in columns, = 2 (mod 16):
                                                                 // row pairs 4 banks apart
    static constexpr int SMEM = (HI * W + XM_TY * WT) * 4;
};

template <int R, int RMAX>
__device__ __forceinline__ void xy_one_scale(const float *s_in, float *s_t1, float *__restrict__ out_plane,
                                             const TapsXY &t, const Dims &d, int x0, int y0, int tid)
{
    using S = XMShape<RMAX>;
    constexpr int R4 = round4(R);
    constexpr int C0 = S::R4M - R4;                 // first staged column this scale needs
    constexpr int W4s = (XM_TX + 2 * R4) / 4;
    constexpr int YB = XM_TY / XM_PY;
    // ---- y pass
    for (int task = tid; task < W4s * YB; task += XM_NT) {
        const int yb = task / W4s, c4 = task - yb * W4s;
        float2 acc[XM_PY][2];
#pragma unroll
        for (int p = 0; p < XM_PY; ++p) acc[p][0] = acc[p][1] = make_float2(0.f, 0.f);
        const float *col = s_in + (yb * XM_PY + (RMAX - R)) * S::W + C0 + 4 * c4;
#pragma unroll
        for (int j = 0; j < XM_PY + 2 * R; ++j) {
            const float4 v = *reinterpret_cast<const float4 *>(col + j * S::W);
#pragma unroll
            for (int p = 0; p < XM_PY; ++p) {
                const int o = j - p;
                if (o >= 0 && o <= 2 * R) {
                    acc[p][0] = ffma2(make_float2(v.x, v.y), t.gy[o], acc[p][0]);
                    acc[p][1] = ffma2(make_float2(v.z, v.w), t.gy[o], acc[p][1]);
                }
            }
        }
#pragma unroll
        for (int jj = 0; jj < XM_PY / 2; ++jj) {
            float *dst = s_t1 + ((yb * (XM_PY / 2) + jj) * S::WT + C0 + 4 * c4) * 2;
            const float2 a0 = acc[2 * jj][0], a1 = acc[2 * jj][1], b0 = acc[2 * jj + 1][0], b1 = acc[2 * jj + 1][1];
            *reinterpret_cast<float4 *>(dst) = make_float4(a0.x, b0.x, a0.y, b0.y);
            *reinterpret_cast<float4 *>(dst + 4) = make_float4(a1.x, b1.x, a1.y, b1.y);
        }
    }
    __syncthreads();
    // ---- x pass
    {
        const int jp = tid & (XM_TY / 2 - 1), xb = tid / (XM_TY / 2);
        constexpr int CS = S::R4M - R;              // staged column of tap o = 0 of output column 0
        constexpr int SH = CS & 1;                  // float4 loads start at an even column
        constexpr int NL = (XM_QX + 2 * R + SH + 1) / 2;
        float2 v[2 * NL];
        const float *src = s_t1 + (jp * S::WT + (CS - SH) + XM_QX * xb) * 2;
#pragma unroll
        for (int k = 0; k < NL; ++k) {
            const float4 q = *reinterpret_cast<const float4 *>(src + 4 * k);
            v[2 * k] = make_float2(q.x, q.y);
            v[2 * k + 1] = make_float2(q.z, q.w);
        }
        float2 acc[XM_QX];
#pragma unroll
        for (int i = 0; i < XM_QX; ++i) acc[i] = make_float2(0.f, 0.f);
#pragma unroll
        for (int o = 0; o <= 2 * R; ++o)
#pragma unroll
            for (int i = 0; i < XM_QX; ++i) acc[i] = ffma2(v[i + o + SH], t.gx[o], acc[i]);
        const int gy = y0 + 2 * jp, gx = x0 + XM_QX * xb;
        if (gx < d.nx) {
            float *dst = out_plane + (long long)gy * d.nx + gx;
            const bool second = gx + 4 < d.nx;
            if (gy < d.ny) {
                *reinterpret_cast<float4 *>(dst) = make_float4(acc[0].x, acc[1].x, acc[2].x, acc[3].x);
                if (second) *reinterpret_cast<float4 *>(dst + 4) = make_float4(acc[4].x, acc[5].x, acc[6].x, acc[7].x);
            }
            if (gy + 1 < d.ny) {
                *reinterpret_cast<float4 *>(dst + d.nx) = make_float4(acc[0].y, acc[1].y, acc[2].y, acc[3].y);
                if (second)
                    *reinterpret_cast<float4 *>(dst + d.nx + 4) = make_float4(acc[4].y, acc[5].y, acc[6].y, acc[7].y);
            }
        }
    }
}

template <int RMAX>
__global__ void __launch_bounds__(XM_NT) k_xy_multi(const float *__restrict__ in,
                                                     const __grid_constant__ XYMultiParams P)
{
    using S = XMShape<RMAX>;
    extern __shared__ __align__(16) float smem[];
    float *s_in = smem;                  // [HI][W]
    float *s_t1 = smem + S::HI * S::W;   // [TY/2][WT][2]
    const Dims &d = P.d;
    const int tid = threadIdx.x;
    const int x0 = blockIdx.x * XM_TX, y0 = blockIdx.y * XM_TY, z = blockIdx.z;
    const long long plane_off = (long long)z * d.plane;

    // stage the input tile + halo: thread <-> one 16-byte column chunk, rows r0, r0 + RP, ...
    {
        constexpr int W4 = S::W / 4, RP = XM_NT / W4;
        if (tid < RP * W4) {
            const int c4 = tid % W4, r0 = tid / W4;
            const int xx = x0 - S::R4M + 4 * c4;
            const bool xok = xx >= 0 && xx < d.nx;
            int yy = y0 - RMAX + r0;
            long long off = plane_off + (long long)yy * d.nx + xx;
            float *dst = s_in + r0 * S::W + 4 * c4;
            for (int r = r0; r < S::HI; r += RP) {
                const bool ok = xok && yy >= 0 && yy < d.ny;
                cp_async16(dst, in + (ok ? off : 0), ok);
                yy += RP;
                off += (long long)RP * d.nx;
                dst += RP * S::W;
            }
        }
        cp_async_wait_all();
        __syncthreads();
    }

    for (int s = 0; s < P.n; ++s) {
        if (s > 0) __syncthreads();      // the previous scale's x pass has read s_t1
        float *out_plane = P.out[s] + plane_off;
        const TapsXY &t = P.t[s];
        switch (P.rc[s]) {
        case 3: xy_one_scale<3, RMAX>(s_in, s_t1, out_plane, t, d, x0, y0, tid); break;
        case 6: if constexpr (RMAX >= 6) xy_one_scale<6, RMAX>(s_in, s_t1, out_plane, t, d, x0, y0, tid); break;
        case 9: if constexpr (RMAX >= 9) xy_one_scale<9, RMAX>(s_in, s_t1, out_plane, t, d, x0, y0, tid); break;
        case 12: if constexpr (RMAX >= 12) xy_one_scale<12, RMAX>(s_in, s_t1, out_plane, t, d, x0, y0, tid); break;
        default: break;
        }
    }
}

// ------------------------------------------------------------------------------------ z pass

constexpr int Z_XT = 128;       // columns per CTA (32 float4 lanes = one warp per plane row)
constexpr int Z_PZ = 8;         // channels per thread
constexpr int Z_WARPS = 8;      // z groups per CTA
constexpr int Z_THREADS = 32 * Z_WARPS;
constexpr int Z_ZB = Z_PZ * Z_WARPS;   // 64 output channels per CTA

template <int RZ>
struct ZShape {
    static constexpr int PLANES = Z_ZB + 2 * RZ;
    static constexpr int SMEM = PLANES * Z_XT * 4;
};

template <int RZ>
__global__ void __launch_bounds__(Z_THREADS) k_z(const float *__restrict__ in, float *__restrict__ out,
                                                 Dims d, Taps t)
{
    using S = ZShape<RZ>;
    extern __shared__ __align__(16) float smem[];  // [PLANES][Z_XT]
    const int tid = threadIdx.x, lane = tid & 31, wz = tid >> 5;
    const int z0 = blockIdx.x * Z_ZB, x0 = blockIdx.y * Z_XT, y = blockIdx.z;
    const int gx = x0 + 4 * lane;
    const bool col_ok = gx < d.nx;
    const float *col_in = in + (long long)y * d.nx + (col_ok ? gx : 0);

    // stage channels z0-RZ .. z0+ZB+RZ-1 of this 128-column strip; outside the cube -> 0 (C-5)
    for (int pz = wz; pz < S::PLANES; pz += Z_WARPS) {
        const int gz = z0 - RZ + pz;
        const bool ok = col_ok && gz >= 0 && gz < d.nz;
        cp_async16(smem + pz * Z_XT + 4 * lane, ok ? col_in + (long long)gz * d.plane : in, ok);
    }
    cp_async_wait_all();
    __syncthreads();

    // Eq. 5: f[z] = sum_o t2[z+o] gz[o]; the thread walks along z, PZ accumulators x 4 columns.
    // Taps are stored at g[o + kTapPad] with kTapPad zeros on both sides.
    float2 acc[Z_PZ][2];
#pragma unroll
    for (int p = 0; p < Z_PZ; ++p) acc[p][0] = acc[p][1] = make_float2(0.f, 0.f);
    const float *base = smem + (wz * Z_PZ) * Z_XT + 4 * lane;
    if constexpr (RZ <= 48) {
        // fully unrolled: every tap index is a compile-time constant-bank offset
#pragma unroll
        for (int j = 0; j < Z_PZ + 2 * RZ; ++j) {
            const float4 v = *reinterpret_cast<const float4 *>(base + j * Z_XT);
#pragma unroll
            for (int p = 0; p < Z_PZ; ++p) {
                const int o = j - p;
                if (o >= 0 && o <= 2 * RZ) {
                    acc[p][0] = ffma2(make_float2(v.x, v.y), t.g[o + kTapPad], acc[p][0]);
                    acc[p][1] = ffma2(make_float2(v.z, v.w), t.g[o + kTapPad], acc[p][1]);
                }
            }
        }
    } else {
        // too long to unroll: walk the PZ + 2 RZ staged channels in chunks of 8; the zero padding of
        // the tap array makes the ramp-up / ramp-down iterations the same code as the steady state
        static_assert((Z_PZ + 2 * RZ) % 8 == 0 && kTapPad >= Z_PZ - 1, "chunking");
#pragma unroll 1
        for (int jc = 0; jc < Z_PZ + 2 * RZ; jc += 8) {
#pragma unroll
            for (int jj = 0; jj < 8; ++jj) {
                const float4 v = *reinterpret_cast<const float4 *>(base + (jc + jj) * Z_XT);
#pragma unroll
                for (int p = 0; p < Z_PZ; ++p) {
                    const float g = t.g[jc + jj - p + kTapPad];
                    acc[p][0] = ffma2(make_float2(v.x, v.y), g, acc[p][0]);
                    acc[p][1] = ffma2(make_float2(v.z, v.w), g, acc[p][1]);
                }
            }
        }
    }
    if (!col_ok) return;
    float *col_out = out + (long long)y * d.nx + gx;
#pragma unroll
    for (int p = 0; p < Z_PZ; ++p) {
        const int gz = z0 + wz * Z_PZ + p;
        if (gz < d.nz)
            *reinterpret_cast<float4 *>(col_out + (long long)gz * d.plane) =
                make_float4(acc[p][0].x, acc[p][0].y, acc[p][1].x, acc[p][1].y);
    }
}

template <int RMAX>
cudaError_t launch_xy_multi(const float *in, const XYMultiParams &P, cudaStream_t st)
{
    static bool configured = false;
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(k_xy_multi<RMAX>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             XMShape<RMAX>::SMEM);
        if (e != cudaSuccess) return e;
        configured = true;
    }
    dim3 grid((P.d.nx + XM_TX - 1) / XM_TX, (P.d.ny + XM_TY - 1) / XM_TY, P.d.nz);
    k_xy_multi<RMAX><<<grid, XM_NT, XMShape<RMAX>::SMEM, st>>>(in, P);
    return cudaGetLastError();
}

template <int RZ>
cudaError_t launch_z(const float *in, float *out, const Dims &d, const Taps &t, cudaStream_t st)
{
    static bool configured = false;
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(k_z<RZ>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             ZShape<RZ>::SMEM);
        if (e != cudaSuccess) return e;
        configured = true;
    }
    dim3 grid((d.nz + Z_ZB - 1) / Z_ZB, (d.nx + Z_XT - 1) / Z_XT, d.ny);
    k_z<RZ><<<grid, Z_THREADS, ZShape<RZ>::SMEM, st>>>(in, out, d, t);
    return cudaGetLastError();
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

// x and y passes of the scales `scales[0..n)` of one cube: in -> out[i] (x/y-filtered cubes)
cudaError_t fast_xy_multi(pgsf_plan *p, const int *scales, int n, const float *in, float *const *out,
                          cudaStream_t st)
{
    const Dims &d = p->dims;
    if (d.ny > 65535 * XM_TY || d.nz > 65535 || n < 1 || n > PGSF_MAX_SCALES) return cudaErrorInvalidConfiguration;
    XYMultiParams P;
    P.d = d;
    P.n = n;
    int rmax = 0;
    for (int i = 0; i < n; ++i) {
        const ScalePlan &sp = p->scales[scales[i]];
        P.rc[i] = sp.rxy_c;
        P.out[i] = out[i];
        P.t[i] = sp.txy;
        if (sp.rxy_c > rmax) rmax = sp.rxy_c;
    }
    for (int i = n; i < PGSF_MAX_SCALES; ++i) { P.rc[i] = 0; P.out[i] = nullptr; }
    char name[32];
    if (n == 1) snprintf(name, sizeof name, "xy_s%d", scales[0]);
    else snprintf(name, sizeof name, "xy_all");
    LaunchScope ls(p, name, st);
    switch (rmax) {
    case 3: return launch_xy_multi<3>(in, P, st);
    case 6: return launch_xy_multi<6>(in, P, st);
    case 9: return launch_xy_multi<9>(in, P, st);
    case 12: return launch_xy_multi<12>(in, P, st);
    default: return cudaErrorNotSupported;
    }
}

// frequency pass of one scale: in (x/y-filtered cube) -> out
cudaError_t fast_z(pgsf_plan *p, int scale, const float *in, float *out, cudaStream_t st)
{
    const Dims &d = p->dims;
    const ScalePlan &sp = p->scales[scale];
    if (d.ny > 65535 || d.nz > 65535 * Z_ZB) return cudaErrorInvalidConfiguration;
    char name[32];
    snprintf(name, sizeof name, "z_s%d", scale);
    LaunchScope ls(p, name, st);
    switch (sp.rz_c) {
    case 6: return launch_z<6>(in, out, d, sp.tz, st);
    case 12: return launch_z<12>(in, out, d, sp.tz, st);
    case 24: return launch_z<24>(in, out, d, sp.tz, st);
    case 48: return launch_z<48>(in, out, d, sp.tz, st);
    case 72: return launch_z<72>(in, out, d, sp.tz, st);
    case 96: return launch_z<96>(in, out, d, sp.tz, st);
    default: return cudaErrorNotSupported;
    }
}

cudaError_t fast_filter3d(pgsf_plan *p, int scale, const float *in, float *out, float *tmp,
                          cudaStream_t st)
{
    float *outs[1] = {tmp};
    cudaError_t e = fast_xy_multi(p, &scale, 1, in, outs, st);
    if (e != cudaSuccess) return e;
    return fast_z(p, scale, tmp, out, st);
}

}  // namespace pgsf
