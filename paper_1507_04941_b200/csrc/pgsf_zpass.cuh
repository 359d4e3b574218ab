// Frequency-axis kernels of the separable form of Eq. 2 (Eq. 5), as templates on the compiled
// radius RZ.  Every radius is instantiated in its own translation unit (pgsf_z_r*.cu) so that the long,
// fully unrolled tap walks compile in parallel.
#pragma once
#include <string.h>
#include "pgsf_device.cuh"
#include "pgsf_tma.cuh"

namespace pgsf {
namespace {

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

// Eq. 5 for one thread: PZ consecutive channels x 4 columns from the staged slab (`base` = the
// thread's first staged channel, i.e. tap -RZ of its first output).  Taps are stored at
// g[o + kTapPad] with kTapPad zeros on both sides.  The walk over the PZ + 2 RZ staged channels is
// unrolled by template recursion for RZ <= 48 (a `#pragma unroll` of 104 iterations is not honoured), so
// every tap is a compile-time constant-bank offset and the body is LDS.128 + 16 FFMA2 per channel.
template <int RZ, int J, int XT>
__device__ __forceinline__ void z_step(const float *__restrict__ base, const Taps &t, float2 (&acc)[Z_PZ][2])
{
    const float4 v = *reinterpret_cast<const float4 *>(base + J * XT);
#pragma unroll
    for (int p = 0; p < Z_PZ; ++p) {
        const int o = J - p;
        if (o >= 0 && o <= 2 * RZ) {
            acc[p][0] = ffma2(make_float2(v.x, v.y), t.g[o + kTapPad], acc[p][0]);
            acc[p][1] = ffma2(make_float2(v.z, v.w), t.g[o + kTapPad], acc[p][1]);
        }
    }
}

template <int RZ, int J0, int N, int XT>
__device__ __forceinline__ void z_steps(const float *__restrict__ base, const Taps &t, float2 (&acc)[Z_PZ][2])
{
    if constexpr (N == 1) {
        z_step<RZ, J0, XT>(base, t, acc);
    } else {
        z_steps<RZ, J0, N / 2, XT>(base, t, acc);
        z_steps<RZ, J0 + N / 2, N - N / 2, XT>(base, t, acc);
    }
}

template <int RZ, int XT = Z_XT, bool FULL = (RZ <= 48)>
__device__ __forceinline__ void z_accumulate(const float *__restrict__ base, const Taps &t, float2 (&acc)[Z_PZ][2])
{
#pragma unroll
    for (int p = 0; p < Z_PZ; ++p) acc[p][0] = acc[p][1] = make_float2(0.f, 0.f);
    if constexpr (FULL) {
        z_steps<RZ, 0, Z_PZ + 2 * RZ, XT>(base, t, acc);
    } else {
        // 150 - 200 channels: walk them in chunks of 8 with the tap index in a uniform register; the zero
        // padding of the tap array makes the ramp-up / ramp-down iterations the same code as the steady state
        static_assert((Z_PZ + 2 * RZ) % 8 == 0 && kTapPad >= Z_PZ - 1, "chunking");
#pragma unroll 1
        for (int jc = 0; jc < Z_PZ + 2 * RZ; jc += 8) {
#pragma unroll
            for (int jj = 0; jj < 8; ++jj) {
                const float4 v = *reinterpret_cast<const float4 *>(base + (jc + jj) * XT);
#pragma unroll
                for (int p = 0; p < Z_PZ; ++p) {
                    const float g = t.g[jc + jj - p + kTapPad];
                    acc[p][0] = ffma2(make_float2(v.x, v.y), g, acc[p][0]);
                    acc[p][1] = ffma2(make_float2(v.z, v.w), g, acc[p][1]);
                }
            }
        }
    }
}

template <int RZ, bool TMA>
__global__ void __launch_bounds__(Z_THREADS) k_z(const float *__restrict__ in, float *__restrict__ out,
                                                 float *__restrict__ ratio, Dims d, Taps t,
                                                 const __grid_constant__ CUtensorMap tmap)
{
    using S = ZShape<RZ>;
    extern __shared__ __align__(128) float smem[];  // [PLANES][Z_XT]
    const int tid = threadIdx.x, lane = tid & 31, wz = tid >> 5;
    const int z0 = blockIdx.x * Z_ZB, x0 = blockIdx.y * Z_XT, y = blockIdx.z;
    const int gx = x0 + 4 * lane;
    const bool col_ok = gx < d.nx;
    const float *col_in = in + (long long)y * d.nx + (col_ok ? gx : 0);

    // stage channels z0-RZ .. z0+ZB+RZ-1 of this 128-column strip; outside the cube -> 0 (C-5)
    if constexpr (TMA) {   // one bulk tensor copy, zero fill by the TMA unit
        __shared__ unsigned long long bar;
        if (tid == 0) mbar_init(&bar, 1);
        __syncthreads();
        if (tid == 0) {
            mbar_arrive_expect_tx(&bar, S::SMEM);
            tma_load_4d(smem, &tmap, x0, y, z0 - RZ, 0, &bar);
        }
        mbar_wait(&bar, 0);
    } else {   // (running source pointer and shared-memory address: a handful of instructions per row)
        const float *src = col_in + (long long)(z0 - RZ + wz) * d.plane;   // dereferenced only where gz is inside the cube
        const long long step = (long long)Z_WARPS * d.plane;
        unsigned dst = (unsigned)__cvta_generic_to_shared(smem + wz * Z_XT + 4 * lane);
        int gz = z0 - RZ + wz;
#pragma unroll 4
        for (int pz = wz; pz < S::PLANES; pz += Z_WARPS, gz += Z_WARPS, src += step, dst += Z_WARPS * Z_XT * 4)
        {
            const bool ok = col_ok && (unsigned)gz < (unsigned)d.nz;
            cp_async16_s(dst, ok ? src : in, ok);   // (a valid address even when nothing is read)
        }
        cp_async_wait_all();
        __syncthreads();
    }

    // Eq. 5: f[z] = sum_o t2[z+o] gz[o]; the thread walks along z, PZ accumulators x 4 columns.
    float2 acc[Z_PZ][2];
    z_accumulate<RZ>(smem + (wz * Z_PZ) * Z_XT + 4 * lane, t, acc);
    if (!col_ok) return;
    if (ratio != nullptr) {
        // Eq. 1: this pass produced the denominator; `ratio` holds the numerator and receives the quotient (0 / 0 -> 0)
        float *col = ratio + (long long)y * d.nx + gx;
#pragma unroll
        for (int p = 0; p < Z_PZ; ++p) {
            const int gz = z0 + wz * Z_PZ + p;
            if (gz >= d.nz) break;
            float4 *q = reinterpret_cast<float4 *>(col + (long long)gz * d.plane);
            const float4 n = *q;
            const float4 dn = make_float4(acc[p][0].x, acc[p][0].y, acc[p][1].x, acc[p][1].y);
            *q = make_float4(dn.x != 0.f ? n.x / dn.x : 0.f, dn.y != 0.f ? n.y / dn.y : 0.f,
                             dn.z != 0.f ? n.z / dn.z : 0.f, dn.w != 0.f ? n.w / dn.w : 0.f);
        }
        return;
    }
    float *col_out = out + (long long)y * d.nx + gx;
#pragma unroll
    for (int p = 0; p < Z_PZ; ++p) {
        const int gz = z0 + wz * Z_PZ + p;
        if (gz < d.nz)
            *reinterpret_cast<float4 *>(col_out + (long long)gz * d.plane) =
                make_float4(acc[p][0].x, acc[p][0].y, acc[p][1].x, acc[p][1].y);
    }
}

// ------------------------------------------------------------------------------------ z pass + z window sums
//
// k_zm<RZ>: the frequency pass of k_z FUSED with the frequency-direction window sums of the local
// statistics ("three directional sums"; the z direction first).  A CTA owns a strip of 128
// columns of one row and marches along the WHOLE frequency axis in steps of 64 channels:
//   filter phase  as k_z: slab of 64 + 2 RZ channels of t2 staged in shared memory, every thread
//                 4 columns x 8 channels of Eq. 5; f goes to HBM (it is an output) and to a 64-channel
//                 slab in shared memory;
//   window phase  thread (column c, quantity q in {f, f^2}) walks the 64 new channels: the channel
//                 entering the window [z - hz, z + hz] comes from the shared-memory slab, the one
//                 leaving it is re-read from the f this CTA wrote 2 hz + 1 channels earlier -- the
//                 strip is narrow, so that plane is still in L2 (fetched with the slab by cp.async).
//                 The running sums are kept in fp64 (see window_run).  Writes Z1 = sum f, Z2 = sum f^2
//                 (window clipped to the cube, C-7).
// Against k_z + k_zbox this saves one HBM read of t2's halo, both HBM reads of f by k_zbox and one
// launch: 8 + 8 + 16 GB instead of 17 + 35 GB per scale at config 3.

// n steps of the sliding window sums of one column, both quantities (sum of f - c0 and of its square), accumulated in
// fp64 as the paper accumulates ("sums in double"): the squares and the sums of 2 hz + 1 fp32 values are exact to
// 2^-53, so nothing of a bright source stays behind once it has left the window.  The FP64 pipe (64 lanes per clock and
// SM on B200, `pgsf_ubench`) is otherwise idle in this kernel; only the fp32 -> fp64 conversions are slow (16 per clock
// and SM), two per channel and column.  pb1 / pb2 = the leaving terms of the previous output, not yet subtracted: they
// are combined with the entering terms off the dependent chain (one DADD per channel and quantity on it).
template <bool SQ, int XT>
__device__ __forceinline__ float *window_run(double &s, double &pb, const float *__restrict__ lead,
                                             const float *__restrict__ trail, float *__restrict__ zp, long long plane, int n,
                                             float c0)
{
#pragma unroll 8
    for (int j = 0; j < n; ++j) {
        const double a = (double)(lead[j * XT] - c0), b = (double)(trail[j * XT] - c0);     // (pivot c0: D-2)
        if constexpr (SQ) {
            s += fma(a, a, -pb);
            pb = b * b;
        } else {
            s += a - pb;
            pb = b;
        }
        *zp = (float)s;
        zp += plane;
    }
    return zp;
}

constexpr int ZM_XT = 64;       // columns per CTA of the marching kernel (16 float4 lanes per channel row)

template <int RZ, int XT, int ZB>
struct ZmShape {
    static constexpr int LX = XT / 4;                       // lanes per channel row
    static constexpr int GROUPS = ZB / Z_PZ;                // groups of 8 channels per step
    static constexpr int THREADS = LX * GROUPS;             // >= 2 XT; the first 2 XT threads run the window phase
    static constexpr int PLANES = ZB + 2 * RZ;            // t2 slab; its first ZB planes are reused as the f slab
    static constexpr int SMEM = (PLANES + ZB) * XT * 4;   // + slab of the channels leaving the window
};

template <int RZ, int XT, int ZB, bool TMA>
__global__ void __launch_bounds__(ZmShape<RZ, XT, ZB>::THREADS) k_zm(const float *__restrict__ in, float *out,
                                                                float *__restrict__ Z1, float *__restrict__ Z2,
                                                                Dims d, int hz, const float *__restrict__ pivot, Taps t,
                                                                int kbeg, int kend, float *__restrict__ state,
                                                                const __grid_constant__ CUtensorMap tmap, int zmap_lo)
{
    const float c0 = __ldg(pivot);   // the window sums are of f - c0 and (f - c0)^2 (D-2)
    using S = ZmShape<RZ, XT, ZB>;
    extern __shared__ __align__(128) float smem[];  // [PLANES][XT] t2 slab / f slab, [ZB][XT] leaving slab
    __shared__ unsigned long long bar;             // TMA: completion of the t2 slab
    unsigned phase = 0;
    if constexpr (TMA) {
        if (threadIdx.x == 0) mbar_init(&bar, 1);
        __syncthreads();
    }
    float *fs = smem;                              // f of this step (written after the filter phase)
    float *ts = smem + S::PLANES * XT;             // f of the channels leaving the window in this step
    const int tid = threadIdx.x, lx = tid % S::LX, wz = tid / S::LX;
    const int x0 = blockIdx.x * XT, y = blockIdx.y;
    {   // one cube of the group per blockIdx.z
        const long long cube_off = (long long)blockIdx.z * d.cube;
        in += cube_off; out += cube_off; Z1 += cube_off; Z2 += cube_off;
    }
    const int gx = x0 + 4 * lx;
    const bool col_ok = gx < d.nx;
    const float *col_in = in + (long long)y * d.nx + (col_ok ? gx : 0);
    float *col_out = out + (long long)y * d.nx + (col_ok ? gx : 0);
    // window phase: one thread per (column, quantity)
    const int c = tid % XT;
    const bool sq = tid >= XT;
    const bool c_ok = x0 + c < d.nx && tid < 2 * XT;
    const long long cb = (long long)y * d.nx + x0 + c;
    float *Zq = sq ? Z2 : Z1;
    double s = 0.0;
    const int nz = d.nz;
    // march steps kbeg .. kend - 1 of the (nz + hz + ZB - 1) / ZB steps of the whole axis (entering channels
    // 0 .. nz + hz - 1; the tail drains the window).  A march cut into sections (pgsf_find_multiscale_host streams the
    // cube through the device) carries the running window sums from one launch to the next in `state`
    // (fp64, [quantity][row][column]), so that the sections perform exactly the arithmetic of one whole march.
    double *st_s = nullptr;
    if (state != nullptr && c_ok) {
        st_s = reinterpret_cast<double *>(state) + (sq ? d.plane : 0) + cb;
        if (kbeg > 0) s = st_s[0];
    }
    const long long gstep = (long long)S::GROUPS * d.plane;   // staging: a warp group takes every GROUPS-th channel

    for (int k = kbeg; k < kend; ++k) {
        const int z0 = k * ZB;
        // channels leaving the window in this step: z0 - 2 hz + j, j = 0..63.  Those written in EARLIER steps
        // (by this CTA: still in L2) are fetched now, together with the t2 slab; those of this step's own
        // f block (2 hz < 64) are read from the f slab instead.
        // (running source pointers and shared-memory addresses: a handful of instructions per staged row)
        {
            const float *src = col_out + (long long)(z0 - 2 * hz + wz) * d.plane;
            unsigned dst = (unsigned)__cvta_generic_to_shared(ts + wz * XT + 4 * lx);
            int zt = z0 - 2 * hz + wz;
#pragma unroll 4
            for (int pz = wz; pz < ZB; pz += S::GROUPS, zt += S::GROUPS, src += gstep, dst += S::GROUPS * XT * 4)
            {
                // (zt < nz: the drain steps have z0 >= nz, and planes nz .. z0-1 of `out` do not exist)
                const bool ok = col_ok && zt >= 0 && zt < z0 && zt < nz;
                cp_async16_s(dst, ok ? src : in, ok);   // (a valid address even when nothing is read)
            }
        }
        if (TMA && z0 < nz) {
            // channels z0-RZ .. z0+ZB+RZ-1 of t2 as one (or two) bulk tensor copies; outside the cube -> 0 (C-5).  The
            // slab was read and rewritten (f slab) through the generic proxy in the previous step: fence, then copy.
            if (tid == 0) {
                constexpr int NBOX = S::PLANES > 256 ? 2 : 1, BZ = S::PLANES / NBOX;
                fence_proxy_async_smem();
                mbar_arrive_expect_tx(&bar, S::PLANES * XT * 4);
#pragma unroll
                for (int bx = 0; bx < NBOX; ++bx)
                    tma_load_4d(smem + bx * BZ * XT, &tmap, x0, y, z0 - RZ + bx * BZ - zmap_lo, blockIdx.z, &bar);
            }
        }
        if (!TMA && z0 < nz) {
            // stage channels z0-RZ .. z0+ZB+RZ-1 of t2; outside the cube -> 0 (C-5)
            const float *src = col_in + (long long)(z0 - RZ + wz) * d.plane;
            unsigned dst = (unsigned)__cvta_generic_to_shared(smem + wz * XT + 4 * lx);
            int gz = z0 - RZ + wz;
#pragma unroll 4
            for (int pz = wz; pz < S::PLANES; pz += S::GROUPS, gz += S::GROUPS, src += gstep, dst += S::GROUPS * XT * 4)
            {
                const bool ok = col_ok && (unsigned)gz < (unsigned)nz;
                cp_async16_s(dst, ok ? src : in, ok);
            }
        }
        cp_async_wait_all();
        if (TMA && z0 < nz) {
            mbar_wait(&bar, phase);
            phase ^= 1;
        }
        __syncthreads();
        if (z0 < nz) {
            float2 acc[Z_PZ][2];
            z_accumulate<RZ, XT, true>(smem + (wz * Z_PZ) * XT + 4 * lx, t, acc);
            __syncthreads();   // every warp is done with the t2 slab: its head becomes the f slab
#pragma unroll
            for (int p = 0; p < Z_PZ; ++p) {
                const int gz = z0 + wz * Z_PZ + p;
                const float4 v = make_float4(acc[p][0].x, acc[p][0].y, acc[p][1].x, acc[p][1].y);
                *reinterpret_cast<float4 *>(fs + (wz * Z_PZ + p) * XT + 4 * lx) = v;
                if (col_ok && gz < nz) *reinterpret_cast<float4 *>(col_out + (long long)gz * d.plane) = v;
            }
            __syncthreads();   // f slab complete
        }
        if (c_ok) {
            if (z0 >= 2 * hz && z0 + ZB <= nz) {
                // interior step: all 64 entering and all 64 leaving channels (and all 64 outputs) are inside the cube
                const int jsplit = min(2 * hz, ZB);   // leaving channel: ts[j] for j < jsplit, else fs[j - 2 hz]
                float *zp = Zq + (long long)(z0 - hz) * d.plane + cb;
                double pb = 0.0;
                if (sq) {
                    zp = window_run<true, XT>(s, pb, fs + c, ts + c, zp, d.plane, jsplit, c0);
                    window_run<true, XT>(s, pb, fs + jsplit * XT + c, fs + c, zp, d.plane, ZB - jsplit, c0);
                } else {
                    zp = window_run<false, XT>(s, pb, fs + c, ts + c, zp, d.plane, jsplit, c0);
                    window_run<false, XT>(s, pb, fs + jsplit * XT + c, fs + c, zp, d.plane, ZB - jsplit, c0);
                }
                s -= pb;
            } else {
                for (int j = 0; j < ZB; ++j) {
                    const int zl = z0 + j;          // channel entering the window of output zo
                    const int zo = zl - hz;
                    if (zl < nz) {
                        const double v = (double)(fs[j * XT + c] - c0);
                        s = sq ? fma(v, v, s) : s + v;
                    }
                    if (zo >= 0 && zo < nz) {
                        Zq[(long long)zo * d.plane + cb] = (float)s;
                        const int jt = j - 2 * hz;  // the channel leaving after this output, relative to z0
                        if (zo - hz >= 0) {         // (a channel in front of the cube never entered the sum)
                            const double v = (double)((jt >= 0 ? fs[jt * XT + c] : ts[j * XT + c]) - c0);
                            s = sq ? fma(-v, v, s) : s - v;
                        }
                    }
                }
            }
        }
        __syncthreads();   // slabs are overwritten by the next step
    }
    if (st_s != nullptr) st_s[0] = s;
}

template <int RZ>
cudaError_t launch_z(const float *in, float *out, float *ratio, const Dims &d, const Taps &t, cudaStream_t st, bool tma)
{
    dim3 grid((d.nz + Z_ZB - 1) / Z_ZB, (d.nx + Z_XT - 1) / Z_XT, d.ny);
    alignas(64) CUtensorMap map;
    if (tma && make_slab_map(&map, in, d.nx, d.ny, d.nz, 1, Z_XT, ZShape<RZ>::PLANES)) {
        cudaError_t e = ensure_dynamic_smem(k_z<RZ, true>, ZShape<RZ>::SMEM);
        if (e != cudaSuccess) return e;
        k_z<RZ, true><<<grid, Z_THREADS, ZShape<RZ>::SMEM, st>>>(in, out, ratio, d, t, map);
        return cudaGetLastError();
    }
    memset(&map, 0, sizeof map);
    cudaError_t e = ensure_dynamic_smem(k_z<RZ, false>, ZShape<RZ>::SMEM);
    if (e != cudaSuccess) return e;
    k_z<RZ, false><<<grid, Z_THREADS, ZShape<RZ>::SMEM, st>>>(in, out, ratio, d, t, map);
    return cudaGetLastError();
}

// channels per march step: 64 (4 warps per CTA) up to RZ = 48; 128 (8 warps) above, where the slab of
// 64 + 2 RZ channels would leave room for two 4-warp CTAs only
template <int RZ>
constexpr int zm_step_channels() { return zm_step_rule(RZ); }

template <int RZ>
cudaError_t launch_zm(const float *in, float *out, float *Z1, float *Z2, const Dims &d, int hz, const float *pivot,
                      const Taps &t, int ncubes, cudaStream_t st, const ZmSection *sec, bool tma)
{
    constexpr int ZB = zm_step_channels<RZ>();
    using S = ZmShape<RZ, ZM_XT, ZB>;
    cudaError_t e;
    const int nsteps = (d.nz + hz + ZB - 1) / ZB;
    int kbeg = 0, kend = nsteps;
    float *state = nullptr;
    if (sec != nullptr) {     // entering channels [c0, c1), both multiples of ZB (c1 beyond the axis = to the end)
        kbeg = sec->c0 / ZB;
        kend = sec->c1 / ZB < nsteps ? sec->c1 / ZB : nsteps;
        state = sec->state;
        if (kbeg >= kend) return cudaSuccess;
    }
    dim3 grid((d.nx + ZM_XT - 1) / ZM_XT, d.ny, ncubes);
    alignas(64) CUtensorMap map;
    constexpr int BZ = S::PLANES > 256 ? S::PLANES / 2 : S::PLANES;
    int zmap_lo = 0;
    bool ok = tma;
    if (ok && sec != nullptr && sec->t2_buf != nullptr) {
        // a section: the buffer holds channels t2_base .. t2_hi - 1; the map covers those that exist in the cube
        const int lo = sec->t2_base > 0 ? sec->t2_base : 0, hi = sec->t2_hi < d.nz ? sec->t2_hi : d.nz;
        zmap_lo = lo;
        ok = make_slab_map(&map, sec->t2_buf + (long long)(lo - sec->t2_base) * d.plane, d.nx, d.ny, hi - lo, 1, ZM_XT, BZ);
    } else if (ok) {
        ok = make_slab_map(&map, in, d.nx, d.ny, d.nz, ncubes, ZM_XT, BZ);
    }
    if (ok) {
        if ((e = ensure_dynamic_smem(k_zm<RZ, ZM_XT, ZB, true>, S::SMEM)) != cudaSuccess) return e;
        k_zm<RZ, ZM_XT, ZB, true><<<grid, S::THREADS, S::SMEM, st>>>(in, out, Z1, Z2, d, hz, pivot, t, kbeg, kend, state,
                                                                     map, zmap_lo);
        return cudaGetLastError();
    }
    memset(&map, 0, sizeof map);
    if ((e = ensure_dynamic_smem(k_zm<RZ, ZM_XT, ZB, false>, S::SMEM)) != cudaSuccess) return e;
    k_zm<RZ, ZM_XT, ZB, false><<<grid, S::THREADS, S::SMEM, st>>>(in, out, Z1, Z2, d, hz, pivot, t, kbeg, kend, state, map, 0);
    return cudaGetLastError();
}

}  // namespace
}  // namespace pgsf

// one pair of plain entry points per radius
#define PGSF_INSTANTIATE_Z(RZ)                                                                              \
    namespace pgsf {                                                                                        \
    cudaError_t launch_z_r##RZ(const float *in, float *out, float *ratio, const Dims &d, const Taps &t,     \
                               cudaStream_t st, bool tma)                                                   \
    {                                                                                                       \
        return launch_z<RZ>(in, out, ratio, d, t, st, tma);                                                 \
    }                                                                                                       \
    cudaError_t launch_zm_r##RZ(const float *in, float *out, float *Z1, float *Z2, const Dims &d, int hz,   \
                                const float *pivot, const Taps &t, int ncubes, cudaStream_t st,             \
                                const ZmSection *sec, bool tma)                                             \
    {                                                                                                       \
        return launch_zm<RZ>(in, out, Z1, Z2, d, hz, pivot, t, ncubes, st, sec, tma);                       \
    }                                                                                                       \
    }
