// k_ztc: the OPTIONAL banded-Toeplitz tensor-core form of the frequency pass (Eq. 5; the filters are
// largest along frequency), fused with the z-direction window sums exactly as k_zm is.  BASELINE.json allows tensor
// cores only here, "for large spectral sigma", and only if the variant beats the CUDA-core path inside the stated
// tolerance; it runs when the plan carries PGSF_FLAG_TENSOR_ZPASS and the compiled z radius is >= 24.
//
// One CTA owns 32 columns of one row and marches along z in steps of 128 channels.  Per step the pass is the GEMM
//     D[m, n] = sum_k A[m, k] B[k, n]      m = output channel (128), n = column (32), k = slab channel (K = 128 + 2 RZ)
// with B the slab of x/y-filtered data as TMA lands it (MN-major, 128-byte swizzle with 32-byte atoms: two 512-byte
// atoms of 4 channels x 32 columns per MMA K step) and A the band matrix A[m, k] = g[k - m].  Row m is stored REVERSED (m' = 127 - m), which
// makes A a Hankel matrix, A'[m', k] = h[m' + k]: every 8 x 4 core matrix depends on 8 a + 4 b only (a = row group,
// b = K chunk), so the whole operand is ONE strip of K / 4 + 30 core matrices addressed through SBO = 256 B,
// LBO = 128 B -- 11 KB instead of 112 KB.  tcgen05.mma.kind::tf32 with fp32 accumulators in TMEM.
//
// Precision: a single TF32 product (10-bit mantissa) misses the filter tolerance by two orders of magnitude, so every
// operand is split x = hi + lo with hi = rna_tf32(x), lo = rna_tf32(x - hi), and three MMAs per K step accumulate
// hi hi + lo hi + hi lo (the dropped lo lo term and the residues are ~2^-22 relative).  The data slab is split in
// place by the CUDA cores (hi) into a second buffer (lo); the taps are split on the host.
#include <stdio.h>
#include <string.h>

#include "pgsf_internal.h"
#include "pgsf_device.cuh"
#include "pgsf_tma.cuh"

namespace pgsf {
namespace {

constexpr int TC_XT = 32;        // columns per CTA (one 128-byte swizzle atom)
constexpr int TC_ZB = 128;       // output channels per step (UMMA M)
constexpr int TC_NT = 128;       // threads: 4 warps = the 4 x 32 TMEM lanes of the epilogue

__device__ __forceinline__ float rna_tf32(float x)
{
    unsigned r;
    asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(x));
    return __uint_as_float(r);
}

// UMMA shared-memory descriptors (SM100 format: start >> 4 | LBO >> 4 << 16 | SBO >> 4 << 32 | version 1 << 46 | layout << 61)
__device__ __forceinline__ unsigned long long umma_desc(unsigned smem_addr, unsigned lbo_bytes, unsigned sbo_bytes, unsigned layout)
{
    return (unsigned long long)((smem_addr >> 4) & 0x3fffu) | ((unsigned long long)((lbo_bytes >> 4) & 0x3fffu) << 16) |
           ((unsigned long long)((sbo_bytes >> 4) & 0x3fffu) << 32) | (1ull << 46) | ((unsigned long long)layout << 61);
}
// instruction descriptor: fp32 accumulate, tf32 x tf32, A K-major, B MN-major, N = 32, M = 128
constexpr unsigned kIdescTf32 = (1u << 4) | (2u << 7) | (2u << 10) | (0u << 15) | (1u << 16) | ((TC_XT >> 3) << 17) | ((TC_ZB >> 4) << 24);

__device__ __forceinline__ void umma_tf32(unsigned d_tmem, unsigned long long adesc, unsigned long long bdesc, unsigned accumulate)
{
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}"
                 ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(kIdescTf32), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void umma_commit(unsigned long long *bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

// this warp's 32 lanes x 32 consecutive TMEM columns -> 32 registers per thread (thread t = lane base + t)
__device__ __forceinline__ void tmem_ld32(unsigned taddr, float (&v)[32])
{
    unsigned r[32];
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 "
                 "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
                 "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
                   "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]),
                   "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]),
                   "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
                 : "r"(taddr) : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
    for (int i = 0; i < 32; ++i) v[i] = __uint_as_float(r[i]);
}

// f slab in shared memory: [channel j][32 columns], the 16-byte chunk of a row XOR-ed with j & 7 (the epilogue writes
// one row per thread, the window phase reads one row per warp: both conflict-free)
__device__ __forceinline__ int fs_idx(int j, int c) { return j * TC_XT + ((((c >> 2) ^ (j & 7)) << 2) | (c & 3)); }

struct ZtcParams {
    Dims d;
    int hz, rz, K;                 // compiled radius, slab channels = 128 + 2 rz
    int kbeg, kend;                // march steps (see k_zm)
    int zmap_lo;                   // channel of plane 0 of the tensor map
    int nbox;                      // TMA boxes per slab (1, or 2 when K > 256)
};

__global__ void __launch_bounds__(TC_NT) k_ztc(float *out, float *__restrict__ Z1, float *__restrict__ Z2,
                                               const float *__restrict__ pivot, const float *__restrict__ strips,
                                               float *__restrict__ state, const __grid_constant__ CUtensorMap tmap,
                                               const ZtcParams p)
{
    extern __shared__ __align__(1024) unsigned char ztc_smem[];
    __shared__ unsigned long long bar_tma, bar_mma;
    __shared__ unsigned tmem_slot;
    const int K = p.K, T = K / 4 + 30;
    float *Bh = reinterpret_cast<float *>(ztc_smem);      // [K][32] data slab, hi part (128-byte swizzle)
    float *Bl = Bh + K * TC_XT;                           // lo part, same layout
    float *fs = Bl + K * TC_XT;                           // [128][32] f of this step (fs_idx)
    float *ts = fs + TC_ZB * TC_XT;                       // [128][32] f of the channels leaving the window
    float *Ah = ts + TC_ZB * TC_XT;                       // band-matrix strips: T core matrices of 128 bytes, hi then lo
    float *Al = Ah + T * 32;
    const int tid = threadIdx.x, warp = tid >> 5;
    const Dims &d = p.d;
    const int x0 = blockIdx.x * TC_XT, y = blockIdx.y, nz = d.nz, hz = p.hz;
    const long long cube_off = (long long)blockIdx.z * d.cube;
    out += cube_off; Z1 += cube_off; Z2 += cube_off;
    const float c0 = __ldg(pivot);

    if (tid == 0) { mbar_init(&bar_tma, 1); mbar_init(&bar_mma, 1); tma_prefetch_desc(&tmap); }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 32;" ::"r"(smem_u32(&tmem_slot)) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    for (int i = tid; i < 2 * T * 32; i += TC_NT) Ah[i] = __ldg(strips + i);
    fence_proxy_async_smem();          // the strips are read by the tensor core (async proxy)
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const unsigned tmem = tmem_slot;
    const unsigned ah_addr = smem_u32(Ah), al_addr = smem_u32(Al), bh_addr = smem_u32(Bh), bl_addr = smem_u32(Bl);

    // window phase: one thread per (column, quantity), as in k_zm
    const int c = tid & 31;
    const bool sq = warp == 1;
    const bool c_ok = warp < 2 && x0 + c < d.nx;
    const long long cb = (long long)y * d.nx + x0 + c;
    float *Zq = sq ? Z2 : Z1;
    float s = 0.f, e = 0.f;
    float *st_s = nullptr;
    if (state != nullptr && c_ok) {
        st_s = state + ((long long)(sq ? 2 : 0) * d.plane + cb);
        if (p.kbeg > 0) { s = st_s[0]; e = st_s[d.plane]; }
    }
    unsigned ph_tma = 0, ph_mma = 0;
    const float *row_out = out + (long long)y * d.nx + x0;     // column x0 of row y, channel 0

    // ---- the pieces of one step (z0 = 128 k) -------------------------------------------------------------------
    auto issue_tma = [&](int z0) {        // slab channels z0 - rz .. z0 + 127 + rz: bulk tensor copies, zeros outside (C-5)
        if (warp == 0) {
            if (tid == 0) {
                fence_proxy_async_smem();
                mbar_arrive_expect_tx(&bar_tma, K * TC_XT * 4);
                const int bz = K / p.nbox;
                for (int b = 0; b < p.nbox; ++b)
                    tma_load_4d(Bh + b * bz * TC_XT, &tmap, x0, y, z0 - p.rz + b * bz - p.zmap_lo, blockIdx.z, &bar_tma);
            }
            __syncwarp();
        }
    };
    auto split_and_mma = [&]() {
        mbar_wait(&bar_tma, ph_tma);
        ph_tma ^= 1;
        // split the slab: hi in place, lo beside it (element-wise, so the swizzle is irrelevant here)
        float4 *bh4 = reinterpret_cast<float4 *>(Bh), *bl4 = reinterpret_cast<float4 *>(Bl);
        for (int i = tid; i < K * 8; i += TC_NT) {
            const float4 v = bh4[i];
            float4 h, l;
            h.x = rna_tf32(v.x); h.y = rna_tf32(v.y); h.z = rna_tf32(v.z); h.w = rna_tf32(v.w);
            l.x = rna_tf32(v.x - h.x); l.y = rna_tf32(v.y - h.y); l.z = rna_tf32(v.z - h.z); l.w = rna_tf32(v.w - h.w);
            bh4[i] = h;
            bl4[i] = l;
        }
        fence_proxy_async_smem();
        tc_fence_before();
        __syncthreads();
        if (warp == 0) {       // one lane issues; its warp waits at the __syncwarp, not spinning on a barrier
            if (tid == 0) {
                tc_fence_after();
                // A: K-major, no swizzle, Hankel strip (LBO 128 B between the two K chunks, SBO 256 B between row groups),
                //    256 bytes further per K step.  B: MN-major TF32 = 128-byte swizzle with 32-byte atoms (the only MN-major
                //    layout for 32-bit operands): two atoms of 4 channels x 32 columns per K step, SBO 512 B between them.
                unsigned long long ah = umma_desc(ah_addr, 128, 256, 0), al = umma_desc(al_addr, 128, 256, 0);
                unsigned long long bh = umma_desc(bh_addr, 1024, 512, 1), bl = umma_desc(bl_addr, 1024, 512, 1);
                for (int ks = 0; ks < K / 8; ++ks) {
                    umma_tf32(tmem, ah, bh, ks > 0);
                    umma_tf32(tmem, al, bh, 1);
                    umma_tf32(tmem, ah, bl, 1);
                    ah += 16; al += 16; bh += 64; bl += 64;        // (start-address field, units of 16 bytes)
                }
                umma_commit(&bar_mma);
            }
            __syncwarp();
        }
    };
    auto stage_leaving = [&](int z0) {    // channels leaving the window in the step that earlier steps wrote (cp.async, L2)
        for (int i = tid; i < TC_ZB * 8; i += TC_NT) {
            const int j = i >> 3, ch = i & 7, zt = z0 - 2 * hz + j;
            const bool ok = zt >= 0 && zt < z0 && zt < nz && x0 + 4 * ch < d.nx;
            cp_async16(ts + j * TC_XT + 4 * ch, ok ? row_out + (long long)zt * d.plane + 4 * ch : out, ok);
        }
    };
    auto epilogue = [&](int z0) {         // TMEM lane L = row m' = 127 - (channel - z0); this thread takes lane tid
        mbar_wait(&bar_mma, ph_mma);
        ph_mma ^= 1;
        tc_fence_after();
        float v[32];
        tmem_ld32(tmem + ((unsigned)(warp * 32) << 16), v);
        const int j = TC_ZB - 1 - tid, gz = z0 + j;
        float *g = out + (long long)gz * d.plane + (long long)y * d.nx + x0;
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            const float4 w = make_float4(v[4 * q], v[4 * q + 1], v[4 * q + 2], v[4 * q + 3]);
            *reinterpret_cast<float4 *>(fs + j * TC_XT + ((q ^ (j & 7)) << 2)) = w;
            if (gz < nz && x0 + 4 * q < d.nx) *reinterpret_cast<float4 *>(g + 4 * q) = w;
        }
        tc_fence_before();
    };
    // window sums of one step.  The running value is s + e (two-sum compensated: the rounding error of every addition is
    // recovered exactly and gathered in e).  In the interior the channel entering and the channel that left one output
    // earlier are combined OFF the dependent chain, so the chain is one addition per channel.
    auto acc_add = [&](float v) {
        const float t = s + v, bp = t - s;
        e += (s - (t - bp)) + (v - bp);
        s = t;
    };
    auto window = [&](int z0) {
        if (!c_ok) return;
        const int cx = ((c >> 2) << 2), cl = c & 3;
        if (z0 >= 2 * hz && z0 + TC_ZB <= nz) {
            const int jsplit = min(2 * hz, TC_ZB);     // leaving channel: ts[j] for j < jsplit, else fs[j - 2 hz]
            float *zp = Zq + (long long)(z0 - hz) * d.plane + cb;
            float pb = 0.f;                            // the leaving term of the previous output, not yet subtracted
#pragma unroll 4
            for (int j = 0; j < TC_ZB; ++j) {
                const float a = fs[j * TC_XT + ((cx ^ ((j & 7) << 2)) | cl)] - c0;
                const int jt = j - 2 * hz;
                const float b = (j < jsplit ? ts[j * TC_XT + c] : fs[jt * TC_XT + ((cx ^ ((jt & 7) << 2)) | cl)]) - c0;
                const float va = sq ? a * a : a, vb = sq ? b * b : b;
                acc_add(va - pb);
                pb = vb;
                *zp = s + e;
                zp += d.plane;
            }
            acc_add(-pb);
        } else {
            for (int j = 0; j < TC_ZB; ++j) {
                const int zl = z0 + j, zo = zl - hz;       // channel entering the window of output zo
                if (zl < nz) {
                    const float a = fs[fs_idx(j, c)] - c0;
                    acc_add(sq ? a * a : a);
                }
                if (zo >= 0 && zo < nz) {
                    Zq[(long long)zo * d.plane + cb] = s + e;
                    const int jt = j - 2 * hz;             // the channel leaving after this output, relative to z0
                    if (zo - hz >= 0) {
                        const float b = (jt >= 0 ? fs[fs_idx(jt, c)] : ts[j * TC_XT + c]) - c0;
                        acc_add(sq ? -(b * b) : -b);
                    }
                }
            }
        }
    };

    // ---- the march: the window sums of step k - 1 run under the MMAs of step k; the slab of step k + 1 is requested
    //      as soon as the MMAs of step k have retired
    bool pending = false;
    int pending_z0 = 0;
    if (p.kbeg < p.kend && p.kbeg * TC_ZB < nz) issue_tma(p.kbeg * TC_ZB);
    for (int k = p.kbeg; k < p.kend; ++k) {
        const int z0 = k * TC_ZB;
        const bool have = z0 < nz;
        if (have) split_and_mma();
        if (pending) window(pending_z0);
        __syncthreads();                  // the window walk is done with the f and leaving slabs
        stage_leaving(z0);
        if (have) {
            epilogue(z0);
            if (k + 1 < p.kend && (k + 1) * TC_ZB < nz) issue_tma((k + 1) * TC_ZB);
        }
        cp_async_wait_all();
        __syncthreads();                  // f slab and leaving slab of step k complete; the accumulator has been read
        pending = true;
        pending_z0 = z0;
    }
    if (pending) window(pending_z0);
    if (st_s != nullptr) { st_s[0] = s; st_s[d.plane] = e; }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 32;" ::"r"(tmem) : "memory");
}

// ------------------------------------------------------------------------------------ k_ztc2
// The same GEMM with 64 columns per CTA and two warp groups, for the radii whose operands fit one CTA per SM
// (RZ <= 72).  Group B (warps 4-7) waits for the slab of step k, splits it and issues its MMAs; group A (warps 0-3:
// one thread per (column, quantity)) meanwhile walks the window sums of step k-1; all eight warps then drain the
// accumulator (warp w: TMEM lanes 32 (w & 3).., columns 32 (w >> 2)..) and stage the leaving slab.
constexpr int T2_XT = 64, T2_NT = 256;
constexpr unsigned kIdescTf32N64 = (1u << 4) | (2u << 7) | (2u << 10) | (1u << 16) | ((T2_XT >> 3) << 17) | ((TC_ZB >> 4) << 24);

__device__ __forceinline__ void umma_tf32_n64(unsigned d_tmem, unsigned long long adesc, unsigned long long bdesc, unsigned accumulate)
{
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}"
                 ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(kIdescTf32N64), "r"(accumulate) : "memory");
}

__global__ void __launch_bounds__(T2_NT, 1) k_ztc2(float *out, float *__restrict__ Z1, float *__restrict__ Z2,
                                                   const float *__restrict__ pivot, const float *__restrict__ strips,
                                                   float *__restrict__ state, const __grid_constant__ CUtensorMap tmap,
                                                   const ZtcParams p)
{
    extern __shared__ __align__(1024) unsigned char ztc_smem[];
    __shared__ unsigned long long bar_tma, bar_mma;
    __shared__ unsigned tmem_slot;
    const int K = p.K, T = K / 4 + 30;
    float *Bh = reinterpret_cast<float *>(ztc_smem);      // [2 column atoms][K][32], hi part (32-byte-atom swizzle)
    float *Bl = Bh + 2 * K * 32;                          // lo part
    float *fs = Bl + 2 * K * 32;                          // [128][64] f of a step, 16-byte chunks XOR-ed with (row & 7)
    float *ts = fs + TC_ZB * T2_XT;                       // [128][64] f of the channels leaving the window
    float *Ah = ts + TC_ZB * T2_XT;
    float *Al = Ah + T * 32;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const bool grpB = warp >= 4;
    const Dims &d = p.d;
    const int x0 = blockIdx.x * T2_XT, y = blockIdx.y, nz = d.nz, hz = p.hz;
    const long long cube_off = (long long)blockIdx.z * d.cube;
    out += cube_off; Z1 += cube_off; Z2 += cube_off;
    const float c0 = __ldg(pivot);

    if (tid == 0) { mbar_init(&bar_tma, 1); mbar_init(&bar_mma, 1); tma_prefetch_desc(&tmap); }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 64;" ::"r"(smem_u32(&tmem_slot)) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    for (int i = tid; i < 2 * T * 32; i += T2_NT) Ah[i] = __ldg(strips + i);
    fence_proxy_async_smem();
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const unsigned tmem = tmem_slot;
    const unsigned ah_addr = smem_u32(Ah), al_addr = smem_u32(Al), bh_addr = smem_u32(Bh), bl_addr = smem_u32(Bl);

    // group A: one thread per (column, quantity)
    const int c = tid & 63;
    const bool sq = tid >= 64;
    const bool c_ok = !grpB && x0 + c < d.nx;
    const long long cb = (long long)y * d.nx + x0 + c;
    float *Zq = sq ? Z2 : Z1;
    float s = 0.f, e = 0.f;
    float *st_s = nullptr;
    if (state != nullptr && c_ok) {
        st_s = state + ((long long)(sq ? 2 : 0) * d.plane + cb);
        if (p.kbeg > 0) { s = st_s[0]; e = st_s[d.plane]; }
    }
    unsigned ph_tma = 0, ph_mma = 0;
    const float *row_out = out + (long long)y * d.nx + x0;

    auto issue_tma = [&](int z0) {        // (called by warp 4)
        if (lane == 0) {
            fence_proxy_async_smem();
            mbar_arrive_expect_tx(&bar_tma, K * T2_XT * 4);
            const int bz = K / p.nbox;
            for (int a = 0; a < 2; ++a)
                for (int b = 0; b < p.nbox; ++b)
                    tma_load_4d(Bh + a * K * 32 + b * bz * 32, &tmap, x0 + 32 * a, y, z0 - p.rz + b * bz - p.zmap_lo,
                                blockIdx.z, &bar_tma);
        }
        __syncwarp();
    };
    auto acc_add = [&](float v) {
        const float t = s + v, bp = t - s;
        e += (s - (t - bp)) + (v - bp);
        s = t;
    };
    auto fidx = [&](int j, int cc) { return j * T2_XT + (((((cc >> 2) & 7) ^ (j & 7)) | ((cc >> 2) & 8)) << 2 | (cc & 3)); };
    auto window = [&](int z0) {
        if (!c_ok) return;
        if (z0 >= 2 * hz && z0 + TC_ZB <= nz && (hz & 3) == 0) {
            const int jsplit = min(2 * hz, TC_ZB);     // (a multiple of 8) leaving channel: ts[j] below it, fs[j - 2 hz] from it on
            float *zp = Zq + (long long)(z0 - hz) * d.plane + cb;
            float pb = 0.f;
            int off[8];                                // column offset inside a row for (row & 7) = 0 .. 7
#pragma unroll
            for (int r = 0; r < 8; ++r) off[r] = ((((c >> 2) & 7) ^ r) | ((c >> 2) & 8)) << 2 | (c & 3);
            for (int jb = 0; jb < jsplit; jb += 8) {
#pragma unroll
                for (int r = 0; r < 8; ++r) {
                    const int j = jb + r;
                    const float a = fs[j * T2_XT + off[r]] - c0, b = ts[j * T2_XT + c] - c0;
                    acc_add((sq ? a * a : a) - pb);
                    pb = sq ? b * b : b;
                    *zp = s + e;
                    zp += d.plane;
                }
            }
            for (int jb = jsplit; jb < TC_ZB; jb += 8) {
#pragma unroll
                for (int r = 0; r < 8; ++r) {
                    const int j = jb + r;              // (j - 2 hz) & 7 == r as well
                    const float a = fs[j * T2_XT + off[r]] - c0, b = fs[(j - 2 * hz) * T2_XT + off[r]] - c0;
                    acc_add((sq ? a * a : a) - pb);
                    pb = sq ? b * b : b;
                    *zp = s + e;
                    zp += d.plane;
                }
            }
            acc_add(-pb);
        } else {
            for (int j = 0; j < TC_ZB; ++j) {
                const int zl = z0 + j, zo = zl - hz;
                if (zl < nz) {
                    const float a = fs[fidx(j, c)] - c0;
                    acc_add(sq ? a * a : a);
                }
                if (zo >= 0 && zo < nz) {
                    Zq[(long long)zo * d.plane + cb] = s + e;
                    const int jt = j - 2 * hz;
                    if (zo - hz >= 0) {
                        const float b = (jt >= 0 ? fs[fidx(jt, c)] : ts[j * T2_XT + c]) - c0;
                        acc_add(sq ? -(b * b) : -b);
                    }
                }
            }
        }
    };

    bool pending = false;
    int pending_z0 = 0;
    if (warp == 4 && p.kbeg < p.kend && p.kbeg * TC_ZB < nz) issue_tma(p.kbeg * TC_ZB);
    for (int k = p.kbeg; k < p.kend; ++k) {
        const int z0 = k * TC_ZB;
        const bool have = z0 < nz;
        if (grpB) {
            if (have) {
                mbar_wait(&bar_tma, ph_tma);
                ph_tma ^= 1;
                float4 *bh4 = reinterpret_cast<float4 *>(Bh), *bl4 = reinterpret_cast<float4 *>(Bl);
                for (int i = tid - 128; i < K * 16; i += 128) {
                    const float4 v = bh4[i];
                    float4 h, l;
                    h.x = rna_tf32(v.x); h.y = rna_tf32(v.y); h.z = rna_tf32(v.z); h.w = rna_tf32(v.w);
                    l.x = rna_tf32(v.x - h.x); l.y = rna_tf32(v.y - h.y); l.z = rna_tf32(v.z - h.z); l.w = rna_tf32(v.w - h.w);
                    bh4[i] = h;
                    bl4[i] = l;
                }
                fence_proxy_async_smem();
                tc_fence_before();
                asm volatile("bar.sync 1, 128;" ::: "memory");
                if (warp == 4) {
                    if (lane == 0) {
                        tc_fence_after();
                        // A: Hankel strip (K-major, LBO 128 B, SBO 256 B).  B: two column atoms K x 128 bytes apart (LBO), 4-channel
                        // atoms 512 B apart (SBO), 1 KB per K step.
                        unsigned long long ah = umma_desc(ah_addr, 128, 256, 0), al = umma_desc(al_addr, 128, 256, 0);
                        unsigned long long bh = umma_desc(bh_addr, K * 128, 512, 1), bl = umma_desc(bl_addr, K * 128, 512, 1);
                        for (int ks = 0; ks < K / 8; ++ks) {
                            umma_tf32_n64(tmem, ah, bh, ks > 0);
                            umma_tf32_n64(tmem, al, bh, 1);
                            umma_tf32_n64(tmem, ah, bl, 1);
                            ah += 16; al += 16; bh += 64; bl += 64;
                        }
                        umma_commit(&bar_mma);
                    }
                    __syncwarp();
                }
            }
        } else if (pending) {
            window(pending_z0);
        }
        __syncthreads();                  // the window walk is done with the f and leaving slabs; the MMAs are in flight
        for (int i = tid; i < TC_ZB * 16; i += T2_NT) {
            const int j = i >> 4, ch = i & 15, zt = z0 - 2 * hz + j;
            const bool ok = zt >= 0 && zt < z0 && zt < nz && x0 + 4 * ch < d.nx;
            cp_async16(ts + j * T2_XT + 4 * ch, ok ? row_out + (long long)zt * d.plane + 4 * ch : out, ok);
        }
        if (have) {
            mbar_wait(&bar_mma, ph_mma);
            ph_mma ^= 1;
            tc_fence_after();
            if (warp == 4 && k + 1 < p.kend && (k + 1) * TC_ZB < nz) issue_tma((k + 1) * TC_ZB);
            float v[32];
            const int quarter = warp & 3, half = warp >> 2;
            tmem_ld32(tmem + ((unsigned)(quarter * 32) << 16) + (unsigned)(half * 32), v);
            const int j = TC_ZB - 1 - (quarter * 32 + lane), gz = z0 + j;
            float *g = out + (long long)gz * d.plane + (long long)y * d.nx + x0 + 32 * half;
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                const float4 w = make_float4(v[4 * q], v[4 * q + 1], v[4 * q + 2], v[4 * q + 3]);
                *reinterpret_cast<float4 *>(fs + j * T2_XT + ((half * 8 + (q ^ (j & 7))) << 2)) = w;
                if (gz < nz && x0 + 32 * half + 4 * q < d.nx) *reinterpret_cast<float4 *>(g + 4 * q) = w;
            }
            tc_fence_before();
        }
        cp_async_wait_all();
        __syncthreads();                  // f slab and leaving slab of step k complete; the accumulator has been read
        pending = true;
        pending_z0 = z0;
    }
    if (!grpB && pending) window(pending_z0);
    if (st_s != nullptr) { st_s[0] = s; st_s[d.plane] = e; }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 64;" ::"r"(tmem) : "memory");
}

}  // namespace

// host: round to the nearest TF32 (ties away from zero, as cvt.rna.tf32.f32)
static float host_rna_tf32(float x)
{
    unsigned u;
    memcpy(&u, &x, 4);
    u = (u + 0x1000u) & 0xffffe000u;
    memcpy(&x, &u, 4);
    return x;
}

bool ztc_radius(int rz_c) { return rz_c >= 24 && rz_c % 4 == 0; }

int ztc_step_channels(const pgsf_plan *p, int scale)
{
    return (p->tensor_z && p->d_tc_strips[scale] != nullptr && ztc_radius(p->scales[scale].rz_c)) ? TC_ZB : 0;
}

// The band-matrix strips of every scale the variant serves: S[t][r][j] = h[4 t + r + j], h[u] = g[u - 127],
// g[0 .. 2 RZ] the taps centred in the compiled window; hi part, then lo part.
cudaError_t ztc_prepare(pgsf_plan *p)
{
    for (int s = 0; s < p->desc.n_scales; ++s) {
        const ScalePlan &sp = p->scales[s];
        p->d_tc_strips[s] = nullptr;
        if (!ztc_radius(sp.rz_c)) continue;
        const int K = TC_ZB + 2 * sp.rz_c, T = K / 4 + 30;
        std::vector<float> hst((size_t)2 * T * 32);
        for (int t = 0; t < T; ++t)
            for (int r = 0; r < 8; ++r)
                for (int j = 0; j < 4; ++j) {
                    const int i = 4 * t + r + j - (TC_ZB - 1);            // tap index k - m
                    const float g = (i >= 0 && i <= 2 * sp.rz_c) ? sp.tz.g[i + kTapPad] : 0.f;
                    const float hi = host_rna_tf32(g);
                    hst[(size_t)(t * 8 + r) * 4 + j] = hi;
                    hst[(size_t)T * 32 + (size_t)(t * 8 + r) * 4 + j] = host_rna_tf32(g - hi);
                }
        cudaError_t e = cudaMalloc(&p->d_tc_strips[s], hst.size() * sizeof(float));
        if (e == cudaSuccess) e = cudaMemcpy(p->d_tc_strips[s], hst.data(), hst.size() * sizeof(float), cudaMemcpyHostToDevice);
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

void ztc_release(pgsf_plan *p)
{
    for (int s = 0; s < PGSF_MAX_SCALES; ++s) { cudaFree(p->d_tc_strips[s]); p->d_tc_strips[s] = nullptr; }
}

// frequency pass + z-direction window sums of one scale on the tensor cores; cudaErrorNotSupported = the caller runs k_zm
cudaError_t fast_ztc(pgsf_plan *p, int scale, const float *in, float *out, float *Z1, float *Z2, int ncubes,
                     cudaStream_t st, const ZmSection *sec)
{
    const ScalePlan &sp = p->scales[scale];
    if (!p->tensor_z || p->d_tc_strips[scale] == nullptr || !ztc_radius(sp.rz_c)) return cudaErrorNotSupported;
    const Dims &d = p->dims;
    ZtcParams zp;
    zp.d = d;
    zp.hz = p->desc.box_half[2];
    zp.rz = sp.rz_c;
    zp.K = TC_ZB + 2 * sp.rz_c;
    zp.nbox = zp.K > 256 ? 2 : 1;
    zp.zmap_lo = 0;
    const int nsteps = (d.nz + zp.hz + TC_ZB - 1) / TC_ZB;
    zp.kbeg = 0;
    zp.kend = nsteps;
    float *state = nullptr;
    alignas(64) CUtensorMap map;
    bool ok;
    if (sec != nullptr) {
        // (pgsf_host.cu sizes its sections in whole steps of every scale's kernel: a section that is not must fail, not
        // fall back to k_zm -- the sections of one march would then mix the carried states of two kernels)
        if (sec->c0 % TC_ZB != 0 || (sec->c1 % TC_ZB != 0 && sec->c1 < (1 << 29))) return cudaErrorInvalidValue;
        zp.kbeg = sec->c0 / TC_ZB;
        zp.kend = sec->c1 / TC_ZB < nsteps ? sec->c1 / TC_ZB : nsteps;
        state = sec->state;
        if (zp.kbeg > 0 && p->tc_march[scale] == 2) return cudaErrorNotSupported;   // the march began on k_zm: stay there
        if (zp.kbeg >= zp.kend) return cudaSuccess;
        const int lo = sec->t2_base > 0 ? sec->t2_base : 0, hi = sec->t2_hi < d.nz ? sec->t2_hi : d.nz;
        zp.zmap_lo = lo;
        ok = sec->t2_buf != nullptr &&
             make_slab_map(&map, sec->t2_buf + (long long)(lo - sec->t2_base) * d.plane, d.nx, d.ny, hi - lo, 1, TC_XT,
                           zp.K / zp.nbox, true);
    } else {
        ok = make_slab_map(&map, in, d.nx, d.ny, d.nz, ncubes, TC_XT, zp.K / zp.nbox, true);
    }
    if (!ok) {     // no tensor map (nx % 4 != 0, no driver entry point): k_zm -- but never in the middle of a march
        if (sec != nullptr && zp.kbeg > 0) return cudaErrorInvalidValue;
        p->tc_march[scale] = 2;
        return cudaErrorNotSupported;
    }
    p->tc_march[scale] = 1;
    const int T = zp.K / 4 + 30;
    const int smem2 = (2 * zp.K * T2_XT + 2 * TC_ZB * T2_XT + 2 * T * 32) * (int)sizeof(float);
    if (smem2 <= 227 * 1024 && !(p->tune & 32)) {          // 64 columns per CTA, two warp groups (PGSF_OPT_TUNE bit 5: k_ztc)
        cudaError_t e2 = ensure_dynamic_smem(k_ztc2, smem2);
        if (e2 != cudaSuccess) return e2;
        char name2[32];
        snprintf(name2, sizeof name2, "ztc_s%d", scale);
        LaunchScope ls2(p, name2, st);
        dim3 grid2((d.nx + T2_XT - 1) / T2_XT, d.ny, ncubes);
        k_ztc2<<<grid2, T2_NT, smem2, st>>>(out, Z1, Z2, p->d_pivot, p->d_tc_strips[scale], state, map, zp);
        return cudaGetLastError();
    }
    const int smem = (2 * zp.K * TC_XT + 2 * TC_ZB * TC_XT + 2 * T * 32) * (int)sizeof(float);
    cudaError_t e = ensure_dynamic_smem(k_ztc, smem);
    if (e != cudaSuccess) return e;
    char name[32];
    snprintf(name, sizeof name, "ztc_s%d", scale);
    LaunchScope ls(p, name, st);
    dim3 grid((d.nx + TC_XT - 1) / TC_XT, d.ny, ncubes);
    k_ztc<<<grid, TC_NT, smem, st>>>(out, Z1, Z2, p->d_pivot, p->d_tc_strips[scale], state, map, zp);
    return cudaGetLastError();
}

}  // namespace pgsf
