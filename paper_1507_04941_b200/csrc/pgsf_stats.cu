// Local statistics + voxel selection for sm_100a ("three directional sums" of the filtered
// data and of its square, then the z-score; P:33 / P:282 threshold and voxel selection; readings
// C-6..C-10).  Two kernels per filtered cube, no other pass over the data:
//
//   k_zbox    frequency direction first.  Every thread owns four adjacent (x, y) columns and marches
//             along z with the window sums  Z1 = sum_{|o|<=hz} f(z+o),  Z2 = sum f(z+o)^2  in registers:
//             the plane entering the window is added, the plane leaving it subtracted (both read from
//             HBM; nothing is staged).  The running sums are Kahan-compensated: a bright source is
//             > 10^3 x the filtered noise in f^2, and an uncompensated fp32 running sum would keep the
//             rounding error made while the source was inside the window long after it has left.
//             Writes Z1, Z2 (two workspace cubes).
//   k_xybox   per z plane: 128 x 32 tile + (hx, hy) halo of Z1 and Z2 staged in shared memory (cp.async,
//             zero fill outside the cube = the clipped window of C-7), x- then y-direction window sums,
//             then m = S1/n, var = S2/n - m^2, selection f > m + k sd (division-free form of
//             pgsf_generic.cu), mask write / OR, count.  The window sums use the van Herk / Gil-Werman
//             decomposition (suffix sum of one block + prefix sum of the next): ~3 additions per output
//             like a sliding sum, but every output is a plain sum of the elements of ITS window, so no
//             cancellation and no error carried over from bright neighbours.
//
// Preconditions (else the generic kernels run): nx % 4 == 0, hx in {0,4,8,12,16}, hy <= 16.
#include <stdio.h>

#include "pgsf_internal.h"

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

// Kahan-compensated s += v (e holds the running low-order error)
__device__ __forceinline__ void kahan_add(float &s, float &e, float v)
{
    const float y = v - e;
    const float t = s + y;
    e = (t - s) - y;
    s = t;
}

__global__ void __launch_bounds__(ZB_NT) k_zbox(const float4 *__restrict__ f, float4 *__restrict__ Z1,
                                                float4 *__restrict__ Z2, ZboxParams p)
{
    const long long c = (long long)blockIdx.x * ZB_NT + threadIdx.x;
    if (c >= p.cols4) return;
    const int chunk = blockIdx.y;
    const int za = chunk * p.zchunk, zb = min(za + p.zchunk, p.d.nz);
    const long long plane4 = p.d.plane / 4;
    const int hz = p.hz, nz = p.d.nz;
    float s1[4] = {0.f, 0.f, 0.f, 0.f}, e1[4] = {0.f, 0.f, 0.f, 0.f};
    float s2[4] = {0.f, 0.f, 0.f, 0.f}, e2[4] = {0.f, 0.f, 0.f, 0.f};
    // planes za-hz .. za+hz-1 of the first window (clipped to the cube, C-7)
    for (int z = max(za - hz, 0); z < min(za + hz, nz); ++z) {
        const float4 v = __ldg(f + (long long)z * plane4 + c);
        const float a[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            kahan_add(s1[u], e1[u], a[u]);
            kahan_add(s2[u], e2[u], a[u] * a[u]);
        }
    }
#pragma unroll 4
    for (int zc = za; zc < zb; ++zc) {
        const int zl = zc + hz, zt = zc - hz;
        float4 l = make_float4(0.f, 0.f, 0.f, 0.f), t = make_float4(0.f, 0.f, 0.f, 0.f);
        if (zl < nz) l = __ldg(f + (long long)zl * plane4 + c);
        if (zt >= 0) t = __ldg(f + (long long)zt * plane4 + c);   // leaves after this output
        const float a[4] = {l.x, l.y, l.z, l.w}, b[4] = {t.x, t.y, t.z, t.w};
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            kahan_add(s1[u], e1[u], a[u]);
            kahan_add(s2[u], e2[u], a[u] * a[u]);
        }
        const long long o = (long long)zc * plane4 + c;
        Z1[o] = make_float4(s1[0] - e1[0], s1[1] - e1[1], s1[2] - e1[2], s1[3] - e1[3]);
        Z2[o] = make_float4(s2[0] - e2[0], s2[1] - e2[1], s2[2] - e2[2], s2[3] - e2[3]);
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            kahan_add(s1[u], e1[u], -b[u]);
            kahan_add(s2[u], e2[u], -(b[u] * b[u]));
        }
    }
}

// ------------------------------------------------------------------------------------ k_xybox

constexpr int ST_TX = 128;
constexpr int ST_TY = 32;
constexpr int ST_NT = 256;
constexpr int ST_L = 32;              // x-direction outputs per thread
constexpr int ST_ROWS = ST_TY / 2;    // y-direction outputs per thread (two threads per column)
constexpr int ST_MAX_HY = 16;

struct XyboxParams {
    Dims d;
    int hy, hz;
    int gx, gy, gz;      // halo excluded from mask and count (C-11)
    int or_into;
    float k2;            // k^2
};

__device__ __forceinline__ void st_cp_async16(void *smem, const void *gmem, bool valid)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    const int bytes = valid ? 16 : 0;  // src-size 0 -> 16 bytes of zeros
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(s), "l"(gmem), "r"(bytes));
}
__device__ __forceinline__ void st_cp_async4(void *smem, const void *gmem, bool valid)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    const int bytes = valid ? 4 : 0;
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4, %2;" ::"r"(s), "l"(gmem), "r"(bytes));
}
__device__ __forceinline__ void st_cp_async_wait()
{
    asm volatile("cp.async.commit_group;\n\tcp.async.wait_group 0;" ::: "memory");
}

__device__ __forceinline__ int clipped_len(int c, int h, int n)
{
    return min(c + h, n - 1) - max(c - h, 0) + 1;
}

// x-direction window sums of one staged row segment, in place:
//   row[i] <- sum_{e = i .. i + 2 HX} row[e],  i = 0 .. ST_L - 1   (row has ST_L + 2 HX valid elements)
// van Herk / Gil-Werman with blocks of WN = 2 HX + 1 elements: h = suffix sum inside a block,
// g = prefix sum inside a block, out[i] = h[i] + g[i + WN - 1] (just h[i] when i starts a block).
// All indices are compile-time; the four segments of a row sit in one warp, hence __syncwarp
// between the last read and the first write.
template <int HX>
__device__ __forceinline__ void xbox_inplace(float *row, bool active)
{
    constexpr int WN = 2 * HX + 1;
    constexpr int N = ST_L + 2 * HX;
    float o[ST_L];
    if (active) {
        float g[N], h[N];
#pragma unroll
        for (int q = 0; q < N / 4; ++q) {
            const float4 v = *reinterpret_cast<const float4 *>(row + 4 * q);
            g[4 * q] = v.x; g[4 * q + 1] = v.y; g[4 * q + 2] = v.z; g[4 * q + 3] = v.w;
        }
#pragma unroll
        for (int e = 0; e < N; ++e) h[e] = g[e];
#pragma unroll
        for (int e = 1; e < N; ++e)
            if (e % WN != 0) g[e] = g[e - 1] + g[e];
#pragma unroll
        for (int e = N - 2; e >= 0; --e)
            if (e % WN != WN - 1) h[e] = h[e + 1] + h[e];
#pragma unroll
        for (int i = 0; i < ST_L; ++i) o[i] = (i % WN == 0) ? h[i] : h[i] + g[i + WN - 1];
    }
    __syncwarp();
    if (active) {
#pragma unroll
        for (int q = 0; q < ST_L / 4; ++q)
            *reinterpret_cast<float4 *>(row + 4 * q) = make_float4(o[4 * q], o[4 * q + 1], o[4 * q + 2], o[4 * q + 3]);
    }
}

// y-direction window sums down one staged column: out[r] = sum_{q = r .. r + 2 hy} col[q * pitch],
// r = 0 .. ST_ROWS - 1.  For 2 hy + 1 >= ST_ROWS the same two-block decomposition as in x (block 0 =
// rows 0 .. 2 hy, block 1 = the rows below); shorter windows are summed directly.
__device__ __forceinline__ void ybox(const float *col, int pitch, int hy, float (&out)[ST_ROWS])
{
    const int wy = 2 * hy;
    if (wy + 1 >= ST_ROWS) {
        float tail = 0.f;                      // rows ST_ROWS .. 2 hy, common to every suffix
        for (int q = wy; q >= ST_ROWS; --q) tail += col[q * pitch];
        float h = tail;
#pragma unroll
        for (int r = ST_ROWS - 1; r >= 0; --r) {
            h += col[r * pitch];
            out[r] = h;                        // suffix of block 0 starting at row r
        }
        float g = 0.f;
#pragma unroll
        for (int r = 1; r < ST_ROWS; ++r) {
            g += col[(r + wy) * pitch];        // prefix of block 1 up to row r + 2 hy
            out[r] += g;
        }
    } else {
#pragma unroll
        for (int r = 0; r < ST_ROWS; ++r) {
            float s = 0.f;
            for (int q = 0; q <= wy; ++q) s += col[(r + q) * pitch];
            out[r] = s;
        }
    }
}

template <int HX>
__global__ void __launch_bounds__(ST_NT, 2) k_xybox(const float *__restrict__ f, const float *__restrict__ Z1,
                                                   const float *__restrict__ Z2, uint8_t *__restrict__ mask,
                                                   float *__restrict__ mean, float *__restrict__ sd,
                                                   unsigned long long *__restrict__ count, XyboxParams p)
{
    constexpr int W = ST_TX + 2 * HX;   // staged columns
    constexpr int W4 = W / 4;
    constexpr int WP = W + 4;           // row pitch: WP/4 odd -> conflict-free 16-byte accesses down a column
    constexpr int RP = ST_NT / W4;      // staged rows per pass of the CTA
    extern __shared__ __align__(16) float smem[];
    const int H = ST_TY + 2 * p.hy;     // staged rows
    float *s_a = smem;                  // Z1 tile + halo, then its x-direction sums
    float *s_b = s_a + H * WP;          // Z2 likewise
    float *s_f = s_b + H * WP;          // centre values f of the tile [ST_TY][ST_TX]
    uint8_t *s_m = reinterpret_cast<uint8_t *>(s_f + ST_TY * ST_TX);   // mask bytes of the tile [ST_TY][ST_TX]
    const Dims &d = p.d;
    const int tid = threadIdx.x;
    const int x0 = blockIdx.x * ST_TX, y0 = blockIdx.y * ST_TY, z = blockIdx.z;
    const long long plane_off = (long long)z * d.plane;

    // stage Z1 / Z2: thread <-> one 16-byte column chunk, rows r0, r0 + RP, ...
    if (tid < RP * W4) {
        const int c4 = tid % W4, r0 = tid / W4;
        const int xx = x0 - HX + 4 * c4;
        const bool xok = xx >= 0 && xx < d.nx;
        int yy = y0 - p.hy + r0;
        long long off = plane_off + (long long)yy * d.nx + xx;
        float *da = s_a + r0 * WP + 4 * c4, *db = s_b + r0 * WP + 4 * c4;
        for (int r = r0; r < H; r += RP) {
            const bool ok = xok && yy >= 0 && yy < d.ny;
            const long long o = ok ? off : 0;
            st_cp_async16(da, Z1 + o, ok);
            st_cp_async16(db, Z2 + o, ok);
            yy += RP;
            off += (long long)RP * d.nx;
            da += RP * WP;
            db += RP * WP;
        }
    }
    // stage the centre values (and, in OR mode, the previous mask) of the tile
    {
        const int c4 = tid & 31, r0 = tid >> 5;
        const int xx = x0 + 4 * c4;
        const bool xok = xx < d.nx;
#pragma unroll
        for (int k = 0; k < ST_TY / 8; ++k) {
            const int r = r0 + 8 * k, yy = y0 + r;
            const bool ok = xok && yy < d.ny;
            const long long o = ok ? plane_off + (long long)yy * d.nx + xx : 0;
            st_cp_async16(s_f + r * ST_TX + 4 * c4, f + o, ok);
            if (p.or_into) st_cp_async4(s_m + r * ST_TX + 4 * c4, mask + o, ok);
        }
    }
    st_cp_async_wait();
    __syncthreads();

    // x direction: one row segment of 32 outputs per thread (8 consecutive rows per quarter warp)
    {
        const int warp = tid >> 5, lane = tid & 31;
        const int xr = warp * 8 + (lane & 7), xs = lane >> 3;
        const bool act = xr < H;
        const int o = act ? xr * WP + xs * ST_L : 0;
        xbox_inplace<HX>(s_a + o, act);
        xbox_inplace<HX>(s_b + o, act);
    }
    __syncthreads();

    // y direction + selection: column cx of the tile, rows ry0 .. ry0 + ST_ROWS - 1
    {
        const int cx = tid & (ST_TX - 1);
        const int ry0 = (tid >> 7) * ST_ROWS;
        const int gx = x0 + cx;
        float S1[ST_ROWS], S2[ST_ROWS];
        ybox(s_a + ry0 * WP + cx, WP, p.hy, S1);
        ybox(s_b + ry0 * WP + cx, WP, p.hy, S2);
        const float nxz = (float)clipped_len(min(gx, d.nx - 1), HX, d.nx) * (float)clipped_len(z, p.hz, d.nz);
        const bool y_inside = y0 - p.hy >= 0 && y0 + ST_TY - 1 + p.hy < d.ny;   // no row of the tile is clipped
        const float n_in = nxz * (float)(2 * p.hy + 1);
        const bool halo = (p.gx | p.gy | p.gz) != 0;
        const bool core_xz = gx >= p.gx && gx < d.nx - p.gx && z >= p.gz && z < d.nz - p.gz;
        const float *vf = s_f + ry0 * ST_TX + cx;
        uint8_t *vm = s_m + ry0 * ST_TX + cx;
#pragma unroll
        for (int i = 0; i < ST_ROWS; ++i) {
            const int gy = y0 + ry0 + i;
            const float n = y_inside ? n_in : nxz * (float)clipped_len(min(gy, d.ny - 1), p.hy, d.ny);
            const float v = vf[i * ST_TX], s1 = S1[i], s2 = S2[i];
            const float a = fmaf(n, v, -s1);
            const float q = fmaxf(fmaf(n, s2, -s1 * s1), 0.f);
            int sel = (a > kFlatGuard * n * fabsf(v)) && (a * a > p.k2 * q);
            if (halo && !(core_xz && gy >= p.gy && gy < d.ny - p.gy)) sel = 0;
            else if (p.or_into) sel |= (vm[i * ST_TX] != 0);
            vm[i * ST_TX] = (uint8_t)sel;
            if ((mean != nullptr || sd != nullptr) && gx < d.nx && gy < d.ny) {
                const long long idx = plane_off + (long long)gy * d.nx + gx;
                const float m = s1 / n;
                if (mean != nullptr) mean[idx] = m;
                if (sd != nullptr) sd[idx] = sqrtf(fmaxf(s2 / n - m * m, 0.f));
            }
        }
    }
    __syncthreads();

    // mask tile -> global, 4 bytes per thread and row pass (one 128-byte row per warp); count = popcount
    unsigned my_count = 0;
    {
        const int c4 = tid & 31, r0 = tid >> 5;
        const int xx = x0 + 4 * c4;
        if (xx < d.nx) {
#pragma unroll
            for (int k = 0; k < ST_TY / 8; ++k) {
                const int r = r0 + 8 * k, yy = y0 + r;
                if (yy < d.ny) {
                    const unsigned w = *reinterpret_cast<const unsigned *>(s_m + r * ST_TX + 4 * c4);
                    *reinterpret_cast<unsigned *>(mask + plane_off + (long long)yy * d.nx + xx) = w;
                    my_count += __popc(w);
                }
            }
        }
    }

    if (count != nullptr) {
        __shared__ unsigned wsum[ST_NT / 32];
        unsigned c = my_count;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
        if ((tid & 31) == 0) wsum[tid >> 5] = c;
        __syncthreads();
        if (tid == 0) {
            unsigned t = 0;
            for (int w = 0; w < ST_NT / 32; ++w) t += wsum[w];
            if (t) atomicAdd(count, (unsigned long long)t);
        }
    }
}

template <int HX>
cudaError_t launch_xybox(const float *f, const float *Z1, const float *Z2, uint8_t *mask, float *mean,
                         float *sd, unsigned long long *count, const XyboxParams &p, cudaStream_t st)
{
    const int H = ST_TY + 2 * p.hy;
    const int smem = 2 * H * (ST_TX + 2 * HX + 4) * (int)sizeof(float) + ST_TY * ST_TX * 5;
    static int configured = 0;
    if (configured < smem) {
        cudaError_t e = cudaFuncSetAttribute(k_xybox<HX>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return e;
        configured = smem;
    }
    dim3 grid((p.d.nx + ST_TX - 1) / ST_TX, (p.d.ny + ST_TY - 1) / ST_TY, p.d.nz);
    k_xybox<HX><<<grid, ST_NT, smem, st>>>(f, Z1, Z2, mask, mean, sd, count, p);
    return cudaGetLastError();
}

}  // namespace

bool fast_stats_supported(const pgsf_plan *p)
{
    const int hx = p->desc.box_half[0], hy = p->desc.box_half[1];
    if (p->desc.nx % 4 != 0) return false;
    if (hx % 4 != 0 || hx > 16 || hy > ST_MAX_HY) return false;
    return (p->desc.ny + ST_TY - 1) / ST_TY <= 65535 && p->desc.nz <= 65535;
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
                                       reinterpret_cast<float4 *>(Z2), zp);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    XyboxParams xp;
    xp.d = d;
    xp.hy = p->desc.box_half[1];
    xp.hz = p->desc.box_half[2];
    xp.gx = p->desc.halo[0];
    xp.gy = p->desc.halo[1];
    xp.gz = p->desc.halo[2];
    xp.or_into = or_into;
    xp.k2 = (float)(p->desc.k * p->desc.k);
    LaunchScope ls(p, "stats_xybox", st);
    switch (p->desc.box_half[0]) {
    case 0: return launch_xybox<0>(f, Z1, Z2, mask, mean, sd, count, xp, st);
    case 4: return launch_xybox<4>(f, Z1, Z2, mask, mean, sd, count, xp, st);
    case 8: return launch_xybox<8>(f, Z1, Z2, mask, mean, sd, count, xp, st);
    case 12: return launch_xybox<12>(f, Z1, Z2, mask, mean, sd, count, xp, st);
    case 16: return launch_xybox<16>(f, Z1, Z2, mask, mean, sd, count, xp, st);
    default: return cudaErrorNotSupported;
    }
}

}  // namespace pgsf
