// Generic kernels: any cube shape, any radius <= PGSF_MAX_RADIUS, any box.  One thread per output
// voxel, every pass through global memory.  They are the path for shapes / radii the tiled sm_100a
// kernels (pgsf_filter.cu, pgsf_stats.cu) do not cover, and a second implementation the parity
// tests run against the same oracle.  Eq. 2 as three 1-D passes; P:152 as three
// directional sums.
#include "pgsf_internal.h"

namespace pgsf {
namespace {

constexpr int kThreads = 256;

__device__ __forceinline__ void decode(long long i, const Dims &d, int &x, int &y, int &z)
{
    x = (int)(i % d.nx);
    long long q = i / d.nx;
    y = (int)(q % d.ny);
    z = (int)(q / d.ny);
}

// out[v] = sum_o in[v + o*e_AXIS] g[o], zero outside the cube (C-5)
template <int AXIS>
__global__ void __launch_bounds__(kThreads) k_conv1d(const float *__restrict__ in,
                                                      float *__restrict__ out, Dims d, Taps t)
{
    long long i = (long long)blockIdx.x * kThreads + threadIdx.x;
    if (i >= d.cube) return;
    int x, y, z;
    decode(i, d, x, y, z);
    const int c = AXIS == 0 ? x : (AXIS == 1 ? y : z);
    const int n = AXIS == 0 ? d.nx : (AXIS == 1 ? d.ny : d.nz);
    const long long stride = AXIS == 0 ? 1 : (AXIS == 1 ? (long long)d.nx : d.plane);
    const int lo = max(-t.r, -c), hi = min(t.r, n - 1 - c);
    float acc = 0.f;
    for (int o = lo; o <= hi; ++o) acc = fmaf(in[i + o * stride], t.g[o + t.r], acc);
    out[i] = acc;
}

// Pivot of the statistics: mean of a lattice of at most kPivotAxis^3 samples of the CENTRAL half of the cube
// along every axis (next to a face the zero padding of the filter pulls f towards 0, which is not the level of
// the data), fp64, fixed summation order.  The pivot is applied only where it is free of cost: when the samples
// sit within a quarter of their mean (|mean| >= 4 sd), f - c is an exact fp32 subtraction for nearly every voxel
// (Sterbenz: c/2 <= f <= 2c); for data scattered around zero the pivot is 0 and nothing changes.
constexpr int kPivotThreads = 256;
constexpr int kPivotAxis = 100;

}  // namespace

// the lattice: first sample, stride and number of samples per axis (host and device)
__host__ __device__ inline void pivot_lattice_hd(const Dims &d, int lo[3], int st[3], int cnt[3])
{
    const int n[3] = {d.nx, d.ny, d.nz};
    for (int a = 0; a < 3; ++a) {
        lo[a] = n[a] / 4;
        const int len = n[a] / 2 > 1 ? n[a] / 2 : 1;
        st[a] = (len + kPivotAxis - 1) / kPivotAxis;
        cnt[a] = (len + st[a] - 1) / st[a];
    }
}
void pivot_lattice(const Dims &d, int lo[3], int st[3], int cnt[3]) { pivot_lattice_hd(d, lo, st, cnt); }

namespace {

// sample i of the lattice comes from fetch(i); one CTA, fixed summation order
// Two deterministic stages: kPivotBlocks CTAs each reduce a contiguous range of the samples (fixed order inside the
// CTA) to a partial (sum, sum of squares) in the plan's constant block; one CTA then adds the partials in index order.
constexpr int kPivotBlocks = 64;
constexpr int kPivotPartialOffset = 128;     // in doubles from the start of the constant block (= byte 1024)

template <class Fetch>
__device__ __forceinline__ void pivot_partial(Fetch fetch, int nsamp, double *__restrict__ partial)
{
    __shared__ double part[kPivotThreads];
    __shared__ double part2[kPivotThreads];
    const int chunk = (nsamp + kPivotBlocks - 1) / kPivotBlocks;
    const int i0 = blockIdx.x * chunk, i1 = min(i0 + chunk, nsamp);
    double acc = 0.0, acc2 = 0.0;
    for (int i = i0 + threadIdx.x; i < i1; i += kPivotThreads) {
        const double v = (double)fetch(i);
        acc += v;
        acc2 += v * v;
    }
    part[threadIdx.x] = acc;
    part2[threadIdx.x] = acc2;
    __syncthreads();
    for (int w = kPivotThreads / 2; w > 0; w >>= 1) {
        if ((int)threadIdx.x < w) { part[threadIdx.x] += part[threadIdx.x + w]; part2[threadIdx.x] += part2[threadIdx.x + w]; }
        __syncthreads();
    }
    if (threadIdx.x == 0) { partial[2 * blockIdx.x] = part[0]; partial[2 * blockIdx.x + 1] = part2[0]; }
}

__global__ void __launch_bounds__(kPivotThreads) k_pivot(const float *__restrict__ data, Dims d, float *__restrict__ cblock)
{
    int lo[3], st[3], cnt[3];
    pivot_lattice_hd(d, lo, st, cnt);
    const int nsamp = cnt[0] * cnt[1] * cnt[2];
    pivot_partial([&](int i) {
        const int ix = i % cnt[0], iy = (i / cnt[0]) % cnt[1], iz = i / (cnt[0] * cnt[1]);
        const long long o = (long long)(lo[0] + ix * st[0]) + (long long)d.nx * ((lo[1] + iy * st[1]) + (long long)d.ny * (lo[2] + iz * st[2]));
        return __ldg(data + o);
    }, nsamp, reinterpret_cast<double *>(cblock) + kPivotPartialOffset);
}

// the same reduction over samples gathered beforehand, in lattice order
__global__ void __launch_bounds__(kPivotThreads) k_pivot_list(const float *__restrict__ list, int nsamp, float *__restrict__ cblock)
{
    pivot_partial([&](int i) { return __ldg(list + i); }, nsamp, reinterpret_cast<double *>(cblock) + kPivotPartialOffset);
}

__global__ void k_pivot_final(float *__restrict__ cblock, int nsamp)
{
    const double *partial = reinterpret_cast<const double *>(cblock) + kPivotPartialOffset;
    double s = 0.0, s2 = 0.0;
    for (int b = 0; b < kPivotBlocks; ++b) { s += partial[2 * b]; s2 += partial[2 * b + 1]; }
    const double m = s / (double)nsamp;
    const double var = fmax(s2 / (double)nsamp - m * m, 0.0);
    cblock[0] = (m * m >= 16.0 * var && m != 0.0) ? (float)m : 0.f;
}

// One directional sum of P:152 over the window clipped to the cube (C-7).
// FIRST: q1 = a - c, q2 = (a - c)^2 with the pivot c; otherwise q1 = a, q2 = b.
template <int AXIS, bool FIRST>
__global__ void __launch_bounds__(kThreads) k_boxsum(const float *__restrict__ a,
                                                      const float *__restrict__ b,
                                                      float *__restrict__ oa, float *__restrict__ ob,
                                                      Dims d, int h, const float *__restrict__ pivot)
{
    const float c0 = FIRST ? __ldg(pivot) : 0.f;
    long long i = (long long)blockIdx.x * kThreads + threadIdx.x;
    if (i >= d.cube) return;
    int x, y, z;
    decode(i, d, x, y, z);
    const int c = AXIS == 0 ? x : (AXIS == 1 ? y : z);
    const int n = AXIS == 0 ? d.nx : (AXIS == 1 ? d.ny : d.nz);
    const long long stride = AXIS == 0 ? 1 : (AXIS == 1 ? (long long)d.nx : d.plane);
    const int lo = max(-h, -c), hi = min(h, n - 1 - c);
    float s1 = 0.f, s2 = 0.f;
    for (int o = lo; o <= hi; ++o) {
        float v = a[i + o * stride] - c0;
        s1 += v;
        if (FIRST) s2 = fmaf(v, v, s2);
        else s2 += b[i + o * stride];
    }
    oa[i] = s1;
    ob[i] = s2;
}

__device__ __forceinline__ int clipped_len(int c, int h, int n)
{
    return min(c + h, n - 1) - max(c - h, 0) + 1;
}

// z-score / voxel selection: division-free form of f > m + k*sd,
//   n f - S1 > k sqrt(max(n S2 - S1^2, 0))   <=>   f > S1/n + k sqrt(max(S2/n - (S1/n)^2, 0)).
__global__ void __launch_bounds__(kThreads) k_threshold(
    const float *__restrict__ f, const float *__restrict__ S1, const float *__restrict__ S2,
    uint8_t *__restrict__ mask, int or_into, float *__restrict__ mean, float *__restrict__ sd,
    unsigned long long *__restrict__ count, Dims d, int hx, int hy, int hz, int gx, int gy, int gz,
    float k, float k2, const float *__restrict__ pivot)
{
    long long i = (long long)blockIdx.x * kThreads + threadIdx.x;
    const float c0 = __ldg(pivot);
    int set = 0;
    if (i < d.cube) {
        int x, y, z;
        decode(i, d, x, y, z);
        const float n = (float)clipped_len(x, hx, d.nx) * (float)clipped_len(y, hy, d.ny) *
                        (float)clipped_len(z, hz, d.nz);
        const float v = f[i] - c0, s1 = S1[i], s2 = S2[i];     // (S1, S2 are sums of f - c0 and (f - c0)^2)
        const float a = fmaf(n, v, -s1);
        const float q = fmaxf(fmaf(n, s2, -s1 * s1), 0.f);
        int sel = (a > kFlatGuard * n * fabsf(v)) && (a * a > k2 * q);
        const bool core = x >= gx && x < d.nx - gx && y >= gy && y < d.ny - gy && z >= gz &&
                          z < d.nz - gz;
        if (!core) sel = 0;
        else if (or_into) sel |= (mask[i] != 0);
        mask[i] = (uint8_t)sel;
        set = sel;
        if (mean != nullptr) {
            const float m = s1 / n;
            mean[i] = m + c0;
            if (sd != nullptr) sd[i] = sqrtf(fmaxf(s2 / n - m * m, 0.f));
        } else if (sd != nullptr) {
            const float m = s1 / n;
            sd[i] = sqrtf(fmaxf(s2 / n - m * m, 0.f));
        }
    }
    if (count != nullptr) {
        unsigned b = __ballot_sync(0xffffffffu, set);
        __shared__ unsigned wsum[kThreads / 32];
        if ((threadIdx.x & 31) == 0) wsum[threadIdx.x >> 5] = __popc(b);
        __syncthreads();
        if (threadIdx.x == 0) {
            unsigned t = 0;
            for (int w = 0; w < kThreads / 32; ++w) t += wsum[w];
            if (t) atomicAdd(count, (unsigned long long)t);
        }
    }
    (void)k;
}

inline unsigned grid_for(long long n) { return (unsigned)((n + kThreads - 1) / kThreads); }

}  // namespace

cudaError_t compute_pivot_list(pgsf_plan *p, const float *d_list, int nsamp, cudaStream_t st)
{
    LaunchScope ls(p, "pivot", st);
    p->launches += 1;          // (two kernels)
    k_pivot_list<<<kPivotBlocks, kPivotThreads, 0, st>>>(d_list, nsamp, p->d_pivot);
    k_pivot_final<<<1, 1, 0, st>>>(p->d_pivot, nsamp);
    return cudaGetLastError();
}

cudaError_t compute_pivot(pgsf_plan *p, const float *data, cudaStream_t st)
{
    LaunchScope ls(p, "pivot", st);
    p->launches += 1;          // (two kernels)
    int lo[3], s3[3], cnt[3];
    pivot_lattice_hd(p->dims, lo, s3, cnt);
    k_pivot<<<kPivotBlocks, kPivotThreads, 0, st>>>(data, p->dims, p->d_pivot);
    k_pivot_final<<<1, 1, 0, st>>>(p->d_pivot, cnt[0] * cnt[1] * cnt[2]);
    return cudaGetLastError();
}

cudaError_t generic_filter3d(pgsf_plan *p, int scale, const float *in, float *out, float *tmp_a,
                             float *tmp_b, cudaStream_t st)
{
    const Dims &d = p->dims;
    const ScalePlan &sp = p->scales[scale];
    const unsigned g = grid_for(d.cube);
    { LaunchScope ls(p, "generic_conv_x", st); k_conv1d<0><<<g, kThreads, 0, st>>>(in, tmp_a, d, sp.taps[0]); }
    { LaunchScope ls(p, "generic_conv_y", st); k_conv1d<1><<<g, kThreads, 0, st>>>(tmp_a, tmp_b, d, sp.taps[1]); }
    { LaunchScope ls(p, "generic_conv_z", st); k_conv1d<2><<<g, kThreads, 0, st>>>(tmp_b, out, d, sp.taps[2]); }
    return cudaGetLastError();
}

cudaError_t generic_threshold(pgsf_plan *p, const float *f, uint8_t *mask, int or_into, float *mean,
                              float *sd, unsigned long long *count, float *tmp4, cudaStream_t st)
{
    const Dims &d = p->dims;
    const unsigned g = grid_for(d.cube);
    float *x1 = tmp4, *x2 = tmp4 + d.cube, *y1 = tmp4 + 2 * d.cube, *y2 = tmp4 + 3 * d.cube;
    const int *h = p->desc.box_half;
    { LaunchScope ls(p, "generic_boxsum_x", st); k_boxsum<0, true><<<g, kThreads, 0, st>>>(f, nullptr, x1, x2, d, h[0], p->d_pivot); }
    { LaunchScope ls(p, "generic_boxsum_y", st); k_boxsum<1, false><<<g, kThreads, 0, st>>>(x1, x2, y1, y2, d, h[1], p->d_pivot); }
    { LaunchScope ls(p, "generic_boxsum_z", st); k_boxsum<2, false><<<g, kThreads, 0, st>>>(y1, y2, x1, x2, d, h[2], p->d_pivot); }
    const float k = (float)p->desc.k;
    {
        LaunchScope ls(p, "generic_threshold", st);
        k_threshold<<<g, kThreads, 0, st>>>(f, x1, x2, mask, or_into, mean, sd, count, d, h[0], h[1], h[2],
                                            p->desc.halo[0], p->desc.halo[1], p->desc.halo[2], k,
                                            (float)(p->desc.k * p->desc.k), p->d_pivot);
    }
    return cudaGetLastError();
}

}  // namespace pgsf
