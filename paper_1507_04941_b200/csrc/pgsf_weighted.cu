// Eq. 1, the weighted convolution (reading C-16 of DESIGN.md):
//
//      c_w[v] = sum_o d[v+o] f[o] w[v+o]  /  sum_o w[v+o]          (mode 0, as printed)
//      c_w[v] = sum_o d[v+o] f[o] w[v+o]  /  sum_o f[o] w[v+o]     (mode 1)
//
// For the outer-product Gaussian both sums are separable: the numerator is Eq. 2 of the product cube d*w,
// i.e. the same x/y and z kernels as pgsf_filter3d; the printed denominator is the sum of w over the box
// of the support (three directional sums), the mode-1 denominator Eq. 2 of w.  This file holds the three
// element-wise / box kernels around those filter calls; pgsf_api.cu sequences them.
#include "pgsf_internal.h"

namespace pgsf {
namespace {

constexpr int kThreads = 256;

// p = d * w
__global__ void __launch_bounds__(kThreads) k_wmul(const float *__restrict__ d, const float *__restrict__ w,
                                                   float *__restrict__ p, long long n4, long long n)
{
    const long long i = (long long)blockIdx.x * kThreads + threadIdx.x;
    if (i < n4) {
        const float4 a = __ldg(reinterpret_cast<const float4 *>(d) + i);
        const float4 b = __ldg(reinterpret_cast<const float4 *>(w) + i);
        reinterpret_cast<float4 *>(p)[i] = make_float4(a.x * b.x, a.y * b.y, a.z * b.z, a.w * b.w);
    }
    const long long t = 4 * n4 + i;     // tail of a cube whose size is not a multiple of 4
    if (i < n - 4 * n4) p[t] = d[t] * w[t];
}

// c = den != 0 ? c / den : 0
__device__ __forceinline__ float wdiv(float c, float q) { return q != 0.f ? c / q : 0.f; }

__global__ void __launch_bounds__(kThreads) k_wdiv(float *__restrict__ c, const float *__restrict__ den, long long n4,
                                                   long long n)
{
    const long long i = (long long)blockIdx.x * kThreads + threadIdx.x;
    if (i < n4) {
        const float4 a = reinterpret_cast<const float4 *>(c)[i];
        const float4 q = __ldg(reinterpret_cast<const float4 *>(den) + i);
        reinterpret_cast<float4 *>(c)[i] = make_float4(wdiv(a.x, q.x), wdiv(a.y, q.y), wdiv(a.z, q.z), wdiv(a.w, q.w));
    }
    const long long t = 4 * n4 + i;
    if (i < n - 4 * n4) c[t] = wdiv(c[t], den[t]);
}

// out[v] = sum_{|o| <= r} in[v + o e_AXIS] over the part of the support inside the cube (C-5)
template <int AXIS>
__global__ void __launch_bounds__(kThreads) k_wbox(const float *__restrict__ in, float *__restrict__ out, Dims d, int r)
{
    const long long i = (long long)blockIdx.x * kThreads + threadIdx.x;
    if (i >= d.cube) return;
    const int x = (int)(i % d.nx);
    const long long q = i / d.nx;
    const int y = (int)(q % d.ny), z = (int)(q / d.ny);
    const int c = AXIS == 0 ? x : (AXIS == 1 ? y : z);
    const int n = AXIS == 0 ? d.nx : (AXIS == 1 ? d.ny : d.nz);
    const long long stride = AXIS == 0 ? 1 : (AXIS == 1 ? (long long)d.nx : d.plane);
    const int lo = max(-r, -c), hi = min(r, n - 1 - c);
    float s = 0.f;
    for (int o = lo; o <= hi; ++o) s += in[i + o * stride];
    out[i] = s;
}

unsigned blocks_for(long long n) { return (unsigned)((n + kThreads - 1) / kThreads); }

}  // namespace

cudaError_t weighted_mul(pgsf_plan *p, const float *d, const float *w, float *prod, cudaStream_t st)
{
    const long long n = p->dims.cube;
    const bool vec = ((reinterpret_cast<uintptr_t>(d) | reinterpret_cast<uintptr_t>(w) | reinterpret_cast<uintptr_t>(prod)) & 15u) == 0;
    const long long n4 = vec ? n / 4 : 0;
    const long long work = n4 > n - 4 * n4 ? n4 : n - 4 * n4;
    LaunchScope ls(p, "w_mul", st);
    k_wmul<<<blocks_for(work > 0 ? work : 1), kThreads, 0, st>>>(d, w, prod, n4, n);
    return cudaGetLastError();
}

// sum of w over the box [-r, r]^3 of the support: w -> a (result), b = scratch cube
cudaError_t weighted_boxsum(pgsf_plan *p, int scale, const float *w, float *a, float *b, cudaStream_t st)
{
    const Dims &d = p->dims;
    const int *r = p->scales[scale].r;
    LaunchScope ls(p, "w_box", st);
    k_wbox<0><<<blocks_for(d.cube), kThreads, 0, st>>>(w, a, d, r[0]);
    k_wbox<1><<<blocks_for(d.cube), kThreads, 0, st>>>(a, b, d, r[1]);
    k_wbox<2><<<blocks_for(d.cube), kThreads, 0, st>>>(b, a, d, r[2]);
    p->launches += 2;
    return cudaGetLastError();
}

cudaError_t weighted_div(pgsf_plan *p, float *c, const float *den, cudaStream_t st)
{
    const long long n = p->dims.cube;
    const bool vec = ((reinterpret_cast<uintptr_t>(c) | reinterpret_cast<uintptr_t>(den)) & 15u) == 0;
    const long long n4 = vec ? n / 4 : 0;
    const long long work = n4 > n - 4 * n4 ? n4 : n - 4 * n4;
    LaunchScope ls(p, "w_div", st);
    k_wdiv<<<blocks_for(work > 0 ? work : 1), kThreads, 0, st>>>(c, den, n4, n);
    return cudaGetLastError();
}

}  // namespace pgsf
