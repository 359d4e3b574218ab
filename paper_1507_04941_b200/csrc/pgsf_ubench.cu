// Micro-benchmark behind the "alu" roofline of DESIGN.md section 6 (not part of libpgsf.so):
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o pgsf_ubench paper_1507_04941_b200/csrc/pgsf_ubench.cu && ./pgsf_ubench
// Measures, per SM and clock, what the FMA pipe retires for FFMA (scalar), FFMA2 (fma.rn.f32x2 with a uniform
// multiplier, the inner instruction of the filter kernels), FADD, FADD2 (add.rn.f32x2, the statistics kernels), DADD / DFMA and
// the fp32 <-> fp64 conversions (fp64 window sums were considered for the statistics), and what shared memory delivers for LDS.128, with enough independent chains and resident warps to hide latencies.
#include <cstdio>
#include <cuda_runtime.h>

constexpr int kIters = 4096, kChains = 8;

__device__ __forceinline__ float2 ffma2(float2 a, float2 g, float2 c)
{
    unsigned long long ra = *reinterpret_cast<unsigned long long *>(&a), rb = *reinterpret_cast<unsigned long long *>(&g),
                       rc = *reinterpret_cast<unsigned long long *>(&c), rd;
    asm volatile("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(rd) : "l"(ra), "l"(rb), "l"(rc));
    return *reinterpret_cast<float2 *>(&rd);
}
__device__ __forceinline__ float2 fadd2(float2 a, float2 b)
{
    unsigned long long ra = *reinterpret_cast<unsigned long long *>(&a), rb = *reinterpret_cast<unsigned long long *>(&b), rd;
    asm volatile("add.rn.f32x2 %0, %1, %2;" : "=l"(rd) : "l"(ra), "l"(rb));
    return *reinterpret_cast<float2 *>(&rd);
}

template <int OP>
__global__ void __launch_bounds__(1024) k_ubench(float *out, float g, long long *cycles)
{
    __shared__ __align__(16) float sm[256 * 4];
    float2 acc[kChains];
    for (int i = 0; i < kChains; ++i) acc[i] = make_float2(threadIdx.x * 1e-3f + i, 1.f);
    for (int i = threadIdx.x; i < 256 * 4; i += 1024) sm[i] = (float)i;
    __syncthreads();
    const float2 gg = make_float2(g, g);
    double dacc[kChains];
    for (int i = 0; i < kChains; ++i) dacc[i] = threadIdx.x * 1e-3 + i;
    const double gd = (double)g;
    const long long t0 = clock64();
    for (int it = 0; it < kIters; ++it) {
#pragma unroll
        for (int i = 0; i < kChains; ++i) {
            if (OP == 0) { acc[i].x = fmaf(acc[i].x, g, 1.f); }                       // FFMA
            else if (OP == 1) { acc[i] = ffma2(acc[i], gg, make_float2(1.f, 1.f)); }  // FFMA2
            else if (OP == 2) { acc[i].x = acc[i].x + g; }                            // FADD
            else if (OP == 3) { acc[i] = fadd2(acc[i], gg); }                         // FADD2
            else if (OP == 5) { dacc[i] = dacc[i] + gd; }                             // DADD
            else if (OP == 6) { dacc[i] = fma(dacc[i], gd, 1.0); }                    // DFMA
            else if (OP == 7) { dacc[i] += (double)acc[i].x; acc[i].x += 1.f; }       // F2F.F64.F32 + DADD (+ FADD)
            else if (OP == 8) { acc[i].x = (float)dacc[i]; dacc[i] += gd; }           // F2F.F32.F64 + DADD
            else {                                                                    // LDS.128
                float4 v;
                asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w)
                             : "r"((unsigned)__cvta_generic_to_shared(&sm[((threadIdx.x + 32 * i + it) & 255) * 4])));
                acc[i].x += v.x;
            }
        }
    }
    const long long t1 = clock64();
    float s = 0.f;
    for (int i = 0; i < kChains; ++i) s += acc[i].x + acc[i].y + (float)dacc[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
    if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
}

template <int OP>
void run(const char *name, double lanes_per_op, const char *unit, int sms)
{
    const int blocks = sms;                     // one CTA of 1024 threads = 32 warps per SM, all starting together
    float *out; long long *cyc;
    cudaMalloc(&out, sizeof(float) * blocks * 1024);
    cudaMalloc(&cyc, sizeof(long long) * blocks);
    k_ubench<OP><<<blocks, 1024>>>(out, 1.0000001f, cyc);
    k_ubench<OP><<<blocks, 1024>>>(out, 1.0000001f, cyc);
    cudaDeviceSynchronize();
    long long *h = new long long[blocks];
    cudaMemcpy(h, cyc, sizeof(long long) * blocks, cudaMemcpyDeviceToHost);
    double mean = 0;
    for (int i = 0; i < blocks; ++i) mean += (double)h[i];
    mean /= blocks;
    // per SM: 1024 threads x kIters x kChains instructions in `mean` cycles
    const double per_clk = 1024.0 * kIters * kChains * lanes_per_op / mean;
    printf("%-8s %8.1f %s per clock and SM   (%.0f cycles per CTA)\n", name, per_clk, unit, mean);
    delete[] h;
    cudaFree(out);
    cudaFree(cyc);
}

int main()
{
    cudaDeviceProp p;
    cudaGetDeviceProperties(&p, 0);
    int clk = 0;
    cudaDeviceGetAttribute(&clk, cudaDevAttrClockRate, 0);
    printf("%s, %d SMs, max SM clock %d MHz\n", p.name, p.multiProcessorCount, clk / 1000);
    run<0>("FFMA", 1, "lane-FMA", p.multiProcessorCount);
    run<1>("FFMA2", 2, "lane-FMA", p.multiProcessorCount);
    run<2>("FADD", 1, "lane-add", p.multiProcessorCount);
    run<3>("FADD2", 2, "lane-add", p.multiProcessorCount);
    run<4>("LDS.128", 16, "bytes", p.multiProcessorCount);
    run<5>("DADD", 1, "lane-add", p.multiProcessorCount);
    run<6>("DFMA", 1, "lane-FMA", p.multiProcessorCount);
    run<7>("F2F64+DADD", 1, "lane-(cvt+add)", p.multiProcessorCount);
    run<8>("F2F32+DADD", 1, "lane-(cvt+add)", p.multiProcessorCount);
    return 0;
}
