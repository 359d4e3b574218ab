// Device helpers shared by the filter kernels (internal; not part of the ABI).
#pragma once
#include <mutex>

#include "pgsf_internal.h"

namespace pgsf {
namespace {

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
// same with the shared-memory address already converted (staging loops that step it by a constant)
__device__ __forceinline__ void cp_async16_s(unsigned smem_addr, const void *gmem, bool valid)
{
    const int bytes = valid ? 16 : 0;
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(smem_addr), "l"(gmem), "r"(bytes));
}
__device__ __forceinline__ void cp_async_wait_all()
{
    asm volatile("cp.async.commit_group;\n\tcp.async.wait_group 0;" ::: "memory");
}

// Compensated s += v by the branch-free two-sum (Knuth): the rounding error of s + v is recovered exactly and gathered
// in c; the value of the sum is s + c.  Unlike Kahan's form this is exact also when |v| > |s| -- a bright source
// entering a window of noise.
__device__ __forceinline__ void twosum_add(float &s, float &c, float v)
{
    const float t = s + v;
    const float bp = t - s;
    const float da = s - (t - bp);
    const float db = v - bp;
    c += da + db;
    s = t;
}

// Kahan-compensated s += v (e holds the running low-order error)
__device__ __forceinline__ void kahan_add(float &s, float &e, float v)
{
    const float y = v - e;
    const float t = s + y;
    e = (t - s) - y;
    s = t;
}



// Opt a kernel in to `bytes` of dynamic shared memory.  The attribute belongs to the (kernel, device) pair,
// so what has been granted is remembered per pair (many kernels share one function-pointer type).
template <class K>
cudaError_t ensure_dynamic_smem(K kernel, int bytes)
{
    struct Grant { const void *fn; int dev; int bytes; };
    static Grant table[256];
    static int used = 0;
    static std::mutex mtx;                    // plans of different host threads share this table
    std::lock_guard<std::mutex> lock(mtx);
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    const void *fn = reinterpret_cast<const void *>(kernel);
    Grant *g = nullptr;
    for (int i = 0; i < used; ++i)
        if (table[i].fn == fn && table[i].dev == dev) { g = &table[i]; break; }
    if (g && g->bytes >= bytes) return cudaSuccess;
    if (bytes > 48 * 1024) {
        e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
        if (e != cudaSuccess) return e;
    }
    if (!g && used < 256) g = &table[used++];
    if (g) { g->fn = fn; g->dev = dev; g->bytes = bytes; }
    return cudaSuccess;
}

}  // namespace
}  // namespace pgsf
