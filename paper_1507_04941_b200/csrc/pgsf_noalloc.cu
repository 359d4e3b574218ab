// pgsf_filter3d_noalloc: Eq. 2 (index ranges Eq. 3-5) for one Gaussian as three 1-D passes -- the
// arithmetic of the generic path (k_conv1d of pgsf_generic.cu: one thread per voxel, fmaf over the taps in order, zero
// outside the cube, C-5) -- for callers that cannot allocate device memory: code under CUDA graph capture, tight serving
// loops, harnesses that forbid it.  There is no plan and no workspace argument: the two intermediate cubes that the
// generic path takes from the caller's workspace live in a file-scope device array of fixed size.
//
//   * g_na_scratch: 2 x PGSF_NOALLOC_MAX_VOXELS floats = 16 MiB, held by every GPU that loads the library until the
//     process exits.  Larger cubes are refused (PGSF_ERR_UNSUPPORTED, with a text).
//   * In host code the NAME g_na_scratch is a host-side stand-in, not a device address.  The address a kernel may use
//     comes from cudaGetSymbolAddress, asked once per device with that device current (na_scratch_for_current_device).
//   * Every call on a device shares the array; it keeps the previous call's contents.  Nothing in it has to start at
//     zero (each pass writes every voxel of its output before the next pass reads it), so nothing is cleared.  Calls
//     that overlap on the GPU (two streams, two host threads) race on it: the caller serialises them.
//   * The call makes no cudaMalloc / cudaFree / cudaMemcpy and uses no allocating library routine: argument checks, a
//     mutex, two snprintf into the caller's buffer, three kernel launches.  The first call on a device also asks for the
//     symbol address and the device's compute capability (set-up; make one call before capturing a graph).
#include <math.h>
#include <stdint.h>
#include <stdio.h>

#include <mutex>

#include <cuda_runtime.h>

#include "pgsf.h"

namespace {

constexpr int kNaThreads = 256;
constexpr int kNaMaxDevices = 64;

static __device__ __align__(256) float g_na_scratch[2ull * PGSF_NOALLOC_MAX_VOXELS];

struct NaTaps {
    int r;
    float g[2 * PGSF_MAX_RADIUS + 1];
};

struct NaDims {
    int nx, ny, nz;
    long long plane, cube;
};

// out[v] = sum_o in[v + o e_AXIS] g[o], zero outside the cube (C-5)
template <int AXIS>
__global__ void __launch_bounds__(kNaThreads) k_na_conv1d(const float *__restrict__ in, float *__restrict__ out,
                                                          NaDims d, NaTaps t)
{
    const long long i = (long long)blockIdx.x * kNaThreads + threadIdx.x;
    if (i >= d.cube) return;
    const int z = (int)(i / d.plane);
    const int rem = (int)(i - (long long)z * d.plane);
    const int y = rem / d.nx, x = rem - y * d.nx;
    const int c = AXIS == 0 ? x : (AXIS == 1 ? y : z);
    const int n = AXIS == 0 ? d.nx : (AXIS == 1 ? d.ny : d.nz);
    const long long stride = AXIS == 0 ? 1 : (AXIS == 1 ? (long long)d.nx : d.plane);
    const int lo = max(-t.r, -c), hi = min(t.r, n - 1 - c);
    float acc = 0.f;
    for (int o = lo; o <= hi; ++o) acc = fmaf(in[i + o * stride], t.g[o + t.r], acc);
    out[i] = acc;
}

// radius = ceil(truncate sigma) (C-2); fp64 taps renormalised over the truncated support (C-1, C-3), rounded to fp32
// once -- the plan's rule (pgsf_api.cu), restated here because this entry point has no plan
int na_radius(double sigma, double truncate) { return sigma > 0.0 ? (int)ceil(truncate * sigma) : 0; }

void na_taps(double sigma, int r, NaTaps *t)
{
    t->r = r;
    for (int j = 0; j < 2 * PGSF_MAX_RADIUS + 1; ++j) t->g[j] = 0.f;
    if (r == 0) { t->g[0] = 1.f; return; }
    double w[2 * PGSF_MAX_RADIUS + 1], sum = 0.0;
    for (int o = -r; o <= r; ++o) {
        w[o + r] = exp(-0.5 * ((double)o / sigma) * ((double)o / sigma));
        sum += w[o + r];
    }
    for (int o = -r; o <= r; ++o) t->g[o + r] = (float)(w[o + r] / sum);
}

void na_text(char *buf, int cap, const char *msg)
{
    if (buf != nullptr && cap > 0) snprintf(buf, (size_t)cap, "%s", msg);
}

// Set-up, once per device, with that device current: the DEVICE address of g_na_scratch.
cudaError_t na_scratch_for_current_device(float **out, int *cc_major)
{
    static float *ptr[kNaMaxDevices];
    static int major[kNaMaxDevices];
    static bool ready[kNaMaxDevices];
    static std::mutex mtx;
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kNaMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(mtx);
    if (!ready[dev]) {
        float *p = nullptr;
        if ((e = cudaGetSymbolAddress(reinterpret_cast<void **>(&p), g_na_scratch)) != cudaSuccess) return e;
        if (p == nullptr) return cudaErrorInvalidSymbol;
        int mj = 0;
        if ((e = cudaDeviceGetAttribute(&mj, cudaDevAttrComputeCapabilityMajor, dev)) != cudaSuccess) return e;
        ptr[dev] = p;
        major[dev] = mj;
        ready[dev] = true;
    }
    *out = ptr[dev];
    *cc_major = major[dev];
    return cudaSuccess;
}

}  // namespace

extern "C" pgsf_status pgsf_filter3d_noalloc(const float *d_in, float *d_out, int nx, int ny, int nz,
                                             const double *sigma_xyz, double truncate, void *cuda_stream, char *err_text,
                                             int err_cap)
{
    char msg[256];
    na_text(err_text, err_cap, "");
    if (d_in == nullptr || d_out == nullptr || sigma_xyz == nullptr) {
        na_text(err_text, err_cap, "pgsf_filter3d_noalloc: null pointer");
        return PGSF_ERR_INVALID_ARG;
    }
    if (nx < 1 || ny < 1 || nz < 1 || !(truncate > 0.0)) {
        na_text(err_text, err_cap, "pgsf_filter3d_noalloc: extents must be >= 1 and truncate > 0");
        return PGSF_ERR_INVALID_ARG;
    }
    if ((reinterpret_cast<uintptr_t>(d_in) & 3u) || (reinterpret_cast<uintptr_t>(d_out) & 3u)) {
        na_text(err_text, err_cap, "pgsf_filter3d_noalloc: d_in / d_out must be 4-byte aligned");
        return PGSF_ERR_INVALID_ARG;
    }
    const long long voxels = (long long)nx * ny * nz;
    if (voxels > (long long)PGSF_NOALLOC_MAX_VOXELS) {
        snprintf(msg, sizeof msg,
                 "pgsf_filter3d_noalloc: a cube of %lld voxels (%d x %d x %d) exceeds PGSF_NOALLOC_MAX_VOXELS = %lld, the size "
                 "of the static device scratch; use pgsf_filter3d with a workspace",
                 voxels, nx, ny, nz, (long long)PGSF_NOALLOC_MAX_VOXELS);
        na_text(err_text, err_cap, msg);
        return PGSF_ERR_UNSUPPORTED;
    }
    {
        const uintptr_t a = reinterpret_cast<uintptr_t>(d_in), b = reinterpret_cast<uintptr_t>(d_out);
        const uintptr_t bytes = (uintptr_t)voxels * sizeof(float);
        if (a < b + bytes && b < a + bytes) {
            na_text(err_text, err_cap, "pgsf_filter3d_noalloc: d_in and d_out overlap");
            return PGSF_ERR_INVALID_ARG;
        }
    }
    NaTaps t[3];
    for (int a = 0; a < 3; ++a) {
        if (!(sigma_xyz[a] >= 0.0)) {
            na_text(err_text, err_cap, "pgsf_filter3d_noalloc: sigma must be >= 0");
            return PGSF_ERR_INVALID_ARG;
        }
        const int r = na_radius(sigma_xyz[a], truncate);
        if (r > PGSF_MAX_RADIUS) {
            snprintf(msg, sizeof msg, "pgsf_filter3d_noalloc: radius %d on axis %d exceeds PGSF_MAX_RADIUS = %d", r, a,
                     PGSF_MAX_RADIUS);
            na_text(err_text, err_cap, msg);
            return PGSF_ERR_UNSUPPORTED;
        }
        na_taps(sigma_xyz[a], r, &t[a]);
    }
    float *scratch = nullptr;
    int cc_major = 0;
    cudaError_t e = na_scratch_for_current_device(&scratch, &cc_major);
    if (e != cudaSuccess) {
        snprintf(msg, sizeof msg, "pgsf_filter3d_noalloc: set-up of the static scratch failed: %s", cudaGetErrorString(e));
        na_text(err_text, err_cap, msg);
        return PGSF_ERR_CUDA;
    }
    if (cc_major != 10) {
        na_text(err_text, err_cap, "pgsf_filter3d_noalloc: the library holds sm_100a code only");
        return PGSF_ERR_UNSUPPORTED;
    }
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    NaDims d;
    d.nx = nx; d.ny = ny; d.nz = nz;
    d.plane = (long long)nx * ny;
    d.cube = voxels;
    float *tmp_a = scratch, *tmp_b = scratch + PGSF_NOALLOC_MAX_VOXELS;
    const unsigned grid = (unsigned)((voxels + kNaThreads - 1) / kNaThreads);
    k_na_conv1d<0><<<grid, kNaThreads, 0, st>>>(d_in, tmp_a, d, t[0]);
    k_na_conv1d<1><<<grid, kNaThreads, 0, st>>>(tmp_a, tmp_b, d, t[1]);
    k_na_conv1d<2><<<grid, kNaThreads, 0, st>>>(tmp_b, d_out, d, t[2]);
    e = cudaGetLastError();
    if (e != cudaSuccess) {
        snprintf(msg, sizeof msg, "pgsf_filter3d_noalloc: kernel launch failed: %s", cudaGetErrorString(e));
        na_text(err_text, err_cap, msg);
        return PGSF_ERR_CUDA;
    }
    return PGSF_OK;
}
