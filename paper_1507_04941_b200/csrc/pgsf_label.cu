// NEXT-4: mask -> candidate objects.  The paper merges the selected voxels into sources and combines them "to a
// single, parameterised catalogue" (selection step P:282) without saying how voxels are joined; reading C-19
// (DESIGN.md): an object is a connected component of the OR mask under 26-connectivity, every cube of a batch on its
// own.  Label = 1 + the smallest linear index (inside its cube) of the component's voxels, 0 = background -- a unique
// labelling, so the result can be compared with the oracle element by element.
//
// Union-find on the device: the label array doubles as the parent array (a root points at itself).  k_lbl_init makes
// every set voxel its own root, k_lbl_merge unites every set voxel with its set neighbours among the 13 that precede
// it in memory (the other 13 pairs are seen from the other side), always hanging the larger root under the smaller
// (atomicMin), so the root of a finished tree is the smallest index of the component; k_lbl_flatten points every voxel
// at its root; k_lbl_final turns roots into labels and counts them.
#include "pgsf_internal.h"

namespace pgsf {
namespace {

constexpr int LB_NT = 256;
constexpr unsigned kNone = 0xffffffffu;

__device__ __forceinline__ unsigned lbl_find(const unsigned *L, unsigned x)
{
    unsigned p = *reinterpret_cast<const volatile unsigned *>(L + x);
    while (p != x) {
        x = p;
        p = *reinterpret_cast<const volatile unsigned *>(L + x);
    }
    return x;
}

__device__ __forceinline__ void lbl_unite(unsigned *L, unsigned a, unsigned b)
{
    while (true) {
        a = lbl_find(L, a);
        b = lbl_find(L, b);
        if (a == b) return;
        if (a < b) { const unsigned t = a; a = b; b = t; }      // a > b: hang a under b
        const unsigned old = atomicMin(L + a, b);
        if (old == a) return;                                   // a was still a root: done
        a = old;                                                // someone else re-parented a meanwhile: go on from there
    }
}

__global__ void __launch_bounds__(LB_NT) k_lbl_init(const uint8_t *__restrict__ mask, unsigned *__restrict__ L, long long cube,
                                                    long long total)
{
    const long long i = (long long)blockIdx.x * LB_NT + threadIdx.x;
    if (i >= total) return;
    L[i] = mask[i] ? (unsigned)(i % cube) : kNone;
}

__global__ void __launch_bounds__(LB_NT) k_lbl_merge(const uint8_t *__restrict__ mask, unsigned *L, Dims d, long long total)
{
    const long long i = (long long)blockIdx.x * LB_NT + threadIdx.x;
    if (i >= total || !mask[i]) return;
    const long long base = i / d.cube * d.cube;                 // this voxel's cube
    const long long v = i - base;
    const int x = (int)(v % d.nx), y = (int)((v / d.nx) % d.ny), z = (int)(v / d.plane);
    unsigned *Lc = L + base;
    const uint8_t *mc = mask + base;
    for (int dz = -1; dz <= 0; ++dz)
        for (int dy = -1; dy <= (dz < 0 ? 1 : 0); ++dy)
            for (int dx = -1; dx <= ((dz < 0 || dy < 0) ? 1 : -1); ++dx) {
                const int xx = x + dx, yy = y + dy, zz = z + dz;
                if (xx < 0 || yy < 0 || zz < 0 || xx >= d.nx || yy >= d.ny) continue;
                const long long u = xx + (long long)d.nx * (yy + (long long)d.ny * zz);
                if (mc[u]) lbl_unite(Lc, (unsigned)v, (unsigned)u);
            }
}

__global__ void __launch_bounds__(LB_NT) k_lbl_flatten(unsigned *L, long long cube, long long total)
{
    const long long i = (long long)blockIdx.x * LB_NT + threadIdx.x;
    if (i >= total) return;
    const unsigned p = L[i];
    if (p == kNone) return;
    const long long base = i / cube * cube;
    L[i] = lbl_find(L + base, p);
}

__global__ void __launch_bounds__(LB_NT) k_lbl_final(unsigned *__restrict__ L, long long cube, long long total,
                                                     unsigned long long *__restrict__ count)
{
    const long long i = (long long)blockIdx.x * LB_NT + threadIdx.x;
    unsigned root = 0;
    if (i < total) {
        const unsigned p = L[i];
        root = (p != kNone && p == (unsigned)(i % cube)) ? 1u : 0u;
        L[i] = p == kNone ? 0u : p + 1u;
    }
    const unsigned n = __popc(__ballot_sync(0xffffffffu, root != 0));
    if (count != nullptr && n && (threadIdx.x & 31) == 0) atomicAdd(count, (unsigned long long)n);
}

}  // namespace

cudaError_t label_objects(pgsf_plan *p, const uint8_t *mask, unsigned *labels, unsigned long long *count, cudaStream_t st)
{
    const Dims &d = p->dims;
    const long long total = d.cube * p->desc.batch;
    const long long blocks = (total + LB_NT - 1) / LB_NT;
    if (blocks > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    cudaError_t e;
    if (count != nullptr && (e = cudaMemsetAsync(count, 0, sizeof(unsigned long long), st)) != cudaSuccess) return e;
    { LaunchScope ls(p, "label_init", st); k_lbl_init<<<(unsigned)blocks, LB_NT, 0, st>>>(mask, labels, d.cube, total); }
    { LaunchScope ls(p, "label_merge", st); k_lbl_merge<<<(unsigned)blocks, LB_NT, 0, st>>>(mask, labels, d, total); }
    { LaunchScope ls(p, "label_flatten", st); k_lbl_flatten<<<(unsigned)blocks, LB_NT, 0, st>>>(labels, d.cube, total); }
    { LaunchScope ls(p, "label_final", st); k_lbl_final<<<(unsigned)blocks, LB_NT, 0, st>>>(labels, d.cube, total, count); }
    return cudaGetLastError();
}

}  // namespace pgsf
