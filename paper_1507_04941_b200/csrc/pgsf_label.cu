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

// grid (blocks per cube, cubes); a thread takes V consecutive voxels of its cube (V = 16: one 16-byte load of the mask,
// when the cube is a multiple of 16 voxels; V = 1 otherwise).  v = index inside the cube (fits 32 bits).
template <int V>
__device__ __forceinline__ void load_mask(const uint8_t *m, uint8_t (&b)[V])
{
    if constexpr (V == 16) {
        const uint4 q = *reinterpret_cast<const uint4 *>(m);
        const unsigned w[4] = {q.x, q.y, q.z, q.w};
#pragma unroll
        for (int i = 0; i < 16; ++i) b[i] = (uint8_t)(w[i >> 2] >> (8 * (i & 3)));
    } else {
        b[0] = m[0];
    }
}

template <int V>
__global__ void __launch_bounds__(LB_NT) k_lbl_init(const uint8_t *__restrict__ mask, unsigned *__restrict__ L, long long cube)
{
    const long long v = ((long long)blockIdx.x * LB_NT + threadIdx.x) * V;
    if (v >= cube) return;
    const long long i = (long long)blockIdx.y * cube + v;
    uint8_t b[V];
    load_mask<V>(mask + i, b);
    unsigned out[V];
#pragma unroll
    for (int k = 0; k < V; ++k) out[k] = b[k] ? (unsigned)(v + k) : kNone;
    if constexpr (V == 16) {
#pragma unroll
        for (int k = 0; k < 4; ++k)
            reinterpret_cast<uint4 *>(L + i)[k] = make_uint4(out[4 * k], out[4 * k + 1], out[4 * k + 2], out[4 * k + 3]);
    } else {
        L[i] = out[0];
    }
}

template <int V>
__global__ void __launch_bounds__(LB_NT) k_lbl_merge(const uint8_t *__restrict__ mask, unsigned *L, Dims d)
{
    const long long v0 = ((long long)blockIdx.x * LB_NT + threadIdx.x) * V;
    if (v0 >= d.cube) return;
    const long long base = (long long)blockIdx.y * d.cube;
    const uint8_t *mc = mask + base;
    uint8_t b[V];
    load_mask<V>(mc + v0, b);
    unsigned any = 0;
#pragma unroll
    for (int k = 0; k < V; ++k) any |= b[k];
    if (!any) return;                                          // (a few voxels in 10^4 are set)
    unsigned *Lc = L + base;
    for (int k = 0; k < V; ++k) {
        if (!b[k]) continue;
        const long long v = v0 + k;
        const int z = (int)(v / d.plane);
        const unsigned r = (unsigned)(v - (long long)z * d.plane);      // (a plane fits 32 bits)
        const int y = (int)(r / (unsigned)d.nx), x = (int)(r - (unsigned)y * (unsigned)d.nx);
        for (int dz = -1; dz <= 0; ++dz)
            for (int dy = -1; dy <= (dz < 0 ? 1 : 0); ++dy)
                for (int dx = -1; dx <= ((dz < 0 || dy < 0) ? 1 : -1); ++dx) {
                    const int xx = x + dx, yy = y + dy, zz = z + dz;
                    if (xx < 0 || yy < 0 || zz < 0 || xx >= d.nx || yy >= d.ny) continue;
                    const long long u = xx + (long long)d.nx * (yy + (long long)d.ny * zz);
                    if (mc[u]) lbl_unite(Lc, (unsigned)v, (unsigned)u);
                }
    }
}

// flatten: only the set voxels have anything to do, and the mask says which they are without reading L
template <int V>
__global__ void __launch_bounds__(LB_NT) k_lbl_flatten(const uint8_t *__restrict__ mask, unsigned *L, long long cube)
{
    const long long v0 = ((long long)blockIdx.x * LB_NT + threadIdx.x) * V;
    if (v0 >= cube) return;
    const long long base = (long long)blockIdx.y * cube;
    uint8_t b[V];
    load_mask<V>(mask + base + v0, b);
    unsigned *Lc = L + base;
    for (int k = 0; k < V; ++k) {
        if (!b[k]) continue;
        const long long v = v0 + k;
        const unsigned p = Lc[v];
        if (p != (unsigned)v) Lc[v] = lbl_find(Lc, p);
    }
}

template <int V>
__global__ void __launch_bounds__(LB_NT) k_lbl_final(const uint8_t *__restrict__ mask, unsigned *__restrict__ L, long long cube,
                                                     unsigned long long *__restrict__ count)
{
    const long long v0 = ((long long)blockIdx.x * LB_NT + threadIdx.x) * V;
    unsigned roots = 0;
    if (v0 < cube) {
        const long long base = (long long)blockIdx.y * cube;
        uint8_t b[V];
        load_mask<V>(mask + base + v0, b);
        unsigned any = 0;
#pragma unroll
        for (int k = 0; k < V; ++k) any |= b[k];
        unsigned *Lc = L + base + v0;
        if (!any) {
            if constexpr (V == 16) {
#pragma unroll
                for (int k = 0; k < 4; ++k) reinterpret_cast<uint4 *>(Lc)[k] = make_uint4(0u, 0u, 0u, 0u);
            } else {
                Lc[0] = 0u;
            }
        } else {
            for (int k = 0; k < V; ++k) {
                const unsigned p = b[k] ? Lc[k] : kNone;
                roots += (b[k] && p == (unsigned)(v0 + k)) ? 1u : 0u;
                Lc[k] = b[k] ? p + 1u : 0u;
            }
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) roots += __shfl_xor_sync(0xffffffffu, roots, o);
    if (count != nullptr && roots && (threadIdx.x & 31) == 0) atomicAdd(count, (unsigned long long)roots);
}

template <int V>
cudaError_t label_launch(pgsf_plan *p, const uint8_t *mask, unsigned *labels, unsigned long long *count, cudaStream_t st)
{
    const Dims &d = p->dims;
    const long long blocks = ((d.cube + V - 1) / V + LB_NT - 1) / LB_NT;
    if (blocks > 0x7fffffffLL || p->desc.batch > 65535) return cudaErrorInvalidConfiguration;
    const dim3 grid((unsigned)blocks, (unsigned)p->desc.batch);
    { LaunchScope ls(p, "label_init", st); k_lbl_init<V><<<grid, LB_NT, 0, st>>>(mask, labels, d.cube); }
    { LaunchScope ls(p, "label_merge", st); k_lbl_merge<V><<<grid, LB_NT, 0, st>>>(mask, labels, d); }
    { LaunchScope ls(p, "label_flatten", st); k_lbl_flatten<V><<<grid, LB_NT, 0, st>>>(mask, labels, d.cube); }
    { LaunchScope ls(p, "label_final", st); k_lbl_final<V><<<grid, LB_NT, 0, st>>>(mask, labels, d.cube, count); }
    return cudaGetLastError();
}

}  // namespace

cudaError_t label_objects(pgsf_plan *p, const uint8_t *mask, unsigned *labels, unsigned long long *count, cudaStream_t st)
{
    cudaError_t e;
    if (count != nullptr && (e = cudaMemsetAsync(count, 0, sizeof(unsigned long long), st)) != cudaSuccess) return e;
    const bool vec = p->dims.cube % 16 == 0 && (reinterpret_cast<uintptr_t>(mask) & 15u) == 0;
    return vec ? label_launch<16>(p, mask, labels, count, st) : label_launch<1>(p, mask, labels, count, st);
}

}  // namespace pgsf
