// Eq. 2 (index ranges Eq. 3-5) for an ARBITRARY, non-separable filter f[oz][oy][ox] by direct
// summation -- the operation the paper's own kernel performs, with fp32 or,
// as in the paper, fp64 accumulators.
//
// k_direct: one CTA = 128 columns x 64 channels of one row y.  For every filter row oy the CTA stages the slab
// of 64 + 2 rz channels x (128 + 2 rx) columns of input row y + oy in shared memory (zero fill outside the
// cube, C-5) together with that row's taps; then, for every ox, each thread walks along z with 4 columns x 8
// channels of accumulators in registers (the register-march of k_z): per staged channel 4 shared-memory words
// (a lane's columns are 32 apart, so every load is one conflict-free wavefront) and 16 FFMA2, the 15 taps a
// block of 8 channels needs held in registers.  Where the paper re-reads a z line
// per (ox, oy) and does one multiply-add per shared-memory read, this does 8.
#include "pgsf_internal.h"
#include "pgsf_device.cuh"

namespace pgsf {
namespace {

// A thread owns PZ consecutive channels x NC columns (lane l: columns l, l + 32, ...); a warp is one channel
// group, a CTA eight of them: tile = 32 NC columns x 8 PZ channels.  <PZ, NC> = <8, 4> in general; <4, 8> for
// rz <= 8, where a walk in blocks of 8 channels x PZ outputs wastes fewer taps outside the band of 2 rz + 1.
constexpr int DR_GROUPS = 8;              // channel groups = warps
constexpr int DR_LX = 32;                 // one warp per channel group
constexpr int DR_THREADS = DR_LX * DR_GROUPS;

struct DirectShape {
    int rxp;     // rx rounded up to a multiple of 4 (16-byte aligned staging)
    int sw;      // staged columns = 32 NC + 2 rxp
    int nj;      // channels walked per thread = PZ + 2 rz rounded up to a multiple of 8
    int planes;  // staged channels = 7 PZ + nj (>= 8 PZ + 2 rz; the surplus is zero filled)
    int tlen;    // padded taps per ox = nj + 8
    int smem_bytes(int rx) const { return (planes * sw + (2 * rx + 1) * tlen) * (int)sizeof(float); }
};

DirectShape direct_shape(int rx, int rz, int pz, int nc)
{
    DirectShape s;
    s.rxp = (rx + 3) & ~3;
    s.sw = 32 * nc + 2 * s.rxp;
    s.nj = (pz + 2 * rz + 7) & ~7;
    s.planes = (DR_GROUPS - 1) * pz + s.nj;
    s.tlen = s.nj + 8;
    return s;
}

template <bool F64, int DR_PZ, int NC>
__global__ void __launch_bounds__(DR_THREADS) k_direct(const float *__restrict__ in, float *__restrict__ out,
                                                        const float *__restrict__ filt, Dims d, int rx, int ry,
                                                        int rz, DirectShape sh)
{
    constexpr int DR_XT = 32 * NC, DR_ZB = DR_PZ * DR_GROUPS;
    extern __shared__ __align__(16) float dr_smem[];
    float *slab = dr_smem;                              // [planes][sw]
    float *taps = dr_smem + sh.planes * sh.sw;          // [2 rx + 1][tlen]: tap of channel offset o at [8 + o + rz]
    const int tid = threadIdx.x, lx = tid % DR_LX, wz = tid / DR_LX;
    const int z0 = blockIdx.x * DR_ZB, x0 = blockIdx.y * DR_XT, y = blockIdx.z;
    const int fx = 2 * rx + 1, fy = 2 * ry + 1, fz = 2 * rz + 1;
    const bool vec = (d.nx & 3) == 0;                   // rows are 16-byte aligned

    using acc_t = typename std::conditional<F64, double, float>::type;
    acc_t acc[DR_PZ][NC];                               // fp64 path
    float2 a2[DR_PZ][NC / 2];                           // fp32 path: pairs of the lane's columns as FFMA2 operands
#pragma unroll
    for (int p = 0; p < DR_PZ; ++p) {
#pragma unroll
        for (int c = 0; c < NC; ++c) acc[p][c] = (acc_t)0;
#pragma unroll
        for (int c = 0; c < NC / 2; ++c) a2[p][c] = make_float2(0.f, 0.f);
    }

    for (int oy = -ry; oy <= ry; ++oy) {
        const int yy = y + oy;
        if (yy < 0 || yy >= d.ny) continue;             // (uniform over the CTA)
        __syncthreads();                                // the previous row's slab and taps are no longer read
        // slab: channels z0 - rz .. , columns x0 - rxp .. of row yy; zero outside the cube and in the surplus
        const float *row = in + (long long)yy * d.nx;
        // (warp wz takes every 8th staged channel, its lanes stride along the row: no integer divisions)
        for (int pz = wz; pz < sh.planes; pz += DR_GROUPS) {
            const int gz = z0 - rz + pz;
            const bool pok = pz < DR_ZB + 2 * rz && gz >= 0 && gz < d.nz;
            const float *src = row + (long long)(pok ? gz : 0) * d.plane;
            float *dst = slab + pz * sh.sw;
            if (vec) {
                for (int ch = lx; 4 * ch < sh.sw; ch += DR_LX) {
                    const int gx = x0 - sh.rxp + 4 * ch;
                    const bool ok = pok && gx >= 0 && gx < d.nx;
                    cp_async16(dst + 4 * ch, ok ? src + gx : in, ok);
                }
            } else {
                for (int c = lx; c < sh.sw; c += DR_LX) {
                    const int gx = x0 - sh.rxp + c;
                    dst[c] = (pok && gx >= 0 && gx < d.nx) ? __ldg(src + gx) : 0.f;
                }
            }
        }
        // taps of filter row oy: taps[ox][8 + o] = f[o][oy][ox], o = oz + rz; zero padding on both sides
        for (int ix = wz; ix < fx; ix += DR_GROUPS)
            for (int i = lx; i < sh.tlen; i += DR_LX) {
                const int o = i - 8;
                taps[ix * sh.tlen + i] = (o >= 0 && o < fz) ? __ldg(filt + ((long long)o * fy + (oy + ry)) * fx + ix) : 0.f;
            }
        cp_async_wait_all();
        __syncthreads();

        for (int ix = 0; ix < fx; ++ix) {
            // data of output column c and channel offset o sits at slab[(channel - z0 + rz + o)][c + rxp + ox]
            const float *base = slab + (wz * DR_PZ) * sh.sw + sh.rxp + lx + (ix - rx);
            const float *tv = taps + ix * sh.tlen;
#pragma unroll 1
            for (int jc = 0; jc < sh.nj; jc += 8) {
                float tw[16];                           // taps jc .. jc + 15 of the padded vector
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    const float4 t4 = *reinterpret_cast<const float4 *>(tv + jc + 4 * i);
                    tw[4 * i] = t4.x; tw[4 * i + 1] = t4.y; tw[4 * i + 2] = t4.z; tw[4 * i + 3] = t4.w;
                }
#pragma unroll
                for (int jj = 0; jj < 8; ++jj) {
                    const float *pv = base + (jc + jj) * sh.sw;
                    float v[NC];
#pragma unroll
                    for (int c = 0; c < NC; ++c) v[c] = pv[32 * c];
#pragma unroll
                    for (int p = 0; p < DR_PZ; ++p) {
                        const float g = tw[jj - p + 8];  // tap of channel offset (jc + jj) - p - rz
                        if constexpr (F64) {
#pragma unroll
                            for (int c = 0; c < NC; ++c) acc[p][c] += (double)v[c] * (double)g;
                        } else {
#pragma unroll
                            for (int c = 0; c < NC / 2; ++c) a2[p][c] = ffma2(make_float2(v[2 * c], v[2 * c + 1]), g, a2[p][c]);
                        }
                    }
                }
            }
        }
    }

    float *rowo = out + (long long)y * d.nx;
#pragma unroll
    for (int p = 0; p < DR_PZ; ++p) {
        const int gz = z0 + wz * DR_PZ + p;
        if (gz >= d.nz) break;
        float *o = rowo + (long long)gz * d.plane;
        float v[NC];
        if constexpr (F64) {
#pragma unroll
            for (int c = 0; c < NC; ++c) v[c] = (float)acc[p][c];
        } else {
#pragma unroll
            for (int c = 0; c < NC / 2; ++c) { v[2 * c] = a2[p][c].x; v[2 * c + 1] = a2[p][c].y; }
        }
#pragma unroll
        for (int c = 0; c < NC; ++c) {
            const int gx = x0 + lx + 32 * c;
            if (gx < d.nx) o[gx] = v[c];
        }
    }
}

}  // namespace

// <PZ, NC> of the launch: narrow bands walk 4 outputs per thread
inline bool direct_narrow(int rz) { return rz <= 8; }

bool direct_supported(const pgsf_plan *p, int rx, int ry, int rz, int *smem)
{
    if (rx < 0 || ry < 0 || rz < 0 || rx > PGSF_MAX_RADIUS || ry > PGSF_MAX_RADIUS || rz > PGSF_MAX_RADIUS) return false;
    const bool nb = direct_narrow(rz);
    const DirectShape sh = direct_shape(rx, rz, nb ? 4 : 8, nb ? 8 : 4);
    *smem = sh.smem_bytes(rx);
    const int xt = nb ? 256 : 128;
    return *smem <= 200 * 1024 && p->dims.ny <= 65535 && (p->dims.nx + xt - 1) / xt <= 65535;
}

template <bool F64, int PZ, int NC>
cudaError_t launch_direct(const float *filt, int rx, int ry, int rz, const float *in, float *out, const Dims &d,
                          cudaStream_t st)
{
    const DirectShape sh = direct_shape(rx, rz, PZ, NC);
    const int smem = sh.smem_bytes(rx);
    cudaError_t e = ensure_dynamic_smem(k_direct<F64, PZ, NC>, smem);
    if (e != cudaSuccess) return e;
    dim3 grid((d.nz + PZ * DR_GROUPS - 1) / (PZ * DR_GROUPS), (d.nx + 32 * NC - 1) / (32 * NC), d.ny);
    k_direct<F64, PZ, NC><<<grid, DR_THREADS, smem, st>>>(in, out, filt, d, rx, ry, rz, sh);
    return cudaGetLastError();
}

// one cube per call
cudaError_t direct_filter3d(pgsf_plan *p, const float *filt, int rx, int ry, int rz, const float *in, float *out,
                            bool fp64, cudaStream_t st)
{
    const Dims &d = p->dims;
    LaunchScope ls(p, fp64 ? "direct_f64" : "direct_f32", st);
    if (direct_narrow(rz))
        return fp64 ? launch_direct<true, 4, 8>(filt, rx, ry, rz, in, out, d, st)
                    : launch_direct<false, 4, 8>(filt, rx, ry, rz, in, out, d, st);
    return fp64 ? launch_direct<true, 8, 4>(filt, rx, ry, rz, in, out, d, st)
                : launch_direct<false, 8, 4>(filt, rx, ry, rz, in, out, d, st);
}

}  // namespace pgsf
