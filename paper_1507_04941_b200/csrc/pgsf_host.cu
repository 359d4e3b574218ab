// pgsf_find_multiscale_host, streamed: a HOST-resident cube goes through the device in sections along the
// frequency axis, with the copies of section i+1 (in) and section i-1 (out) running under the compute of section i.
//
// The paper cuts the cube into sections sized to the board's memory, "section = core + halo", and runs
// host-to-device copy, kernel and device-to-host copy one after the other (Fig. 1).  Here:
//   * sections are ranges [c0, c1) of ENTERING channels of the frequency march (multiples of k_zm's step);
//   * nothing is recomputed at the seams: the march of k_zm is cut at step boundaries and carries its running
//     window sums from one launch to the next (ZmSection::state), the x/y-filtered planes and the filtered planes a
//     later section still needs (2 RZ and 2 hz of them) stay on the device and are rolled to the front of their
//     buffers, so every input plane crosses PCIe exactly once and every kernel performs exactly the arithmetic of the
//     resident call -- mask, count and filtered cubes are bit-identical to pgsf_find_multiscale;
//   * three streams: H2D of the next chunk of input planes (two buffers), compute, D2H of the finished mask
//     planes (two buffers; they trail the input by hz channels) and, when asked for, of the filtered planes.
// Device memory: about (6 + 2 S) sections of planes instead of (3 + S) cubes, so a cube that does not fit the
// device (or the budget of PGSF_OPT_HOST_DEVICE_BUDGET) still runs.
#include <stdio.h>
#include <string.h>

#include <algorithm>

#include "pgsf_internal.h"

struct pgsf_host_stage {
    int sec;                                  // entering channels per section
    int rmax;                                 // largest compiled z radius of the plan
    int cap_in, cap_t2[PGSF_MAX_SCALES], cap_f;
    float *d_in[2];
    float *t2[PGSF_MAX_SCALES], *f[PGSF_MAX_SCALES], *state[PGSF_MAX_SCALES];
    float *Z1, *Z2;
    uint8_t *mask[2];
    unsigned long long *d_count;
    float *d_pivlist, *h_pivlist;
    cudaStream_t s_comp, s_in, s_out;
    cudaEvent_t ev_in[2], ev_in_free[2], ev_comp[2], ev_out[2], ev_piv;
    size_t bytes;
};

namespace pgsf {

void host_stage_release(pgsf_plan *p)
{
    pgsf_host_stage *h = p->hs;
    if (!h) return;
    for (int i = 0; i < 2; ++i) {
        cudaFree(h->d_in[i]);
        cudaFree(h->mask[i]);
        if (h->ev_in[i]) cudaEventDestroy(h->ev_in[i]);
        if (h->ev_in_free[i]) cudaEventDestroy(h->ev_in_free[i]);
        if (h->ev_comp[i]) cudaEventDestroy(h->ev_comp[i]);
        if (h->ev_out[i]) cudaEventDestroy(h->ev_out[i]);
    }
    for (int s = 0; s < PGSF_MAX_SCALES; ++s) { cudaFree(h->t2[s]); cudaFree(h->f[s]); cudaFree(h->state[s]); }
    cudaFree(h->Z1);
    cudaFree(h->Z2);
    cudaFree(h->d_count);
    cudaFree(h->d_pivlist);
    if (h->h_pivlist) cudaFreeHost(h->h_pivlist);
    if (h->ev_piv) cudaEventDestroy(h->ev_piv);
    if (h->s_comp) cudaStreamDestroy(h->s_comp);
    if (h->s_in) cudaStreamDestroy(h->s_in);
    if (h->s_out) cudaStreamDestroy(h->s_out);
    cudaGetLastError();
    delete h;
    p->hs = nullptr;
}

namespace {

pgsf_status hfail(pgsf_plan *p, pgsf_status st, const char *what, cudaError_t e)
{
    char buf[256];
    snprintf(buf, sizeof buf, "%s: %s", what, cudaGetErrorString(e));
    p->err = buf;
    cudaGetLastError();
    return st;
}

int round_up(int v, int m) { return (v + m - 1) / m * m; }

// bytes of device staging for sections of `sec` entering channels
size_t stage_bytes(const pgsf_plan *p, int sec, int rmax)
{
    const size_t plane = (size_t)p->dims.plane;
    const int S = p->desc.n_scales, hz = p->desc.box_half[2];
    size_t planes = 2 * (size_t)(sec + rmax) + 2 * (size_t)sec;             // input (x2), Z1, Z2
    for (int s = 0; s < S; ++s) planes += (size_t)(sec + p->scales[s].rz_c + rmax) + (size_t)(sec + 2 * hz) + 4;
    return planes * plane * sizeof(float) + 2 * (size_t)sec * plane + (1u << 23);
}

pgsf_status stage_create(pgsf_plan *p)
{
    const int S = p->desc.n_scales, hz = p->desc.box_half[2], nz = p->desc.nz;
    int rmax = 0, zb = 64;
    for (int s = 0; s < S; ++s) {
        rmax = std::max(rmax, p->scales[s].rz_c);
        zb = std::max(zb, zm_step_channels_of(p->scales[s].rz_c));
        zb = std::max(zb, ztc_step_channels(p, s));      // (PGSF_FLAG_TENSOR_ZPASS: 128-channel steps)
    }
    // a section must be a whole number of march steps and at least as long as what is rolled over to the next one
    const int keep = std::max(std::max(2 * rmax, 2 * hz), zb);
    const int total = nz + hz;
    int sec = p->host_section_planes > 0 ? (int)p->host_section_planes : (total + 15) / 16;
    sec = round_up(std::max(sec, keep), zb);
    size_t budget = (size_t)p->host_budget;
    if (budget == 0) {
        size_t fr = 0, tot = 0;
        cudaError_t e = cudaMemGetInfo(&fr, &tot);
        if (e != cudaSuccess) return hfail(p, PGSF_ERR_CUDA, "cudaMemGetInfo", e);
        budget = fr / 10 * 8;
    }
    if (p->host_section_planes == 0)
        while (stage_bytes(p, sec, rmax) > budget && sec > round_up(keep, zb)) sec -= zb;
    if (stage_bytes(p, sec, rmax) > budget) {
        char buf[256];
        snprintf(buf, sizeof buf, "sections of %d channels need %zu bytes of device staging, the budget is %zu", sec,
                 stage_bytes(p, sec, rmax), budget);
        p->err = buf;
        return PGSF_ERR_OOM;
    }
    pgsf_host_stage *h = new (std::nothrow) pgsf_host_stage();
    if (!h) { p->err = "host stage allocation failed"; return PGSF_ERR_OOM; }
    memset(h, 0, sizeof *h);
    p->hs = h;
    h->sec = sec;
    h->rmax = rmax;
    h->bytes = stage_bytes(p, sec, rmax);
    const size_t plane = (size_t)p->dims.plane;
    h->cap_in = sec + rmax;
    h->cap_f = sec + 2 * hz;
    cudaError_t e = cudaSuccess;
    auto alloc = [&](void **ptr, size_t bytes) { if (e == cudaSuccess) e = cudaMalloc(ptr, bytes ? bytes : 256); };
    for (int i = 0; i < 2; ++i) {
        alloc(reinterpret_cast<void **>(&h->d_in[i]), (size_t)h->cap_in * plane * sizeof(float));
        alloc(reinterpret_cast<void **>(&h->mask[i]), (size_t)sec * plane);
    }
    for (int s = 0; s < S; ++s) {
        h->cap_t2[s] = sec + p->scales[s].rz_c + rmax;
        alloc(reinterpret_cast<void **>(&h->t2[s]), (size_t)h->cap_t2[s] * plane * sizeof(float));
        alloc(reinterpret_cast<void **>(&h->f[s]), (size_t)h->cap_f * plane * sizeof(float));
        alloc(reinterpret_cast<void **>(&h->state[s]), 4 * plane * sizeof(float));
    }
    alloc(reinterpret_cast<void **>(&h->Z1), (size_t)sec * plane * sizeof(float));
    alloc(reinterpret_cast<void **>(&h->Z2), (size_t)sec * plane * sizeof(float));
    alloc(reinterpret_cast<void **>(&h->d_count), sizeof(unsigned long long));
    alloc(reinterpret_cast<void **>(&h->d_pivlist), sizeof(float) << 20);
    if (e == cudaSuccess) e = cudaMallocHost(reinterpret_cast<void **>(&h->h_pivlist), sizeof(float) << 20);
    if (e != cudaSuccess) {
        host_stage_release(p);
        return hfail(p, PGSF_ERR_OOM, "device staging allocation failed", e);
    }
    if ((e = cudaStreamCreateWithFlags(&h->s_comp, cudaStreamNonBlocking)) == cudaSuccess &&
        (e = cudaStreamCreateWithFlags(&h->s_in, cudaStreamNonBlocking)) == cudaSuccess)
        e = cudaStreamCreateWithFlags(&h->s_out, cudaStreamNonBlocking);
    for (int i = 0; i < 2 && e == cudaSuccess; ++i) {
        if ((e = cudaEventCreateWithFlags(&h->ev_in[i], cudaEventDisableTiming)) != cudaSuccess) break;
        if ((e = cudaEventCreateWithFlags(&h->ev_in_free[i], cudaEventDisableTiming)) != cudaSuccess) break;
        if ((e = cudaEventCreateWithFlags(&h->ev_comp[i], cudaEventDisableTiming)) != cudaSuccess) break;
        e = cudaEventCreateWithFlags(&h->ev_out[i], cudaEventDisableTiming);
    }
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&h->ev_piv, cudaEventDisableTiming);
    if (e != cudaSuccess) {
        host_stage_release(p);
        return hfail(p, PGSF_ERR_CUDA, "stream / event creation failed", e);
    }
    return PGSF_OK;
}

// virtual cube pointer: plane `base` of the cube lives at the start of `buf`
template <class T>
T *virt(T *buf, long long base, size_t plane)
{
    return reinterpret_cast<T *>(reinterpret_cast<uintptr_t>(buf) - (uintptr_t)((long long)sizeof(T) * base * (long long)plane));
}

}  // namespace

pgsf_status host_streamed(pgsf_plan *p, const float *h_in, float *const *h_filtered, uint8_t *h_mask,
                          unsigned long long *h_count, bool *handled)
{
    *handled = false;
    if (!p->fast_filter || !stats_sparse_or(p)) return PGSF_OK;     // the generic kernels take whole cubes
    *handled = true;
    if (!p->hs) {
        pgsf_status rc = stage_create(p);
        if (rc != PGSF_OK) return rc;
    }
    pgsf_host_stage *h = p->hs;
    const int S = p->desc.n_scales, hz = p->desc.box_half[2], nz = p->desc.nz, B = p->desc.batch;
    const int sec = h->sec, rmax = h->rmax;
    const size_t plane = (size_t)p->dims.plane, cube = (size_t)p->dims.cube;
    const int nsec = (nz + hz + sec - 1) / sec;
    bool any_f = false;
    if (h_filtered)
        for (int s = 0; s < S; ++s) any_f = any_f || h_filtered[s] != nullptr;
    cudaError_t e;
#define HCHECK(call, what) do { if ((e = (call)) != cudaSuccess) return hfail(p, PGSF_ERR_CUDA, what, e); } while (0)
    HCHECK(cudaMemsetAsync(h->d_count, 0, sizeof(unsigned long long), h->s_comp), "cudaMemsetAsync(count)");
    int idx[PGSF_MAX_SCALES];
    for (int s = 0; s < S; ++s) idx[s] = s;
    const int G = p->group;
    long long q = 0;              // running section number: selects the input / mask buffer
    bool piv_pending = false;
    for (int b = 0; b < B; ++b) {
        const float *h_cube = h_in + (size_t)b * cube;
        if (b % G == 0) {
            // pivot of the statistics of this group of cubes (D-2): the lattice of the group's first cube.
            // Page-locked input is read in place by the very kernel the resident call runs; otherwise the samples are
            // gathered here, in lattice order, and reduced by the same code.
            cudaPointerAttributes attr;
            const bool mapped = cudaPointerGetAttributes(&attr, h_cube) == cudaSuccess &&
                                attr.type == cudaMemoryTypeHost && attr.devicePointer != nullptr;
            cudaGetLastError();
            if (mapped) {
                HCHECK(compute_pivot(p, static_cast<const float *>(attr.devicePointer), h->s_comp), "pivot launch");
            } else {
                if (piv_pending) HCHECK(cudaEventSynchronize(h->ev_piv), "pivot list synchronize");
                int lo[3], st[3], cnt[3];
                pivot_lattice(p->dims, lo, st, cnt);
                const int nsamp = cnt[0] * cnt[1] * cnt[2];
                for (int i = 0; i < nsamp; ++i) {
                    const int ix = i % cnt[0], iy = (i / cnt[0]) % cnt[1], iz = i / (cnt[0] * cnt[1]);
                    h->h_pivlist[i] = h_cube[(size_t)(lo[0] + ix * st[0]) +
                                             (size_t)p->dims.nx * ((size_t)(lo[1] + iy * st[1]) + (size_t)p->dims.ny * (size_t)(lo[2] + iz * st[2]))];
                }
                HCHECK(cudaMemcpyAsync(h->d_pivlist, h->h_pivlist, sizeof(float) * nsamp, cudaMemcpyHostToDevice, h->s_comp),
                       "H2D pivot samples");
                HCHECK(cudaEventRecord(h->ev_piv, h->s_comp), "event record");
                piv_pending = true;
                HCHECK(compute_pivot_list(p, h->d_pivlist, nsamp, h->s_comp), "pivot launch");
            }
        }
        int hi_prev = 0;          // input planes [0, hi_prev) of this cube are on the device (x/y passes done)
        for (int i = 0; i < nsec; ++i, ++q) {
            const int bi = (int)(q & 1);
            const int c0 = i * sec, c1 = c0 + sec;
            const bool last = i == nsec - 1;
            const int hi = std::min(c1 + rmax, nz);
            const int p0 = hi_prev, p1 = std::max(hi, hi_prev);
            // ---- H2D: the new input planes [p0, p1)
            if (p1 > p0) {
                if (q >= 2) HCHECK(cudaStreamWaitEvent(h->s_in, h->ev_in_free[bi], 0), "stream wait");
                HCHECK(cudaMemcpyAsync(h->d_in[bi], h_cube + (size_t)p0 * plane, (size_t)(p1 - p0) * plane * sizeof(float),
                                       cudaMemcpyHostToDevice, h->s_in), "H2D copy");
                HCHECK(cudaEventRecord(h->ev_in[bi], h->s_in), "event record");
            }
            // ---- compute
            cudaStream_t sc = h->s_comp;
            if (q >= 2) HCHECK(cudaStreamWaitEvent(sc, h->ev_out[bi], 0), "stream wait");          // mask buffer is free
            if (any_f && q >= 1) HCHECK(cudaStreamWaitEvent(sc, h->ev_out[bi ^ 1], 0), "stream wait");   // f planes are out
            const int zs0 = std::max(c0 - hz, 0), zs1 = last ? nz : std::min(c1 - hz, nz);
            for (int s = 0; s < S && i > 0; ++s) {
                // roll what the next section still needs to the front of its buffer
                const int rz = p->scales[s].rz_c;
                const int keep_t2 = hi_prev - (c0 - rz);        // planes [c0 - rz, hi_prev); they sat `sec` planes in
                if (keep_t2 > 0)
                    HCHECK(cudaMemcpyAsync(h->t2[s], h->t2[s] + (size_t)sec * plane, (size_t)keep_t2 * plane * sizeof(float),
                                           cudaMemcpyDeviceToDevice, sc), "roll of the x/y-filtered planes");
                HCHECK(cudaMemcpyAsync(h->f[s], h->f[s] + (size_t)sec * plane, (size_t)(2 * hz) * plane * sizeof(float),
                                       cudaMemcpyDeviceToDevice, sc), "roll of the filtered planes");
            }
            float *t2v[PGSF_MAX_SCALES], *t2w[PGSF_MAX_SCALES];
            for (int s = 0; s < S; ++s) {
                t2v[s] = virt(h->t2[s], (long long)c0 - p->scales[s].rz_c, plane);
                t2w[s] = t2v[s] + (size_t)p0 * plane;           // where plane p0 goes
            }
            if (p1 > p0) {
                HCHECK(cudaStreamWaitEvent(sc, h->ev_in[bi], 0), "stream wait");
                HCHECK(fast_xy_multi(p, idx, S, h->d_in[bi], t2w, 1, sc, false, nullptr, p1 - p0), "xy filter launch");
                HCHECK(cudaEventRecord(h->ev_in_free[bi], sc), "event record");
            }
            hi_prev = p1;
            for (int s = 0; s < S; ++s) {
                float *fv = virt(h->f[s], (long long)c0 - 2 * hz, plane);
                float *z1v = virt(h->Z1, (long long)c0 - hz, plane), *z2v = virt(h->Z2, (long long)c0 - hz, plane);
                ZmSection zs{c0, last ? (1 << 30) : c1, h->state[s], h->t2[s], c0 - p->scales[s].rz_c, hi_prev};
                HCHECK(fast_zm(p, s, t2v[s], fv, z1v, z2v, 1, sc, &zs), "z filter + window launch");
                if (zs1 > zs0)
                    HCHECK(xyb_threshold(p, fv + (size_t)zs0 * plane, z1v + (size_t)zs0 * plane, z2v + (size_t)zs0 * plane,
                                         h->mask[bi], s == 0 ? 0 : 2, nullptr, nullptr, h->d_count, 1, sc, zs1 - zs0, zs0),
                           "threshold launch");
            }
            HCHECK(cudaEventRecord(h->ev_comp[bi], sc), "event record");
            // ---- D2H: the finished mask planes [zs0, zs1) and the filtered planes [c0, min(c1, nz))
            HCHECK(cudaStreamWaitEvent(h->s_out, h->ev_comp[bi], 0), "stream wait");
            if (zs1 > zs0)
                HCHECK(cudaMemcpyAsync(h_mask + (size_t)b * cube + (size_t)zs0 * plane, h->mask[bi], (size_t)(zs1 - zs0) * plane,
                                       cudaMemcpyDeviceToHost, h->s_out), "D2H mask copy");
            const int f1 = std::min(c1, nz);
            if (any_f && f1 > c0)
                for (int s = 0; s < S; ++s)
                    if (h_filtered[s])
                        HCHECK(cudaMemcpyAsync(h_filtered[s] + (size_t)b * cube + (size_t)c0 * plane,
                                               h->f[s] + (size_t)(2 * hz) * plane, (size_t)(f1 - c0) * plane * sizeof(float),
                                               cudaMemcpyDeviceToHost, h->s_out), "D2H filtered copy");
            HCHECK(cudaEventRecord(h->ev_out[bi], h->s_out), "event record");
        }
    }
    unsigned long long cnt = 0;
    HCHECK(cudaStreamSynchronize(h->s_out), "stream synchronize");
    HCHECK(cudaMemcpyAsync(&cnt, h->d_count, sizeof cnt, cudaMemcpyDeviceToHost, h->s_comp), "D2H count copy");
    HCHECK(cudaStreamSynchronize(h->s_comp), "stream synchronize");
    HCHECK(cudaStreamSynchronize(h->s_in), "stream synchronize");
#undef HCHECK
    if (h_count) *h_count = cnt;
    return PGSF_OK;
}

}  // namespace pgsf
