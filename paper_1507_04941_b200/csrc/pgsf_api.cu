// C ABI of libpgsf.so: plan construction (host), argument validation, kernel dispatch.
// See include/pgsf.h for the contract of every entry point.
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <string.h>

#include <new>

#include "pgsf_internal.h"

namespace {

thread_local std::string g_create_err;

pgsf_status fail(pgsf_plan *p, pgsf_status st, const char *fmt, ...)
{
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    if (p) p->err = buf;
    else g_create_err = buf;
    return st;
}

pgsf_status cuda_fail(pgsf_plan *p, cudaError_t e, const char *what)
{
    return fail(p, PGSF_ERR_CUDA, "%s: %s", what, cudaGetErrorString(e));
}

// radius = ceil(truncate * sigma) in fp64 (C-2); sigma = 0 -> 0
int radius_of(double sigma, double truncate)
{
    if (!(sigma > 0.0)) return 0;
    return (int)ceil(truncate * sigma);
}

// fp64 taps, renormalised over the truncated support (C-1, C-3), rounded to fp32 once.
void make_taps(double sigma, int r, float *g /* 2r+1 */)
{
    if (r == 0) { g[0] = 1.f; return; }
    double w[pgsf::kMaxTaps];
    double sum = 0.0;
    for (int o = -r; o <= r; ++o) {
        w[o + r] = exp(-0.5 * ((double)o / sigma) * ((double)o / sigma));
        sum += w[o + r];
    }
    for (int o = -r; o <= r; ++o) g[o + r] = (float)(w[o + r] / sum);
}

cudaEvent_t take_event(pgsf_plan *p)
{
    cudaEvent_t e = nullptr;
    if (!p->prof_free.empty()) {
        e = p->prof_free.back();
        p->prof_free.pop_back();
    } else if (cudaEventCreate(&e) != cudaSuccess) {
        cudaGetLastError();
        e = nullptr;
    }
    return e;
}

bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

struct Range { const char *name; const void *ptr; size_t bytes; };

// first pair of overlapping byte ranges (NULL / empty ranges are skipped), or false
bool find_overlap(const Range *r, int n, int *a, int *b)
{
    for (int i = 0; i < n; ++i)
        for (int j = i + 1; j < n; ++j) {
            if (!r[i].ptr || !r[j].ptr || !r[i].bytes || !r[j].bytes) continue;
            const char *pi = static_cast<const char *>(r[i].ptr), *pj = static_cast<const char *>(r[j].ptr);
            if (pi < pj + r[j].bytes && pj < pi + r[i].bytes) { *a = i; *b = j; return true; }
        }
    return false;
}

size_t round256(size_t v) { return (v + 255u) & ~(size_t)255u; }

}  // namespace

namespace pgsf {

void host_release(pgsf_plan *p)
{
    host_stage_release(p);
    cudaFree(p->h_d_in);
    cudaFree(p->h_d_mask);
    cudaFree(p->h_d_count);
    cudaFree(p->h_d_ws);
    p->h_d_in = nullptr;
    p->h_d_mask = nullptr;
    p->h_d_count = nullptr;
    p->h_d_ws = nullptr;
    for (int s = 0; s < PGSF_MAX_SCALES; ++s) { cudaFree(p->h_d_f[s]); p->h_d_f[s] = nullptr; }
    if (p->h_stream) cudaStreamDestroy(p->h_stream);
    p->h_stream = nullptr;
    cudaGetLastError();
}

LaunchScope::LaunchScope(pgsf_plan *plan, const char *name, cudaStream_t stream) : p(plan), st(stream), b(nullptr)
{
    p->launches += 1;
    if (!p->prof_on) return;
    int id = -1;
    for (size_t i = 0; i < p->prof_acc.size(); ++i)
        if (p->prof_acc[i].name == name) { id = (int)i; break; }
    if (id < 0) {
        p->prof_acc.push_back(ProfAcc{name, 0ULL, 0.0});
        id = (int)p->prof_acc.size() - 1;
    }
    cudaEvent_t a = take_event(p);
    b = take_event(p);
    if (!a || !b) { if (a) p->prof_free.push_back(a); if (b) p->prof_free.push_back(b); b = nullptr; return; }
    cudaEventRecord(a, st);
    p->prof_recs.push_back(ProfRec{id, a, b});
}

LaunchScope::~LaunchScope()
{
    if (b) cudaEventRecord(b, st);
}

}  // namespace pgsf

extern "C" {

pgsf_status pgsf_plan_create(pgsf_plan **out, const pgsf_plan_desc *desc, int device)
{
    if (out == nullptr) return fail(nullptr, PGSF_ERR_INVALID_ARG, "out is NULL");
    *out = nullptr;
    if (desc == nullptr) return fail(nullptr, PGSF_ERR_INVALID_ARG, "desc is NULL");
    if (desc->nx < 1 || desc->ny < 1 || desc->nz < 1 || desc->batch < 1)
        return fail(nullptr, PGSF_ERR_INVALID_ARG, "extents and batch must be >= 1");
    if ((long long)desc->nx * desc->ny >= (1LL << 31))
        return fail(nullptr, PGSF_ERR_UNSUPPORTED, "nx*ny must be < 2^31");
    if (desc->n_scales < 1 || desc->n_scales > PGSF_MAX_SCALES)
        return fail(nullptr, PGSF_ERR_INVALID_ARG, "n_scales must be in 1..%d", PGSF_MAX_SCALES);
    if (desc->sigmas == nullptr) return fail(nullptr, PGSF_ERR_INVALID_ARG, "sigmas is NULL");
    if (!(desc->truncate > 0.0)) return fail(nullptr, PGSF_ERR_INVALID_ARG, "truncate must be > 0");
    if (!(desc->k >= 0.0)) return fail(nullptr, PGSF_ERR_INVALID_ARG, "k must be >= 0");
    const int ext[3] = {desc->nx, desc->ny, desc->nz};
    for (int a = 0; a < 3; ++a) {
        if (desc->box_half[a] < 0 || desc->halo[a] < 0)
            return fail(nullptr, PGSF_ERR_INVALID_ARG, "box_half and halo must be >= 0");
        if (desc->halo[a] > 0 && 2 * desc->halo[a] >= ext[a])
            return fail(nullptr, PGSF_ERR_INVALID_ARG, "2*halo must be < extent");
        if (desc->box_half[a] > PGSF_MAX_BOX_HALF)
            return fail(nullptr, PGSF_ERR_UNSUPPORTED, "box_half above %d", PGSF_MAX_BOX_HALF);
    }
    for (int i = 0; i < desc->n_scales * 3; ++i) {
        const double s = desc->sigmas[i];
        if (!(s >= 0.0) || !isfinite(s))
            return fail(nullptr, PGSF_ERR_INVALID_ARG, "sigma must be finite and >= 0");
        if (radius_of(s, desc->truncate) > PGSF_MAX_RADIUS)
            return fail(nullptr, PGSF_ERR_UNSUPPORTED, "radius ceil(truncate*sigma) above %d",
                        PGSF_MAX_RADIUS);
    }
    const bool dry = (desc->flags & PGSF_FLAG_DRY_RUN) != 0;
    cudaDeviceProp prop;
    prop.multiProcessorCount = 148;
    if (!dry) {
        int ndev = 0;
        cudaError_t e = cudaGetDeviceCount(&ndev);
        if (e != cudaSuccess) return cuda_fail(nullptr, e, "cudaGetDeviceCount (no CPU fallback exists)");
        if (device < 0 || device >= ndev)
            return fail(nullptr, PGSF_ERR_CUDA, "device %d not present (%d devices)", device, ndev);
        e = cudaGetDeviceProperties(&prop, device);
        if (e != cudaSuccess) return cuda_fail(nullptr, e, "cudaGetDeviceProperties");
        if (prop.major != 10)
            return fail(nullptr, PGSF_ERR_UNSUPPORTED, "device is sm_%d%d; this library is built for sm_100a",
                        prop.major, prop.minor);
    }

    pgsf_plan *p = new (std::nothrow) pgsf_plan();
    if (!p) return fail(nullptr, PGSF_ERR_OOM, "plan allocation failed");
    p->desc = *desc;
    memcpy(p->sigmas, desc->sigmas, sizeof(double) * 3 * desc->n_scales);
    p->desc.sigmas = p->sigmas;
    p->device = device;
    p->dry = dry;
    p->sm_count = prop.multiProcessorCount;
    p->dims.nx = desc->nx;
    p->dims.ny = desc->ny;
    p->dims.nz = desc->nz;
    p->dims.plane = (long long)desc->nx * desc->ny;
    p->dims.cube = p->dims.plane * desc->nz;
    p->launches = 0;
    p->prof_on = false;
    p->d_pivot = nullptr;
    p->h_d_in = nullptr;
    p->h_d_mask = nullptr;
    p->h_d_count = nullptr;
    p->h_d_ws = nullptr;
    p->h_stream = nullptr;
    p->hs = nullptr;
    p->tensor_z = false;
    for (int s = 0; s < PGSF_MAX_SCALES; ++s) { p->d_tc_strips[s] = nullptr; p->tc_march[s] = 0; }
    for (int s = 0; s < PGSF_MAX_SCALES; ++s) p->h_d_f[s] = nullptr;

    const bool force_generic = (desc->flags & PGSF_FLAG_FORCE_GENERIC) != 0;
    // The tiled kernels put ny, nz (x batch group) on grid.y / grid.z: shapes beyond those limits run the generic
    // kernels (decided here, so that no launch can fail with an invalid configuration later).
    const bool grid_ok = desc->ny <= 65535 && desc->nz <= 65535;
    bool fast = !force_generic && (desc->nx % 4 == 0) && grid_ok;
    char why[160];
    if (force_generic) p->why_filter = "PGSF_FLAG_FORCE_GENERIC";
    else if (desc->nx % 4 != 0) p->why_filter = "nx % 4 != 0";
    else if (!grid_ok) p->why_filter = "ny or nz above 65535";
    for (int s = 0; s < desc->n_scales; ++s) {
        pgsf::ScalePlan &sp = p->scales[s];
        memset(&sp, 0, sizeof sp);
        for (int a = 0; a < 3; ++a) {
            const double sg = desc->sigmas[3 * s + a];
            sp.r[a] = radius_of(sg, desc->truncate);
            sp.taps[a].r = sp.r[a];
            make_taps(sg, sp.r[a], sp.taps[a].g);
        }
        const int rxy = sp.r[0] > sp.r[1] ? sp.r[0] : sp.r[1];
        if (!pgsf::fast_xy_radius(rxy, &sp.rxy_c) || !pgsf::fast_z_radius(sp.r[2], &sp.rz_c)) {
            if (fast) {
                snprintf(why, sizeof why, "scale %d: radii (%d, %d, %d) outside the compiled x/y <= 12, z <= 96", s,
                         sp.r[0], sp.r[1], sp.r[2]);
                p->why_filter = why;
            }
            fast = false;
            continue;
        }
        // centre the true taps in the compiled window; the padding taps are exact zeros, so the
        // extra FMAs add +0 and do not change the result
        for (int o = -sp.r[0]; o <= sp.r[0]; ++o) sp.txy.gx[o + sp.rxy_c] = sp.taps[0].g[o + sp.r[0]];
        for (int o = -sp.r[1]; o <= sp.r[1]; ++o) sp.txy.gy[o + sp.rxy_c] = sp.taps[1].g[o + sp.r[1]];
        sp.tz.r = sp.rz_c;
        for (int o = -sp.r[2]; o <= sp.r[2]; ++o) sp.tz.g[o + sp.rz_c + pgsf::kTapPad] = sp.taps[2].g[o + sp.r[2]];
        for (int o = -sp.r[0]; o <= sp.r[0]; ++o) sp.txy_box.gx[o + sp.rxy_c] = 1.f;
        for (int o = -sp.r[1]; o <= sp.r[1]; ++o) sp.txy_box.gy[o + sp.rxy_c] = 1.f;
        sp.tz_box.r = sp.rz_c;
        for (int o = -sp.r[2]; o <= sp.r[2]; ++o) sp.tz_box.g[o + sp.rz_c + pgsf::kTapPad] = 1.f;
    }
    p->fast_filter = fast;
    p->fast_stats = !force_generic && grid_ok && pgsf::fast_stats_supported(p, &p->why_stats);
    if (force_generic) p->why_stats = "PGSF_FLAG_FORCE_GENERIC";
    else if (!grid_ok) p->why_stats = "ny or nz above 65535";
    p->host_section_planes = 0;
    p->host_budget = 0;
    p->tune = 0;

    // workspace: [scratch filtered cube][filter temporaries][statistics temporaries]
    p->ws_cube_bytes = round256((size_t)p->dims.cube * sizeof(float));
    // Batches: the fast path of pgsf_find_multiscale runs `group` cubes per launch (the kernels of one
    // 60-M-voxel sub-cube do not fill the machine), bounded by 2^32 voxels and by grid.z <= 65535 planes.
    p->group = 1;
    if (p->fast_filter && p->fast_stats && desc->batch > 1) {
        long long g = (1LL << 32) / p->dims.cube;
        if (g > 65535 / desc->nz) g = 65535 / desc->nz;
        if (g > desc->batch) g = desc->batch;
        p->group = g < 1 ? 1 : (int)g;
    }
    p->group_max = p->group;
    if (!dry) {
        cudaError_t e = cudaSetDevice(device);
        // constant block: [0] the pivot, bytes 64.. zeros (k_xyb's source for columns outside the cube), bytes 1024.. the
        // partial sums of the pivot reduction
        if (e == cudaSuccess) e = cudaMalloc(&p->d_pivot, 4096);
        if (e == cudaSuccess) e = cudaMemset(p->d_pivot, 0, 4096);
        if (e != cudaSuccess) {
            cudaGetLastError();
            delete p;
            return fail(nullptr, PGSF_ERR_OOM, "plan constants: %s", cudaGetErrorString(e));
        }
    }
    if (!dry && (desc->flags & PGSF_FLAG_TENSOR_ZPASS) && p->fast_filter && p->fast_stats) {
        const cudaError_t e = pgsf::ztc_prepare(p);
        if (e != cudaSuccess) {
            cudaGetLastError();
            pgsf::ztc_release(p);
            cudaFree(p->d_pivot);
            delete p;
            return fail(nullptr, PGSF_ERR_OOM, "tensor-core operands: %s", cudaGetErrorString(e));
        }
        p->tensor_z = true;
    }
    const size_t cubes = 1 + (p->fast_filter ? (size_t)p->group : 2) + (p->fast_stats ? 2 * (size_t)p->group : 4);
    p->ws_bytes = cubes * p->ws_cube_bytes;
    *out = p;
    return PGSF_OK;
}

pgsf_status pgsf_plan_destroy(pgsf_plan *p)
{
    if (!p) return PGSF_OK;
    if (!p->dry) {
        cudaSetDevice(p->device);      // (events, streams and staging buffers belong to the plan's device)
        pgsf::host_release(p);
        pgsf::ztc_release(p);
        cudaFree(p->d_pivot);
        for (auto &r : p->prof_recs) { cudaEventDestroy(r.a); cudaEventDestroy(r.b); }
        for (auto e : p->prof_free) cudaEventDestroy(e);
        cudaGetLastError();
    }
    delete p;
    return PGSF_OK;
}

pgsf_status pgsf_plan_set_option(pgsf_plan *p, int option, long long value)
{
    if (!p) return PGSF_ERR_INVALID_ARG;
    switch (option) {
    case PGSF_OPT_GROUP_CUBES:
        if (value < 1 || value > p->group_max)
            return fail(p, PGSF_ERR_INVALID_ARG, "PGSF_OPT_GROUP_CUBES must be in 1..%d", p->group_max);
        p->group = (int)value;
        return PGSF_OK;
    case PGSF_OPT_HOST_SECTION_PLANES:
        if (value < 0 || value > p->desc.nz)
            return fail(p, PGSF_ERR_INVALID_ARG, "PGSF_OPT_HOST_SECTION_PLANES must be in 0..nz");
        if (value != p->host_section_planes && !p->dry) { cudaSetDevice(p->device); pgsf::host_release(p); }
        p->host_section_planes = value;
        return PGSF_OK;
    case PGSF_OPT_HOST_DEVICE_BUDGET:
        if (value < 0) return fail(p, PGSF_ERR_INVALID_ARG, "PGSF_OPT_HOST_DEVICE_BUDGET must be >= 0");
        if (value != p->host_budget && !p->dry) { cudaSetDevice(p->device); pgsf::host_release(p); }
        p->host_budget = value;
        return PGSF_OK;
    case PGSF_OPT_TUNE:
        if (value < 0 || value > 0xffff) return fail(p, PGSF_ERR_INVALID_ARG, "PGSF_OPT_TUNE must be in 0..65535");
        p->tune = (int)value;
        return PGSF_OK;
    default:
        return fail(p, PGSF_ERR_INVALID_ARG, "unknown option %d", option);
    }
}

int pgsf_plan_path(const pgsf_plan *p, char *text, int cap)
{
    if (!p || !text || cap < 1) return -1;
    const bool tiled = p->fast_filter && p->fast_stats;
    snprintf(text, (size_t)cap, "filter: %s%s%s; stats: %s%s%s",
             p->fast_filter ? (p->tensor_z ? "tiled (k_xym + k_z / k_zm, k_ztc on the tensor cores for z radii >= 13)" : "tiled (k_xym + k_z / k_zm)")
                            : "generic (k_conv1d) because ", p->fast_filter ? "" : p->why_filter.c_str(), "",
             p->fast_stats ? (pgsf::stats_sparse_or(p) ? "tiled (k_zm / k_zbox + k_xyb)" : "tiled (k_zm / k_zbox + k_ymarch)")
                           : "generic (k_boxsum + k_threshold) because ",
             p->fast_stats ? "" : p->why_stats.c_str(), "");
    return tiled ? 1 : 0;
}

pgsf_status pgsf_plan_set_profiling(pgsf_plan *p, int enable)
{
    if (!p) return PGSF_ERR_INVALID_ARG;
    for (auto &r : p->prof_recs) { p->prof_free.push_back(r.a); p->prof_free.push_back(r.b); }
    p->prof_recs.clear();
    p->prof_acc.clear();
    p->prof_on = enable != 0;
    return PGSF_OK;
}

pgsf_status pgsf_plan_profile_collect(pgsf_plan *p, int *n_entries)
{
    if (!p || !n_entries) return PGSF_ERR_INVALID_ARG;
    for (auto &r : p->prof_recs) {
        cudaError_t e = cudaEventSynchronize(r.b);
        float ms = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, r.a, r.b);
        if (e != cudaSuccess) return cuda_fail(p, e, "profile collect");
        p->prof_acc[r.name_id].launches += 1;
        p->prof_acc[r.name_id].ms += ms;
        p->prof_free.push_back(r.a);
        p->prof_free.push_back(r.b);
    }
    p->prof_recs.clear();
    *n_entries = (int)p->prof_acc.size();
    return PGSF_OK;
}

pgsf_status pgsf_plan_profile_entry(const pgsf_plan *p, int index, char *name, int cap,
                                    unsigned long long *launches, double *ms_total)
{
    if (!p || index < 0 || index >= (int)p->prof_acc.size() || !name || cap < 1)
        return PGSF_ERR_INVALID_ARG;
    const pgsf::ProfAcc &a = p->prof_acc[index];
    snprintf(name, cap, "%s", a.name.c_str());
    if (launches) *launches = a.launches;
    if (ms_total) *ms_total = a.ms;
    return PGSF_OK;
}

size_t pgsf_plan_workspace_bytes(const pgsf_plan *p) { return p ? p->ws_bytes : 0; }

const char *pgsf_last_error(const pgsf_plan *p) { return p ? p->err.c_str() : g_create_err.c_str(); }

unsigned long long pgsf_plan_launch_count(const pgsf_plan *p) { return p ? p->launches : 0ULL; }

pgsf_status pgsf_plan_get_taps(const pgsf_plan *p, int scale, int axis, float *taps, int cap,
                               int *radius)
{
    if (!p || scale < 0 || scale >= p->desc.n_scales || axis < 0 || axis > 2 || !taps || !radius)
        return PGSF_ERR_INVALID_ARG;
    const int r = p->scales[scale].r[axis];
    *radius = r;
    if (cap < 2 * r + 1) return PGSF_ERR_INVALID_ARG;
    memcpy(taps, p->scales[scale].taps[axis].g, sizeof(float) * (2 * r + 1));
    return PGSF_OK;
}

}  // extern "C"

namespace {

struct Workspace {
    float *scratch;  // 1 cube
    float *ftmp;     // 1 or 2 cubes
    float *stmp;     // 2 or 4 cubes
};

Workspace carve(const pgsf_plan *p, void *ws)
{
    Workspace w;
    char *b = static_cast<char *>(ws);
    w.scratch = reinterpret_cast<float *>(b);
    w.ftmp = reinterpret_cast<float *>(b + p->ws_cube_bytes);
    w.stmp = reinterpret_cast<float *>(b + p->ws_cube_bytes * (1 + (p->fast_filter ? (size_t)p->group_max : 2)));
    return w;
}

pgsf_status check_ws(pgsf_plan *p, void *ws)
{
    if (p->ws_bytes > 0 && ws == nullptr) return fail(p, PGSF_ERR_INVALID_ARG, "d_workspace is NULL");
    if ((reinterpret_cast<uintptr_t>(ws) & 255u) != 0)
        return fail(p, PGSF_ERR_INVALID_ARG, "d_workspace must be 256-byte aligned");
    return PGSF_OK;
}

pgsf_status filter_one(pgsf_plan *p, int scale, const float *in, float *out, const Workspace &w,
                       cudaStream_t st)
{
    cudaError_t e;
    if (p->fast_filter) e = pgsf::fast_filter3d(p, scale, in, out, w.ftmp, st);
    else e = pgsf::generic_filter3d(p, scale, in, out, w.ftmp, w.ftmp + p->ws_cube_bytes / sizeof(float), st);
    if (e != cudaSuccess) return cuda_fail(p, e, "filter launch");
    return PGSF_OK;
}

// statistics + selection of `batch` consecutive cubes starting at f / mask (/ mean / sd)
pgsf_status threshold_batch(pgsf_plan *p, const float *f, uint8_t *mask, int or_into, float *mean,
                            float *sd, unsigned long long *count, int batch, const Workspace &w,
                            cudaStream_t st)
{
    cudaError_t e = cudaSuccess;
    for (int bi = 0; bi < batch && e == cudaSuccess; ++bi) {
        const size_t off = (size_t)bi * p->dims.cube;
        float *m = mean ? mean + off : nullptr, *s = sd ? sd + off : nullptr;
        e = pgsf::compute_pivot(p, f + off, st);
        if (e != cudaSuccess) break;
        if (p->fast_stats) e = pgsf::fast_threshold(p, f + off, mask + off, or_into, m, s, count, w.stmp, st);
        else e = pgsf::generic_threshold(p, f + off, mask + off, or_into, m, s, count, w.stmp, st);
    }
    if (e != cudaSuccess) return cuda_fail(p, e, "threshold launch");
    return PGSF_OK;
}

}  // namespace

extern "C" {

pgsf_status pgsf_filter3d(pgsf_plan *p, int scale, const float *d_in, float *d_out, void *d_ws,
                          void *stream)
{
    if (!p) return PGSF_ERR_INVALID_ARG;
    if (scale < 0 || scale >= p->desc.n_scales) return fail(p, PGSF_ERR_INVALID_ARG, "scale out of range");
    if (!d_in || !d_out) return fail(p, PGSF_ERR_INVALID_ARG, "NULL cube pointer");
    if (!aligned16(d_in) || !aligned16(d_out))
        return fail(p, PGSF_ERR_INVALID_ARG, "cube pointers must be 16-byte aligned");
    const size_t bytes = (size_t)p->dims.cube * p->desc.batch * sizeof(float);
    const char *a = reinterpret_cast<const char *>(d_in), *b = reinterpret_cast<const char *>(d_out);
    if (a < b + bytes && b < a + bytes) return fail(p, PGSF_ERR_INVALID_ARG, "d_out overlaps d_in");
    pgsf_status s = check_ws(p, d_ws);
    if (s != PGSF_OK) return s;
    if (p->dry) return fail(p, PGSF_ERR_CUDA, "PGSF_FLAG_DRY_RUN plan: arguments are valid, but no device is attached");
    cudaError_t e = cudaSetDevice(p->device);
    if (e != cudaSuccess) return cuda_fail(p, e, "cudaSetDevice");
    const Workspace w = carve(p, d_ws);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    for (int bi = 0; bi < p->desc.batch; ++bi) {
        s = filter_one(p, scale, d_in + (size_t)bi * p->dims.cube, d_out + (size_t)bi * p->dims.cube, w, st);
        if (s != PGSF_OK) return s;
    }
    return PGSF_OK;
}

pgsf_status pgsf_filter3d_weighted(pgsf_plan *p, int scale, const float *d_in, const float *d_w, float *d_out,
                                   int mode, void *d_ws, void *stream)
{
    if (!p) return PGSF_ERR_INVALID_ARG;
    if (scale < 0 || scale >= p->desc.n_scales) return fail(p, PGSF_ERR_INVALID_ARG, "scale out of range");
    if (mode != PGSF_WEIGHTED_AS_PRINTED && mode != PGSF_WEIGHTED_NORMALISED)
        return fail(p, PGSF_ERR_INVALID_ARG, "mode must be PGSF_WEIGHTED_AS_PRINTED or PGSF_WEIGHTED_NORMALISED");
    if (!d_in || !d_w || !d_out) return fail(p, PGSF_ERR_INVALID_ARG, "NULL cube pointer");
    if (!aligned16(d_in) || !aligned16(d_w) || !aligned16(d_out))
        return fail(p, PGSF_ERR_INVALID_ARG, "cube pointers must be 16-byte aligned");
    const size_t bytes = (size_t)p->dims.cube * p->desc.batch * sizeof(float);
    const char *o = reinterpret_cast<const char *>(d_out);
    for (const float *src : {d_in, d_w}) {
        const char *a = reinterpret_cast<const char *>(src);
        if (a < o + bytes && o < a + bytes) return fail(p, PGSF_ERR_INVALID_ARG, "d_out overlaps an input");
    }
    pgsf_status s = check_ws(p, d_ws);
    if (s != PGSF_OK) return s;
    if (p->dry) return fail(p, PGSF_ERR_CUDA, "PGSF_FLAG_DRY_RUN plan: arguments are valid, but no device is attached");
    cudaError_t e = cudaSetDevice(p->device);
    if (e != cudaSuccess) return cuda_fail(p, e, "cudaSetDevice");
    const Workspace w = carve(p, d_ws);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    float *den = w.stmp, *tmp = w.stmp + p->dims.cube;      // (the statistics cubes are free here)
    for (int bi = 0; bi < p->desc.batch; ++bi) {
        const size_t off = (size_t)bi * p->dims.cube;
        // numerator: Eq. 2 of the product cube (fast path: the product is formed while the x/y pass stages its input)
        if (p->fast_filter) {
            if ((e = pgsf::fast_filter3d(p, scale, d_in + off, d_out + off, w.ftmp, st, false, d_w + off)) != cudaSuccess)
                return cuda_fail(p, e, "weighted filter launch");
        } else {
            if ((e = pgsf::weighted_mul(p, d_in + off, d_w + off, w.scratch, st)) != cudaSuccess)
                return cuda_fail(p, e, "weighted product launch");
            if ((s = filter_one(p, scale, w.scratch, d_out + off, w, st)) != PGSF_OK) return s;
        }
        // denominator: box sum of w (as printed) or Eq. 2 of w
        if (p->fast_filter) {
            // the filter kernels with all-ones (or the Gaussian) taps; their frequency pass divides d_out in place
            e = pgsf::fast_filter3d(p, scale, d_w + off, den, w.ftmp, st, mode == PGSF_WEIGHTED_AS_PRINTED, nullptr,
                                    d_out + off);
            if (e != cudaSuccess) return cuda_fail(p, e, "weight sum launch");
            continue;
        }
        if (mode == PGSF_WEIGHTED_AS_PRINTED) {
            if ((e = pgsf::weighted_boxsum(p, scale, d_w + off, den, tmp, st)) != cudaSuccess)
                return cuda_fail(p, e, "weight box sum launch");
        } else if ((s = filter_one(p, scale, d_w + off, den, w, st)) != PGSF_OK) {
            return s;
        }
        if ((e = pgsf::weighted_div(p, d_out + off, den, st)) != cudaSuccess) return cuda_fail(p, e, "division launch");
    }
    return PGSF_OK;
}

pgsf_status pgsf_filter3d_direct(pgsf_plan *p, const float *d_filter, int rx, int ry, int rz, const float *d_in,
                                 float *d_out, unsigned flags, void *stream)
{
    if (!p) return PGSF_ERR_INVALID_ARG;
    if (!d_filter || !d_in || !d_out) return fail(p, PGSF_ERR_INVALID_ARG, "NULL pointer");
    if (rx < 0 || ry < 0 || rz < 0) return fail(p, PGSF_ERR_INVALID_ARG, "radii must be >= 0");
    if (flags & ~(unsigned)PGSF_DIRECT_FP64_ACCUM) return fail(p, PGSF_ERR_INVALID_ARG, "unknown flag");
    if (!aligned16(d_in) || !aligned16(d_out) || (reinterpret_cast<uintptr_t>(d_filter) & 3u))
        return fail(p, PGSF_ERR_INVALID_ARG, "cube pointers must be 16-byte, the filter 4-byte aligned");
    const size_t bytes = (size_t)p->dims.cube * p->desc.batch * sizeof(float);
    const char *a = reinterpret_cast<const char *>(d_in), *b = reinterpret_cast<const char *>(d_out);
    if (a < b + bytes && b < a + bytes) return fail(p, PGSF_ERR_INVALID_ARG, "d_out overlaps d_in");
    int smem = 0;
    if (!pgsf::direct_supported(p, rx, ry, rz, &smem))
        return fail(p, PGSF_ERR_UNSUPPORTED, "filter radii (%d, %d, %d) need %d bytes of shared memory or exceed %d",
                    rx, ry, rz, smem, PGSF_MAX_RADIUS);
    if (p->dry) return fail(p, PGSF_ERR_CUDA, "PGSF_FLAG_DRY_RUN plan: arguments are valid, but no device is attached");
    cudaError_t e = cudaSetDevice(p->device);
    if (e != cudaSuccess) return cuda_fail(p, e, "cudaSetDevice");
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    for (int bi = 0; bi < p->desc.batch; ++bi) {
        const size_t off = (size_t)bi * p->dims.cube;
        e = pgsf::direct_filter3d(p, d_filter, rx, ry, rz, d_in + off, d_out + off, (flags & PGSF_DIRECT_FP64_ACCUM) != 0, st);
        if (e != cudaSuccess) return cuda_fail(p, e, "direct filter launch");
    }
    return PGSF_OK;
}

pgsf_status pgsf_local_threshold(pgsf_plan *p, const float *d_f, uint8_t *d_mask, int or_into,
                                 float *d_mean, float *d_std, unsigned long long *d_count, void *d_ws,
                                 void *stream)
{
    if (!p) return PGSF_ERR_INVALID_ARG;
    if (!d_f || !d_mask) return fail(p, PGSF_ERR_INVALID_ARG, "NULL cube or mask pointer");
    if (!aligned16(d_f) || !aligned16(d_mask) || !aligned16(d_mean) || !aligned16(d_std))
        return fail(p, PGSF_ERR_INVALID_ARG, "pointers must be 16-byte aligned");
    if (d_count && (reinterpret_cast<uintptr_t>(d_count) & 7u))
        return fail(p, PGSF_ERR_INVALID_ARG, "d_count must be 8-byte aligned");
    pgsf_status s = check_ws(p, d_ws);
    if (s != PGSF_OK) return s;
    if (p->dry) return fail(p, PGSF_ERR_CUDA, "PGSF_FLAG_DRY_RUN plan: arguments are valid, but no device is attached");
    cudaError_t e = cudaSetDevice(p->device);
    if (e != cudaSuccess) return cuda_fail(p, e, "cudaSetDevice");
    const Workspace w = carve(p, d_ws);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (d_count) {
        e = cudaMemsetAsync(d_count, 0, sizeof(unsigned long long), st);
        if (e != cudaSuccess) return cuda_fail(p, e, "cudaMemsetAsync(count)");
    }
    return threshold_batch(p, d_f, d_mask, or_into, d_mean, d_std, d_count, p->desc.batch, w, st);
}

pgsf_status pgsf_find_multiscale(pgsf_plan *p, const float *d_in, float *const *d_filtered,
                                 uint8_t *d_mask, unsigned long long *d_count, void *d_ws, void *stream)
{
    if (!p) return PGSF_ERR_INVALID_ARG;
    if (!d_in || !d_mask) return fail(p, PGSF_ERR_INVALID_ARG, "NULL cube or mask pointer");
    if (!aligned16(d_in) || !aligned16(d_mask))
        return fail(p, PGSF_ERR_INVALID_ARG, "pointers must be 16-byte aligned");
    if (d_count && (reinterpret_cast<uintptr_t>(d_count) & 7u))
        return fail(p, PGSF_ERR_INVALID_ARG, "d_count must be 8-byte aligned");
    const int S = p->desc.n_scales;
    if (d_filtered)
        for (int s = 0; s < S; ++s)
            if (d_filtered[s] && !aligned16(d_filtered[s]))
                return fail(p, PGSF_ERR_INVALID_ARG, "d_filtered[%d] must be 16-byte aligned", s);
    pgsf_status rc = check_ws(p, d_ws);
    if (rc != PGSF_OK) return rc;
    {
        // the filtered cubes double as scratch (pgsf.h), so every buffer of the call must be disjoint
        static const char *fname[PGSF_MAX_SCALES] = {"d_filtered[0]", "d_filtered[1]", "d_filtered[2]", "d_filtered[3]",
                                                     "d_filtered[4]", "d_filtered[5]", "d_filtered[6]", "d_filtered[7]"};
        const size_t nvox = (size_t)p->dims.cube * p->desc.batch;
        Range r[4 + PGSF_MAX_SCALES];
        int n = 0;
        r[n++] = Range{"d_in", d_in, nvox * sizeof(float)};
        r[n++] = Range{"d_mask", d_mask, nvox};
        r[n++] = Range{"d_count", d_count, sizeof(unsigned long long)};
        r[n++] = Range{"d_workspace", d_ws, p->ws_bytes};
        if (d_filtered)
            for (int s = 0; s < S; ++s) r[n++] = Range{fname[s], d_filtered[s], nvox * sizeof(float)};
        int a = 0, b = 0;
        if (find_overlap(r, n, &a, &b))
            return fail(p, PGSF_ERR_INVALID_ARG, "%s overlaps %s", r[a].name, r[b].name);
    }
    if (p->dry) return fail(p, PGSF_ERR_CUDA, "PGSF_FLAG_DRY_RUN plan: arguments are valid, but no device is attached");
    cudaError_t e = cudaSetDevice(p->device);
    if (e != cudaSuccess) return cuda_fail(p, e, "cudaSetDevice");
    const Workspace w = carve(p, d_ws);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (d_count) {
        e = cudaMemsetAsync(d_count, 0, sizeof(unsigned long long), st);
        if (e != cudaSuccess) return cuda_fail(p, e, "cudaMemsetAsync(count)");
    }
    const int B = p->desc.batch;
    bool all_kept = d_filtered != nullptr;
    for (int s = 0; s < S && all_kept; ++s) all_kept = d_filtered[s] != nullptr;
    if (p->fast_filter && all_kept) {
        // x and y passes of all scales from ONE read of the input; the x/y-filtered cube of scale s
        // is parked in the output cube of scale s+1 (the last one in the workspace), so the z passes
        // run in order s = 0..S-1, each freeing the cube the next one writes to.  Batches go through in
        // groups of p->group cubes per launch.
        int idx[PGSF_MAX_SCALES];
        for (int s = 0; s < S; ++s) idx[s] = s;
        const int G = p->fast_stats ? p->group : 1;
        for (int b0 = 0; b0 < B; b0 += G) {
            const int nb = B - b0 < G ? B - b0 : G;
            const size_t off = (size_t)b0 * p->dims.cube;
            float *park[PGSF_MAX_SCALES];
            for (int s = 0; s < S; ++s) park[s] = (s + 1 < S) ? d_filtered[s + 1] + off : w.ftmp;
            cudaError_t ce = pgsf::fast_xy_multi(p, idx, S, d_in + off, park, nb, st);
            if (ce != cudaSuccess) return cuda_fail(p, ce, "xy filter launch");
            // pivot of the statistics of every scale of this group: the level of the input (the taps sum to 1)
            if (p->fast_stats && (ce = pgsf::compute_pivot(p, d_in + off, st)) != cudaSuccess)
                return cuda_fail(p, ce, "pivot launch");
            for (int s = 0; s < S; ++s) {
                if (p->fast_stats) {
                    // frequency pass and z-direction window sums in one march; then the x/y window sums
                    float *Z1 = w.stmp, *Z2 = w.stmp + (size_t)p->group_max * p->dims.cube;
                    ce = pgsf::fast_zm(p, s, park[s], d_filtered[s] + off, Z1, Z2, nb, st);
                    if (ce != cudaSuccess) return cuda_fail(p, ce, "z filter + window launch");
                    // scales after the first OR into the mask: sparsely where the kernel can (then every scale adds
                    // its newly set voxels to the count), else densely with the count taken by the last scale
                    const bool sparse = pgsf::stats_sparse_or(p);
                    ce = pgsf::fast_threshold_xy(p, d_filtered[s] + off, Z1, Z2, d_mask + off,
                                                 s == 0 ? 0 : (sparse ? 2 : 1), nullptr, nullptr,
                                                 (sparse || s == S - 1) ? d_count : nullptr, nb, st);
                    if (ce != cudaSuccess) return cuda_fail(p, ce, "threshold launch");
                    continue;
                }
                ce = pgsf::fast_z(p, s, park[s], d_filtered[s] + off, st);
                if (ce != cudaSuccess) return cuda_fail(p, ce, "z filter launch");
                rc = threshold_batch(p, d_filtered[s] + off, d_mask + off, s > 0, nullptr, nullptr,
                                     (s == S - 1) ? d_count : nullptr, 1, w, st);
                if (rc != PGSF_OK) return rc;
            }
        }
        return PGSF_OK;
    }
    for (int bi = 0; bi < B; ++bi) {
        const size_t off = (size_t)bi * p->dims.cube;
        for (int s = 0; s < S; ++s) {
            float *f = (d_filtered && d_filtered[s]) ? d_filtered[s] + off : w.scratch;
            if (p->fast_filter && p->fast_stats) {
                // filtered cubes not (all) kept: no room to park the x/y passes of all scales, so one x/y launch
                // per scale; the frequency pass still carries the z-direction window sums
                float *t2[1] = {w.ftmp};
                float *Z1 = w.stmp, *Z2 = w.stmp + (size_t)p->group_max * p->dims.cube;
                cudaError_t ce = s == 0 ? pgsf::compute_pivot(p, d_in + off, st) : cudaSuccess;
                if (ce == cudaSuccess) ce = pgsf::fast_xy_multi(p, &s, 1, d_in + off, t2, 1, st);
                if (ce == cudaSuccess) ce = pgsf::fast_zm(p, s, w.ftmp, f, Z1, Z2, 1, st);
                if (ce == cudaSuccess)
                {
                    const bool sparse = pgsf::stats_sparse_or(p);
                    ce = pgsf::fast_threshold_xy(p, f, Z1, Z2, d_mask + off, s == 0 ? 0 : (sparse ? 2 : 1), nullptr,
                                                 nullptr, (sparse || s == S - 1) ? d_count : nullptr, 1, st);
                }
                if (ce != cudaSuccess) return cuda_fail(p, ce, "filter / threshold launch");
                continue;
            }
            rc = filter_one(p, s, d_in + off, f, w, st);
            if (rc != PGSF_OK) return rc;
            rc = threshold_batch(p, f, d_mask + off, s > 0, nullptr, nullptr, (s == S - 1) ? d_count : nullptr,
                                 1, w, st);
            if (rc != PGSF_OK) return rc;
        }
    }
    return PGSF_OK;
}

pgsf_status pgsf_label_objects(pgsf_plan *p, const uint8_t *d_mask, uint32_t *d_labels, unsigned long long *d_count,
                               void *stream)
{
    if (!p) return PGSF_ERR_INVALID_ARG;
    if (!d_mask || !d_labels) return fail(p, PGSF_ERR_INVALID_ARG, "NULL mask or label pointer");
    if (!aligned16(d_labels)) return fail(p, PGSF_ERR_INVALID_ARG, "d_labels must be 16-byte aligned");
    if (d_count && (reinterpret_cast<uintptr_t>(d_count) & 7u))
        return fail(p, PGSF_ERR_INVALID_ARG, "d_count must be 8-byte aligned");
    if ((unsigned long long)p->dims.cube > 0xfffffffeULL)
        return fail(p, PGSF_ERR_UNSUPPORTED, "a cube of more than 2^32 - 2 voxels cannot be labelled with 32-bit labels");
    {
        const size_t nvox = (size_t)p->dims.cube * p->desc.batch;
        Range r[3] = {{"d_mask", d_mask, nvox}, {"d_labels", d_labels, nvox * sizeof(uint32_t)},
                      {"d_count", d_count, sizeof(unsigned long long)}};
        int a = 0, b = 0;
        if (find_overlap(r, 3, &a, &b)) return fail(p, PGSF_ERR_INVALID_ARG, "%s overlaps %s", r[a].name, r[b].name);
    }
    if (p->dry) return fail(p, PGSF_ERR_CUDA, "PGSF_FLAG_DRY_RUN plan: arguments are valid, but no device is attached");
    cudaError_t e = cudaSetDevice(p->device);
    if (e != cudaSuccess) return cuda_fail(p, e, "cudaSetDevice");
    e = pgsf::label_objects(p, d_mask, d_labels, d_count, static_cast<cudaStream_t>(stream));
    if (e != cudaSuccess) return cuda_fail(p, e, "label launch");
    return PGSF_OK;
}

pgsf_status pgsf_find_multiscale_host(pgsf_plan *p, const float *h_in, float *const *h_filtered,
                                      uint8_t *h_mask, unsigned long long *h_count)
{
    if (!p) return PGSF_ERR_INVALID_ARG;
    if (!h_in || !h_mask) return fail(p, PGSF_ERR_INVALID_ARG, "NULL host pointer");
    if (p->dry) return fail(p, PGSF_ERR_CUDA, "PGSF_FLAG_DRY_RUN plan: arguments are valid, but no device is attached");
    cudaError_t e = cudaSetDevice(p->device);
    if (e != cudaSuccess) return cuda_fail(p, e, "cudaSetDevice");
    {
        // the tiled kernels stream the cube through the device in sections (pgsf_host.cu); other plans stage it whole
        bool handled = false;
        const pgsf_status rs = pgsf::host_streamed(p, h_in, h_filtered, h_mask, h_count, &handled);
        if (handled) return rs;
    }
    const size_t nvox = (size_t)p->dims.cube * p->desc.batch;
    const int S = p->desc.n_scales;
    if (!p->h_d_in) {
        if ((e = cudaStreamCreateWithFlags(&p->h_stream, cudaStreamNonBlocking)) != cudaSuccess) {
            p->h_stream = nullptr;
            return cuda_fail(p, e, "cudaStreamCreate");
        }
        if ((e = cudaMalloc(&p->h_d_in, nvox * sizeof(float))) != cudaSuccess ||
            (e = cudaMalloc(&p->h_d_mask, nvox)) != cudaSuccess ||
            (e = cudaMalloc(&p->h_d_count, sizeof(unsigned long long))) != cudaSuccess ||
            (e = cudaMalloc(&p->h_d_ws, p->ws_bytes ? p->ws_bytes : 256)) != cudaSuccess) {
            pgsf::host_release(p);     // all or nothing: the next call starts from scratch
            return fail(p, PGSF_ERR_OOM, "device staging allocation failed: %s", cudaGetErrorString(e));
        }
    }
    float *dptr[PGSF_MAX_SCALES] = {nullptr};
    if (h_filtered) {
        for (int s = 0; s < S; ++s) {
            if (!h_filtered[s]) continue;
            if (!p->h_d_f[s] && (e = cudaMalloc(&p->h_d_f[s], nvox * sizeof(float))) != cudaSuccess) {
                p->h_d_f[s] = nullptr;
                cudaGetLastError();
                return fail(p, PGSF_ERR_OOM, "device staging allocation failed: %s", cudaGetErrorString(e));
            }
            dptr[s] = p->h_d_f[s];
        }
    }
    cudaStream_t st = p->h_stream;
    if ((e = cudaMemcpyAsync(p->h_d_in, h_in, nvox * sizeof(float), cudaMemcpyHostToDevice, st)) != cudaSuccess)
        return cuda_fail(p, e, "H2D copy");
    pgsf_status rc = pgsf_find_multiscale(p, p->h_d_in, h_filtered ? dptr : nullptr, p->h_d_mask,
                                          p->h_d_count, p->h_d_ws, st);
    if (rc != PGSF_OK) return rc;
    if ((e = cudaMemcpyAsync(h_mask, p->h_d_mask, nvox, cudaMemcpyDeviceToHost, st)) != cudaSuccess)
        return cuda_fail(p, e, "D2H mask copy");
    if (h_filtered)
        for (int s = 0; s < S; ++s)
            if (h_filtered[s] &&
                (e = cudaMemcpyAsync(h_filtered[s], dptr[s], nvox * sizeof(float), cudaMemcpyDeviceToHost, st)) != cudaSuccess)
                return cuda_fail(p, e, "D2H filtered copy");
    unsigned long long cnt = 0;
    if ((e = cudaMemcpyAsync(&cnt, p->h_d_count, sizeof cnt, cudaMemcpyDeviceToHost, st)) != cudaSuccess)
        return cuda_fail(p, e, "D2H count copy");
    if ((e = cudaStreamSynchronize(st)) != cudaSuccess) return cuda_fail(p, e, "stream synchronize");
    if (h_count) *h_count = cnt;
    return PGSF_OK;
}

}  // extern "C"
