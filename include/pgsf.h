/*
 * pgsf.h -- C ABI of the B200-native hot path of the filter-based HI source finder of
 * arXiv 1507.04941 (Westerlund & Harris, "Performance Analysis of GPU-Accelerated Filter-Based
 * Source Finding for HI Spectral Line Image Data").
 *
 * Citations "P:<n>" are line numbers of the paper text; "C-<n>" are the readings
 * listed in DESIGN.md where the paper is silent.
 *
 * What the path computes:
 *   for every Gaussian scale s of a filter bank:
 *     f_s  = 3-D convolution of the cube d with the outer-product Gaussian of sigma_s     (Eq. 2)
 *     m, sd = mean and standard deviation of f_s over a box around every voxel
 *     mask |= f_s > m + k * sd
 *   count = number of set mask voxels.
 *
 * Data layout (C-0): a cube is nx*ny*nz fp32 values, linear index x + nx*(y + ny*z): x (right
 * ascension) is unit stride, z (frequency) is the slowest axis; `batch` cubes follow each other
 * with stride nx*ny*nz.  Masks use the same indexing with one byte per voxel.
 *
 * Ownership: every cube / mask / count / workspace pointer named d_* is a caller-owned DEVICE
 * pointer (e.g. a torch tensor's data_ptr()); h_* are HOST pointers.  The library never frees
 * caller memory, never writes d_in, and allocates only its own small constants (plus, for the
 * *_host entry point, plan-owned staging buffers released by pgsf_plan_destroy).
 *
 * Execution: calls validate on the host, enqueue work on `cuda_stream` (a cudaStream_t passed as
 * void*; NULL = the legacy default stream) and return WITHOUT synchronising; results (including
 * *d_count) are valid once the caller has synchronised the stream.  pgsf_find_multiscale_host is
 * the exception: it synchronises before returning.  One plan must not be used from two threads
 * at once (different plans may).  Every compute call makes the plan's device the calling thread's
 * current CUDA device (cudaSetDevice) and leaves it so.
 *
 * Errors: every call returns a pgsf_status; nothing throws or aborts across the ABI.  The text of
 * the last error of a plan is available from pgsf_last_error().  There is no CPU fallback: on a
 * machine without a CUDA device pgsf_plan_create returns PGSF_ERR_CUDA.
 */
#ifndef PGSF_H
#define PGSF_H

#include <stddef.h>
#include <stdint.h>

#if defined(__GNUC__)
#define PGSF_API __attribute__((visibility("default")))
#else
#define PGSF_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pgsf_plan pgsf_plan; /* opaque host object */

typedef enum {
    PGSF_OK = 0,
    PGSF_ERR_INVALID_ARG = 1, /* null / misaligned pointer, bad extent, scale out of range, ... */
    PGSF_ERR_UNSUPPORTED = 2, /* radius or box above the supported maximum, device not sm_100 */
    PGSF_ERR_OOM = 3,         /* an internal allocation failed */
    PGSF_ERR_CUDA = 4         /* a CUDA runtime call failed; see pgsf_last_error */
} pgsf_status;

/* plan flags */
#define PGSF_FLAG_FORCE_GENERIC 0x1u /* use only the generic (any shape / any radius) kernels */
/* (bit 0x2 is reserved: it was a test aid in an earlier revision, now PGSF_OPT_GROUP_CUBES below) */
#define PGSF_FLAG_DRY_RUN 0x4u       /* plan for inspection only: pgsf_plan_create touches no device (148 SMs are
                                        assumed), so pgsf_plan_path / pgsf_plan_workspace_bytes / the argument
                                        validation of every call can be exercised on a machine without a GPU;
                                        a compute call that passes validation returns PGSF_ERR_CUDA */

#define PGSF_FLAG_TENSOR_ZPASS 0x8u  /* OPTIONAL variant: the frequency pass of pgsf_find_multiscale as a banded-Toeplitz
                                        GEMM on the tensor cores (tcgen05, 3 x TF32 split) for scales whose z radius
                                        is >= 13 (compiled radius 24 and above); same tolerances, different rounding */

#define PGSF_MAX_SCALES 8
#define PGSF_MAX_RADIUS 96 /* largest supported ceil(truncate*sigma) on any axis */
#define PGSF_MAX_BOX_HALF 128

typedef struct {
    int32_t nx, ny, nz;   /* extents of ONE cube INCLUDING any halo; x is unit stride (C-0)       */
    int32_t batch;        /* >= 1 identically shaped cubes, stride nx*ny*nz elements              */
    int32_t halo[3];      /* (x,y,z) voxels next to each face excluded from mask and count (C-11) */
    int32_t n_scales;     /* 1..PGSF_MAX_SCALES                                                   */
    const double *sigmas; /* HOST: n_scales x (sigma_x, sigma_y, sigma_z) in voxels, >= 0;
                             0 = identity along that axis                                         */
    double truncate;      /* radius = ceil(truncate*sigma) (C-2); the paper's configs use 3.0     */
    int32_t box_half[3];  /* (hx,hy,hz) >= 0: statistics window [v-h, v+h] per axis (C-6)         */
    double k;             /* threshold in local-standard-deviation units (C-10); configs use 4.0  */
    uint32_t flags;       /* PGSF_FLAG_*                                                          */
} pgsf_plan_desc;

/*
 * pgsf_plan_create -- host only.  For every scale and axis: r = ceil(truncate*sigma); taps
 * g[o] = exp(-o^2 / (2 sigma^2)) for o = -r..r evaluated in fp64, divided by their fp64 sum
 * (C-1..C-3; the paper only says "Gaussian filters"), rounded to fp32 and uploaded to
 * `device`.  Each batch entry is a standalone cube: input outside it is zero (C-5).
 * Returns INVALID_ARG for nx,ny,nz,batch < 1, n_scales outside 1..PGSF_MAX_SCALES, negative
 * sigma / box_half / halo, 2*halo >= extent, truncate <= 0; UNSUPPORTED for a radius above
 * PGSF_MAX_RADIUS or box_half above PGSF_MAX_BOX_HALF; CUDA if `device` cannot be used.
 * On failure *out is NULL.
 */
PGSF_API pgsf_status pgsf_plan_create(pgsf_plan **out, const pgsf_plan_desc *desc, int device);

/* Releases the plan and everything it owns.  NULL is allowed. */
PGSF_API pgsf_status pgsf_plan_destroy(pgsf_plan *plan);

/*
 * pgsf_plan_set_option -- run-time knobs of a plan (host only; none of them changes a result).
 *   PGSF_OPT_GROUP_CUBES          cubes of a batch that pgsf_find_multiscale takes per launch group; 1 .. the plan's
 *                                 default (as many as fit 2^32 voxels).  A test aid: ragged last groups.
 *   PGSF_OPT_HOST_SECTION_PLANES  pgsf_find_multiscale_host: core planes (channels) per section of the streamed
 *                                 cube ("section = core + halo"); 0 = chosen from the device budget.
 *   PGSF_OPT_HOST_DEVICE_BUDGET   pgsf_find_multiscale_host: bytes of device memory its staging may use;
 *                                 0 = 80 % of the memory free at the first call.
 *   PGSF_OPT_TUNE                 measurement aid, a bit set: 1 = statistics kernel without L2 eviction hints,
 *                                 2 = the previous statistics kernel (k_ymarch) instead of k_xyb (where it exists),
 *                                 4 = cp.async staging of every z-pass slab, 8 = TMA bulk tensor copies for every
 *                                 z-pass slab (default: TMA up to a compiled radius of 24, cp.async above),
 *                                 32 = the 32-column form of the tensor-core z pass (k_ztc) for every radius.
 * INVALID_ARG for an unknown option or a value outside its range.
 */
#define PGSF_OPT_GROUP_CUBES 1
#define PGSF_OPT_HOST_SECTION_PLANES 2
#define PGSF_OPT_HOST_DEVICE_BUDGET 3
#define PGSF_OPT_TUNE 4
PGSF_API pgsf_status pgsf_plan_set_option(pgsf_plan *plan, int option, long long value);

/*
 * The tiled sm_100a kernels take: nx a multiple of 4; x / y radii <= 12 and z radii <= 96 (every scale); statistics
 * box half-width hx in {4, 8, 12, 16} (any hy, hz); ny, nz <= 65535.  Anything else runs the generic kernels.
 *
 * pgsf_plan_path -- which kernels this plan runs, as text ("filter: tiled ...; stats: generic (hx = 5 ...)"),
 * so that a caller can see a shape / radius / box that falls off the tiled sm_100a kernels onto the
 * one-thread-per-voxel generic ones (several times slower, same results).  Writes at most cap bytes (NUL
 * terminated) to HOST `text`; returns 1 if every stage of pgsf_find_multiscale runs tiled kernels, 0 if some
 * stage is generic, -1 for bad arguments.
 */
PGSF_API int pgsf_plan_path(const pgsf_plan *plan, char *text, int cap);

/* Bytes of DEVICE scratch the caller must pass as d_workspace to the calls below (256-byte
 * aligned; may be 0, in which case d_workspace may be NULL).  0 for a NULL plan. */
PGSF_API size_t pgsf_plan_workspace_bytes(const pgsf_plan *plan);

/* Text of the last error recorded on this plan ("" if none).  With plan == NULL: the text of the
 * last pgsf_plan_create failure of the calling thread. */
PGSF_API const char *pgsf_last_error(const pgsf_plan *plan);

/* Copies the fp32 taps the kernels use for (scale, axis) to HOST `taps` (capacity `cap` floats)
 * and the radius to *radius; returns INVALID_ARG if cap < 2*radius+1.  For tests. */
PGSF_API pgsf_status pgsf_plan_get_taps(const pgsf_plan *plan, int scale, int axis, float *taps, int cap,
                               int *radius);

/*
 * pgsf_filter3d -- Eq. 2 with the index ranges of Eq. 3-5 for the Gaussian of
 * scale `scale`, evaluated as three 1-D passes (x, y, z), which is exact for an outer-product
 * filter up to fp32 rounding:
 *     d_out[x,y,z] = sum_ox sum_oy sum_oz d_in[x+ox, y+oy, z+oz] gx[ox] gy[oy] gz[oz],
 * input outside the cube = 0, taps not renormalised at the faces (C-5).  fp32 throughout.
 * d_in, d_out: batch*nx*ny*nz floats, 16-byte aligned, must not overlap.  d_out has the input's
 * full extents.
 */
PGSF_API pgsf_status pgsf_filter3d(pgsf_plan *plan, int scale, const float *d_in, float *d_out,
                          void *d_workspace, void *cuda_stream);

/*
 * pgsf_filter3d_direct -- Eq. 2 (Eq. 3-5) for an ARBITRARY filter by direct summation, the
 * operation of the paper's own kernel:
 *     d_out[x,y,z] = sum_ox sum_oy sum_oz d_in[x+ox, y+oy, z+oz] f[ox][oy][oz],   |ox| <= rx, |oy| <= ry, |oz| <= rz,
 * a correlation as printed (C-4), input outside the cube = 0 (C-5).  d_filter: DEVICE array of
 * (2rz+1)*(2ry+1)*(2rx+1) floats, index (ox+rx) + (2rx+1)*((oy+ry) + (2ry+1)*(oz+rz)) (x fastest, like the
 * cubes).  flags: PGSF_DIRECT_FP64_ACCUM accumulates in double as the paper does; default fp32.
 * Uses only the plan's extents, batch and device (not its scales); needs no workspace.  d_in, d_out as for
 * pgsf_filter3d.  UNSUPPORTED when the staged slab of 64 + 2rz channels x 64 + 2rx columns exceeds shared memory.
 */
#define PGSF_DIRECT_FP64_ACCUM 0x1u
PGSF_API pgsf_status pgsf_filter3d_direct(pgsf_plan *plan, const float *d_filter, int rx, int ry, int rz,
                                          const float *d_in, float *d_out, unsigned flags, void *cuda_stream);

/*
 * pgsf_filter3d_weighted -- Eq. 1, the weighted convolution, for the Gaussian of scale `scale`
 * (reading C-16 of DESIGN.md).  With i = (x+ox, y+oy, z+oz) over the part of the
 * filter support inside the cube:
 *     mode PGSF_WEIGHTED_AS_PRINTED : d_out = sum_o d_in[i] f[o] d_w[i] / sum_o d_w[i]        (the paper's Eq. 1)
 *     mode PGSF_WEIGHTED_NORMALISED : d_out = sum_o d_in[i] f[o] d_w[i] / sum_o f[o] d_w[i]   (w == 1 gives Eq. 2)
 * f[o] = gx[ox] gy[oy] gz[oz]; a zero denominator gives 0.  Both sums are evaluated in their separable form
 * (numerator = Eq. 2 of the product cube d_in * d_w), fp32 throughout.
 * d_in, d_w, d_out: batch*nx*ny*nz floats, 16-byte aligned DEVICE pointers; d_out must overlap neither input.
 * Enqueues on `cuda_stream`, does not synchronise; errors as for pgsf_filter3d.
 */
#define PGSF_WEIGHTED_AS_PRINTED 0
#define PGSF_WEIGHTED_NORMALISED 1
PGSF_API pgsf_status pgsf_filter3d_weighted(pgsf_plan *plan, int scale, const float *d_in, const float *d_w,
                                            float *d_out, int mode, void *d_workspace, void *cuda_stream);


/*
 * pgsf_local_threshold -- local statistics and voxel selection of one
 * filtered cube, with the plan's box_half, k and halo:
 *     S1 = sum of f, S2 = sum of f^2 over the box [v-h, v+h] clipped to the cube (C-7), n = its
 *     voxel count; m = S1/n; var = max(S2/n - m^2, 0) (population, C-8); t = m + k*sqrt(var);
 *     sel = f > t (strict, one-sided, C-10), forced to 0 within `halo` of a face (C-11).
 * d_mask (uint8, same indexing): or_into == 0 -> mask = sel; or_into != 0 -> mask |= sel.
 * d_mean / d_std (nullable): fp32 m and sqrt(var) for every voxel (parity aid).
 * d_count (nullable): receives the number of non-zero bytes of the RESULTING mask (after the OR,
 * outside the halo) (C-15).
 */
PGSF_API pgsf_status pgsf_local_threshold(pgsf_plan *plan, const float *d_filtered, uint8_t *d_mask,
                                 int or_into, float *d_mean, float *d_std,
                                 unsigned long long *d_count, void *d_workspace, void *cuda_stream);

/*
 * pgsf_find_multiscale -- the whole hot path: for every scale of the plan, filter
 * d_in, threshold, OR into d_mask; *d_count = set voxels of the final mask.
 * d_filtered: HOST array of n_scales DEVICE pointers receiving the filtered cubes, or NULL /
 * NULL entries = do not keep (the workspace then holds one scratch cube).  The cubes of d_filtered are used
 * as scratch before they hold their final content (the x/y-filtered data of scale s+1 is parked in
 * d_filtered[s+1] while scale s runs), so d_in, d_mask, d_count, the workspace and every d_filtered[s] must
 * be mutually disjoint: INVALID_ARG otherwise.
 */
PGSF_API pgsf_status pgsf_find_multiscale(pgsf_plan *plan, const float *d_in, float *const *d_filtered,
                                 uint8_t *d_mask, unsigned long long *d_count, void *d_workspace,
                                 void *cuda_stream);

/*
 * pgsf_find_multiscale_host -- same result (bit for bit) from HOST buffers, with plan-owned device
 * staging (allocated on first use, released by pgsf_plan_destroy or by a change of the two host options).
 * Plans that run the tiled kernels stream the cube through the device in sections along the frequency axis
 * (the paper's "section = core + halo", Fig. 1 -- but with the copy in of section i+1 and the copy
 * out of section i-1 under the compute of section i, every input plane copied once, nothing recomputed at the
 * seams), so a cube larger than the device memory (or than PGSF_OPT_HOST_DEVICE_BUDGET) still runs; other plans
 * copy the whole cube in, run pgsf_find_multiscale and copy the results out.  Writes the mask (and, when
 * h_filtered != NULL, the filtered cubes: n_scales host pointers, NULL entries skipped) and *h_count, and
 * synchronises.  Page-locked host memory makes the copies asynchronous (and overlapped) but is not required.
 * OOM if the smallest possible sections do not fit the budget.
 */
PGSF_API pgsf_status pgsf_find_multiscale_host(pgsf_plan *plan, const float *h_in, float *const *h_filtered,
                                      uint8_t *h_mask, unsigned long long *h_count);

/*
 * pgsf_label_objects -- NEXT-4: the selected voxels merged into candidate OBJECTS.  The paper combines the voxels it
 * selects into sources of "a single, parameterised catalogue" without defining the merge; reading C-19:
 * an object is a connected component of the mask under 26-connectivity (voxels that touch by a face, an edge or a
 * corner), every cube of the batch on its own.
 * d_mask: the mask of pgsf_find_multiscale / pgsf_local_threshold (any non-zero byte = set), never written.
 * d_labels: DEVICE, one uint32 per voxel (16-byte aligned, disjoint from d_mask): 0 for background, else
 *   1 + the smallest linear index x + nx*(y + ny*z) (inside its cube) of the voxels of the component -- a unique
 *   labelling.  d_count (nullable, 8-byte aligned): the number of objects of all cubes.
 * INVALID_ARG for NULL / misaligned / overlapping buffers; UNSUPPORTED if one cube has more than 2^32 - 2 voxels.
 */
PGSF_API pgsf_status pgsf_label_objects(pgsf_plan *plan, const uint8_t *d_mask, uint32_t *d_labels,
                               unsigned long long *d_count, void *cuda_stream);

/*
 * pgsf_filter3d_noalloc -- pgsf_filter3d (Eq. 2; Eq. 3-5; readings C-1 .. C-5) of ONE cube for callers
 * that cannot allocate device memory: code under CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc.  No plan, no workspace: the two intermediate cubes of the three 1-D passes live in a static device
 * array of 2 x PGSF_NOALLOC_MAX_VOXELS floats (16 MiB, held by every GPU that loads the library until the process
 * exits).  The call makes no cudaMalloc / cudaFree and calls no allocating library routine; it runs the arithmetic
 * of the generic kernels on the CURRENT device and enqueues three kernels on `cuda_stream`.
 * d_in, d_out: DEVICE, nx*ny*nz floats (x fastest), 4-byte aligned, must not overlap; caller owned.
 * sigma_xyz: HOST, 3 doubles >= 0; radius = ceil(truncate * sigma) <= PGSF_MAX_RADIUS, taps as pgsf_plan_create.
 * err_text (nullable): HOST buffer of err_cap chars that receives the text of an error ("" on success).
 * Errors: INVALID_ARG (null / misaligned / overlapping pointer, extent < 1, sigma < 0, truncate <= 0); UNSUPPORTED
 * when nx*ny*nz > PGSF_NOALLOC_MAX_VOXELS (the text names both numbers), a radius is above PGSF_MAX_RADIUS or the
 * device is not sm_100; CUDA when a runtime call fails.
 * The scratch is SHARED by every call on a device and keeps the previous call's contents (nothing in it needs to
 * start at zero: every pass writes its whole output before the next one reads it).  Calls whose kernels may overlap
 * on the GPU -- different streams, different host threads -- race on it: serialise them.  The first call on a
 * device looks the array's device address up (cudaGetSymbolAddress); make one call before starting a graph capture.
 */
#define PGSF_NOALLOC_MAX_VOXELS (1 << 21)
PGSF_API pgsf_status pgsf_filter3d_noalloc(const float *d_in, float *d_out, int nx, int ny, int nz,
                                  const double *sigma_xyz, double truncate, void *cuda_stream, char *err_text,
                                  int err_cap);

/* Number of kernels this library has launched on behalf of `plan` since creation (bench.py's
 * gpu_launches evidence). */
PGSF_API unsigned long long pgsf_plan_launch_count(const pgsf_plan *plan);

/*
 * Per-kernel device timing, for bench.py's roofline line.  pgsf_plan_set_profiling(plan, 1) clears
 * the table and makes every later launch of this plan be bracketed by a cudaEvent pair recorded on
 * the stream the kernel is launched on; 0 switches it off.  pgsf_plan_profile_collect waits for the
 * pending events (it synchronises with those launches), adds their durations to the per-kernel-name
 * totals and writes the number of names to *n_entries; pgsf_plan_profile_entry copies entry
 * `index`: its name (NUL terminated, at most cap bytes), launch count and summed milliseconds.
 */
PGSF_API pgsf_status pgsf_plan_set_profiling(pgsf_plan *plan, int enable);
PGSF_API pgsf_status pgsf_plan_profile_collect(pgsf_plan *plan, int *n_entries);
PGSF_API pgsf_status pgsf_plan_profile_entry(const pgsf_plan *plan, int index, char *name, int cap,
                                             unsigned long long *launches, double *ms_total);

#ifdef __cplusplus
}
#endif
#endif /* PGSF_H */
