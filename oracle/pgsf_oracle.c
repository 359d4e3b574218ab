/*
 * pgsf_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, fp64 CPU oracle for the hot path of arXiv 1507.04941 (Westerlund & Harris):
 * multi-scale 3D Gaussian filtering of an fp32 cube followed by the local mean / standard
 * deviation threshold.  Written from /root/reference/PAPER.md ("P:<line>") and the readings
 * C-0..C-15 listed in DESIGN.md.  It shares NO code with the CUDA path: only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call it.
 *
 * Two levels:
 *   L0 "definition": the formulas written out as printed -- direct six-deep loop for Eq. 2
 *       (index ranges Eq. 3-5) and a brute-force scan of every voxel's window for
 *       the local statistics.  Tiny cubes only.
 *   L1 "plain separable": three 1-D gather passes (x, then y, then z) and the "three directional
 *       sums" of P:152 (per-line fp64 prefix sums), with a region mode so that bricks of an
 *       8 GiB cube can be checked.  L1 is pinned to L0 in tests/test_oracle_pins.py.
 *
 * Memory order (reading C-0): linear index = x + nx*(y + ny*z); x is unit stride.
 * All accumulation is double.  Input cubes are float (the paper stores fp32).
 *
 * Also here: Eq. 1, the weighted convolution (NEXT-1 of SURVEY.md 8(f)), at both levels, and Eq. 2
 * for an arbitrary non-separable filter array (NEXT-2).
 *
 * Pins: tests/test_oracle_pins.py (S1-S15, W1-W6, G1-G3 and L1-L4 of DESIGN.md).  Nothing here is "parity unpinned"
 * except agreement with the authors' own PGSF output on their simulated cube, which is not
 * available (no code, no data).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef int64_t i64;

/* ---------------------------------------------------------------- threads (for the timed baseline) */
int pgsf_oracle_set_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
    return omp_get_max_threads();
#else
    (void)n;
    return 1;
#endif
}

/* ---------------------------------------------------------------- taps (C-1, C-2, C-3) */

/* Radius r = ceil(truncate * sigma), evaluated in fp64; sigma <= 0 -> r = 0 (identity axis).
 * Eq. 3-5 give o in [-F/2, F/2]; F = 2r+1, F/2 in integer division = r. */
int pgsf_oracle_radius(double sigma, double truncate)
{
    if (!(sigma > 0.0)) return 0;
    return (int)ceil(truncate * sigma);
}

/* g[o + r] = exp(-o^2 / (2 sigma^2)) / sum, o = -r..r: a point-sampled Gaussian ("Gaussian
 * filters"), truncated at r and renormalised to sum 1 (BASELINE.json configs[0]). */
void pgsf_oracle_taps(double sigma, int r, double *g)
{
    if (r == 0 || !(sigma > 0.0)) {
        for (int o = -r; o <= r; ++o) g[o + r] = (o == 0) ? 1.0 : 0.0;
        return;
    }
    double sum = 0.0;
    for (int o = -r; o <= r; ++o) {
        g[o + r] = exp(-((double)o * (double)o) / (2.0 * sigma * sigma));
        sum += g[o + r];
    }
    for (int o = -r; o <= r; ++o) g[o + r] /= sum;
}

/* ---------------------------------------------------------------- L0: the definitions */

/* Eq. 2 with the ranges of Eq. 3-5, f[ox][oy][oz] = gx[ox]*gy[oy]*gz[oz]
 * (outer-product Gaussian), input outside the cube = 0 (C-5), taps NOT renormalised at edges.
 *   c_u[x][y][z] = sum_ox sum_oy sum_oz d[x+ox][y+oy][z+oz] * f[ox][oy][oz]                    */
void pgsf_oracle_filter_direct(const float *d, int nx, int ny, int nz,
                               const double *gx, int rx, const double *gy, int ry,
                               const double *gz, int rz, double *c)
{
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                double sum = 0.0;
                for (int oz = -rz; oz <= rz; ++oz) {
                    int iz = z + oz;
                    if (iz < 0 || iz >= nz) continue;
                    for (int oy = -ry; oy <= ry; ++oy) {
                        int iy = y + oy;
                        if (iy < 0 || iy >= ny) continue;
                        for (int ox = -rx; ox <= rx; ++ox) {
                            int ix = x + ox;
                            if (ix < 0 || ix >= nx) continue;
                            double f = gx[ox + rx] * gy[oy + ry] * gz[oz + rz];
                            sum += (double)d[(i64)ix + (i64)nx * ((i64)iy + (i64)ny * iz)] * f;
                        }
                    }
                }
                c[(i64)x + (i64)nx * ((i64)y + (i64)ny * z)] = sum;
            }
}

/* Local statistics by definition ("calculated independently for each voxel from a
 * user-specified range of image data around the voxel": mean and standard deviation give
 * the threshold).  Window = box [x-hx,x+hx] x [y-hy,y+hy] x [z-hz,z+hz] clipped to the cube (C-6,
 * C-7), centre included; population variance clamped at 0 (C-8); t = m + k*sd; mask = c > t,
 * strict (C-10). */
void pgsf_oracle_threshold_brute(const double *c, int nx, int ny, int nz,
                                 int hx, int hy, int hz, double k,
                                 double *mean, double *sd, double *thr, uint8_t *mask)
{
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                double s1 = 0.0, s2 = 0.0;
                i64 n = 0;
                for (int wz = z - hz; wz <= z + hz; ++wz) {
                    if (wz < 0 || wz >= nz) continue;
                    for (int wy = y - hy; wy <= y + hy; ++wy) {
                        if (wy < 0 || wy >= ny) continue;
                        for (int wx = x - hx; wx <= x + hx; ++wx) {
                            if (wx < 0 || wx >= nx) continue;
                            double v = c[(i64)wx + (i64)nx * ((i64)wy + (i64)ny * wz)];
                            s1 += v;
                            s2 += v * v;
                            n += 1;
                        }
                    }
                }
                double m = s1 / (double)n;
                double var = s2 / (double)n - m * m;
                if (var < 0.0) var = 0.0;
                double s = sqrt(var);
                double t = m + k * s;
                i64 i = (i64)x + (i64)nx * ((i64)y + (i64)ny * z);
                if (mean) mean[i] = m;
                if (sd) sd[i] = s;
                if (thr) thr[i] = t;
                if (mask) mask[i] = (c[i] > t) ? 1 : 0;
            }
}

/* ---------------------------------------------------------------- L1: plain separable, region mode */

static int imax(int a, int b) { return a > b ? a : b; }
static int imin(int a, int b) { return a < b ? a : b; }

/*
 * Separable form of Eq. 2 for an outer-product filter: t1 = x-pass of d, t2 = y-pass of t1,
 * c = z-pass of t2, each a plain gather loop in fp64, zero outside the CUBE (C-5).
 *
 * Region mode: `sub` holds the input for cube coordinates [slo, shi) (x fastest); the output is
 * produced for [lo, hi) only, written densely (x fastest) to `out`.  Reads falling inside the
 * cube but outside `sub` are an error (return -1): the caller must supply the brick +- radius,
 * clipped to the cube.  cube = {nx, ny, nz}.
 */
int pgsf_oracle_filter_region(const float *sub, const int *slo, const int *shi, const int *cube,
                              const double *gx, int rx, const double *gy, int ry,
                              const double *gz, int rz,
                              const int *lo, const int *hi, double *out)
{
    const int nx = cube[0], ny = cube[1], nz = cube[2];
    /* extents of the intermediate passes, clipped to the cube */
    const int ylo = imax(0, lo[1] - ry), yhi = imin(ny, hi[1] + ry);
    const int zlo = imax(0, lo[2] - rz), zhi = imin(nz, hi[2] + rz);
    const int xlo_in = imax(0, lo[0] - rx), xhi_in = imin(nx, hi[0] + rx);
    if (xlo_in < slo[0] || xhi_in > shi[0] || ylo < slo[1] || yhi > shi[1] || zlo < slo[2] ||
        zhi > shi[2])
        return -1;
    const i64 snx = shi[0] - slo[0], sny = shi[1] - slo[1];
    const i64 wx = hi[0] - lo[0], wy = hi[1] - lo[1], wz = hi[2] - lo[2];
    const i64 t1y = yhi - ylo, tz = zhi - zlo;
    double *t1 = (double *)malloc(sizeof(double) * (size_t)(wx * t1y * tz));
    double *t2 = (double *)malloc(sizeof(double) * (size_t)(wx * wy * tz));
    if (!t1 || !t2) { free(t1); free(t2); return -2; }

    /* x-pass: t1[x,y,z] = sum_o d[x+o,y,z] gx[o]   (Eq. 2 with Eq. 3) */
#pragma omp parallel for schedule(static)
    for (int z = zlo; z < zhi; ++z)
        for (int y = ylo; y < yhi; ++y)
            for (int x = lo[0]; x < hi[0]; ++x) {
                double s = 0.0;
                for (int o = -rx; o <= rx; ++o) {
                    int ix = x + o;
                    if (ix < 0 || ix >= nx) continue;
                    s += (double)sub[(ix - slo[0]) + snx * ((i64)(y - slo[1]) + sny * (z - slo[2]))] *
                         gx[o + rx];
                }
                t1[(x - lo[0]) + wx * ((i64)(y - ylo) + t1y * (z - zlo))] = s;
            }
    /* y-pass: t2[x,y,z] = sum_o t1[x,y+o,z] gy[o]   (Eq. 4) */
#pragma omp parallel for schedule(static)
    for (int z = zlo; z < zhi; ++z)
        for (int y = lo[1]; y < hi[1]; ++y)
            for (int x = lo[0]; x < hi[0]; ++x) {
                double s = 0.0;
                for (int o = -ry; o <= ry; ++o) {
                    int iy = y + o;
                    if (iy < 0 || iy >= ny) continue;
                    s += t1[(x - lo[0]) + wx * ((i64)(iy - ylo) + t1y * (z - zlo))] * gy[o + ry];
                }
                t2[(x - lo[0]) + wx * ((i64)(y - lo[1]) + wy * (z - zlo))] = s;
            }
    /* z-pass: c[x,y,z] = sum_o t2[x,y,z+o] gz[o]   (Eq. 5) */
#pragma omp parallel for schedule(static)
    for (int z = lo[2]; z < hi[2]; ++z)
        for (int y = lo[1]; y < hi[1]; ++y)
            for (int x = lo[0]; x < hi[0]; ++x) {
                double s = 0.0;
                for (int o = -rz; o <= rz; ++o) {
                    int iz = z + o;
                    if (iz < 0 || iz >= nz) continue;
                    s += t2[(x - lo[0]) + wx * ((i64)(y - lo[1]) + wy * (iz - zlo))] * gz[o + rz];
                }
                out[(x - lo[0]) + wx * ((i64)(y - lo[1]) + wy * (z - lo[2]))] = s;
            }
    (void)wz;
    free(t1);
    free(t2);
    return 0;
}

/*
 * Local mean / sd / threshold / mask on a region, as the "three directional sums" of P:152:
 * sums of c and c^2 along x, then y, then z over the window clipped to the CUBE (C-7), each by a
 * per-line fp64 prefix sum; n = product of the per-axis clipped window lengths.
 *
 * `csub` holds the filtered data for cube coordinates [clo, chi); it must cover [lo,hi) +- h
 * clipped to the cube (else return -1).  Outputs (any may be NULL) are dense over [lo, hi).
 */
int pgsf_oracle_threshold_region(const double *csub, const int *clo, const int *chi,
                                 const int *cube, const int *h, double k,
                                 const int *lo, const int *hi,
                                 double *mean, double *sd, double *thr, uint8_t *mask)
{
    const int nx = cube[0], ny = cube[1], nz = cube[2];
    const int hx = h[0], hy = h[1], hz = h[2];
    const int xlo = imax(0, lo[0] - hx), xhi = imin(nx, hi[0] + hx);
    const int ylo = imax(0, lo[1] - hy), yhi = imin(ny, hi[1] + hy);
    const int zlo = imax(0, lo[2] - hz), zhi = imin(nz, hi[2] + hz);
    if (xlo < clo[0] || xhi > chi[0] || ylo < clo[1] || yhi > chi[1] || zlo < clo[2] || zhi > chi[2])
        return -1;
    const i64 cnx = chi[0] - clo[0], cny = chi[1] - clo[1];
    const i64 wx = hi[0] - lo[0], wy = hi[1] - lo[1], wz = hi[2] - lo[2];
    const i64 ay = yhi - ylo, az = zhi - zlo; /* extents of the x-summed arrays */
    /* A1/A2: sums along x for x in [lo,hi), y in [ylo,yhi), z in [zlo,zhi) */
    double *A1 = (double *)malloc(sizeof(double) * (size_t)(wx * ay * az));
    double *A2 = (double *)malloc(sizeof(double) * (size_t)(wx * ay * az));
    /* B1/B2: then along y, for y in [lo,hi) */
    double *B1 = (double *)malloc(sizeof(double) * (size_t)(wx * wy * az));
    double *B2 = (double *)malloc(sizeof(double) * (size_t)(wx * wy * az));
    if (!A1 || !A2 || !B1 || !B2) { free(A1); free(A2); free(B1); free(B2); return -2; }

    /* directional sum 1: along x */
#pragma omp parallel
    {
        double *p1 = (double *)malloc(sizeof(double) * (size_t)(xhi - xlo + 1));
        double *p2 = (double *)malloc(sizeof(double) * (size_t)(xhi - xlo + 1));
#pragma omp for schedule(static)
        for (int z = zlo; z < zhi; ++z)
            for (int y = ylo; y < yhi; ++y) {
                const double *line = csub + (cnx * ((i64)(y - clo[1]) + cny * (z - clo[2])) - clo[0]);
                p1[0] = 0.0; p2[0] = 0.0;
                for (int x = xlo; x < xhi; ++x) {
                    double v = line[x];
                    p1[x - xlo + 1] = p1[x - xlo] + v;
                    p2[x - xlo + 1] = p2[x - xlo] + v * v;
                }
                for (int x = lo[0]; x < hi[0]; ++x) {
                    int a = imax(0, x - hx), b = imin(nx - 1, x + hx);
                    i64 o = (x - lo[0]) + wx * ((i64)(y - ylo) + ay * (z - zlo));
                    A1[o] = p1[b + 1 - xlo] - p1[a - xlo];
                    A2[o] = p2[b + 1 - xlo] - p2[a - xlo];
                }
            }
        free(p1); free(p2);
    }
    /* directional sum 2: along y */
#pragma omp parallel
    {
        double *p1 = (double *)malloc(sizeof(double) * (size_t)(ay + 1));
        double *p2 = (double *)malloc(sizeof(double) * (size_t)(ay + 1));
#pragma omp for schedule(static)
        for (int z = zlo; z < zhi; ++z)
            for (int x = lo[0]; x < hi[0]; ++x) {
                p1[0] = 0.0; p2[0] = 0.0;
                for (int y = ylo; y < yhi; ++y) {
                    i64 o = (x - lo[0]) + wx * ((i64)(y - ylo) + ay * (z - zlo));
                    p1[y - ylo + 1] = p1[y - ylo] + A1[o];
                    p2[y - ylo + 1] = p2[y - ylo] + A2[o];
                }
                for (int y = lo[1]; y < hi[1]; ++y) {
                    int a = imax(0, y - hy), b = imin(ny - 1, y + hy);
                    i64 o = (x - lo[0]) + wx * ((i64)(y - lo[1]) + wy * (z - zlo));
                    B1[o] = p1[b + 1 - ylo] - p1[a - ylo];
                    B2[o] = p2[b + 1 - ylo] - p2[a - ylo];
                }
            }
        free(p1); free(p2);
    }
    /* directional sum 3: along z, then the z-score / threshold */
#pragma omp parallel
    {
        double *p1 = (double *)malloc(sizeof(double) * (size_t)(az + 1));
        double *p2 = (double *)malloc(sizeof(double) * (size_t)(az + 1));
#pragma omp for schedule(static)
        for (int y = lo[1]; y < hi[1]; ++y)
            for (int x = lo[0]; x < hi[0]; ++x) {
                p1[0] = 0.0; p2[0] = 0.0;
                for (int z = zlo; z < zhi; ++z) {
                    i64 o = (x - lo[0]) + wx * ((i64)(y - lo[1]) + wy * (z - zlo));
                    p1[z - zlo + 1] = p1[z - zlo] + B1[o];
                    p2[z - zlo + 1] = p2[z - zlo] + B2[o];
                }
                const int xa = imax(0, x - hx), xb = imin(nx - 1, x + hx);
                const int ya = imax(0, y - hy), yb = imin(ny - 1, y + hy);
                for (int z = lo[2]; z < hi[2]; ++z) {
                    int a = imax(0, z - hz), b = imin(nz - 1, z + hz);
                    double s1 = p1[b + 1 - zlo] - p1[a - zlo];
                    double s2 = p2[b + 1 - zlo] - p2[a - zlo];
                    double n = (double)(xb - xa + 1) * (double)(yb - ya + 1) * (double)(b - a + 1);
                    double m = s1 / n;
                    double var = s2 / n - m * m;
                    if (var < 0.0) var = 0.0;
                    double s = sqrt(var);
                    double t = m + k * s;
                    i64 o = (x - lo[0]) + wx * ((i64)(y - lo[1]) + wy * (z - lo[2]));
                    double cv = csub[(x - clo[0]) + cnx * ((i64)(y - clo[1]) + cny * (z - clo[2]))];
                    if (mean) mean[o] = m;
                    if (sd) sd[o] = s;
                    if (thr) thr[o] = t;
                    if (mask) mask[o] = (cv > t) ? 1 : 0;
                }
            }
        free(p1); free(p2);
    }
    (void)wz;
    free(A1); free(A2); free(B1); free(B2);
    return 0;
}

/* ---------------------------------------------------------------- weighted convolution (Eq. 1) */

/*
 * Eq. 1 as printed, with i = (x+ox, y+oy, z+oz) running over the filter support inside the cube:
 *
 *      c_w[x][y][z] =  sum_o d[i] f[o] w[i]  /  sum_o w[i]
 *
 * (reading C-16 of DESIGN.md).  The printed denominator carries no f: with w == 1 it yields
 * c_u / (number of support voxels), not c_u.  mode 1 is the normalisation by sum_o f[o] w[i] that makes
 * w == 1 reproduce c_u (offered as a flag; the paper prints mode 0).  Positions outside the cube contribute
 * to neither sum (C-5); a zero denominator gives 0.  L0: direct six-deep loops.
 */
void pgsf_oracle_wfilter_direct(const float *d, const float *w, int nx, int ny, int nz,
                                const double *gx, int rx, const double *gy, int ry,
                                const double *gz, int rz, int mode, double *c)
{
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                double num = 0.0, den = 0.0;
                for (int oz = -rz; oz <= rz; ++oz) {
                    int iz = z + oz;
                    if (iz < 0 || iz >= nz) continue;
                    for (int oy = -ry; oy <= ry; ++oy) {
                        int iy = y + oy;
                        if (iy < 0 || iy >= ny) continue;
                        for (int ox = -rx; ox <= rx; ++ox) {
                            int ix = x + ox;
                            if (ix < 0 || ix >= nx) continue;
                            const i64 i = (i64)ix + (i64)nx * ((i64)iy + (i64)ny * iz);
                            const double f = gx[ox + rx] * gy[oy + ry] * gz[oz + rz];
                            num += (double)d[i] * f * (double)w[i];
                            den += mode ? f * (double)w[i] : (double)w[i];
                        }
                    }
                }
                c[(i64)x + (i64)nx * ((i64)y + (i64)ny * z)] = den != 0.0 ? num / den : 0.0;
            }
}

/* one 1-D pass along `axis` over a dense double cube: out[v] = sum_{|o|<=r} in[v + o e_axis] g[o + r]
 * (g == NULL: plain sum, the box of the printed denominator), positions outside the cube skipped */
static void pass1d(const double *in, double *out, int nx, int ny, int nz, int axis, const double *g, int r)
{
    const int n[3] = {nx, ny, nz};
    const i64 stride[3] = {1, nx, (i64)nx * ny};
#pragma omp parallel for schedule(static)
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                const int c[3] = {x, y, z};
                const i64 i = (i64)x + (i64)nx * ((i64)y + (i64)ny * z);
                double s = 0.0;
                for (int o = -r; o <= r; ++o) {
                    const int j = c[axis] + o;
                    if (j < 0 || j >= n[axis]) continue;
                    s += in[i + o * stride[axis]] * (g ? g[o + r] : 1.0);
                }
                out[i] = s;
            }
}

/*
 * L1: Eq. 1 through the separable form.  For an outer-product f the numerator is Eq. 2 applied to the
 * product cube d*w (three 1-D passes, as pgsf_oracle_filter_region); the printed denominator is the sum
 * of w over the box of the support (three 1-D plain sums), the mode-1 denominator Eq. 2 applied to w.
 * Returns 0, or -2 when out of memory.
 */
int pgsf_oracle_wfilter(const float *d, const float *w, int nx, int ny, int nz,
                        const double *gx, int rx, const double *gy, int ry, const double *gz, int rz,
                        int mode, double *c)
{
    const i64 n = (i64)nx * ny * nz;
    double *a = (double *)malloc(sizeof(double) * (size_t)n);
    double *b = (double *)malloc(sizeof(double) * (size_t)n);
    double *den = (double *)malloc(sizeof(double) * (size_t)n);
    if (!a || !b || !den) { free(a); free(b); free(den); return -2; }
    for (i64 i = 0; i < n; ++i) a[i] = (double)d[i] * (double)w[i];
    pass1d(a, b, nx, ny, nz, 0, gx, rx);
    pass1d(b, a, nx, ny, nz, 1, gy, ry);
    pass1d(a, c, nx, ny, nz, 2, gz, rz);          /* numerator in c */
    for (i64 i = 0; i < n; ++i) a[i] = (double)w[i];
    pass1d(a, b, nx, ny, nz, 0, mode ? gx : NULL, rx);
    pass1d(b, a, nx, ny, nz, 1, mode ? gy : NULL, ry);
    pass1d(a, den, nx, ny, nz, 2, mode ? gz : NULL, rz);
    for (i64 i = 0; i < n; ++i) c[i] = den[i] != 0.0 ? c[i] / den[i] : 0.0;
    free(a); free(b); free(den);
    return 0;
}

/* ---------------------------------------------------------------- Eq. 2 for an ARBITRARY filter (NEXT-2) */

/*
 * Eq. 2 with the index ranges of Eq. 3-5 for a general, non-separable filter array
 * f[oz][oy][ox] (x fastest, (2rz+1) x (2ry+1) x (2rx+1) doubles) -- what the paper's own kernel evaluates
 * ("for each X and Y position in the filter ... for each Z position").  As printed it is a
 * correlation, d[x+ox] f[ox] (C-4): the orientation matters once f is not symmetric.  Input outside the
 * cube = 0 (C-5).  fp64 accumulation.
 */
void pgsf_oracle_filter_general(const float *d, int nx, int ny, int nz, const double *f, int rx, int ry, int rz,
                                double *c)
{
    const int fx = 2 * rx + 1, fy = 2 * ry + 1;
#pragma omp parallel for schedule(static)
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                double sum = 0.0;
                for (int oz = -rz; oz <= rz; ++oz) {
                    const int iz = z + oz;
                    if (iz < 0 || iz >= nz) continue;
                    for (int oy = -ry; oy <= ry; ++oy) {
                        const int iy = y + oy;
                        if (iy < 0 || iy >= ny) continue;
                        for (int ox = -rx; ox <= rx; ++ox) {
                            const int ix = x + ox;
                            if (ix < 0 || ix >= nx) continue;
                            sum += (double)d[(i64)ix + (i64)nx * ((i64)iy + (i64)ny * iz)] *
                                   f[(ox + rx) + (i64)fx * ((oy + ry) + (i64)fy * (oz + rz))];
                        }
                    }
                }
                c[(i64)x + (i64)nx * ((i64)y + (i64)ny * z)] = sum;
            }
}

/* ---------------------------------------------------------------- NEXT-4: mask -> candidate objects
 * The paper merges the selected voxels into sources and "combin[es] the results to a single, parameterised
 * catalogue" (the selection step is P:282) without saying how voxels are joined.  Reading C-19: an
 * object is a connected component of the OR mask under 26-connectivity (voxels touching by a face, an edge or a corner
 * belong together), every cube of a batch on its own.  Label of a component = 1 + the smallest linear index
 * x + nx (y + ny z) of its voxels; background = 0.  Plain flood fill in index order, so the first voxel met of a
 * component IS its smallest index.  Returns the number of components. */
i64 pgsf_oracle_label26(const uint8_t *mask, int nx, int ny, int nz, uint32_t *labels)
{
    const i64 n = (i64)nx * ny * nz;
    i64 *stack = (i64 *)malloc(sizeof(i64) * (size_t)(n > 0 ? n : 1));
    i64 count = 0;
    memset(labels, 0, sizeof(uint32_t) * (size_t)n);
    for (i64 i = 0; i < n; ++i) {
        if (!mask[i] || labels[i]) continue;
        const uint32_t lab = (uint32_t)(i + 1);
        i64 top = 0;
        stack[top++] = i;
        labels[i] = lab;
        ++count;
        while (top > 0) {
            const i64 v = stack[--top];
            const int x = (int)(v % nx), y = (int)((v / nx) % ny), z = (int)(v / ((i64)nx * ny));
            for (int dz = -1; dz <= 1; ++dz)
                for (int dy = -1; dy <= 1; ++dy)
                    for (int dx = -1; dx <= 1; ++dx) {
                        const int xx = x + dx, yy = y + dy, zz = z + dz;
                        if (xx < 0 || yy < 0 || zz < 0 || xx >= nx || yy >= ny || zz >= nz) continue;
                        const i64 u = xx + (i64)nx * (yy + (i64)ny * zz);
                        if (mask[u] && !labels[u]) { labels[u] = lab; stack[top++] = u; }
                    }
        }
    }
    free(stack);
    return count;
}
