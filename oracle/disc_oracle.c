/*
 * disc_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * Plain, slow, obviously-correct CPU restatement of the DISC hot path
 * (Zhen et al., "CT to Cone-beam CT Deformable Registration With Simultaneous
 * Intensity Correction", arxiv 1204.6295; citations are PAPER.md:LINE).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may build, load or call this file.  It shares no code, header,
 * table or constant generator with paper_1204_6295_b200/ (the CUDA path) and
 * neither imports the other.
 *
 * Conventions: volumes are float32, x fastest,
 * idx = (z*ny + y)*nx + x; displacement is planar disp[c][z][y][x], c=0,1,2 =
 * x,y,z, in voxel units of its level.  Arithmetic inside a step is fp64; the
 * images m, s' and the field r are rounded to fp32 once, at the end of a step.
 * Patch loops are naive (every voxel visits its whole patch, as the paper's own
 * kernel does); variance is two-pass.  OpenMP over z only.
 *
 * Every function is pinned by tests/test_oracle_pins.py and
 * tests/test_oracle_pins_ext.py (closed forms, invariants, brute force, hand
 * values, scipy special cases) -- no function is "parity unpinned" except
 * registration accuracy on the paper's clinical data, which
 * is not reproducible here and not claimed.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define IDX(x, y, z) (((size_t)(z) * ny + (y)) * nx + (x))

static inline int clampi(int v, int lo, int hi) { return v < lo ? lo : (v > hi ? hi : v); }

int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------------
 * (b) warp: m(x) = I_m(x + r(x)), trilinear, sample position clamped to the
 * volume.  PAPER.md:69 (I_m(x+v(x)) = I_s(x), pull-back), :75 "update the
 * moving image", :171 kernel 5.  Reading A11: p = clamp(x + r, 0, n-1) per
 * axis, i0 = min(floor(p), n-2), t = p - i0; an axis of length 1 has weight 0.
 * ---------------------------------------------------------------------- */
static inline void cell(double p, int n, int *i0, int *i1, double *t) {
    if (p < 0.0) p = 0.0;
    if (p > (double)(n - 1)) p = (double)(n - 1);
    if (n < 2) { *i0 = 0; *i1 = 0; *t = 0.0; return; }
    int i = (int)floor(p);
    if (i > n - 2) i = n - 2;
    *i0 = i; *i1 = i + 1; *t = p - (double)i;
}

static double trilinear(const float *I, int nx, int ny, int nz, double px, double py, double pz) {
    int x0, x1, y0, y1, z0, z1; double tx, ty, tz;
    cell(px, nx, &x0, &x1, &tx); cell(py, ny, &y0, &y1, &ty); cell(pz, nz, &z0, &z1, &tz);
    double c00 = (1 - tx) * I[IDX(x0, y0, z0)] + tx * I[IDX(x1, y0, z0)];
    double c10 = (1 - tx) * I[IDX(x0, y1, z0)] + tx * I[IDX(x1, y1, z0)];
    double c01 = (1 - tx) * I[IDX(x0, y0, z1)] + tx * I[IDX(x1, y0, z1)];
    double c11 = (1 - tx) * I[IDX(x0, y1, z1)] + tx * I[IDX(x1, y1, z1)];
    double c0 = (1 - ty) * c00 + ty * c10;
    double c1 = (1 - ty) * c01 + ty * c11;
    return (1 - tz) * c0 + tz * c1;
}

void oracle_warp(const float *I, const float *disp, int nx, int ny, int nz, float *out) {
    size_t N = (size_t)nx * ny * nz;
#pragma omp parallel for schedule(static)
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                size_t i = IDX(x, y, z);
                out[i] = (float)trilinear(I, nx, ny, nz, x + (double)disp[i], y + (double)disp[N + i],
                                          z + (double)disp[2 * N + i]);
            }
}

/* ------------------------------------------------------------------------
 * (a1) patch moments.  PAPER.md:95 Eq. (3): E(X^p) = (1/n) sum x_i^p, p=1,2;
 * PAPER.md:458 (A.4): STD = sqrt(E(X^2) - E(X)^2), i.e. population variance.
 * Patch = cube of radius R centred at x, truncated to the
 * volume (reading A4): n(x) = number of in-volume voxels.  Two-pass variance
 * sum (x - mu)^2 / n, which equals E(X^2) - E(X)^2 in exact arithmetic.
 * ---------------------------------------------------------------------- */
static inline void patch_stats3(const float *v, int nx, int ny, int nz, const int R[3], int x, int y, int z,
                                double *mean, double *var) {
    int x0 = x - R[0] < 0 ? 0 : x - R[0], x1 = x + R[0] > nx - 1 ? nx - 1 : x + R[0];
    int y0 = y - R[1] < 0 ? 0 : y - R[1], y1 = y + R[1] > ny - 1 ? ny - 1 : y + R[1];
    int z0 = z - R[2] < 0 ? 0 : z - R[2], z1 = z + R[2] > nz - 1 ? nz - 1 : z + R[2];
    double n = (double)(x1 - x0 + 1) * (y1 - y0 + 1) * (z1 - z0 + 1);
    double s = 0.0;
    for (int c = z0; c <= z1; ++c)
        for (int b = y0; b <= y1; ++b)
            for (int a = x0; a <= x1; ++a) s += v[IDX(a, b, c)];
    double mu = s / n, q = 0.0;
    for (int c = z0; c <= z1; ++c)
        for (int b = y0; b <= y1; ++b)
            for (int a = x0; a <= x1; ++a) { double d = v[IDX(a, b, c)] - mu; q += d * d; }
    *mean = mu; *var = q / n;
}

/* the cubic patch of the hot path: the same radius on every axis */
static inline void patch_stats(const float *v, int nx, int ny, int nz, int R, int x, int y, int z,
                               double *mean, double *var) {
    const int R3[3] = {R, R, R};
    patch_stats3(v, nx, ny, nz, R3, x, y, z, mean, var);
}

void oracle_box_moments(const float *v, int nx, int ny, int nz, int R, double *mean, double *var) {
#pragma omp parallel for schedule(dynamic, 1)
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) patch_stats(v, nx, ny, nz, R, x, y, z, &mean[IDX(x, y, z)], &var[IDX(x, y, z)]);
}

/* moments at a list of voxel indices only (sampled checks at sizes where the full loop takes minutes) */
void oracle_box_moments_at(const float *v, int nx, int ny, int nz, int R, const long long *idx, int nidx,
                           double *mean, double *var) {
#pragma omp parallel for schedule(dynamic, 16)
    for (int k = 0; k < nidx; ++k) {
        long long i = idx[k];
        int x = (int)(i % nx), y = (int)((i / nx) % ny), z = (int)(i / ((long long)nx * ny));
        patch_stats(v, nx, ny, nz, R, x, y, z, &mean[k], &var[k]);
    }
}

/* ------------------------------------------------------------------------
 * (a2) correction.  PAPER.md:117-119 Eqs. (5)-(6): a = STD(M)/STD(S),
 * b = E(M) - a E(S); I'_s = a I_s + b applied to the ORIGINAL
 * static image.  Written as I' = a (I_s - mu_s) + mu_m (north_star formula,
 * identical algebra).  Reading A5: a = 0 where var_s <= eps_var.
 * ---------------------------------------------------------------------- */
static inline double correct_one(double Is, double mu_s, double var_s, double mu_m, double var_m, double eps_var) {
    double a = var_s > eps_var ? sqrt(var_m / var_s) : 0.0;
    return a * (Is - mu_s) + mu_m;
}

void oracle_correct_from_moments(const float *cbct, const double *mu_s, const double *var_s, const double *mu_m,
                                 const double *var_m, size_t N, double eps_var, float *out) {
#pragma omp parallel for schedule(static)
    for (long long i = 0; i < (long long)N; ++i)
        out[i] = (float)correct_one(cbct[i], mu_s[i], var_s[i], mu_m[i], var_m[i], eps_var);
}

void oracle_correct(const float *cbct, const float *m, int nx, int ny, int nz, int R, double eps_var, float *out) {
#pragma omp parallel for schedule(dynamic, 1)
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                double mus, vs, mum, vm;
                patch_stats(cbct, nx, ny, nz, R, x, y, z, &mus, &vs);
                patch_stats(m, nx, ny, nz, R, x, y, z, &mum, &vm);
                out[IDX(x, y, z)] = (float)correct_one(cbct[IDX(x, y, z)], mus, vs, mum, vm, eps_var);
            }
}

void oracle_correct_at(const float *cbct, const float *m, int nx, int ny, int nz, int R, double eps_var,
                       const long long *idx, int nidx, double *out) {
#pragma omp parallel for schedule(dynamic, 16)
    for (int k = 0; k < nidx; ++k) {
        long long i = idx[k];
        int x = (int)(i % nx), y = (int)((i / nx) % ny), z = (int)(i / ((long long)nx * ny));
        double mus, vs, mum, vm;
        patch_stats(cbct, nx, ny, nz, R, x, y, z, &mus, &vs);
        patch_stats(m, nx, ny, nz, R, x, y, z, &mum, &vm);
        out[k] = correct_one(cbct[i], mus, vs, mum, vm, eps_var);
    }
}

/* ------------------------------------------------------------------------
 * (c) force + update.  PAPER.md:73 Eq. (1), first (passive) term with the
 * corrected static image s' (Alg. A1 steps 3->4), then
 * "add dr to the total moving vector r".  Readings A1/A7/A8:
 * g = central difference with clamped indices, d = s' - m,
 * r_c += d g_c / (|g|^2 + d^2 + eps_den)  (sign that descends for the
 * pull-back warp m(x) = I_m(x + r(x))).
 * ---------------------------------------------------------------------- */
void oracle_force_update(const float *m, const float *s, int nx, int ny, int nz, double eps_den, float *disp) {
    size_t N = (size_t)nx * ny * nz;
#pragma omp parallel for schedule(static)
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                size_t i = IDX(x, y, z);
                double gx = 0.5 * ((double)s[IDX(clampi(x + 1, 0, nx - 1), y, z)] - (double)s[IDX(clampi(x - 1, 0, nx - 1), y, z)]);
                double gy = 0.5 * ((double)s[IDX(x, clampi(y + 1, 0, ny - 1), z)] - (double)s[IDX(x, clampi(y - 1, 0, ny - 1), z)]);
                double gz = 0.5 * ((double)s[IDX(x, y, clampi(z + 1, 0, nz - 1))] - (double)s[IDX(x, y, clampi(z - 1, 0, nz - 1))]);
                double d = (double)s[i] - (double)m[i];
                double den = gx * gx + gy * gy + gz * gz + d * d + eps_den;
                disp[i] = (float)((double)disp[i] + d * gx / den);
                disp[N + i] = (float)((double)disp[N + i] + d * gy / den);
                disp[2 * N + i] = (float)((double)disp[2 * N + i] + d * gz / den);
            }
}

/* NEXT-2: the double-force variant, both terms of Eq. (1): the passive force with the gradient
 * of the (corrected) static image plus the active force with the gradient of the deformed moving image I_m^(k),
 * each with its own denominator.  Same sign convention (reading A1), same central differences with clamped
 * indices (A8) and the same eps_den in both denominators (A7):
 *   d = s' - m,  r_c += d g_c / (|g|^2 + d^2 + eps) + d h_c / (|h|^2 + d^2 + eps),  g = grad s', h = grad m. */
void oracle_force_update_double(const float *m, const float *s, int nx, int ny, int nz, double eps_den, float *disp) {
    size_t N = (size_t)nx * ny * nz;
#pragma omp parallel for schedule(static)
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                size_t i = IDX(x, y, z);
                size_t xp = IDX(clampi(x + 1, 0, nx - 1), y, z), xm = IDX(clampi(x - 1, 0, nx - 1), y, z);
                size_t yp = IDX(x, clampi(y + 1, 0, ny - 1), z), ym = IDX(x, clampi(y - 1, 0, ny - 1), z);
                size_t zp = IDX(x, y, clampi(z + 1, 0, nz - 1)), zm = IDX(x, y, clampi(z - 1, 0, nz - 1));
                double g[3] = {0.5 * ((double)s[xp] - (double)s[xm]), 0.5 * ((double)s[yp] - (double)s[ym]),
                               0.5 * ((double)s[zp] - (double)s[zm])};
                double h[3] = {0.5 * ((double)m[xp] - (double)m[xm]), 0.5 * ((double)m[yp] - (double)m[ym]),
                               0.5 * ((double)m[zp] - (double)m[zm])};
                double d = (double)s[i] - (double)m[i];
                double den_s = g[0] * g[0] + g[1] * g[1] + g[2] * g[2] + d * d + eps_den;
                double den_m = h[0] * h[0] + h[1] * h[1] + h[2] * h[2] + d * d + eps_den;
                for (int c = 0; c < 3; ++c)
                    disp[c * N + i] = (float)((double)disp[c * N + i] + d * g[c] / den_s + d * h[c] / den_m);
            }
}

/* NEXT-3: the two sums of the paper's convergence measure (section 2.3):
 *   l^(k) = sum_x |dr^(k+1)(x)| / sum_x |r^(k)(x)|,
 * dr = the increment the force is about to add (before any smoothing), r = the total field before the update.
 * Reading A16: |.| is the Euclidean norm of the 3-vector at a voxel.  fp64 throughout. */
void oracle_force_norms(const float *m, const float *s, const float *disp, int nx, int ny, int nz, double eps_den,
                        int double_force, double *sum_dr, double *sum_r) {
    size_t N = (size_t)nx * ny * nz;
    float *tmp = (float *)calloc(3 * N, sizeof(float));
    double a = 0.0, b = 0.0;
    /* the increment alone: the update applied to a zero field (evaluated in fp64, stored as the fp32 value that the
     * update would add), summed in fp64 */
    if (double_force) oracle_force_update_double(m, s, nx, ny, nz, eps_den, tmp);
    else oracle_force_update(m, s, nx, ny, nz, eps_den, tmp);
    for (size_t i = 0; i < N; ++i) {
        double dx = tmp[i], dy = tmp[N + i], dz = tmp[2 * N + i];
        double rx = disp[i], ry = disp[N + i], rz = disp[2 * N + i];
        a += sqrt(dx * dx + dy * dy + dz * dz);
        b += sqrt(rx * rx + ry * ry + rz * rz);
    }
    free(tmp);
    *sum_dr = a; *sum_r = b;
}

/* ------------------------------------------------------------------------
 * (d) Gaussian regularisation of the total field r (Alg. A1 step 6,
 * PAPER.md:194).  Reading A10: K = ceil(3 sigma), w_i ~ exp(-i^2 / 2 sigma^2)
 * computed in fp64, normalised to sum 1, then rounded to fp32; replicate
 * (clamped-index) border; passes x, y, z; direct convolution.
 * ---------------------------------------------------------------------- */
int oracle_gauss_radius(double sigma) { return (int)ceil(3.0 * sigma); }

void oracle_gauss_weights(double sigma, float *w /* 2K+1 */) {
    int K = oracle_gauss_radius(sigma);
    double s = 0.0;
    for (int i = -K; i <= K; ++i) s += exp(-(double)(i * i) / (2.0 * sigma * sigma));
    for (int i = -K; i <= K; ++i) w[i + K] = (float)(exp(-(double)(i * i) / (2.0 * sigma * sigma)) / s);
}

static void conv_axis(const double *in, double *out, int nx, int ny, int nz, int axis, const float *w, int K) {
#pragma omp parallel for schedule(static)
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                double acc = 0.0;
                for (int k = -K; k <= K; ++k) {
                    int a = x, b = y, c = z;
                    if (axis == 0) a = clampi(x + k, 0, nx - 1);
                    else if (axis == 1) b = clampi(y + k, 0, ny - 1);
                    else c = clampi(z + k, 0, nz - 1);
                    acc += (double)w[k + K] * in[IDX(a, b, c)];
                }
                out[IDX(x, y, z)] = acc;
            }
}

void oracle_smooth_field(float *disp, int nx, int ny, int nz, double sigma) {
    size_t N = (size_t)nx * ny * nz;
    int K = oracle_gauss_radius(sigma);
    float *w = (float *)malloc(sizeof(float) * (2 * K + 1));
    oracle_gauss_weights(sigma, w);
    double *a = (double *)malloc(sizeof(double) * N), *b = (double *)malloc(sizeof(double) * N);
    for (int c = 0; c < 3; ++c) {
        float *r = disp + c * N;
        for (size_t i = 0; i < N; ++i) a[i] = r[i];
        conv_axis(a, b, nx, ny, nz, 0, w, K);
        conv_axis(b, a, nx, ny, nz, 1, w, K);
        conv_axis(a, b, nx, ny, nz, 2, w, K);
        for (size_t i = 0; i < N; ++i) r[i] = (float)b[i];
    }
    free(a); free(b); free(w);
}

/* ------------------------------------------------------------------------
 * pyramid (reading A9).  Down: 2x2x2 block mean.
 * Up (field): r_fine(i) = 2 * trilinear(r_coarse, clamp(i/2 - 1/4)) per axis
 * (cell-centre aligned), values doubled because the field is in voxel units.
 * ---------------------------------------------------------------------- */
void oracle_downsample(const float *v, int nx, int ny, int nz, float *out) {
    int mx = nx / 2, my = ny / 2, mz = nz / 2;
#pragma omp parallel for schedule(static)
    for (int z = 0; z < mz; ++z)
        for (int y = 0; y < my; ++y)
            for (int x = 0; x < mx; ++x) {
                double s = 0.0;
                for (int c = 0; c < 2; ++c)
                    for (int b = 0; b < 2; ++b)
                        for (int a = 0; a < 2; ++a) s += v[IDX(2 * x + a, 2 * y + b, 2 * z + c)];
                out[((size_t)z * my + y) * mx + x] = (float)(s / 8.0);
            }
}

void oracle_upsample_field(const float *dc, int cx, int cy, int cz, float *out) {
    int nx = 2 * cx, ny = 2 * cy, nz = 2 * cz;
    size_t Nc = (size_t)cx * cy * cz, N = (size_t)nx * ny * nz;
    for (int comp = 0; comp < 3; ++comp) {
        const float *src = dc + comp * Nc;
        float *dst = out + comp * N;
#pragma omp parallel for schedule(static)
        for (int z = 0; z < nz; ++z)
            for (int y = 0; y < ny; ++y)
                for (int x = 0; x < nx; ++x)
                    dst[IDX(x, y, z)] = (float)(2.0 * trilinear(src, cx, cy, cz, x / 2.0 - 0.25, y / 2.0 - 0.25, z / 2.0 - 0.25));
    }
}

/* ------------------------------------------------------------------------
 * driver: Algorithm A1 minus the global shift (a no-op on
 * this path, pin P8), minus step 2 (mask/interpolation, NEXT-1) and with a
 * fixed iteration count instead of the while-test (reading A14).  Per level,
 * `iters` x { warp, moments+correct, force+update, smooth }; up-sample r
 * between levels; out_corr = correct(cbct_0, warp(ct_0, r)) (reading A12).
 * The CBCT moments are those of the level's ORIGINAL cbct, so
 * they are computed once per level with the same naive loop.
 * `trace` (optional, may be NULL): receives sum|r| after every iteration.
 * ---------------------------------------------------------------------- */
/* The general driver.  stop_eps >= 0 enables the paper's stopping criterion: inside a
 * level, l^(k) is evaluated in every iteration k = 0,1,.. (from that iteration's dr and the field before the
 * update; l = +inf while sum|r| = 0); the iteration in which  l^(k-10) - l^(k) <= stop_eps  first holds (k >= 10)
 * is completed and is the level's last.  `iters` stays the per-level maximum.  The text's criterion is followed;
 * Alg. A1's `while` prints it inverted (PAPER.md:187 vs :167).
 * iters_per_level (optional): explicit iteration counts, index = level (0 = finest), overriding `iters`.
 * iters_run (optional, [levels]): iterations actually run per level.  ltrace (optional, [levels*iters]): l^(k),
 * level-major from the coarsest level, `iters` slots per level. */
void oracle_register_full(const float *ct, const float *cbct, int nx, int ny, int nz, int R, double sigma, int levels,
                          int iters, double eps_var, double eps_den, int double_force, double stop_eps,
                          const int *iters_per_level, int *iters_run, double *ltrace, float *out_disp,
                          float *out_corr, double *trace) {
    const float **pct = (const float **)malloc(sizeof(float *) * levels);
    const float **pcb = (const float **)malloc(sizeof(float *) * levels);
    pct[0] = ct; pcb[0] = cbct;
    for (int l = 1; l < levels; ++l) {
        int fx = nx >> (l - 1), fy = ny >> (l - 1), fz = nz >> (l - 1);
        size_t Nl = (size_t)(fx / 2) * (fy / 2) * (fz / 2);
        float *a = (float *)malloc(sizeof(float) * Nl), *b = (float *)malloc(sizeof(float) * Nl);
        oracle_downsample(pct[l - 1], fx, fy, fz, a);
        oracle_downsample(pcb[l - 1], fx, fy, fz, b);
        pct[l] = a; pcb[l] = b;
    }
    float *r = NULL;
    int it_total = 0;
    for (int l = levels - 1; l >= 0; --l) {
        int lx = nx >> l, ly = ny >> l, lz = nz >> l;
        size_t N = (size_t)lx * ly * lz;
        if (r == NULL) {
            r = (float *)calloc(3 * N, sizeof(float));            /* PAPER.md:181 r = 0 */
        } else {
            float *rf = (float *)malloc(sizeof(float) * 3 * N);
            oracle_upsample_field(r, lx / 2, ly / 2, lz / 2, rf);
            free(r); r = rf;
        }
        float *m = (float *)malloc(sizeof(float) * N), *sp = (float *)malloc(sizeof(float) * N);
        double *mus = (double *)malloc(sizeof(double) * N), *vs = (double *)malloc(sizeof(double) * N);
        double *mum = (double *)malloc(sizeof(double) * N), *vm = (double *)malloc(sizeof(double) * N);
        oracle_box_moments(pcb[l], lx, ly, lz, R, mus, vs);
        int n_it = iters_per_level ? iters_per_level[l] : iters, k_run = 0;
        double *hist = (double *)malloc(sizeof(double) * (n_it > 0 ? n_it : 1));
        for (int k = 0; k < n_it; ++k) {
            int stop = 0;
            oracle_warp(pct[l], r, lx, ly, lz, m);                                   /* I_m^(k) */
            oracle_box_moments(m, lx, ly, lz, R, mum, vm);                           /* A1 step 1 */
            oracle_correct_from_moments(pcb[l], mus, vs, mum, vm, N, eps_var, sp);   /* A1 step 3 */
            if (stop_eps >= 0.0 || ltrace) {
                double sdr, sr;
                oracle_force_norms(m, sp, r, lx, ly, lz, eps_den, double_force, &sdr, &sr);
                hist[k] = sr > 0.0 ? sdr / sr : INFINITY;
                if (ltrace) ltrace[(size_t)(levels - 1 - l) * iters + k] = hist[k];
                if (stop_eps >= 0.0 && k >= 10 && hist[k - 10] - hist[k] <= stop_eps) stop = 1;
            }
            if (double_force) oracle_force_update_double(m, sp, lx, ly, lz, eps_den, r); /* Eq. (1), both terms */
            else oracle_force_update(m, sp, lx, ly, lz, eps_den, r);                 /* A1 steps 4-5 */
            oracle_smooth_field(r, lx, ly, lz, sigma);                               /* A1 step 6 */
            if (trace) {
                double s = 0.0;
                for (size_t i = 0; i < 3 * N; ++i) s += fabs((double)r[i]);
                trace[it_total] = s;
            }
            ++it_total;
            k_run = k + 1;
            if (stop) break;
        }
        free(hist);
        if (iters_run) iters_run[l] = k_run;
        if (l == 0) {
            memcpy(out_disp, r, sizeof(float) * 3 * N);
            if (out_corr) {
                oracle_warp(pct[0], r, lx, ly, lz, m);
                oracle_box_moments(m, lx, ly, lz, R, mum, vm);
                oracle_correct_from_moments(pcb[0], mus, vs, mum, vm, N, eps_var, out_corr);
            }
        }
        free(m); free(sp); free(mus); free(vs); free(mum); free(vm);
    }
    free(r);
    for (int l = 1; l < levels; ++l) { free((void *)pct[l]); free((void *)pcb[l]); }
    free(pct); free(pcb);
}

void oracle_register_mode(const float *ct, const float *cbct, int nx, int ny, int nz, int R, double sigma, int levels,
                          int iters, double eps_var, double eps_den, int double_force, float *out_disp,
                          float *out_corr, double *trace) {
    oracle_register_full(ct, cbct, nx, ny, nz, R, sigma, levels, iters, eps_var, eps_den, double_force, -1.0, NULL, NULL,
                         NULL, out_disp, out_corr, trace);
}

/* north_star's schedule: the Thirion (single, passive) force */
void oracle_register(const float *ct, const float *cbct, int nx, int ny, int nz, int R, double sigma, int levels,
                     int iters, double eps_var, double eps_den, float *out_disp, float *out_corr, double *trace) {
    oracle_register_mode(ct, cbct, nx, ny, nz, R, sigma, levels, iters, eps_var, eps_den, 0, out_disp, out_corr, trace);
}

/* ========================================================================
 * Extensions for SURVEY.md section 8(f): NEXT-4 (per-axis patch radius and
 * pyramid factor), NEXT-1 (reliability mask + interpolation of a, b), the
 * Fig.-9 diagnostics, and the summed-area moments used between the first and
 * last iteration of a level in config 4's whole-schedule check (SURVEY.md
 * section 8(c) "Oracle cost").  Same conventions as above.
 * ====================================================================== */

/* NEXT-4: non-cubic patches (PAPER.md:386 lists 3x3x3 ... 25x25x7): radius R[c] along axis c. */
void oracle_box_moments3(const float *v, int nx, int ny, int nz, const int R[3], double *mean, double *var) {
#pragma omp parallel for schedule(dynamic, 1)
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) patch_stats3(v, nx, ny, nz, R, x, y, z, &mean[IDX(x, y, z)], &var[IDX(x, y, z)]);
}

/* The same truncated-patch moments by EXACT summed-area tables: an independently written O(1)-per-voxel routine,
 * pinned against the naive loops above (tests/test_oracle_pins_ext.py::test_sat_moments_match_naive).  Every voxel is
 * taken as the integer q = round(v * 2^30) (exact for 2^-7 <= |v| < 2^14; smaller values are rounded to 2^-30 HU), the
 * tables of q and q^2 are three separable cumulative sums in 128-bit integers, the box sums are the 8-corner
 * inclusion-exclusion, and  n^2 var = n S2 - S1^2  (A.4) is formed exactly before the one conversion to
 * fp64 -- no cancellation error at all, which matters in flat regions: there sigma_m ~ 0 and an error of 1e-6 HU^2 in
 * the variance (what fp64 tables give on a 512x512x128 volume) becomes 1e-3 HU in the corrected image and, through the
 * demons force of a flat region, several 1e-3 voxel per iteration.  Returns 0; returns 1 WITHOUT writing mean and var
 * when a value is not finite or |v| >= 2^14 HU (the fixed-point range): the caller must not use the outputs then. */
typedef __int128 i128;

int oracle_box_moments_sat(const float *v, int nx, int ny, int nz, const int R[3], double *mean, double *var) {
    const size_t N = (size_t)nx * ny * nz;
    const int px = nx + 1, py = ny + 1, pz = nz + 1;
    const size_t NP = (size_t)px * py * pz;
#define PIDX(x, y, z) (((size_t)(z) * py + (y)) * px + (x))
    for (size_t i = 0; i < N; ++i)
        if (!(fabsf(v[i]) < 16384.0f)) return 1;
    i128 *P1 = (i128 *)calloc(NP, sizeof(i128)), *P2 = (i128 *)calloc(NP, sizeof(i128));
    /* P[z+1][y+1][x+1] = sum over the box [0..x] x [0..y] x [0..z]; index 0 planes stay zero */
#pragma omp parallel for schedule(static)
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y) {
            i128 r1 = 0, r2 = 0;                                        /* cumulative sum along x */
            for (int x = 0; x < nx; ++x) {
                long long q = llrint(ldexp((double)v[IDX(x, y, z)], 30));
                r1 += q; r2 += (i128)q * q;
                P1[PIDX(x + 1, y + 1, z + 1)] = r1; P2[PIDX(x + 1, y + 1, z + 1)] = r2;
            }
        }
#pragma omp parallel for schedule(static)
    for (int z = 1; z <= nz; ++z)                                       /* ... along y */
        for (int y = 2; y <= ny; ++y)
            for (int x = 1; x <= nx; ++x) {
                P1[PIDX(x, y, z)] += P1[PIDX(x, y - 1, z)]; P2[PIDX(x, y, z)] += P2[PIDX(x, y - 1, z)];
            }
#pragma omp parallel for schedule(static)
    for (int y = 1; y <= ny; ++y)                                       /* ... along z */
        for (int z = 2; z <= nz; ++z)
            for (int x = 1; x <= nx; ++x) {
                P1[PIDX(x, y, z)] += P1[PIDX(x, y, z - 1)]; P2[PIDX(x, y, z)] += P2[PIDX(x, y, z - 1)];
            }
    const double s30 = ldexp(1.0, -30), s60 = ldexp(1.0, -60);
#pragma omp parallel for schedule(static)
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                int x0 = clampi(x - R[0], 0, nx - 1), x1 = clampi(x + R[0], 0, nx - 1) + 1;
                int y0 = clampi(y - R[1], 0, ny - 1), y1 = clampi(y + R[1], 0, ny - 1) + 1;
                int z0 = clampi(z - R[2], 0, nz - 1), z1 = clampi(z + R[2], 0, nz - 1) + 1;
                long long n = (long long)(x1 - x0) * (y1 - y0) * (z1 - z0);
#define BOX(P) (P[PIDX(x1, y1, z1)] - P[PIDX(x0, y1, z1)] - P[PIDX(x1, y0, z1)] - P[PIDX(x1, y1, z0)] \
              + P[PIDX(x0, y0, z1)] + P[PIDX(x0, y1, z0)] + P[PIDX(x1, y0, z0)] - P[PIDX(x0, y0, z0)])
                i128 S1 = BOX(P1), S2 = BOX(P2);
#undef BOX
                i128 num = (i128)n * S2 - S1 * S1;                      /* n^2 var 2^60, exact and >= 0 */
                mean[IDX(x, y, z)] = (double)S1 * s30 / (double)n;
                var[IDX(x, y, z)] = (double)num * s60 / ((double)n * (double)n);
            }
#undef PIDX
    free(P1); free(P2);
    return 0;
}

/* NEXT-4: pyramid with a per-axis factor f[c] in {1, 2} (the paper's own preprocessing halves only the transverse
 * plane).  Down: block mean over f[0] x f[1] x f[2] voxels.  Up: along an axis with factor 2 the
 * cell-centre-aligned coordinate i/2 - 1/4 and component value x2 (reading A9); along an axis with factor 1 the
 * coordinate i and component value x1 -- component c is in voxel units of axis c. */
void oracle_downsample3(const float *v, int nx, int ny, int nz, const int f[3], float *out) {
    int mx = nx / f[0], my = ny / f[1], mz = nz / f[2];
#pragma omp parallel for schedule(static)
    for (int z = 0; z < mz; ++z)
        for (int y = 0; y < my; ++y)
            for (int x = 0; x < mx; ++x) {
                double s = 0.0;
                for (int c = 0; c < f[2]; ++c)
                    for (int b = 0; b < f[1]; ++b)
                        for (int a = 0; a < f[0]; ++a) s += v[IDX(f[0] * x + a, f[1] * y + b, f[2] * z + c)];
                out[((size_t)z * my + y) * mx + x] = (float)(s / (double)(f[0] * f[1] * f[2]));
            }
}

void oracle_upsample_field3(const float *dc, int cx, int cy, int cz, const int f[3], float *out) {
    int nx = f[0] * cx, ny = f[1] * cy, nz = f[2] * cz;
    size_t Nc = (size_t)cx * cy * cz, N = (size_t)nx * ny * nz;
    for (int comp = 0; comp < 3; ++comp) {
        const float *src = dc + comp * Nc;
        float *dst = out + comp * N;
        double scale = (double)f[comp];
#pragma omp parallel for schedule(static)
        for (int z = 0; z < nz; ++z)
            for (int y = 0; y < ny; ++y)
                for (int x = 0; x < nx; ++x) {
                    double px = f[0] == 2 ? x / 2.0 - 0.25 : (double)x;
                    double py = f[1] == 2 ? y / 2.0 - 0.25 : (double)y;
                    double pz = f[2] == 2 ? z / 2.0 - 0.25 : (double)z;
                    dst[IDX(x, y, z)] = (float)(scale * trilinear(src, cx, cy, cz, px, py, pz));
                }
    }
}

/* ------------------------------------------------------------------------
 * NEXT-1: reliability mask and interpolation / extrapolation of a, b
 * (Eqs. (5)-(10); parameters PAPER.md:161, :165).
 * ---------------------------------------------------------------------- */

/* Eqs. (5), (6) from given patch moments: a = STD(M)/STD(S) (0 where var_s <= eps_var, reading A5),
 * b = E(M) - a E(S). */
void oracle_ab_from_moments(const double *mu_s, const double *var_s, const double *mu_m, const double *var_m, size_t N,
                            double eps_var, double *a, double *b) {
#pragma omp parallel for schedule(static)
    for (long long i = 0; i < (long long)N; ++i) {
        double ai = var_s[i] > eps_var ? sqrt(var_m[i] / var_s[i]) : 0.0;
        a[i] = ai; b[i] = mu_m[i] - ai * mu_s[i];
    }
}

/* Eq. (7) (printed as a broken `cases`): xi = 1 where |I_m^(k)(x) - I_s(x)| > HU_0 or
 * a(x) < a_min or a(x) > a_max, 0 elsewhere.  Comparisons in fp64 (the difference of two fp32 values is exact). */
void oracle_mask(const float *m, const float *cbct, const double *a, size_t N, double hu0, double a_min, double a_max,
                 unsigned char *xi) {
#pragma omp parallel for schedule(static)
    for (long long i = 0; i < (long long)N; ++i) {
        double d = fabs((double)m[i] - (double)cbct[i]);
        xi[i] = (d > hu0 || a[i] < a_min || a[i] > a_max) ? 1 : 0;
    }
}

/* Eqs. (8)-(10): "Initially, we set a(x)=0 and b(x)=0 for xi(x)=1"; then every voxel with xi = 1
 * takes the weighted average of the a, b of the AVAILABLE voxels (xi = 0, or filled by an earlier pass) inside the
 * cube T of radius RT centred at it (truncated to the volume), w_i = exp(-(I_s(i) - I_s(x))^2 / h^2); the pass is
 * repeated "since for some voxels the values of xi may be 1 for all voxels in their neighbor T".  Values at
 * xi = 0 voxels are never changed.  Readings (A18): a pass reads only what was available when it
 * started (Jacobi); the weights are normalised by the largest one, w_i = exp(-((D_i)^2 - min_j (D_j)^2) / h^2), which
 * is the same quotient as Eqs. (8)-(9) and cannot underflow to 0/0; passes stop when nothing is left, when a pass
 * fills nothing, or after max_passes; what is still unfilled keeps a = b = 0.
 * xi (in/out): 1 = masked and unfilled; on return 1 only where no value could be found.  Returns the passes run. */
int oracle_fill_ab(const float *cbct, int nx, int ny, int nz, unsigned char *xi, double *a, double *b, int RT, double h,
                   int max_passes) {
    const size_t N = (size_t)nx * ny * nz;
    unsigned char *nxt = (unsigned char *)malloc(N);
    double *na = (double *)malloc(sizeof(double) * N), *nb = (double *)malloc(sizeof(double) * N);
    for (size_t i = 0; i < N; ++i)
        if (xi[i]) { a[i] = 0.0; b[i] = 0.0; }
    int pass = 0;
    for (; pass < max_passes; ++pass) {
        long long left = 0, filled = 0;
        for (size_t i = 0; i < N; ++i) left += xi[i];
        if (left == 0) break;
        memcpy(nxt, xi, N);
#pragma omp parallel for schedule(dynamic, 1) reduction(+ : filled)
        for (int z = 0; z < nz; ++z)
            for (int y = 0; y < ny; ++y)
                for (int x = 0; x < nx; ++x) {
                    size_t i0 = IDX(x, y, z);
                    if (!xi[i0]) continue;
                    double s0 = cbct[i0], dmin = INFINITY;
                    int x0 = clampi(x - RT, 0, nx - 1), x1 = clampi(x + RT, 0, nx - 1);
                    int y0 = clampi(y - RT, 0, ny - 1), y1 = clampi(y + RT, 0, ny - 1);
                    int z0 = clampi(z - RT, 0, nz - 1), z1 = clampi(z + RT, 0, nz - 1);
                    for (int c = z0; c <= z1; ++c)
                        for (int bb = y0; bb <= y1; ++bb)
                            for (int aa = x0; aa <= x1; ++aa) {
                                size_t i = IDX(aa, bb, c);
                                if (xi[i]) continue;
                                double d = (double)cbct[i] - s0;
                                if (d * d < dmin) dmin = d * d;
                            }
                    if (dmin == INFINITY) continue;               /* every voxel of T is still masked */
                    double sw = 0.0, sa = 0.0, sb = 0.0;
                    for (int c = z0; c <= z1; ++c)
                        for (int bb = y0; bb <= y1; ++bb)
                            for (int aa = x0; aa <= x1; ++aa) {
                                size_t i = IDX(aa, bb, c);
                                if (xi[i]) continue;
                                double d = (double)cbct[i] - s0;
                                double w = exp(-(d * d - dmin) / (h * h));  /* Eq. (10) */
                                sw += w; sa += w * a[i]; sb += w * b[i];
                            }
                    na[i0] = sa / sw; nb[i0] = sb / sw;           /* Eqs. (8), (9) */
                    nxt[i0] = 0;
                    ++filled;
                }
        for (size_t i = 0; i < N; ++i)
            if (xi[i] && !nxt[i]) { a[i] = na[i]; b[i] = nb[i]; }
        memcpy(xi, nxt, N);
        if (filled == 0) { ++pass; break; }
    }
    free(nxt); free(na); free(nb);
    return pass;
}

/* I'_s = a I_s + b on the original static image. */
void oracle_apply_ab(const float *cbct, const double *a, const double *b, size_t N, float *out) {
#pragma omp parallel for schedule(static)
    for (long long i = 0; i < (long long)N; ++i) out[i] = (float)(a[i] * (double)cbct[i] + b[i]);
}

/* Delta HU = mean(CT) - mean(CBCT), the constant that shifts the CBCT to the CT's mean intensity. */
double oracle_delta_hu(const float *ct, const float *cbct, size_t N) {
    double s1 = 0.0, s2 = 0.0;
    for (size_t i = 0; i < N; ++i) { s1 += ct[i]; s2 += cbct[i]; }
    return (s1 - s2) / (double)N;
}

static int cmp_double(const void *p, const void *q) {
    double a = *(const double *)p, b = *(const double *)q;
    return a < b ? -1 : (a > b ? 1 : 0);
}

/* "A is calculated before starting DIR and the median value a_m of A is used".  Reading A17: the
 * median runs over the voxels where Eq. (5) is a ratio of two positive deviations (var_s > eps_var and
 * var_m > eps_var) and is the lower median (order statistic floor((n-1)/2)); 1 if there is no such voxel. */
double oracle_median_a(const double *a, const double *var_s, const double *var_m, size_t N, double eps_var) {
    double *t = (double *)malloc(sizeof(double) * (N ? N : 1));
    size_t n = 0;
    for (size_t i = 0; i < N; ++i)
        if (var_s[i] > eps_var && var_m[i] > eps_var) t[n++] = a[i];
    double med = 1.0;
    if (n) { qsort(t, n, sizeof(double), cmp_double); med = t[(n - 1) / 2]; }
    free(t);
    return med;
}

/* ------------------------------------------------------------------------
 * The general driver: Algorithm A1 with every option.
 * ---------------------------------------------------------------------- */
typedef struct {
    int R[3];             /* patch radius per axis */
    int fac[3];           /* pyramid factor per axis, 1 or 2 */
    double sigma;         /* Gaussian sigma in voxels */
    int levels, iters;
    double eps_var, eps_den;
    int double_force;     /* both terms of Eq. (1) */
    double stop_eps;      /* < 0: fixed iteration count */
    int moments_policy;   /* 0: naive patch loops always; 1: summed-area tables except in the first and last iteration of a level */
    /* NEXT-1 */
    int mask;             /* 1: A1 "globally adjust", step 2 and Eq. (7) are on */
    double hu0;           /* < 0: HU_0 = 2 |Delta HU| */
    double a_min, a_max;  /* a_min < 0: 0.5 a_m and 1.5 a_m with a_m = median(A) before the DIR */
    int fill_radius;      /* radius of T (PAPER.md:131; its size is lost from the text, :165) */
    double h;             /* Eq. (10); never given */
    int max_fill_passes;
} oracle_params;

typedef struct {
    double delta_hu, hu0, a_m, a_min, a_max;   /* what the mask used */
} oracle_info;

static void level_dims(const oracle_params *p, int nx, int ny, int nz, int l, int *lx, int *ly, int *lz) {
    *lx = nx; *ly = ny; *lz = nz;
    for (int i = 0; i < l; ++i) { *lx /= p->fac[0]; *ly /= p->fac[1]; *lz /= p->fac[2]; }
}

static void moments_by_policy(const oracle_params *p, int k, int n_it, const float *v, int lx, int ly, int lz, double *mean,
                              double *var) {
    /* the summed-area routine refuses values outside its fixed-point range: the naive loops take over */
    if (p->moments_policy == 1 && k > 0 && k < n_it - 1 && oracle_box_moments_sat(v, lx, ly, lz, p->R, mean, var) == 0) return;
    oracle_box_moments3(v, lx, ly, lz, p->R, mean, var);
}

/* A1 steps 1 (second half) to 3 from given patch moments: a, b by Eqs. (5)-(6); with the mask on, Eq. (7), the
 * interpolation of Eqs. (8)-(10) and I'_s = a I_s + b; without it the same correction written as
 * a (I_s - mu_s) + mu_m (the hot path's form). */
static void correct_step(const oracle_params *p, const oracle_info *inf, const float *cbct, const float *m, int lx, int ly,
                         int lz, const double *mus, const double *vs, const double *mum, const double *vm, double *a,
                         double *b, unsigned char *xi, float *sp) {
    const size_t N = (size_t)lx * ly * lz;
    oracle_ab_from_moments(mus, vs, mum, vm, N, p->eps_var, a, b);
    if (p->mask) {
        oracle_mask(m, cbct, a, N, inf->hu0, inf->a_min, inf->a_max, xi);                      /* Eq. (7) */
        oracle_fill_ab(cbct, lx, ly, lz, xi, a, b, p->fill_radius, p->h, p->max_fill_passes);   /* A1 step 2 */
        oracle_apply_ab(cbct, a, b, N, sp);                                                    /* A1 step 3 */
    } else {
        oracle_correct_from_moments(cbct, mus, vs, mum, vm, N, p->eps_var, sp);                 /* A1 step 3 */
    }
}

/* Outputs (each may be NULL except out_disp): out_corr [N0]; iters_run [levels]; ltrace, mean_a, mean_b
 * [levels*iters], level-major from the coarsest level (l(k), and Fig. 9 (e),(f): the averages of a and b over all
 * voxels in every iteration); info. */
void oracle_register_ex(const float *ct, const float *cbct_in, int nx, int ny, int nz, const oracle_params *p,
                        float *out_disp, float *out_corr, int *iters_run, double *ltrace, double *mean_a, double *mean_b,
                        oracle_info *info) {
    const int levels = p->levels;
    const size_t N0 = (size_t)nx * ny * nz;
    oracle_info inf = {0.0, 0.0, 1.0, 0.0, 0.0};
    float *cbct0 = (float *)malloc(sizeof(float) * N0);
    memcpy(cbct0, cbct_in, sizeof(float) * N0);
    if (p->mask) {
        /* A1 "Globally adjust the intensity of CBCT" */
        inf.delta_hu = oracle_delta_hu(ct, cbct_in, N0);
        for (size_t i = 0; i < N0; ++i) cbct0[i] = (float)((double)cbct_in[i] + inf.delta_hu);
        inf.hu0 = p->hu0 >= 0.0 ? p->hu0 : 2.0 * fabs(inf.delta_hu);
        if (p->a_min >= 0.0) { inf.a_min = p->a_min; inf.a_max = p->a_max; }
        else {
            /* A before the DIR (r = 0, full resolution), a_m = median(A) */
            double *mus = (double *)malloc(sizeof(double) * N0), *vs = (double *)malloc(sizeof(double) * N0);
            double *mum = (double *)malloc(sizeof(double) * N0), *vm = (double *)malloc(sizeof(double) * N0);
            double *a = (double *)malloc(sizeof(double) * N0), *b = (double *)malloc(sizeof(double) * N0);
            oracle_box_moments3(cbct0, nx, ny, nz, p->R, mus, vs);
            oracle_box_moments3(ct, nx, ny, nz, p->R, mum, vm);
            oracle_ab_from_moments(mus, vs, mum, vm, N0, p->eps_var, a, b);
            inf.a_m = oracle_median_a(a, vs, vm, N0, p->eps_var);
            inf.a_min = 0.5 * inf.a_m; inf.a_max = 1.5 * inf.a_m;
            free(mus); free(vs); free(mum); free(vm); free(a); free(b);
        }
    }
    const float **pct = (const float **)malloc(sizeof(float *) * levels);
    const float **pcb = (const float **)malloc(sizeof(float *) * levels);
    pct[0] = ct; pcb[0] = cbct0;
    for (int l = 1; l < levels; ++l) {
        int fx, fy, fz;
        level_dims(p, nx, ny, nz, l - 1, &fx, &fy, &fz);
        size_t Nl = (size_t)(fx / p->fac[0]) * (fy / p->fac[1]) * (fz / p->fac[2]);
        float *a = (float *)malloc(sizeof(float) * Nl), *b = (float *)malloc(sizeof(float) * Nl);
        oracle_downsample3(pct[l - 1], fx, fy, fz, p->fac, a);
        oracle_downsample3(pcb[l - 1], fx, fy, fz, p->fac, b);
        pct[l] = a; pcb[l] = b;
    }
    float *r = NULL;
    for (int l = levels - 1; l >= 0; --l) {
        int lx, ly, lz;
        level_dims(p, nx, ny, nz, l, &lx, &ly, &lz);
        size_t N = (size_t)lx * ly * lz;
        if (r == NULL) r = (float *)calloc(3 * N, sizeof(float));
        else {
            float *rf = (float *)malloc(sizeof(float) * 3 * N);
            oracle_upsample_field3(r, lx / p->fac[0], ly / p->fac[1], lz / p->fac[2], p->fac, rf);
            free(r); r = rf;
        }
        float *m = (float *)malloc(sizeof(float) * N), *sp = (float *)malloc(sizeof(float) * N);
        double *mus = (double *)malloc(sizeof(double) * N), *vs = (double *)malloc(sizeof(double) * N);
        double *mum = (double *)malloc(sizeof(double) * N), *vm = (double *)malloc(sizeof(double) * N);
        double *a = (double *)malloc(sizeof(double) * N), *b = (double *)malloc(sizeof(double) * N);
        unsigned char *xi = (unsigned char *)malloc(N);
        oracle_box_moments3(pcb[l], lx, ly, lz, p->R, mus, vs);
        const int n_it = p->iters;
        int k_run = 0;
        double *hist = (double *)malloc(sizeof(double) * (n_it > 0 ? n_it : 1));
        for (int k = 0; k < n_it; ++k) {
            oracle_warp(pct[l], r, lx, ly, lz, m);                                  /* I_m^(k) */
            moments_by_policy(p, k, n_it, m, lx, ly, lz, mum, vm);                  /* A1 step 1 */
            correct_step(p, &inf, pcb[l], m, lx, ly, lz, mus, vs, mum, vm, a, b, xi, sp);   /* A1 steps 1-3 */
            if (mean_a || mean_b) {
                double sa = 0.0, sb = 0.0;
                for (size_t i = 0; i < N; ++i) { sa += a[i]; sb += b[i]; }
                if (mean_a) mean_a[(size_t)(levels - 1 - l) * n_it + k] = sa / (double)N;
                if (mean_b) mean_b[(size_t)(levels - 1 - l) * n_it + k] = sb / (double)N;
            }
            int stop = 0;
            if (p->stop_eps >= 0.0 || ltrace) {
                double sdr, sr;
                oracle_force_norms(m, sp, r, lx, ly, lz, p->eps_den, p->double_force, &sdr, &sr);
                hist[k] = sr > 0.0 ? sdr / sr : INFINITY;
                if (ltrace) ltrace[(size_t)(levels - 1 - l) * n_it + k] = hist[k];
                if (p->stop_eps >= 0.0 && k >= 10 && hist[k - 10] - hist[k] <= p->stop_eps) stop = 1;
            }
            if (p->double_force) oracle_force_update_double(m, sp, lx, ly, lz, p->eps_den, r);
            else oracle_force_update(m, sp, lx, ly, lz, p->eps_den, r);             /* A1 steps 4-5 */
            oracle_smooth_field(r, lx, ly, lz, p->sigma);                           /* A1 step 6 */
            k_run = k + 1;
            if (stop) break;
        }
        if (l == 0 && out_corr) {                                                   /* reading A12 */
            oracle_warp(pct[0], r, lx, ly, lz, m);
            oracle_box_moments3(m, lx, ly, lz, p->R, mum, vm);
            correct_step(p, &inf, pcb[0], m, lx, ly, lz, mus, vs, mum, vm, a, b, xi, out_corr);
        }
        free(hist);
        if (iters_run) iters_run[l] = k_run;
        if (l == 0) memcpy(out_disp, r, sizeof(float) * 3 * N);
        free(m); free(sp); free(mus); free(vs); free(mum); free(vm); free(a); free(b); free(xi);
    }
    free(r);
    for (int l = 1; l < levels; ++l) { free((void *)pct[l]); free((void *)pcb[l]); }
    free(pct); free(pcb); free(cbct0);
    if (info) *info = inf;
}
