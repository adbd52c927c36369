/*
 * synth_inputs/phantom_gen.c -- seeded synthetic INPUT generator (harness only).
 *
 * Builds the prostate-like phantoms of BASELINE.json `configs` under the
 * geometry reading of SURVEY.md section 8(d): a voxel grid, four structures
 * (PTV / rectum / bladder / body), coplanar parallel fields cut into square
 * beamlets and an analytic pencil-beam dose-deposition matrix
 *     D = exp(-mu * depth) * exp(-r^2 / (2 sigma^2)),
 * truncated at tau * max(D), stored as CSR (rows = voxels, cols = beamlets,
 * columns ascending).  These matrices STAND IN for the clinical prostate case of
 * PAPER.md:150 (section 3.1), which is not available.
 *
 * This file holds none of the optimiser's arithmetic (no objective, gradient,
 * projection or line search).  It serves both the oracle and the CUDA library
 * with the very same arrays; neither of them includes or links it.
 *
 * Math in fp64; values are cast to fp32 on output.  Deterministic for a given
 * libm (rows are independent, so the OpenMP schedule does not matter).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef struct {
    int32_t nx, ny, nz;   /* grid */
    double h;             /* voxel spacing, mm */
    int32_t geom;         /* 0: box phantom of config 0; 1: elliptic-cylinder phantom of configs 1-4 */
    int32_t n_beams;      /* coplanar, equispaced, parallel (non-divergent) */
    double beamlet;       /* beamlet edge, mm */
    double half_field;    /* F: the field is [-F, F]^2 in (u, v) */
    double sigma;         /* lateral Gaussian sigma, mm */
    double tau;           /* entries < tau * max are dropped */
    double mu;            /* attenuation per mm of depth */
} phantom_cfg;

#define SID_PTV 0
#define SID_RECTUM 1
#define SID_BLADDER 2
#define SID_BODY 3
#define SID_NONE 255

static void voxel_centre(const phantom_cfg *c, int64_t id, double *x, double *y, double *z) {
    int64_t ix = id % c->nx, iy = (id / c->nx) % c->ny, iz = id / ((int64_t)c->nx * c->ny);
    *x = ((double)ix + 0.5 - 0.5 * c->nx) * c->h;
    *y = ((double)iy + 0.5 - 0.5 * c->ny) * c->h;
    *z = ((double)iz + 0.5 - 0.5 * c->nz) * c->h;
}

/* Structure id of every grid voxel (priority PTV > rectum > bladder > body); SID_NONE outside the body. */
void phantom_structures(const phantom_cfg *c, uint8_t *sid_grid) {
    const int64_t n = (int64_t)c->nx * c->ny * c->nz;
    const double Lx = c->nx * c->h, Ly = c->ny * c->h;
#pragma omp parallel for schedule(static)
    for (int64_t id = 0; id < n; ++id) {
        double x, y, z;
        voxel_centre(c, id, &x, &y, &z);
        uint8_t s = SID_NONE;
        if (c->geom == 0) {
            if (x * x + y * y + z * z <= 20.0 * 20.0) s = SID_PTV;
            else if (x * x + (y - 30.0) * (y - 30.0) <= 10.0 * 10.0 && fabs(z) <= 30.0) s = SID_RECTUM;
            else if (x * x + (y + 38.0) * (y + 38.0) + z * z <= 18.0 * 18.0) s = SID_BLADDER;
            else s = SID_BODY;
        } else {
            const double A = 0.4 * Lx, B = 0.4 * Ly;
            if ((x / 30.0) * (x / 30.0) + (y / 25.0) * (y / 25.0) + (z / 30.0) * (z / 30.0) <= 1.0) s = SID_PTV;
            else if (x * x + (y - 40.0) * (y - 40.0) <= 15.0 * 15.0 && fabs(z) <= 45.0) s = SID_RECTUM;
            else if (x * x + (y + 52.0) * (y + 52.0) + z * z <= 27.0 * 27.0) s = SID_BLADDER;
            else if ((x / A) * (x / A) + (y / B) * (y / B) <= 1.0) s = SID_BODY;
        }
        sid_grid[id] = s;
    }
}

/* Where the line {u fixed} of a beam with direction (s, -c) enters the body outline. */
static double entry_t(const phantom_cfg *c, double cs, double sn, double u) {
    const double Lx = c->nx * c->h, Ly = c->ny * c->h;
    if (c->geom == 0) {
        /* x(t) = u cs + t sn ; y(t) = u sn - t cs ; box [-Lx/2, Lx/2] x [-Ly/2, Ly/2] */
        double t_in = -1e300;
        if (fabs(sn) > 1e-12) {
            double t1 = (-0.5 * Lx - u * cs) / sn, t2 = (0.5 * Lx - u * cs) / sn;
            double lo = t1 < t2 ? t1 : t2;
            if (lo > t_in) t_in = lo;
        }
        if (fabs(cs) > 1e-12) {
            double t1 = (-0.5 * Ly - u * sn) / (-cs), t2 = (0.5 * Ly - u * sn) / (-cs);
            double lo = t1 < t2 ? t1 : t2;
            if (lo > t_in) t_in = lo;
        }
        return t_in;
    } else {
        const double A = 0.4 * Lx, B = 0.4 * Ly;
        const double qa = sn * sn / (A * A) + cs * cs / (B * B);
        const double qb = 2.0 * u * cs * sn * (1.0 / (A * A) - 1.0 / (B * B));
        const double qc = u * u * (cs * cs / (A * A) + sn * sn / (B * B)) - 1.0;
        double disc = qb * qb - 4.0 * qa * qc;
        if (disc < 0.0) disc = 0.0;
        return (-qb - sqrt(disc)) / (2.0 * qa);
    }
}

/* One row of D.  mode 0: return the row maximum; mode 1: count entries >= thr; mode 2: write them. */
static double row_pass(const phantom_cfg *c, int64_t vox, double R, double thr, int mode,
                       int64_t *count, int32_t *col, float *val) {
    double x, y, z;
    voxel_centre(c, vox, &x, &y, &z);
    const int m = (int)floor(2.0 * c->half_field / c->beamlet + 0.5);
    const double F = c->half_field, b = c->beamlet;
    const double inv2s2 = 1.0 / (2.0 * c->sigma * c->sigma);
    double rmax = 0.0;
    int64_t n = 0;
    double eu[64], ev[64];
    for (int k = 0; k < c->n_beams; ++k) {
        const double th = 2.0 * M_PI * (double)k / (double)c->n_beams;
        const double cs = cos(th), sn = sin(th);
        const double t = x * sn - y * cs, u = x * cs + y * sn, v = z;
        int a_lo = (int)ceil((u - R + F) / b - 0.5), a_hi = (int)floor((u + R + F) / b - 0.5);
        int c_lo = (int)ceil((v - R + F) / b - 0.5), c_hi = (int)floor((v + R + F) / b - 0.5);
        if (a_lo < 0) a_lo = 0;
        if (c_lo < 0) c_lo = 0;
        if (a_hi > m - 1) a_hi = m - 1;
        if (c_hi > m - 1) c_hi = m - 1;
        if (a_lo > a_hi || c_lo > c_hi) continue;
        if (a_hi - a_lo >= 64) a_hi = a_lo + 63;
        if (c_hi - c_lo >= 64) c_hi = c_lo + 63;
        double depth = t - entry_t(c, cs, sn, u);
        if (depth < 0.0) depth = 0.0;
        const double ed = exp(-c->mu * depth);
        for (int a = a_lo; a <= a_hi; ++a) {
            const double du = u - (-F + (a + 0.5) * b);
            eu[a - a_lo] = exp(-du * du * inv2s2);
        }
        for (int q = c_lo; q <= c_hi; ++q) {
            const double dv = v - (-F + (q + 0.5) * b);
            ev[q - c_lo] = exp(-dv * dv * inv2s2);
        }
        for (int a = a_lo; a <= a_hi; ++a)
            for (int q = c_lo; q <= c_hi; ++q) {
                const double w = ed * eu[a - a_lo] * ev[q - c_lo];
                if (mode == 0) {
                    if (w > rmax) rmax = w;
                } else if (w >= thr) {
                    if (mode == 2) {
                        col[n] = (k * m + a) * m + q;
                        val[n] = (float)w;
                    }
                    ++n;
                }
            }
    }
    if (count) *count = n;
    return rmax;
}

/* Global maximum entry of D over the given voxels (first of the two passes). */
double phantom_dose_max(const phantom_cfg *c, int64_t n_v, const int64_t *vox) {
    double gmax = 0.0;
    const double R = 1.5 * c->beamlet; /* the maximum sits next to a beamlet axis */
#pragma omp parallel for schedule(dynamic, 4096) reduction(max : gmax)
    for (int64_t j = 0; j < n_v; ++j) {
        double r = row_pass(c, vox[j], R, 0.0, 0, NULL, NULL, NULL);
        if (r > gmax) gmax = r;
    }
    return gmax;
}

static double cut_radius(const phantom_cfg *c, double gmax) {
    return c->sigma * sqrt(2.0 * log(1.0 / (c->tau * gmax))) + 1e-9;
}

/* Entries per row after truncation at tau * gmax. */
void phantom_dose_count(const phantom_cfg *c, int64_t n_v, const int64_t *vox, double gmax, int64_t *row_nnz) {
    const double R = cut_radius(c, gmax), thr = c->tau * gmax;
#pragma omp parallel for schedule(dynamic, 4096)
    for (int64_t j = 0; j < n_v; ++j) row_pass(c, vox[j], R, thr, 1, &row_nnz[j], NULL, NULL);
}

/* Fill CSR arrays given row_ptr (int64 prefix sums of row_nnz). */
void phantom_dose_fill(const phantom_cfg *c, int64_t n_v, const int64_t *vox, double gmax,
                       const int64_t *row_ptr, int32_t *col, float *val) {
    const double R = cut_radius(c, gmax), thr = c->tau * gmax;
#pragma omp parallel for schedule(dynamic, 4096)
    for (int64_t j = 0; j < n_v; ++j) {
        int64_t n;
        row_pass(c, vox[j], R, thr, 2, &n, col + row_ptr[j], val + row_ptr[j]);
    }
}

/*
 * Largest eigenvalue of D^T diag(w) D by power iteration from the all-ones
 * vector (fp64, n_iter steps).  Used only to pick the line-search start
 * lambda0, a PARAMETER handed to both sides.
 */
double phantom_power_iter(int64_t n_v, int64_t n_b, const int32_t *row_ptr, const int32_t *col,
                          const float *val, const double *w_row, int n_iter) {
    double *y = (double *)malloc(sizeof(double) * (size_t)n_b);
    double *z = (double *)malloc(sizeof(double) * (size_t)n_b);
    double *dz = (double *)malloc(sizeof(double) * (size_t)n_v);
    for (int64_t i = 0; i < n_b; ++i) y[i] = 1.0;
    double lam = 0.0;
    for (int it = 0; it < n_iter; ++it) {
        double nrm = 0.0;
        for (int64_t i = 0; i < n_b; ++i) nrm += y[i] * y[i];
        nrm = sqrt(nrm);
        for (int64_t i = 0; i < n_b; ++i) y[i] /= nrm;
#pragma omp parallel for schedule(static)
        for (int64_t j = 0; j < n_v; ++j) {
            double s = 0.0;
            for (int64_t p = row_ptr[j]; p < row_ptr[j + 1]; ++p) s += (double)val[p] * y[col[p]];
            dz[j] = w_row[j] * s;
        }
        memset(z, 0, sizeof(double) * (size_t)n_b);
        for (int64_t j = 0; j < n_v; ++j) {
            const double s = dz[j];
            if (s != 0.0)
                for (int64_t p = row_ptr[j]; p < row_ptr[j + 1]; ++p) z[col[p]] += (double)val[p] * s;
        }
        lam = 0.0;
        for (int64_t i = 0; i < n_b; ++i) lam += y[i] * z[i];
        memcpy(y, z, sizeof(double) * (size_t)n_b);
    }
    free(y);
    free(z);
    free(dz);
    return lam;
}
