/*
 * Seeded synthetic INPUT generators for the VMAT hot path (test + benchmark inputs only).
 *
 * This file holds none of the method's arithmetic (no dose sums, penalties, prices,
 * leaf searches or master solves): it only manufactures the sparse dose-deposition
 * matrix D and the isolated-kernel sweep matrices that BASELINE.json:configs describe.
 * One generator feeds both the CPU oracle and the CUDA library, so both sides see the
 * same bits.
 *
 * D model (BASELINE.json:configs[0], concretised in DESIGN.md "Input recipe"):
 *   parallel rays in the axial plane, gantry axis = grid z through the grid centre,
 *   beam k at angle theta_k = k*360/N deg travels along d = (cos, sin, 0); leaf columns
 *   run along u = (-sin, cos, 0), leaf rows stack along z.  Beamlet (k,r,c) is the ray
 *   through  a_c*u + b_r*zhat,  a_c = (c-(C-1)/2)*bw,  b_r = (r-(R-1)/2)*bw.
 *   A voxel centre p inside the body cylinder (radius Rb about the z axis) at lateral
 *   position a = p.u, along-beam position t = p.d has depth = t + sqrt(Rb^2 - a^2) and
 *     value = exp(-mu*depth) * exp(-rho^2/(2 sigma^2)) * (1 + noise*U(-1,1)),
 *   rho^2 = (a-a_c)^2 + (z-b_r)^2, kernel support rho <= 4.5 sigma, entries below
 *   cutoff * (row maximum) dropped.  U(-1,1) is a counter-based hash of
 *   (seed, beamlet, voxel), so generation is order independent.
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC gen.c -o libvmat_inputs.so -lm
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    int32_t nx, ny, nz;       /* voxel grid, x fastest: j = (iz*ny + iy)*nx + ix   */
    double  voxel_mm;
    int32_t n_beams, n_rows, n_cols; /* N, R, C ; beamlet i = (k*R + r)*C + c        */
    double  beamlet_mm;       /* bw                                                 */
    double  body_radius_mm;   /* Rb                                                 */
    double  mu_per_mm;        /* 0.05                                               */
    double  sigma_bw;         /* 0.6 (sigma in beamlet widths)                      */
    double  noise;            /* 0.02                                               */
    double  cutoff;           /* 1e-3                                               */
    uint64_t seed;
} vin_geometry;

static inline uint64_t mix64(uint64_t x) {            /* splitmix64 finaliser */
    x += 0x9E3779B97F4A7C15ull;
    x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ull;
    x = (x ^ (x >> 27)) * 0x94D049BB133111EBull;
    return x ^ (x >> 31);
}
/* uniform in (-1,1), a pure function of (seed, a, b) */
static inline double hash_u11(uint64_t seed, uint64_t a, uint64_t b) {
    uint64_t h = mix64(mix64(seed ^ mix64(a)) ^ (b * 0xD6E8FEB86659FD93ull));
    return ((double)(h >> 11) + 0.5) * (2.0 / 9007199254740992.0) - 1.0;
}

/* Enumerate one beamlet row.  If col/val are NULL only the count is returned.
 * Two sweeps over the candidate set: (1) exact row maximum, (2) keep >= cutoff*max. */
static int64_t beamlet_row(const vin_geometry *g, int64_t i, int32_t *col, float *val) {
    const int R = g->n_rows, C = g->n_cols;
    const int k = (int)(i / ((int64_t)R * C));
    const int r = (int)((i / C) % R);
    const int c = (int)(i % C);
    const double th = (double)k * 360.0 / (double)g->n_beams * (M_PI / 180.0);
    const double cs = cos(th), sn = sin(th);
    const double bw = g->beamlet_mm, vs = g->voxel_mm, Rb = g->body_radius_mm;
    const double a_c = ((double)c - 0.5 * (C - 1)) * bw;
    const double b_r = ((double)r - 0.5 * (R - 1)) * bw;
    const double sigma = g->sigma_bw * bw, inv2s2 = 1.0 / (2.0 * sigma * sigma);
    const double rho_max = 4.5 * sigma, rho_max2 = rho_max * rho_max;
    const double x0 = -0.5 * g->nx * vs, y0 = -0.5 * g->ny * vs, z0 = -0.5 * g->nz * vs;

    if (fabs(a_c) - rho_max >= Rb) return 0;            /* ray (with its halo) misses the body */

    int iz_lo = (int)floor((b_r - rho_max - z0) / vs - 0.5);
    int iz_hi = (int)ceil((b_r + rho_max - z0) / vs - 0.5);
    if (iz_lo < 0) iz_lo = 0;
    if (iz_hi > g->nz - 1) iz_hi = g->nz - 1;
    int iy_lo = (int)floor((-Rb - y0) / vs - 0.5), iy_hi = (int)ceil((Rb - y0) / vs - 0.5);
    if (iy_lo < 0) iy_lo = 0;
    if (iy_hi > g->ny - 1) iy_hi = g->ny - 1;

    double vmax = 0.0;
    int64_t n = 0;
    for (int pass = 0; pass < 2; ++pass) {
        const double keep = g->cutoff * vmax;
        if (pass == 1 && !(vmax > 0.0)) return 0;
        for (int iz = iz_lo; iz <= iz_hi; ++iz) {
            const double z = z0 + (iz + 0.5) * vs, dz = z - b_r;
            const double rxy2 = rho_max2 - dz * dz;
            if (rxy2 < 0.0) continue;
            const double rxy = sqrt(rxy2);
            for (int iy = iy_lo; iy <= iy_hi; ++iy) {
                const double y = y0 + (iy + 0.5) * vs;
                const double bx2 = Rb * Rb - y * y;
                if (bx2 < 0.0) continue;
                double xl = -sqrt(bx2), xh = -xl;                    /* body chord   */
                /* |a - a_c| <= rxy with a = -sn*x + cs*y  ->  x interval when sn != 0  */
                if (fabs(sn) > 1e-12) {
                    double e0 = (cs * y - a_c - rxy) / sn, e1 = (cs * y - a_c + rxy) / sn;
                    if (e0 > e1) { double t = e0; e0 = e1; e1 = t; }
                    if (e0 > xl) xl = e0;
                    if (e1 < xh) xh = e1;
                } else if (fabs(cs * y - a_c) > rxy) continue;
                int ix_lo = (int)floor((xl - x0) / vs - 0.5) - 1, ix_hi = (int)ceil((xh - x0) / vs - 0.5) + 1;
                if (ix_lo < 0) ix_lo = 0;
                if (ix_hi > g->nx - 1) ix_hi = g->nx - 1;
                for (int ix = ix_lo; ix <= ix_hi; ++ix) {
                    const double x = x0 + (ix + 0.5) * vs;
                    const double rr2 = x * x + y * y;
                    if (rr2 > Rb * Rb) continue;                      /* outside body */
                    const double a = -sn * x + cs * y, t = cs * x + sn * y;
                    const double da = a - a_c, rho2 = da * da + dz * dz;
                    if (rho2 > rho_max2) continue;                    /* kernel support */
                    const double depth = t + sqrt(Rb * Rb - a * a > 0.0 ? Rb * Rb - a * a : 0.0);
                    const int64_t j = ((int64_t)iz * g->ny + iy) * g->nx + ix;
                    const double v = exp(-g->mu_per_mm * depth - rho2 * inv2s2) *
                                     (1.0 + g->noise * hash_u11(g->seed, (uint64_t)i, (uint64_t)j));
                    if (pass == 0) { if (v > vmax) vmax = v; }
                    else if (v >= keep) {
                        if (col) { col[n] = (int32_t)j; val[n] = (float)v; }
                        ++n;
                    }
                }
            }
        }
    }
    return n;
}

/* Pass A: per-row counts -> row_ptr (B+1, int64).  Returns nnz. */
int64_t vin_dose_matrix_count(const vin_geometry *g, int64_t *row_ptr) {
    const int64_t B = (int64_t)g->n_beams * g->n_rows * g->n_cols;
    row_ptr[0] = 0;
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < B; ++i) row_ptr[i + 1] = beamlet_row(g, i, NULL, NULL);
    for (int64_t i = 0; i < B; ++i) row_ptr[i + 1] += row_ptr[i];
    return row_ptr[B];
}
/* Pass B: fill col_idx / val (caller allocated, nnz entries) using row_ptr from pass A. */
void vin_dose_matrix_fill(const vin_geometry *g, const int64_t *row_ptr, int32_t *col, float *val) {
    const int64_t B = (int64_t)g->n_beams * g->n_rows * g->n_cols;
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < B; ++i) beamlet_row(g, i, col + row_ptr[i], val + row_ptr[i]);
}

/* ---- BASELINE.json:configs[3] — isolated pricing-kernel sweep matrices ------------------
 * rows with length U[len_lo,len_hi]; voxel indices in sorted, non-overlapping contiguous
 * runs of U[run_lo,run_hi] placed uniformly in [0,V); values U(0,1).                       */
static inline uint64_t rng_next(uint64_t *s) { *s += 0x9E3779B97F4A7C15ull; return mix64(*s); }
static inline double rng_u01(uint64_t *s) { return ((double)(rng_next(s) >> 11) + 0.5) / 9007199254740992.0; }
static inline int64_t rng_range(uint64_t *s, int64_t lo, int64_t hi) { /* inclusive */
    return lo + (int64_t)(rng_u01(s) * (double)(hi - lo + 1));
}

void vin_sweep_row_lengths(int64_t n_rows, int32_t len_lo, int32_t len_hi, uint64_t seed, int64_t *row_ptr) {
    row_ptr[0] = 0;
    for (int64_t i = 0; i < n_rows; ++i) {
        uint64_t s = mix64(seed ^ mix64(0x5157EEull + (uint64_t)i));
        row_ptr[i + 1] = row_ptr[i] + rng_range(&s, len_lo, len_hi);
    }
}
void vin_sweep_fill(int64_t n_rows, const int64_t *row_ptr, int64_t V, int32_t run_lo, int32_t run_hi,
                    uint64_t seed, int32_t *col, float *val) {
#pragma omp parallel for schedule(dynamic, 256)
    for (int64_t i = 0; i < n_rows; ++i) {
        uint64_t s = mix64(seed ^ mix64(0xC01D1Dull + (uint64_t)i));
        const int64_t L = row_ptr[i + 1] - row_ptr[i];
        int32_t *c = col + row_ptr[i];
        float *v = val + row_ptr[i];
        int32_t runs[1024];
        int m = 0;
        for (int64_t left = L; left > 0 && m < 1024; ++m) {
            int64_t len = rng_range(&s, run_lo, run_hi);
            if (len > left || m == 1023) len = left;
            runs[m] = (int32_t)len;
            left -= len;
        }
        /* m+1 gaps summing to V-L: sorted uniform cut points */
        int64_t cuts[1024];
        const int64_t G = V - L;
        for (int q = 0; q < m; ++q) {
            int64_t x = (int64_t)(rng_u01(&s) * (double)(G + 1));
            if (x > G) x = G;
            int p = q;
            while (p > 0 && cuts[p - 1] > x) { cuts[p] = cuts[p - 1]; --p; }
            cuts[p] = x;
        }
        int64_t pos = 0, w = 0;
        for (int q = 0; q < m; ++q) {
            const int64_t start = cuts[q] + pos;   /* gap prefix + entries placed so far */
            for (int32_t e = 0; e < runs[q]; ++e) { c[w] = (int32_t)(start + e); v[w] = (float)rng_u01(&s); ++w; }
            pos += runs[q];
        }
    }
}
/* standard normal vector (Box-Muller on the counter hash), e.g. w ~ N(0,1) */
void vin_normal(int64_t n, uint64_t seed, float *out) {
#pragma omp parallel for
    for (int64_t i = 0; i < n; ++i) {
        uint64_t s = mix64(seed ^ mix64(0x90121Aull + (uint64_t)i));
        const double u1 = rng_u01(&s), u2 = rng_u01(&s);
        out[i] = (float)(sqrt(-2.0 * log(u1)) * cos(2.0 * M_PI * u2));
    }
}
int vin_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
