/*
 * vmat_oracle.c — CPU ORACLE for the column-generation VMAT hot path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may call it.  It shares no code, header,
 * table or helper with the CUDA library under paper_1005_4396_b200/csrc (and neither side
 * includes or imports the other).
 *
 * Plain, slow, double precision.  Written from the paper (arxiv 1005.4396, Men, Romeijn, Jia,
 * Jiang); every function cites the passage of /root/reference/PAPER.md it follows ("PAPER.md:N")
 * or the DESIGN.md reading (S-number) it takes where the paper is silent.  D's fp32 entries and
 * the fp32 voxel parameters are used exactly (widened to double).
 *
 * Pins (tests/test_oracle_*.py, run with -m "not gpu"): dense hand products and scipy.sparse for
 * O2/O4; central finite differences and closed forms for O3; brute-force interval enumeration and
 * the textbook minimum-sum subarray for O5; the one-sided finite difference of the full cost for
 * O6; KKT conditions, scipy NNLS and one/two-aperture closed forms for O7; monotone cost and the
 * leaf-travel invariant for O8; for the dose-rate feasibility post-pass: feasibility at
 * exit, gamma = gamma_0 factor^rounds, infeasibility one round earlier (an independent master solve at
 * the previous gamma), and the two-beam closed form of the smoothed optimum.
 * PARITY UNPINNED: whole-plan numbers (the paper prints no worked example; Table 1 needs clinical
 * data that is not available).
 *
 * Build: gcc -O2 -fopenmp -ffp-contract=off -shared -fPIC vmat_oracle.c -o libvmat_oracle.so -lm
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    int64_t V, N, R, C;            /* voxels, beams, leaf rows per beam, beamlets per row; i=(k*R+r)*C+c */
    const int64_t *row_ptr;        /* B+1, beamlet-major CSR of D                          */
    const int32_t *col;            /* nnz voxel ids, ascending within a row                              */
    const float   *val;            /* nnz D_ij                                                           */
    const float   *T, *alpha, *beta; /* V each (Eq. 1)                                   */
    const double  *theta;          /* N gantry angles in degrees, ascending (reading S4)    */
    int32_t delta;                 /* max leaf travel in beamlets per angular step (reading S6)          */
    double  gamma;                 /* weight of the smoothing term (Eq. 3)               */
    int32_t g_occupied_only;       /* 0: Eq. 2 over all N angles, y = 0 at un-occupied beams (reading S2, default);
                                      1: over successive OCCUPIED beams only (the other reading of S2)    */
} vo_problem;

/* ------------------------------------------------------------------------------------------
 * O2 dose.  z_j = sum_k y_k sum_{i in A_k} D_ij            (Eq. 3)
 * A_k = beamlets (k,r,c) with left[k*R+r] <= c < right[k*R+r] of an occupied beam k.
 * ------------------------------------------------------------------------------------------ */
void vo_dose(const vo_problem *p, const uint8_t *occ, const int32_t *left, const int32_t *right,
             const double *y, double *z) {
    for (int64_t j = 0; j < p->V; ++j) z[j] = 0.0;
    for (int64_t k = 0; k < p->N; ++k) {
        if (!occ[k]) continue;
        for (int64_t r = 0; r < p->R; ++r)
            for (int64_t c = left[k * p->R + r]; c < right[k * p->R + r]; ++c) {
                const int64_t i = (k * p->R + r) * p->C + c;
                for (int64_t e = p->row_ptr[i]; e < p->row_ptr[i + 1]; ++e)
                    z[p->col[e]] += y[k] * (double)p->val[e];
            }
    }
}

/* ------------------------------------------------------------------------------------------
 * O3 voxel penalty and its derivative            (Eq. 1)
 *   F(z_j) = alpha_j max(0,T_j-z_j)^2 + beta_j max(0,z_j-T_j)^2
 *   w_j = dF/dz_j = -2 alpha_j max(0,T_j-z_j) + 2 beta_j max(0,z_j-T_j)
 * Returns F = sum_j F(z_j); w may be NULL.
 * ------------------------------------------------------------------------------------------ */
double vo_penalty(int64_t V, const double *z, const float *T, const float *alpha, const float *beta, double *w) {
    double F = 0.0;
#pragma omp parallel for reduction(+ : F) schedule(static)
    for (int64_t j = 0; j < V; ++j) {
        const double under = fmax(0.0, (double)T[j] - z[j]);
        const double over = fmax(0.0, z[j] - (double)T[j]);
        F += (double)alpha[j] * under * under + (double)beta[j] * over * over;
        if (w) w[j] = -2.0 * (double)alpha[j] * under + 2.0 * (double)beta[j] * over;
    }
    return F;
}

/* ------------------------------------------------------------------------------------------
 * O3 dose-rate smoothing                          (Eq. 2)
 *   G(y) = sum_{k=1}^{N-1} (y_{k+1}-y_k)^2 / (theta_{k+1}-theta_k)
 * over ALL N beams, y_k = 0 at un-occupied beams (reading S2), no wrap-around (S3), theta in
 * degrees (S4).  dG[k] = dG/dy_k with each operation individually rounded, in this order:
 *   dG[k] = 0; if k>0: dG[k] += 2*(y_k-y_{k-1})/(th_k-th_{k-1}); if k<N-1: dG[k] -= 2*(y_{k+1}-y_k)/(th_{k+1}-th_k)
 * dG may be NULL.
 * ------------------------------------------------------------------------------------------ */
double vo_smooth(int64_t N, const double *y, const double *theta, double *dG) {
    double G = 0.0;
    for (int64_t k = 0; k + 1 < N; ++k) {
        const double d = y[k + 1] - y[k];
        G += d * d / (theta[k + 1] - theta[k]);
    }
    if (dG)
        for (int64_t k = 0; k < N; ++k) {
            double s = 0.0;
            if (k > 0) s = s + 2.0 * (y[k] - y[k - 1]) / (theta[k] - theta[k - 1]);
            if (k + 1 < N) s = s - 2.0 * (y[k + 1] - y[k]) / (theta[k + 1] - theta[k]);
            dG[k] = s;
        }
    return G;
}

/* ------------------------------------------------------------------------------------------
 * O3, the other reading of S2: "successive gantry angles" are the successive angles that HOLD an
 * aperture; an un-occupied beam is not part of the arc yet and takes no part in Eq. 2:
 *   G(y) = sum over successive occupied beams p < k of (y_k - y_p)^2 / (theta_k - theta_p).
 * dG[k] for an occupied beam is dG/dy_k.  For an UN-occupied beam it is the derivative, at y_k = 0, of G with beam k
 * put into the arc between its nearest occupied neighbours: the smoothing part of the price of an aperture there
 * (reading S10).  Entering at y_k = 0 then changes G (unless the neighbours are at 0 too), so the post-master cost
 * of the loop is no longer guaranteed to be non-increasing in this reading.  Operations individually rounded, in
 * the order of vo_smooth.  dG may be NULL.
 * ------------------------------------------------------------------------------------------ */
double vo_smooth_occ(int64_t N, const double *y, const double *theta, const uint8_t *occ, double *dG) {
    double G = 0.0;
    int64_t prev = -1;
    for (int64_t k = 0; k < N; ++k) {
        if (!occ[k]) continue;
        if (prev >= 0) {
            const double d = y[k] - y[prev];
            G += d * d / (theta[k] - theta[prev]);
        }
        prev = k;
    }
    if (dG)
        for (int64_t k = 0; k < N; ++k) {
            int64_t p = k - 1, n = k + 1;
            while (p >= 0 && !occ[p]) --p;
            while (n < N && !occ[n]) ++n;
            const double yk = occ[k] ? y[k] : 0.0;
            double s = 0.0;
            if (p >= 0) s = s + 2.0 * (yk - y[p]) / (theta[k] - theta[p]);
            if (n < N) s = s - 2.0 * (y[n] - yk) / (theta[n] - theta[k]);
            dG[k] = s;
        }
    return G;
}

/* G and dG in the reading the problem asks for */
static double smooth_of(const vo_problem *p, const uint8_t *occ, const double *y, double *dG) {
    return p->g_occupied_only ? vo_smooth_occ(p->N, y, p->theta, occ, dG) : vo_smooth(p->N, y, p->theta, dG);
}

/* ------------------------------------------------------------------------------------------
 * O4 beamlet prices from the KKT conditions
 *   g_i = sum_j D_ij w_j  for every beamlet of every UN-occupied beam; 0 for occupied beams.
 * ------------------------------------------------------------------------------------------ */
void vo_prices(const vo_problem *p, const double *w, const uint8_t *occ, double *g) {
    const int64_t RC = p->R * p->C;
#pragma omp parallel for schedule(dynamic, 256)
    for (int64_t i = 0; i < p->N * RC; ++i) {
        double s = 0.0;
        if (!occ || !occ[i / RC])
            for (int64_t e = p->row_ptr[i]; e < p->row_ptr[i + 1]; ++e) s += (double)p->val[e] * w[p->col[e]];
        g[i] = s;
    }
}

/* O5 quantisation: q = llrint((double)g32 * 2^30), exact and order free. */
void vo_quantise(int64_t n, const float *g32, int64_t *q) {
    for (int64_t i = 0; i < n; ++i) q[i] = llrint((double)g32[i] * 1073741824.0);
}

/* ------------------------------------------------------------------------------------------
 * O5 leaf-travel box of one row of un-occupied beam k ("maximum leaf motion speed",
 * "By checking the shapes of existing neighboring MLC apertures"; reading S6: nearest occupied
 * beam on each side, travel budget delta*|k-k'|).  box = {Lmin, Lmax, Rmin, Rmax}.
 * ------------------------------------------------------------------------------------------ */
void vo_leaf_box(const vo_problem *p, const uint8_t *occ, const int32_t *left, const int32_t *right,
                 int64_t k, int64_t r, int64_t box[4]) {
    int64_t Lmin = 0, Lmax = p->C, Rmin = 0, Rmax = p->C;
    int64_t km = k - 1, kp = k + 1;
    while (km >= 0 && !occ[km]) --km;
    while (kp < p->N && !occ[kp]) ++kp;
    if (km >= 0) {
        const int64_t b = (int64_t)p->delta * (k - km), l = left[km * p->R + r], rr = right[km * p->R + r];
        if (l - b > Lmin) Lmin = l - b;
        if (l + b < Lmax) Lmax = l + b;
        if (rr - b > Rmin) Rmin = rr - b;
        if (rr + b < Rmax) Rmax = rr + b;
    }
    if (kp < p->N) {
        const int64_t b = (int64_t)p->delta * (kp - k), l = left[kp * p->R + r], rr = right[kp * p->R + r];
        if (l - b > Lmin) Lmin = l - b;
        if (l + b < Lmax) Lmax = l + b;
        if (rr - b > Rmin) Rmin = rr - b;
        if (rr + b < Rmax) Rmax = rr + b;
    }
    box[0] = Lmin; box[1] = Lmax; box[2] = Rmin; box[3] = Rmax;
}

/* ------------------------------------------------------------------------------------------
 * O5 best contiguous open interval of one leaf row, ONE left-to-right pass (PAPER.md:111:
 * "passing through all feasible beamlets in a row of a given beam from left to right only once").
 * q[c] = fixed-point price of beamlet c.  Open set = {c : l <= c < r'}, 0 <= l <= r' <= C,
 * Lmin<=l<=Lmax, Rmin<=r'<=Rmax.  Minimises the key (P[r']-P[l], r'-l, l) lexicographically
 * (value, then fewest open beamlets, then lowest index: readings S8, S9), P = prefix sums of q.
 * Sweep r' upward keeping the running maximum of P[l] over admissible l <= r' (later l wins ties,
 * which is the narrower interval).  Returns 0, or -1 if the box admits no interval.
 * ------------------------------------------------------------------------------------------ */
int vo_row_search(int64_t C, const int64_t *q, int64_t Lmin, int64_t Lmax, int64_t Rmin, int64_t Rmax,
                  int32_t *l_out, int32_t *r_out, int64_t *value_out) {
    int64_t P = 0, maxP = 0, argl = -1;
    int64_t bv = 0, bw = 0, bl = -1, br = -1;
    for (int64_t pos = 0; pos <= C; ++pos) {
        if (pos > 0) P += q[pos - 1];                              /* P[pos] */
        if (pos >= Lmin && pos <= Lmax && (argl < 0 || P >= maxP)) { maxP = P; argl = pos; }
        if (pos >= Rmin && pos <= Rmax && argl >= 0) {
            const int64_t v = P - maxP, wd = pos - argl;
            if (bl < 0 || v < bv || (v == bv && (wd < bw || (wd == bw && argl < bl)))) { bv = v; bw = wd; bl = argl; br = pos; }
        }
    }
    if (bl < 0) return -1;
    *l_out = (int32_t)bl; *r_out = (int32_t)br; *value_out = bv;
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * O5 + O6 pricing step: best deliverable aperture over all un-occupied beams ("the
 * most promising MLC aperture from all un-occupied beam directions").
 *   g32      B fp32 prices (the hand-over format between pricing and search)
 *   y        N current intensities (0 at un-occupied beams)
 * For each un-occupied beam k:  value_k = sum_r (row minimum, int64),
 *   price_k = ldexp((double)value_k, -30) + gamma * dG/dy_k          (reading S10: the reduced cost)
 * with each operation individually rounded (-ffp-contract=off).  Chooses the smallest price,
 * lowest k on ties (S9).  Outputs (any may be NULL): beam_price[N] (+inf at occupied beams),
 * all_left/all_right [N*R] (row optimum of every un-occupied beam; untouched at occupied),
 * best_left/best_right [R].  A beam with a row whose leaf-travel box admits no interval is undeliverable
 * ("all the deliverability constraints"): price +inf, rows reported as (-1, -1), never chosen.
 * Returns the chosen beam, or -1 if no un-occupied beam is deliverable.
 * ------------------------------------------------------------------------------------------ */
int64_t vo_price_step(const vo_problem *p, const float *g32, const uint8_t *occ, const int32_t *left,
                      const int32_t *right, const double *y, double *best_price, int32_t *best_left,
                      int32_t *best_right, double *beam_price, int32_t *all_left, int32_t *all_right) {
    const int64_t N = p->N, R = p->R, C = p->C;
    double *dG = (double *)malloc(sizeof(double) * N);
    int64_t *q = (int64_t *)malloc(sizeof(int64_t) * C);
    int32_t *tl = (int32_t *)malloc(sizeof(int32_t) * R), *tr = (int32_t *)malloc(sizeof(int32_t) * R);
    smooth_of(p, occ, y, dG);
    int64_t best = -1;
    double bp = 0.0;
    for (int64_t k = 0; k < N; ++k) {
        if (beam_price) beam_price[k] = INFINITY;
        if (occ[k]) continue;
        int64_t total = 0;
        int deliverable = 1;
        for (int64_t r = 0; r < R; ++r) {
            int64_t box[4], v = 0;
            vo_leaf_box(p, occ, left, right, k, r, box);
            vo_quantise(C, g32 + (k * R + r) * C, q);
            if (vo_row_search(C, q, box[0], box[1], box[2], box[3], &tl[r], &tr[r], &v) != 0) {
                /* the box admits no interval (only possible if the occupied apertures themselves break the
                 * leaf-travel limit): this beam has no deliverable aperture and cannot be chosen */
                deliverable = 0; tl[r] = -1; tr[r] = -1; v = 0;
            }
            total += v;
            if (all_left) { all_left[k * R + r] = tl[r]; all_right[k * R + r] = tr[r]; }
        }
        if (!deliverable) continue;                                /* beam_price[k] stays +inf */
        const double smooth = p->gamma * dG[k];
        const double price = ldexp((double)total, -30) + smooth;
        if (beam_price) beam_price[k] = price;
        if (best < 0 || price < bp) {
            best = k; bp = price;
            if (best_left) { memcpy(best_left, tl, sizeof(int32_t) * R); memcpy(best_right, tr, sizeof(int32_t) * R); }
        }
    }
    if (best >= 0 && best_price) *best_price = bp;
    free(dG); free(q); free(tl); free(tr);
    return best;
}

/* ------------------------------------------------------------------------------------------
 * Aperture-dose column d_k = sum_{i in A_k} D_i.  (implied by the master problem over fixed A_k,
 * PAPER.md:113), stored sparse: ascending voxel ids + values.  Returns the column length.
 * idx/val need room for V entries; scratch is V doubles, all zero on entry and on exit.
 * ------------------------------------------------------------------------------------------ */
int64_t vo_aperture_column(const vo_problem *p, int64_t k, const int32_t *left, const int32_t *right,
                           double *scratch, uint8_t *mark, int32_t *idx, double *val) {
    int64_t lo = p->V, hi = -1, n = 0;
    for (int64_t r = 0; r < p->R; ++r)
        for (int64_t c = left[k * p->R + r]; c < right[k * p->R + r]; ++c) {
            const int64_t i = (k * p->R + r) * p->C + c;
            for (int64_t e = p->row_ptr[i]; e < p->row_ptr[i + 1]; ++e) {
                const int64_t j = p->col[e];
                scratch[j] += (double)p->val[e];
                mark[j] = 1;
                if (j < lo) lo = j;
                if (j > hi) hi = j;
            }
        }
    for (int64_t j = lo; j <= hi; ++j)
        if (mark[j]) { idx[n] = (int32_t)j; val[n] = scratch[j]; ++n; scratch[j] = 0.0; mark[j] = 0; }
    return n;
}

/* sparse aperture-dose columns of the occupied beams */
typedef struct {
    int64_t N, V;
    int64_t *len;       /* N, 0 for un-occupied */
    int32_t **idx;      /* N */
    double **val;       /* N */
    double *scratch;    /* V */
    uint8_t *mark;      /* V */
} vo_columns;

static vo_columns *columns_new(int64_t N, int64_t V) {
    vo_columns *c = (vo_columns *)calloc(1, sizeof(vo_columns));
    c->N = N; c->V = V;
    c->len = (int64_t *)calloc(N, sizeof(int64_t));
    c->idx = (int32_t **)calloc(N, sizeof(int32_t *));
    c->val = (double **)calloc(N, sizeof(double *));
    c->scratch = (double *)calloc(V, sizeof(double));
    c->mark = (uint8_t *)calloc(V, 1);
    return c;
}
static void columns_free(vo_columns *c) {
    for (int64_t k = 0; k < c->N; ++k) { free(c->idx[k]); free(c->val[k]); }
    free(c->len); free(c->idx); free(c->val); free(c->scratch); free(c->mark); free(c);
}
static void columns_add(vo_columns *c, const vo_problem *p, int64_t k, const int32_t *left, const int32_t *right) {
    int32_t *idx = (int32_t *)malloc(sizeof(int32_t) * p->V);
    double *val = (double *)malloc(sizeof(double) * p->V);
    const int64_t n = vo_aperture_column(p, k, left, right, c->scratch, c->mark, idx, val);
    free(c->idx[k]); free(c->val[k]);
    c->idx[k] = (int32_t *)malloc(sizeof(int32_t) * (n ? n : 1));
    c->val[k] = (double *)malloc(sizeof(double) * (n ? n : 1));
    memcpy(c->idx[k], idx, sizeof(int32_t) * n);
    memcpy(c->val[k], val, sizeof(double) * n);
    c->len[k] = n;
    free(idx); free(val);
}

/* z = sum_k y_k d_k over occupied beams (O2 written with the precomputed inner sums) */
static void columns_dose(const vo_columns *c, const uint8_t *occ, const double *y, double *z) {
    for (int64_t j = 0; j < c->V; ++j) z[j] = 0.0;
    for (int64_t k = 0; k < c->N; ++k)
        if (occ[k])
            for (int64_t e = 0; e < c->len[k]; ++e) z[c->idx[k][e]] += y[k] * c->val[k][e];
}

/* full gradient of Phi = F + gamma G with respect to y at occupied beams: grad_k = d_k.w + gamma dG_k */
static void master_gradient(const vo_problem *p, const vo_columns *c, const uint8_t *occ, const double *w,
                            const double *dG, double *grad) {
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t k = 0; k < c->N; ++k) {
        double s = 0.0;
        if (occ[k]) {
            for (int64_t e = 0; e < c->len[k]; ++e) s += c->val[k][e] * w[c->idx[k][e]];
            s += p->gamma * dG[k];
        }
        grad[k] = s;
    }
}

typedef struct {
    double eps;           /* stop when max|projected gradient| <= eps*max(1, the same norm at entry) */
    int64_t max_inner;    /* iteration cap                                                           */
    double lb, ub;        /* bounds on the dose rates of occupied beams: lb <= y_k <= ub (default 0, +inf)  */
    /* outputs */
    int64_t inner;        /* iterations done                                                         */
    int64_t backtracks;   /* step halvings                                                           */
    double pg_entry, pg_exit; /* max|projected gradient| at entry / exit                             */
    double F, G, cost;    /* at exit                                                                 */
} vo_master_info;

/* ------------------------------------------------------------------------------------------
 * O7 master problem ("The master problem is to solve our VMAT optimization model
 * (3) with optimized A_k. The gradient projection method is used"; Eq. 3):
 *     minimise  Phi(y) = F(z(y)) + gamma G(y)   over  y_k >= 0 (occupied), y_k = 0 (un-occupied).
 * Convex, so the optimal COST is unique; the result is DEFINED as that minimiser (reading S11) and
 * pinned by the KKT conditions.  Method: gradient projection (Rosen / Bazaraa, paper ref 21) on
 * the bounds y >= 0, warm started from the incoming y, with Polak-Ribiere conjugate directions on
 * the current face (restart = plain projected steepest descent whenever the active set changes):
 *   grad = Dc w + gamma dG;  projected gradient pg_k = grad_k, except 0 where y_k = 0 and grad_k >= 0
 *   direction d (first: -pg);  q = Dc^T d
 *   trial step t = -phi'(0)/phi''(0),  phi'(0) = grad.d,
 *        phi''(0) = 2 sum_j omega_j q_j^2 + 2 gamma d^T L d,  omega_j = alpha_j (z_j<T_j), beta_j (z_j>T_j), else 0
 *   clipped to t_max = min_{d_k<0} y_k/(-d_k);  halved until the sufficient-decrease test holds on the
 *   TRUE Phi (c1 = 1e-4);  y += t d (clamped at 0), z += t q.
 * Two products with Dc per inner iteration = the "aperture-dose GEMV pair".
 * y is updated in place; z (V) receives sum_k y_k d_k recomputed from the final y.
 *
 * Variant (PAPER.md:159 names "the maximum and minimum dose rate constraints" and leaves them
 * out of "this preliminary work"): bounds lb <= y_k <= ub on the occupied beams (reading R4 of DESIGN.md:
 * un-occupied beams deliver nothing, y_k = 0).  Gradient projection on a box instead of on y >= 0: pg_k = 0
 * also where y_k = ub and grad_k <= 0, t_max also limited by (ub - y_k)/d_k for d_k > 0.  With lb = 0,
 * ub = +inf every expression below reduces to the one above, bit for bit.
 * ------------------------------------------------------------------------------------------ */
static void master_solve(const vo_problem *p, const vo_columns *cols, const uint8_t *occ, double *y, double *z,
                         vo_master_info *info) {
    const int64_t N = p->N, V = p->V;
    double *w = (double *)malloc(sizeof(double) * V), *q = (double *)malloc(sizeof(double) * V);
    double *zn = (double *)malloc(sizeof(double) * V), *wn = (double *)malloc(sizeof(double) * V);
    double *dG = (double *)malloc(sizeof(double) * N), *grad = (double *)malloc(sizeof(double) * N);
    double *gradn = (double *)malloc(sizeof(double) * N), *pg = (double *)malloc(sizeof(double) * N);
    double *pgn = (double *)malloc(sizeof(double) * N), *d = (double *)calloc(N, sizeof(double));
    double *yn = (double *)malloc(sizeof(double) * N);
    const double c1 = 1e-4;
    const double lb = info->lb, ub = info->ub;

    for (int64_t k = 0; k < N; ++k) {
        if (!occ[k]) y[k] = 0.0;
        else if (y[k] < lb) y[k] = lb;
        else if (y[k] > ub) y[k] = ub;
    }
    columns_dose(cols, occ, y, z);
    double F = vo_penalty(V, z, p->T, p->alpha, p->beta, w);
    double G = smooth_of(p, occ, y, dG);
    double Phi = F + p->gamma * G;
    master_gradient(p, cols, occ, w, dG, grad);
    double pgmax = 0.0;
    for (int64_t k = 0; k < N; ++k) {
        pg[k] = (!occ[k] || (y[k] <= lb && grad[k] >= 0.0) || (y[k] >= ub && grad[k] <= 0.0)) ? 0.0 : grad[k];
        d[k] = -pg[k];
        if (fabs(pg[k]) > pgmax) pgmax = fabs(pg[k]);
    }
    info->pg_entry = pgmax;
    const double tol = info->eps * fmax(1.0, pgmax);
    info->inner = 0; info->backtracks = 0;

    while (pgmax > tol && info->inner < info->max_inner) {
        /* slope; fall back to steepest descent if d is not a descent direction */
        double phi1 = 0.0;
        for (int64_t k = 0; k < N; ++k) phi1 += grad[k] * d[k];
        if (!(phi1 < 0.0)) {
            phi1 = 0.0;
            for (int64_t k = 0; k < N; ++k) { d[k] = -pg[k]; phi1 += grad[k] * d[k]; }
            if (!(phi1 < 0.0)) break;
        }
        /* q = Dc^T d */
        for (int64_t j = 0; j < V; ++j) q[j] = 0.0;
        for (int64_t k = 0; k < N; ++k)
            if (occ[k] && d[k] != 0.0)
                for (int64_t e = 0; e < cols->len[k]; ++e) q[cols->idx[k][e]] += d[k] * cols->val[k][e];
        /* curvature of the quadratic piece at t = 0 */
        double curvF = 0.0;
#pragma omp parallel for reduction(+ : curvF) schedule(static)
        for (int64_t j = 0; j < V; ++j) {
            const double om = z[j] < (double)p->T[j] ? (double)p->alpha[j] : (z[j] > (double)p->T[j] ? (double)p->beta[j] : 0.0);
            curvF += om * q[j] * q[j];
        }
        const double phi2 = 2.0 * curvF + 2.0 * p->gamma * smooth_of(p, occ, d, NULL); /* d^T L d = G(d) */
        double tmax = INFINITY;
        for (int64_t k = 0; k < N; ++k) {
            if (d[k] < 0.0 && (y[k] - lb) / (-d[k]) < tmax) tmax = (y[k] - lb) / (-d[k]);
            if (d[k] > 0.0 && (ub - y[k]) / d[k] < tmax) tmax = (ub - y[k]) / d[k];
        }
        double t = phi2 > 0.0 ? -phi1 / phi2 : (isfinite(tmax) ? tmax : 1.0);
        int hit = 0;
        if (t >= tmax) { t = tmax; hit = 1; }
        /* backtracking on the true cost */
        int accepted = 0;
        double Fn = 0.0, Gn = 0.0, Phin = 0.0;
        for (int half = 0; half < 80; ++half) {
            for (int64_t k = 0; k < N; ++k) {
                yn[k] = y[k] + t * d[k];
                if (!occ[k]) continue;
                if (yn[k] < lb || (hit && d[k] < 0.0 && (y[k] - lb) / (-d[k]) <= tmax)) yn[k] = lb;
                else if (yn[k] > ub || (hit && d[k] > 0.0 && (ub - y[k]) / d[k] <= tmax)) yn[k] = ub;
            }
#pragma omp parallel for schedule(static)
            for (int64_t j = 0; j < V; ++j) zn[j] = z[j] + t * q[j];
            Fn = vo_penalty(V, zn, p->T, p->alpha, p->beta, wn);
            Gn = smooth_of(p, occ, yn, dG);
            Phin = Fn + p->gamma * Gn;
            if (Phin <= Phi + c1 * t * phi1) { accepted = 1; break; }
            /* below the resolution of Phi: accept on the slope instead (|phi'(t)| <= 0.9 |phi'(0)|) */
            if (Phin <= Phi + 1e-13 * fabs(Phi)) {
                master_gradient(p, cols, occ, wn, dG, gradn);
                double phi1n = 0.0;
                for (int64_t k = 0; k < N; ++k) phi1n += gradn[k] * d[k];
                if (fabs(phi1n) <= 0.9 * fabs(phi1)) { accepted = 1; break; }
            }
            t *= 0.5; hit = 0; ++info->backtracks;
        }
        if (!accepted) break;
        /* take the step */
        int changed = hit;
        for (int64_t k = 0; k < N; ++k) y[k] = yn[k];
        memcpy(z, zn, sizeof(double) * V);
        memcpy(w, wn, sizeof(double) * V);
        F = Fn; G = Gn; Phi = Phin;
        master_gradient(p, cols, occ, w, dG, gradn);
        double num = 0.0, den = 0.0;
        pgmax = 0.0;
        for (int64_t k = 0; k < N; ++k) {
            pgn[k] = (!occ[k] || (y[k] <= lb && gradn[k] >= 0.0) || (y[k] >= ub && gradn[k] <= 0.0)) ? 0.0 : gradn[k];
            if ((pgn[k] == 0.0) != (pg[k] == 0.0)) changed = 1;        /* a bound was hit or released */
            num += pgn[k] * (pgn[k] - pg[k]);
            den += pg[k] * pg[k];
            if (fabs(pgn[k]) > pgmax) pgmax = fabs(pgn[k]);
        }
        const double bpr = (changed || !(den > 0.0) || num <= 0.0) ? 0.0 : num / den;   /* PR+, restart on face change */
        for (int64_t k = 0; k < N; ++k) {
            d[k] = -pgn[k] + bpr * d[k];
            if (!occ[k] || (y[k] <= lb && d[k] < 0.0) || (y[k] >= ub && d[k] > 0.0)) d[k] = 0.0;      /* stay feasible */
            grad[k] = gradn[k]; pg[k] = pgn[k];
        }
        ++info->inner;
    }
    info->pg_exit = pgmax;
    columns_dose(cols, occ, y, z);                                     /* z from the final y, no drift */
    info->F = vo_penalty(V, z, p->T, p->alpha, p->beta, NULL);
    info->G = smooth_of(p, occ, y, NULL);
    info->cost = info->F + p->gamma * info->G;
    free(w); free(q); free(zn); free(wn); free(dG); free(grad); free(gradn); free(pg); free(pgn); free(d); free(yn);
}

/* Stand-alone O7: master solve for a given aperture set. */
void vo_master(const vo_problem *p, const uint8_t *occ, const int32_t *left, const int32_t *right, double *y,
               double *z, vo_master_info *info) {
    vo_columns *cols = columns_new(p->N, p->V);
    for (int64_t k = 0; k < p->N; ++k) if (occ[k]) columns_add(cols, p, k, left, right);
    master_solve(p, cols, occ, y, z, info);
    columns_free(cols);
}

/* ---- hard dose-rate feasibility after the last aperture -----------------------------
 * "In the optimization model, we add dose rate constraints as penalty-based soft constraints in the cost
 *  function.  However, these constraints need to be satisfied as hard constraints. [...] if the final
 *  solution is not feasible, the coefficient gamma in the objective function will be automatically
 *  increased and then the intensity for each aperture will be re-optimized till the solution is feasible."
 * The constraint itself is PAPER.md:80: "the dose rate variation between neighboring angles is constrained
 * within a certain range".  Readings (R1-R3): the range is
 *     |y_{k+1} - y_k| <= rho * (theta_{k+1} - theta_k)   for k = 1..N-1   (rho: intensity change per degree),
 * "increased" is a multiplication of gamma by `factor` (the paper gives no rule), and the incoming y is
 * tested first: a feasible plan is returned untouched with zero rounds.
 *
 * ratio = max_k |y_{k+1} - y_k| / (rho (theta_{k+1} - theta_k));  feasible iff ratio <= 1 + tol. */
double vo_rate_ratio(int64_t N, const double *y, const double *theta, double rho) {
    double r = 0.0;
    for (int64_t k = 0; k + 1 < N; ++k) {
        const double v = fabs(y[k + 1] - y[k]) / (rho * (theta[k + 1] - theta[k]));
        if (v > r) r = v;
    }
    return r;
}

typedef struct {
    double  rho, factor, tol;      /* in */
    int64_t max_rounds;            /* in */
    double  eps;                   /* in: master tolerance */
    int64_t max_inner;             /* in */
    int64_t rounds;                /* out: number of times gamma was raised and the master re-solved */
    int64_t feasible;              /* out */
    double  gamma;                 /* out: gamma at exit = gamma_0 * factor^rounds */
    double  ratio;                 /* out: ratio at exit */
    double  F, G, cost;            /* out: at exit, cost = F + gamma G with the gamma at exit */
} vo_rate_info;

void vo_enforce_rate(const vo_problem *p, const uint8_t *occ, const int32_t *left, const int32_t *right, double *y,
                     double *z, vo_rate_info *info) {
    vo_problem q = *p;
    vo_columns *cols = columns_new(p->N, p->V);
    for (int64_t k = 0; k < p->N; ++k) if (occ[k]) columns_add(cols, p, k, left, right);
    double ratio = vo_rate_ratio(p->N, y, p->theta, info->rho);
    int64_t rounds = 0;
    while (ratio > 1.0 + info->tol && rounds < info->max_rounds) {
        q.gamma *= info->factor;                                   /* "gamma ... automatically increased"   */
        vo_master_info mi;
        mi.eps = info->eps;
        mi.max_inner = info->max_inner;
        mi.lb = 0.0;
        mi.ub = INFINITY;
        master_solve(&q, cols, occ, y, z, &mi);                    /* "intensity ... re-optimized"          */
        ++rounds;
        ratio = vo_rate_ratio(p->N, y, p->theta, info->rho);       /* "till the solution is feasible"       */
    }
    columns_dose(cols, occ, y, z);
    info->rounds = rounds;
    info->feasible = ratio <= 1.0 + info->tol;
    info->gamma = q.gamma;
    info->ratio = ratio;
    info->F = vo_penalty(p->V, z, p->T, p->alpha, p->beta, NULL);
    info->G = smooth_of(p, occ, y, NULL);
    info->cost = info->F + q.gamma * info->G;
    columns_free(cols);
}

/* Full gradient dPhi/dy_k at the occupied beams for a given plan (used by the KKT pin). */
void vo_cost_gradient(const vo_problem *p, const uint8_t *occ, const int32_t *left, const int32_t *right,
                      const double *y, double *grad, double *cost3) {
    vo_columns *cols = columns_new(p->N, p->V);
    double *z = (double *)malloc(sizeof(double) * p->V), *w = (double *)malloc(sizeof(double) * p->V);
    double *dG = (double *)malloc(sizeof(double) * p->N);
    for (int64_t k = 0; k < p->N; ++k) if (occ[k]) columns_add(cols, p, k, left, right);
    columns_dose(cols, occ, y, z);
    const double F = vo_penalty(p->V, z, p->T, p->alpha, p->beta, w);
    const double G = smooth_of(p, occ, y, dG);
    master_gradient(p, cols, occ, w, dG, grad);
    if (cost3) { cost3[0] = F; cost3[1] = G; cost3[2] = F + p->gamma * G; }
    free(z); free(w); free(dG);
    columns_free(cols);
}

/* per-iteration record of the column-generation loop */
typedef struct {
    int64_t max_iters;
    double eps;               /* master tolerance */
    int64_t max_inner;
    int64_t stop_when_priced_out; /* option of reading S5: stop as soon as the best price is >= 0 */
    double lb, ub;            /* bounds on the dose rates of occupied beams in every master solve (variant of
                                 PAPER.md:159, reading R4; 0 and +inf = the paper's y >= 0)                  */
    /* outputs, arrays caller-allocated with max_iters entries (leaf arrays max_iters*R) */
    int64_t iters;            /* outer iterations done */
    int32_t *beam;            /* chosen beam */
    double *price;            /* its price */
    double *F, *G, *cost;     /* after the master solve */
    int64_t *inner;           /* master inner iterations */
    int32_t *it_left, *it_right; /* leaf pairs of the chosen aperture */
    double seconds_price, seconds_master;
} vo_trace;

static double now_s(void) {
#ifdef _OPENMP
    return omp_get_wtime();
#else
    return 0.0;
#endif
}

/* ------------------------------------------------------------------------------------------
 * O1 + O8 column-generation loop (Fig. 1 is missing from the extraction).
 * O1: start from the empty plan, y = 0, z = 0 (reading S1).  Each iteration: gradient (O3),
 * prices (O4, rounded to fp32 for the search), best aperture (O5, O6), occupy that beam with
 * y_k = 0, master (O7).  Stops when every beam is occupied or after max_iters (reading S5); with
 * stop_when_priced_out also as soon as no aperture has a negative price (the textbook column-generation
 * stop, offered as an option because the paper wants an aperture at every angle).
 * State arrays (occ N, left/right N*R, y N, z V) are caller allocated; on entry they hold the
 * plan to continue from (all zero for a fresh run).  With bounds lb <= y_k <= ub on the occupied beams (variant,
 * reading R4) the prices are unchanged (the reduced cost of the paper at the current y); a beam that enters is
 * brought into the box by its first master solve.
 * ------------------------------------------------------------------------------------------ */
void vo_solve(const vo_problem *p, uint8_t *occ, int32_t *left, int32_t *right, double *y, double *z, vo_trace *tr) {
    const int64_t N = p->N, R = p->R, B = p->N * p->R * p->C;
    vo_columns *cols = columns_new(N, p->V);
    double *w = (double *)malloc(sizeof(double) * p->V), *g = (double *)malloc(sizeof(double) * B);
    float *g32 = (float *)malloc(sizeof(float) * B);
    int32_t *bl = (int32_t *)malloc(sizeof(int32_t) * R), *br = (int32_t *)malloc(sizeof(int32_t) * R);
    for (int64_t k = 0; k < N; ++k) if (occ[k]) columns_add(cols, p, k, left, right);
    columns_dose(cols, occ, y, z);
    tr->iters = 0; tr->seconds_price = 0.0; tr->seconds_master = 0.0;
    for (int64_t it = 0; it < tr->max_iters; ++it) {
        double t0 = now_s();
        vo_penalty(p->V, z, p->T, p->alpha, p->beta, w);
        vo_prices(p, w, occ, g);
        for (int64_t i = 0; i < B; ++i) g32[i] = (float)g[i];
        double price = 0.0;
        const int64_t k = vo_price_step(p, g32, occ, left, right, y, &price, bl, br, NULL, NULL, NULL);
        if (k < 0) break;
        if (tr->stop_when_priced_out && !(price < 0.0)) break;
        occ[k] = 1; y[k] = 0.0;
        memcpy(left + k * R, bl, sizeof(int32_t) * R);
        memcpy(right + k * R, br, sizeof(int32_t) * R);
        columns_add(cols, p, k, left, right);
        double t1 = now_s();
        vo_master_info info; memset(&info, 0, sizeof(info));
        info.eps = tr->eps; info.max_inner = tr->max_inner;
        info.lb = tr->lb; info.ub = tr->ub;                        /* the new beam enters at y = 0 and is brought to lb */
        master_solve(p, cols, occ, y, z, &info);
        double t2 = now_s();
        tr->seconds_price += t1 - t0; tr->seconds_master += t2 - t1;
        if (tr->beam) tr->beam[it] = (int32_t)k;
        if (tr->price) tr->price[it] = price;
        if (tr->F) tr->F[it] = info.F;
        if (tr->G) tr->G[it] = info.G;
        if (tr->cost) tr->cost[it] = info.cost;
        if (tr->inner) tr->inner[it] = info.inner;
        if (tr->it_left) { memcpy(tr->it_left + it * R, bl, sizeof(int32_t) * R); memcpy(tr->it_right + it * R, br, sizeof(int32_t) * R); }
        tr->iters = it + 1;
    }
    free(w); free(g); free(g32); free(bl); free(br);
    columns_free(cols);
}

int vo_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
void vo_set_num_threads(int n) {
#ifdef _OPENMP
    omp_set_num_threads(n);
#else
    (void)n;
#endif
}
