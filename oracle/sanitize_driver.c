/*
 * sanitize_driver.c — TEST INFRASTRUCTURE: runs every entry point of the CPU oracle (vmat_oracle.c, included below)
 * on a small seeded random problem so that the whole file can be built with
 *     gcc -O1 -g -fsanitize=address,undefined -fno-sanitize-recover=all -ffp-contract=off sanitize_driver.c -lm
 * and executed under AddressSanitizer / UndefinedBehaviorSanitizer (tests/test_oracle_sanitizers.py, SURVEY.md
 * section 5).  It checks nothing numerically (the pins do that); it exits 0 if every call returns.
 */
#include "vmat_oracle.c"

#include <stdio.h>

static uint64_t rng_state = 0x9E3779B97F4A7C15ull;
static double rnd(void) {              /* xorshift64*, uniform in [0,1) */
    rng_state ^= rng_state >> 12; rng_state ^= rng_state << 25; rng_state ^= rng_state >> 27;
    return (double)((rng_state * 0x2545F4914F6CDD1Dull) >> 11) / 9007199254740992.0;
}

int main(void) {
    const int64_t V = 90, N = 7, R = 3, C = 9, B = N * R * C;
    int64_t *row_ptr = (int64_t *)calloc(B + 1, sizeof(int64_t));
    int32_t *col = (int32_t *)malloc(sizeof(int32_t) * B * V);
    float *val = (float *)malloc(sizeof(float) * B * V);
    int64_t nnz = 0;
    for (int64_t i = 0; i < B; ++i) {
        if (i % 11 != 3)                                   /* a few empty rows */
            for (int64_t j = 0; j < V; ++j)
                if (rnd() < 0.2) { col[nnz] = (int32_t)j; val[nnz] = (float)(0.05 + rnd()); ++nnz; }
        row_ptr[i + 1] = nnz;
    }
    float *T = (float *)malloc(sizeof(float) * V), *al = (float *)malloc(sizeof(float) * V), *be = (float *)malloc(sizeof(float) * V);
    for (int64_t j = 0; j < V; ++j) { T[j] = (float)(0.2 + 0.8 * rnd()); al[j] = rnd() < 0.5 ? (float)(0.5 + rnd()) : 0.f; be[j] = (float)(0.1 + rnd()); }
    double *theta = (double *)malloc(sizeof(double) * N);
    for (int64_t k = 0; k < N; ++k) theta[k] = 2.0 * (double)k + 0.5 * rnd();
    vo_problem p = {V, N, R, C, row_ptr, col, val, T, al, be, theta, 2, 0.3, 0};

    uint8_t *occ = (uint8_t *)calloc(N, 1);
    int32_t *left = (int32_t *)calloc(N * R, sizeof(int32_t)), *right = (int32_t *)calloc(N * R, sizeof(int32_t));
    double *y = (double *)calloc(N, sizeof(double)), *z = (double *)calloc(V, sizeof(double));
    int32_t *beam = (int32_t *)malloc(sizeof(int32_t) * N), *il = (int32_t *)malloc(sizeof(int32_t) * N * R), *ir = (int32_t *)malloc(sizeof(int32_t) * N * R);
    double *price = (double *)malloc(sizeof(double) * N), *F = (double *)malloc(sizeof(double) * N), *G = (double *)malloc(sizeof(double) * N), *cost = (double *)malloc(sizeof(double) * N);
    int64_t *inner = (int64_t *)malloc(sizeof(int64_t) * N);

    /* the loop in two legs (resume from a plan), then every stand-alone entry point on the finished plan */
    vo_trace tr; memset(&tr, 0, sizeof(tr));
    tr.max_iters = 3; tr.eps = 1e-9; tr.max_inner = 2000; tr.lb = 0.0; tr.ub = INFINITY;
    tr.beam = beam; tr.price = price; tr.F = F; tr.G = G; tr.cost = cost; tr.inner = inner; tr.it_left = il; tr.it_right = ir;
    vo_solve(&p, occ, left, right, y, z, &tr);
    tr.max_iters = N;
    vo_solve(&p, occ, left, right, y, z, &tr);

    double *w = (double *)malloc(sizeof(double) * V), *g = (double *)malloc(sizeof(double) * B), *dG = (double *)malloc(sizeof(double) * N);
    float *g32 = (float *)malloc(sizeof(float) * B);
    vo_dose(&p, occ, left, right, y, z);
    vo_penalty(V, z, T, al, be, w);
    vo_smooth(N, y, theta, dG);
    occ[2] = 0; occ[5] = 0; y[2] = 0.0; y[5] = 0.0;
    vo_prices(&p, w, occ, g);
    for (int64_t i = 0; i < B; ++i) g32[i] = (float)g[i];
    double bp = 0.0, *beam_price = (double *)malloc(sizeof(double) * N);
    int32_t *bl = (int32_t *)malloc(sizeof(int32_t) * R), *br = (int32_t *)malloc(sizeof(int32_t) * R);
    int32_t *al_ = (int32_t *)malloc(sizeof(int32_t) * N * R), *ar_ = (int32_t *)malloc(sizeof(int32_t) * N * R);
    vo_price_step(&p, g32, occ, left, right, y, &bp, bl, br, beam_price, al_, ar_);
    occ[2] = 1; occ[5] = 1;
    vo_master_info mi; memset(&mi, 0, sizeof(mi));
    mi.eps = 1e-9; mi.max_inner = 2000; mi.lb = 0.01; mi.ub = 0.5;
    vo_master(&p, occ, left, right, y, z, &mi);
    double c3[3], *grad = (double *)malloc(sizeof(double) * N);
    vo_cost_gradient(&p, occ, left, right, y, grad, c3);
    vo_rate_info ri; memset(&ri, 0, sizeof(ri));
    ri.rho = 0.25 * vo_rate_ratio(N, y, theta, 1.0); ri.factor = 2.0; ri.tol = 1e-6; ri.max_rounds = 8; ri.eps = 1e-9; ri.max_inner = 2000;
    vo_enforce_rate(&p, occ, left, right, y, z, &ri);
    int64_t box[4];
    vo_leaf_box(&p, occ, left, right, 3, 1, box);
    /* the other reading of Eq. 2 (smoothing over the occupied beams only): the loop again from an empty plan */
    p.g_occupied_only = 1;
    memset(occ, 0, N); memset(y, 0, sizeof(double) * N);
    tr.max_iters = N;
    vo_solve(&p, occ, left, right, y, z, &tr);
    vo_smooth_occ(N, y, theta, occ, dG);
    printf("sanitize_driver ok: %lld iterations, cost %.6f, %lld rounds\n", (long long)tr.iters, c3[2], (long long)ri.rounds);

    free(row_ptr); free(col); free(val); free(T); free(al); free(be); free(theta); free(occ); free(left); free(right);
    free(y); free(z); free(beam); free(il); free(ir); free(price); free(F); free(G); free(cost); free(inner); free(w);
    free(g); free(dG); free(g32); free(beam_price); free(bl); free(br); free(al_); free(ar_); free(grad);
    return 0;
}
