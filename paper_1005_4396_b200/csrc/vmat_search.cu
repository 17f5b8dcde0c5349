// vmat_search.cu — step (d): per leaf row the contiguous open interval of least total price
// inside the leaf-travel box, the per-beam sum and the choice of the best un-occupied beam
// ("passing through all feasible beamlets in a row of a given beam from left to
// right only once", "By checking the shapes of existing neighboring MLC apertures", "the most
// promising MLC aperture from all un-occupied beam directions").
//
// Integer work throughout: prices are quantised to int64 fixed point, q_c = rn(g_c * 2^30), so
// prefix sums are exact and independent of evaluation order (reading S9 / O5).  One
// warp owns one leaf row: positions 0..C are dealt to the lanes in blocks of M, the prefix sums
// P, the running maximum of P[l] over admissible l (later l wins ties) and the minimum of the key
// (P[r']-P[l], r'-l, l) are warp-shuffle scans/reductions.  A block owns kRowsPerBlock rows of one
// beam; row optima are added to the beam's total with integer atomics (exact, order free); the last
// block of a beam forms its price, the last block of all picks the beam (smallest price, lowest k
// on ties) and commits it on request.
#include <math_constants.h>

#include "vmat_internal.cuh"

namespace vmat {

namespace {

constexpr unsigned kFull = 0xffffffffu;
constexpr int kSearchThreads = 256;
constexpr int kRowsPerBlock = kSearchThreads / 32;   // one warp per leaf row
constexpr int kMaxListChunks = 64;                   // chunks of 32 beams in the list of un-occupied beams (vmat_create: N <= 2048)

__device__ __forceinline__ long long shfl_up_ll(long long v, int o) {
    return __shfl_up_sync(kFull, v, o);
}

// Warp-cooperative search of one row.  All lanes return the same (value, l, r'); l = -1 if the box
// admits no interval.
template <int M>
__device__ __forceinline__ void row_search_warp(const float *__restrict__ g_row, int C, int Lmin, int Lmax, int Rmin,
                                                int Rmax, int lane, long long &value, int &l_out, int &r_out) {
    // inclusive local prefix sums of the quantised prices; position p uses price p-1
    long long loc[M];
    long long sum = 0;
#pragma unroll
    for (int t = 0; t < M; ++t) {
        const int pos = lane * M + t;
        long long qv = 0;
        if (pos >= 1 && pos <= C) qv = __double2ll_rn((double)g_row[pos - 1] * 1073741824.0);
        sum += qv;
        loc[t] = sum;
    }
    long long incl = sum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const long long n = shfl_up_ll(incl, o);
        if (lane >= o) incl += n;
    }
    const long long off = incl - sum;   // P at the lane's first position = off + loc[0]

    // lane aggregate of the running maximum of P[l] over admissible l, later l wins ties
    int av = 0, ap = -1;
    long long aP = 0;
#pragma unroll
    for (int t = 0; t < M; ++t) {
        const int pos = lane * M + t;
        const long long P = off + loc[t];
        if (pos <= C && pos >= Lmin && pos <= Lmax && (!av || P >= aP)) {
            av = 1;
            aP = P;
            ap = pos;
        }
    }
    // inclusive scan of the aggregates across lanes: combine(earlier, later) keeps `later` iff it is
    // valid and (earlier is invalid or later.P >= earlier.P)
    int sv = av, sp = ap;
    long long sP = aP;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int nv = __shfl_up_sync(kFull, sv, o), np = __shfl_up_sync(kFull, sp, o);
        const long long nP = shfl_up_ll(sP, o);
        if (lane >= o && !(sv && (!nv || sP >= nP))) {
            sv = nv;
            sP = nP;
            sp = np;
        }
    }
    int cv = __shfl_up_sync(kFull, sv, 1), cp = __shfl_up_sync(kFull, sp, 1);
    long long cP = shfl_up_ll(sP, 1);
    if (lane == 0) {
        cv = 0;
        cp = -1;
        cP = 0;
    }
    // sweep the lane's positions: update the running maximum with pos as l, then try pos as r'
    int bv = 0, bw = 0, bl = -1;
    long long bval = 0;
#pragma unroll
    for (int t = 0; t < M; ++t) {
        const int pos = lane * M + t;
        const long long P = off + loc[t];
        if (pos <= C && pos >= Lmin && pos <= Lmax && (!cv || P >= cP)) {
            cv = 1;
            cP = P;
            cp = pos;
        }
        if (pos <= C && pos >= Rmin && pos <= Rmax && cv) {
            const long long v = P - cP;
            const int wd = pos - cp;
            if (!bv || v < bval || (v == bval && (wd < bw || (wd == bw && cp < bl)))) {
                bv = 1;
                bval = v;
                bw = wd;
                bl = cp;
            }
        }
    }
    // lexicographic minimum of (value, width, l) over the lanes
#pragma unroll
    for (int o = 16; o; o >>= 1) {
        const int ov = __shfl_xor_sync(kFull, bv, o), ow = __shfl_xor_sync(kFull, bw, o),
                  ol = __shfl_xor_sync(kFull, bl, o);
        const long long oval = __shfl_xor_sync(kFull, bval, o);
        if (ov && (!bv || oval < bval || (oval == bval && (ow < bw || (ow == bw && ol < bl))))) {
            bv = 1;
            bval = oval;
            bw = ow;
            bl = ol;
        }
    }
    value = bv ? bval : 0;
    l_out = bv ? bl : -1;
    r_out = bv ? bl + bw : -1;
}

struct SearchArgs {
    const float *g;
    const uint8_t *occ_in;
    uint8_t *occ;
    int32_t *free_list;                // ascending list of un-occupied beams, rebuilt on commit
    int32_t *left, *right;
    double *y;
    const double *theta;
    int N, R, C, delta;
    int occ_only;                      // reading of Eq. 2: smoothing over successive occupied beams only
    double gamma;
    int32_t *cand_left, *cand_right;   // N*R row optima
    double *beam_price;                // N
    int32_t *out_left, *out_right;     // optional copies for the caller (may alias cand_*)
    double *out_price;
    Sel *sel;
    unsigned int *ticket;              // beams finished
    unsigned long long *beam_total;    // N: sum of the row optima of a beam (all zero between launches)
    unsigned int *beam_ticket;         // N: blocks of a beam finished (all zero between launches)
    int commit;
    int32_t *tr_beam;                  // trace slots (or null)
    double *tr_price;
    int trace_it;
};

// (price, beam) with the smaller price, the lower beam on ties; beam < 0 = no candidate
__device__ __forceinline__ void take_better(double &bp, int &bk, double op, int ok) {
    if (ok >= 0 && (bk < 0 || op < bp || (op == bp && ok < bk))) {
        bp = op;
        bk = ok;
    }
}

template <int M>
__global__ void __launch_bounds__(kSearchThreads) k_leaf_search(const SearchArgs a) {
    // Launched behind the pricing product by programmatic dependent launch: everything up to pdl_wait() below runs
    // while that grid drains and may read only what earlier launches of the stream left (occupancy, leaves), not g.
    __shared__ int s_km, s_kp, s_last, s_bad;
    __shared__ unsigned long long s_total;
    __shared__ double s_price[kRowsPerBlock];
    __shared__ int s_beam[kRowsPerBlock];
    __shared__ int s_cnt[kMaxListChunks];
    const int N = a.N, R = a.R, C = a.C;
    const int RB = (R + kRowsPerBlock - 1) / kRowsPerBlock;       // blocks per beam
    const int k = blockIdx.x / RB, rb = blockIdx.x - k * RB;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const bool occupied = a.occ[k] != 0;
    if (occupied && rb > 0) return;                               // block 0 of an occupied beam reports +inf
    bool beam_done = false;                                       // this block finishes its beam (thread 0)
    if (occupied) {
        pdl_wait();
        pdl_trigger();
    }

    if (!occupied) {
        if (tid == 0) {
            s_km = -1;
            s_kp = N;
            s_bad = 0;
            s_total = 0ull;
        }
        __syncthreads();
        // nearest occupied beam on each side (reading S6)
        int km_t = -1, kp_t = N;
        for (int kk = tid; kk < N; kk += kSearchThreads)
            if (a.occ[kk]) {
                if (kk < k) km_t = max(km_t, kk);
                if (kk > k) kp_t = min(kp_t, kk);
            }
        km_t = __reduce_max_sync(kFull, km_t);
        kp_t = __reduce_min_sync(kFull, kp_t);
        if (lane == 0) {   // one shared-memory atomic per warp that saw an occupied beam
            if (km_t >= 0) atomicMax(&s_km, km_t);
            if (kp_t < N) atomicMin(&s_kp, kp_t);
        }
        __syncthreads();
        const int km = s_km, kp = s_kp;
        const int r = rb * kRowsPerBlock + warp;
        int Lmin = 0, Lmax = C, Rmin = 0, Rmax = C;
        if (r < R) {
            if (km >= 0) {
                const int b = a.delta * (k - km), l = a.left[km * R + r], rr = a.right[km * R + r];
                Lmin = max(Lmin, l - b);
                Lmax = min(Lmax, l + b);
                Rmin = max(Rmin, rr - b);
                Rmax = min(Rmax, rr + b);
            }
            if (kp < N) {
                const int b = a.delta * (kp - k), l = a.left[kp * R + r], rr = a.right[kp * R + r];
                Lmin = max(Lmin, l - b);
                Lmax = min(Lmax, l + b);
                Rmin = max(Rmin, rr - b);
                Rmax = min(Rmax, rr + b);
            }
        }
        pdl_wait();      // the prices
        pdl_trigger();   // the column build may be scheduled; it waits for the choice itself
        if (r < R) {
            long long value;
            int bl, br;
            row_search_warp<M>(a.g + ((size_t)k * R + r) * C, C, Lmin, Lmax, Rmin, Rmax, lane, value, bl, br);
            if (lane == 0) {
                a.cand_left[k * R + r] = bl;
                a.cand_right[k * R + r] = br;
                if (a.out_left) {
                    a.out_left[k * R + r] = bl;
                    a.out_right[k * R + r] = br;
                }
                atomicAdd(&s_total, (unsigned long long)value);   // exact, order free
                // The box admits no interval: the beam has no deliverable aperture.  Cannot happen
                // while the occupied apertures respect the leaf-travel limit among themselves, which vmat_set_plan
                // checks and the loop preserves (S6); kept so that such a beam could never be chosen.
                if (bl < 0) s_bad = 1;
            }
        }
        __syncthreads();
        if (tid == 0) {
            atomicAdd(a.beam_total + k, s_total);
            if (s_bad) atomicOr(a.beam_ticket + k, 0x80000000u);   // bit 31: a row of this beam is undeliverable
            __threadfence();
            const unsigned int seen = atomicAdd(a.beam_ticket + k, 1u);
            if ((seen & 0x7fffffffu) == (unsigned)RB - 1u) {
                __threadfence();
                beam_done = true;
                const long long total = (long long)atomicExch(a.beam_total + k, 0ull);   // all RB sums are in; reset
                a.beam_ticket[k] = 0u;
                // price_k = 2^-30 * total + gamma * dG/dy_k, every operation individually rounded
                // (Eq. 2; reading S10); same order of operations as the definition
                // (the neighbours of beam k in Eq. 2: the angles next to it, or, in the occupied-only reading, the
                // nearest occupied beams, between which an aperture at k would enter the arc; y_k = 0 here)
                const int pm = a.occ_only ? s_km : k - 1, pp = a.occ_only ? s_kp : k + 1;
                double dG = 0.0;
                if (pm >= 0)
                    dG = __dadd_rn(dG, __ddiv_rn(__dmul_rn(2.0, __dsub_rn(a.y[k], a.y[pm])),
                                                 __dsub_rn(a.theta[k], a.theta[pm])));
                if (pp < N)
                    dG = __dsub_rn(dG, __ddiv_rn(__dmul_rn(2.0, __dsub_rn(a.y[pp], a.y[k])),
                                                 __dsub_rn(a.theta[pp], a.theta[k])));
                const double smooth = __dmul_rn(a.gamma, dG);
                const bool undeliverable = (seen >> 31) != 0u || s_bad;
                const double price = undeliverable ? CUDART_INF : __dadd_rn(ldexp(__ll2double_rn(total), -30), smooth);
                a.beam_price[k] = price;
                if (a.out_price) a.out_price[k] = price;
            }
        }
    } else if (tid == 0) {
        beam_done = true;
        a.beam_price[k] = CUDART_INF;
        if (a.out_price) a.out_price[k] = CUDART_INF;
    }

    // the block that finishes the last beam chooses among all of them
    if (tid == 0) {
        s_last = 0;
        if (beam_done) {
            __threadfence();
            s_last = atomicAdd(a.ticket, 1u) == (unsigned)N - 1u;
        }
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    double bp = CUDART_INF;
    int bk = -1;
    for (int kk = tid; kk < N; kk += kSearchThreads) {
        const double pr = __ldcg(a.beam_price + kk);
        if (!a.occ[kk] && pr < CUDART_INF && (bk < 0 || pr < bp)) {   // ascending kk: the lowest index wins ties
            bp = pr;
            bk = kk;
        }
    }
#pragma unroll
    for (int o = 16; o; o >>= 1) take_better(bp, bk, __shfl_down_sync(kFull, bp, o), __shfl_down_sync(kFull, bk, o));
    if (lane == 0) {
        s_price[warp] = bp;
        s_beam[warp] = bk;
    }
    __syncthreads();
    if (warp == 0) {
        bp = lane < kRowsPerBlock ? s_price[lane] : CUDART_INF;
        bk = lane < kRowsPerBlock ? s_beam[lane] : -1;
#pragma unroll
        for (int o = 16; o; o >>= 1)
            take_better(bp, bk, __shfl_down_sync(kFull, bp, o), __shfl_down_sync(kFull, bk, o));
        if (lane == 0) {
            s_price[0] = bp;
            s_beam[0] = bk;
        }
    }
    __syncthreads();
    const int best = s_beam[0];
    const double best_price = s_price[0];
    if (tid == 0) {
        a.sel->beam = best;
        a.sel->price = best >= 0 ? best_price : 0.0;
        *a.ticket = 0u;
        if (a.tr_beam) {
            a.tr_beam[a.trace_it] = best;
            a.tr_price[a.trace_it] = best >= 0 ? best_price : 0.0;
        }
    }
    if (a.commit && best >= 0) {
        // occupy the beam with this aperture at y_k = 0
        for (int r = tid; r < R; r += kSearchThreads) {
            a.left[best * R + r] = __ldcg(a.cand_left + best * R + r);
            a.right[best * R + r] = __ldcg(a.cand_right + best * R + r);
        }
        // the pricing product of the next iteration walks this list: chunks of 32 beams, counted by one
        // warp each, then written behind the chunks before them
        const int nch = (N + 31) / 32;
        for (int ch = warp; ch < nch; ch += kRowsPerBlock) {
            const int kk = ch * 32 + lane;
            const bool f = kk < N && kk != best && !a.occ[kk];
            const unsigned m = __ballot_sync(kFull, f);
            if (lane == 0) s_cnt[ch] = __popc(m);
        }
        __syncthreads();
        for (int ch = warp; ch < nch; ch += kRowsPerBlock) {
            int base = 0;
            for (int c0 = lane; c0 < ch; c0 += 32) base += s_cnt[c0];
            base = __reduce_add_sync(kFull, base);
            const int kk = ch * 32 + lane;
            const bool f = kk < N && kk != best && !a.occ[kk];
            const unsigned m = __ballot_sync(kFull, f);
            if (f) a.free_list[base + __popc(m & ((1u << lane) - 1u))] = kk;
        }
        if (tid == 0) {   // no reader above looks at occ[best]
            a.occ[best] = 1;
            a.y[best] = 0.0;
        }
    }
}

}  // namespace

int launch_leaf_search(vmat_plan *p, const float *g, int32_t *all_left, int32_t *all_right, double *beam_price,
                       int commit, int trace_it) {
    SearchArgs a;
    a.g = g;
    a.occ_in = p->occ;
    a.occ = p->occ;
    a.free_list = p->free_list;
    a.left = p->left;
    a.right = p->right;
    a.y = p->y;
    a.theta = p->theta;
    a.N = (int)p->N;
    a.R = (int)p->R;
    a.C = (int)p->C;
    a.delta = p->delta;
    a.gamma = p->gamma;
    a.occ_only = p->opt.occupied_only_G ? 1 : 0;
    a.cand_left = p->cand_left;
    a.cand_right = p->cand_right;
    a.beam_price = p->beam_price;
    a.out_left = all_left;
    a.out_right = all_right;
    a.out_price = beam_price;
    a.sel = p->sel;
    a.ticket = p->ticket;
    a.beam_total = p->beam_total;
    a.beam_ticket = p->beam_ticket;
    a.commit = commit;
    a.tr_beam = trace_it >= 0 ? p->tr_beam : nullptr;
    a.tr_price = p->tr_price;
    a.trace_it = trace_it;
    const int M = (int)((p->C + 1 + 31) / 32);
    const dim3 grid((unsigned)(p->N * ((p->R + kRowsPerBlock - 1) / kRowsPerBlock))), block(kSearchThreads);
    switch (M) {
        case 1: VMAT_CUDA(p, launch_pdl(k_leaf_search<1>, grid, block, p->stream, a)); break;
        case 2: VMAT_CUDA(p, launch_pdl(k_leaf_search<2>, grid, block, p->stream, a)); break;
        case 3: VMAT_CUDA(p, launch_pdl(k_leaf_search<3>, grid, block, p->stream, a)); break;
        case 4: VMAT_CUDA(p, launch_pdl(k_leaf_search<4>, grid, block, p->stream, a)); break;
        case 5: VMAT_CUDA(p, launch_pdl(k_leaf_search<5>, grid, block, p->stream, a)); break;
        case 6: VMAT_CUDA(p, launch_pdl(k_leaf_search<6>, grid, block, p->stream, a)); break;
        case 7: VMAT_CUDA(p, launch_pdl(k_leaf_search<7>, grid, block, p->stream, a)); break;
        case 8: VMAT_CUDA(p, launch_pdl(k_leaf_search<8>, grid, block, p->stream, a)); break;
        default: return fail(p, VMAT_EINVAL, "n_cols exceeds VMAT_MAX_COLS");
    }
    ++p->launches;
    VMAT_CUDA(p, cudaGetLastError());
    return VMAT_OK;
}

}  // namespace vmat
