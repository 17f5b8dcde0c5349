// vmat_newton.cu — step (e), master mode 1: semismooth Newton on the reduced problem (k_newton).  The pieces it shares
// with mode 0 (arguments, shared-memory carve-up, products with the columns) are in vmat_master_common.cuh; the host
// side that configures and launches either kernel is in vmat_master.cu and reaches this file through the newton_*
// hooks at the end.
#include "vmat_master_common.cuh"

namespace vmat {

// ------------------------------------------------------------------------------------------------
// Mode 1: semismooth Newton on the reduced problem (k_newton)
// ------------------------------------------------------------------------------------------------
// F is piecewise quadratic in the dose, so on the piece of the current dose the master problem is the quadratic
//     min_{lb <= y <= ub}  g.(y' - y) + 1/2 (y' - y)^T (2 H_F + 2 gamma L) (y' - y),
//     H_F[k][k'] = sum_s omega_s d_k[s] d_k'[s],  omega_s = alpha_s (z_s < T_s), beta_s (z_s > T_s), else 0,
// over the K <= N occupied beams: a problem in K unknowns that needs no pass over the columns at all once H_F is
// known.  One block of the grid (the last one) solves that quadratic, step by step: it forms the face of the box the
// step starts from (the occupied beams not at a bound with the true gradient pointing outwards: about half of an
// arc's beams sit at y = 0), holds H_F over those free beams in its shared memory and runs conjugate gradients on the
// face (Jacobi-preconditioned, fp64 vectors; a beam that reaches a bound leaves it); the other blocks evaluate the
// TRUE cost and gradient at the point it proposes, in one pass each (z = sum_k y_k d_k formed from y itself, so
// there is no z += t q drift and no closing pass).  The piece changes only where a voxel crosses its T_s, so a
// master solve takes two or three such passes instead of the twenty-odd of mode 0 (same minimiser: reading S11).
//
// H_F lives in global memory in 64-bit fixed point (integer adds: order free, so a solve stays bit-reproducible) and
// is kept current INCREMENTALLY: every pass compares omega at its dose with the omega the matrix was built with
// (a.omref) and, chunk by chunk, adds  sum_{s flipped} (omega_new - omega_ref)_s d_k[s] d_k'[s]  for the pairs of
// columns that touch the chunk; a column that is not in the matrix yet (the aperture the leaf search has just
// committed; all of them after vmat_set_plan) enters with all its slots.  Measured on configs[1]: 24 of 830 chunks
// see a flip in a late pass.
//
// Hand-over between the solving block and the working blocks: a message in global memory (struct Mail + the
// coefficients) published by a release store of a monotone epoch counter the workers spin on, and a monotone arrival
// counter the solver spins on; no grid-wide barrier.  Both counters run on from launch to launch (bases in a.sync).
struct Mail {
    double scF, scG;   // fixed-point scales of the pass to run
    int state;         // kRunTrial: evaluate at the coefficients that follow; kFinish: stop
    int dst;           // kRunTrial: write z, w to buffer pair dst (0: a.z / a.w, 1: a.zn / a.wn)
    int cur;           // kFinish: the buffer pair that holds the accepted point
    int pad;
};

namespace {

__device__ __forceinline__ unsigned long long ld_acquire_u64(const unsigned long long *p) {
    unsigned long long v;
    asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_u64(unsigned long long *p, unsigned long long v) {
    asm volatile("st.release.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
// spin until *p >= want.  The wait is bounded (about ten seconds): all blocks of a cooperative launch are resident,
// so the other side always arrives; the bound only keeps a defect from hanging the device.  false = gave up.
__device__ __forceinline__ bool spin_until(const unsigned long long *p, unsigned long long want) {
    for (unsigned n = 0; ld_acquire_u64(p) < want; ++n) {
        if (n > (1u << 23)) return false;
        __nanosleep(n < 64 ? 20 : 200);
    }
    return true;
}

// H_F += the change the group's chunks owe it (see above): the pairs of columns already in the matrix take the
// flipped slots of a chunk.  all_slots: the pairs with a column that is not in the matrix yet take every slot of the
// chunk with the new omega (the slow, general way in; a single new column comes in through newton_pass's second
// gradient product instead).
__device__ __forceinline__ void hess_update(const MasterArgs &a, const Smem &sm, int Ku, int g, bool all_slots) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    __shared__ int s_m;
    for (int cs = 0; cs < kGroup; ++cs) {
        const int c = chunk_of(a, g, cs);
        if (c >= a.nchunks) break;
        const int j = g * kGroup + cs;
        const int nf = sm.fl_wc[cs * 4] + sm.fl_wc[cs * 4 + 1] + sm.fl_wc[cs * 4 + 2] + sm.fl_wc[cs * 4 + 3];
        if (nf == 0 && !all_slots) continue;   // the same for the whole block
        // the columns that touch the chunk: staged segments first, then the unstaged ones
        const int nS = sm.coff[j + 1] - sm.coff[j];
        for (int n = tid; n < nS; n += kMasterThreads) sm.hm[n] = sm.cseg[sm.coff[j] + n];
        if (a.ul_cap > 0) {
            const int nU = sm.uoff[j + 1] - sm.uoff[j];
            for (int n = tid; n < nU; n += kMasterThreads) sm.hm[nS + n] = 0xffff | ((int)sm.ul[sm.uoff[j] + n] << 16);
            if (tid == 0) s_m = nS + nU;
        } else if (warp == 0) {
            int run = nS;
            for (int u0 = 0; u0 < Ku; u0 += 32) {
                const int u = u0 + lane, i = u < Ku ? sm.unc[u] : 0;
                const bool f = u < Ku && touches(sm, a.N, i, j);
                const unsigned mk = __ballot_sync(kFull, f);
                if (f) sm.hm[run + __popc(mk & ((1u << lane) - 1u))] = 0xffff | (i << 16);
                run += __popc(mk);
            }
            if (lane == 0) s_m = run;
        }
        __syncthreads();
        const int m = s_m;
        const float *om = sm.ombuf + cs * kSeg, *fd = sm.fl_dw + cs * kChunk;
        const unsigned char *fs = sm.fl_slot + cs * kChunk;
        const float *dch = a.Dd + (size_t)c * a.N * kChunk;   // the chunk's segments in global memory
        // pairs (ia <= ib) of the m members, dealt to the threads row by row of the upper triangle
        const int npair = m * (m + 1) / 2;
        for (int pq = tid; pq < npair; pq += kMasterThreads) {
            // row ia of the triangle starts at ia m - ia (ia - 1) / 2
            int ia = (int)((2.0f * m + 1.0f - sqrtf((2.0f * m + 1.0f) * (2.0f * m + 1.0f) - 8.0f * (float)pq)) * 0.5f);
            while (ia > 0 && ia * m - ia * (ia - 1) / 2 > pq) --ia;
            while ((ia + 1) * m - (ia + 1) * ia / 2 <= pq) ++ia;
            const int ib = ia + pq - (ia * m - ia * (ia - 1) / 2);
            const int ea = sm.hm[ia], eb = sm.hm[ib], ca = ea >> 16, cb = eb >> 16;
            const bool both = sm.hv[ca] && sm.hv[cb];
            if (both ? nf == 0 : !all_slots) continue;
            const float *pa = (ea & 0xffff) == 0xffff ? dch + (size_t)sm.sk[ca] * kChunk : sm.tile + (size_t)(ea & 0xffff) * kSeg;
            const float *pb = (eb & 0xffff) == 0xffff ? dch + (size_t)sm.sk[cb] * kChunk : sm.tile + (size_t)(eb & 0xffff) * kSeg;
            double acc = 0.0;
            if (both) {
                for (int f = 0; f < nf; ++f) {
                    const int sl = fs[f];
                    acc = fma((double)fd[f], (double)(pa[sl] * pb[sl]), acc);
                }
            } else {
                for (int sl = 0; sl < kChunk; ++sl) {
                    const float w = om[sl];
                    if (w != 0.f) acc = fma((double)w, (double)(pa[sl] * pb[sl]), acc);
                }
            }
            if (acc != 0.0) {
                const int ka = sm.sk[ca], kb = sm.sk[cb];
                atomicAdd(reinterpret_cast<unsigned long long *>(a.hess) + (size_t)min(ka, kb) * a.N + max(ka, kb),
                          (unsigned long long)__double2ll_rn(acc * a.hscale));
            }
        }
        __syncthreads();
    }
}

// One pass of a working block: z = sum_k coef_k d_k for its slots -> zdst; w, F and omega there; its share of
// grad = Dc w (record `rec`, fixed point); the flips of omega against a.omref and the update of H_F they call for.
// fresh: compact index of the ONE occupied column that is not in H_F yet (the aperture the leaf search has just
// committed), -1 if there is none, -2 if there are several (then they enter through hess_update, slot by slot).
// The row of the one new column is a second gradient product, H_F[new][i] = d_i . (omega d_new).
__device__ __forceinline__ void newton_pass(const MasterArgs &a, const Smem &sm, int K, int Ku, int ngroups, float *zdst,
                                            float *wdst, long long *rec, double scF, double scG, double *red, int fresh) {
    const bool res = a.rslots > 0;
    const int tid = threadIdx.x, lane = tid & 31;
    const bool one = fresh >= 0;
    for (int i = tid; i < 2 * a.N; i += kMasterThreads) {
        sm.gacc[i] = 0.0;
        if (one) sm.gaccu[i] = 0.0;
    }
    if (a.ul_cap > 0)
        for (int i = tid; i < a.N; i += kMasterThreads) {
            sm.gfx[i] = 0;
            if (one) sm.gfxu[i] = 0;
        }
    double F = 0.0;
    __syncthreads();
    for (int g = 0; g < ngroups; ++g) {
        float zv[kOutPerThread], dw[kOutPerThread];
        unsigned bal[kOutPerThread];
        combine_group(a, sm, Ku, g, zv);
#pragma unroll
        for (int r = 0; r < kOutPerThread; ++r) {
            const int o = tid + r * kMasterThreads, c = chunk_of(a, g, o >> 7);
            float wv = 0.f, omn = 0.f;
            dw[r] = 0.f;
            if (c < a.nchunks) {
                const size_t s = (size_t)c * kChunk + (o & (kChunk - 1));
                const int ls = g * (kGroup * kChunk) + o;
                const float z = zv[r];
                float Tv, al, be;
                if (res) Tv = sm.rT[ls], al = sm.ral[ls], be = sm.rbe[ls];
                else Tv = a.T[s], al = a.alpha[s], be = a.beta[s];
                double f;
                penalty(z, Tv, al, be, wv, f);
                F += f;
                omn = z < Tv ? al : (z > Tv ? be : 0.f);
                const float omo = res ? sm.rom[ls] : a.omref[s];   // every slot belongs to one thread of one block
                dw[r] = omn - omo;
                if (dw[r] != 0.f) {
                    a.omref[s] = omn;
                    if (res) sm.rom[ls] = omn;
                }
                zdst[s] = z;
                wdst[s] = wv;
            }
            sm.wbuf[(o >> 7) * kSeg + (o & (kChunk - 1))] = wv;
            if (one) {   // omega d_new: the new column's own value at this slot, if it touches the chunk at all
                const int j = g * kGroup + (o >> 7);
                float dn = 0.f;
                if (c < a.nchunks && touches(sm, a.N, fresh, j)) {
                    const int bs = sm.base[fresh];
                    dn = bs == kNoCache ? __ldg(a.Dd + ((size_t)c * a.N + sm.sk[fresh]) * kChunk + (o & (kChunk - 1)))
                                        : sm.tile[(size_t)(bs + seg_rank(sm, a.N, fresh, j)) * kSeg + (o & (kChunk - 1))];
                }
                sm.ubuf[(o >> 7) * kSeg + (o & (kChunk - 1))] = omn * dn;
            } else if (fresh == -2) sm.ombuf[(o >> 7) * kSeg + (o & (kChunk - 1))] = omn;
            bal[r] = __ballot_sync(kFull, dw[r] != 0.f);
            if (lane == 0) sm.fl_wc[(o >> 7) * 4 + ((o & (kChunk - 1)) >> 5)] = __popc(bal[r]);
        }
        __syncthreads();
        // the flipped slots of every chunk, in slot order (a fixed order: the sums over them are reproducible)
        int any = 0;
#pragma unroll
        for (int r = 0; r < kOutPerThread; ++r) {
            if (dw[r] != 0.f) {
                const int o = tid + r * kMasterThreads, cs = o >> 7, q = (o & (kChunk - 1)) >> 5;
                int pos = __popc(bal[r] & ((1u << lane) - 1u));
                for (int x = 0; x < q; ++x) pos += sm.fl_wc[cs * 4 + x];
                sm.fl_slot[cs * kChunk + pos] = (unsigned char)(o & (kChunk - 1));
                sm.fl_dw[cs * kChunk + pos] = dw[r];
                any = 1;
            }
        }
        grad_staged(sm, g, sm.wbuf, sm.gpart);
        if (one) grad_staged(sm, g, sm.ubuf, sm.gpartu);
        if (Ku > 0 && a.ul_cap > 0) {
            grad_unstaged_listed(a, sm, g, sm.wbuf, sm.gfx, scG);
            if (one) grad_unstaged_listed(a, sm, g, sm.ubuf, sm.gfxu, a.hscale);
        } else if (Ku > 0) {
            grad_unstaged_masked(a, sm, g, Ku, sm.wbuf, sm.gacc);
            if (one) grad_unstaged_masked(a, sm, g, Ku, sm.ubuf, sm.gaccu);
        }
        // the barrier that ends the group's products also tells whether any of its slots flipped
        if (__syncthreads_or(any) || fresh == -2) hess_update(a, sm, Ku, g, fresh == -2);
    }
    F = block_sum(F, red);
    if (tid == 0) fx_add(rec, F, scF);
    for (int i = tid; i < K; i += kMasterThreads) {
        const bool fx = a.ul_cap > 0 && sm.base[i] == kNoCache;   // already in fixed point
        if (fx) atomicAdd(reinterpret_cast<unsigned long long *>(rec + 2 + i), (unsigned long long)sm.gfx[i]);
        else fx_add(rec + 2 + i, grad_total(sm, sm.gpart, sm.gacc, i, a.N), scG);
        if (one) {   // row of the new column
            const int ka = sm.sk[i], kb = sm.sk[fresh];
            unsigned long long *dst = reinterpret_cast<unsigned long long *>(a.hess) + (size_t)min(ka, kb) * a.N + max(ka, kb);
            if (fx) {
                if (sm.gfxu[i]) atomicAdd(dst, (unsigned long long)sm.gfxu[i]);
            } else {
                const double v = grad_total(sm, sm.gpartu, sm.gaccu, i, a.N);
                if (v != 0.0) atomicAdd(dst, (unsigned long long)__double2ll_rn(v * a.hscale));
            }
        }
    }
}

// ---- the solving block ---------------------------------------------------------------------------------
constexpr int kSolveRed = 8;   // values per warp row of the solver's reduction scratch

// sums s[0..MS) and one maximum over the block, every thread receives them; fixed order.  Only the first nv <= 16
// warps hold data (one beam per thread); the others skip the first level.
template <int MS>
__device__ __forceinline__ void solver_reduce(double (&s)[MS], double &mx, double *buf, int &tog, int nv) {
    static_assert(MS < kSolveRed, "scratch row too short");
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double *b = buf + tog * (kMasterWarps * kSolveRed);
    tog ^= 1;
    if (warp < nv) {
#pragma unroll
        for (int o = 16; o; o >>= 1) {
#pragma unroll
            for (int m = 0; m < MS; ++m) s[m] += __shfl_xor_sync(kFull, s[m], o);
            mx = fmax(mx, __shfl_xor_sync(kFull, mx, o));
        }
        if (lane == 0) {
#pragma unroll
            for (int m = 0; m < MS; ++m) b[warp * kSolveRed + m] = s[m];
            b[warp * kSolveRed + kSolveRed - 1] = mx;
        }
    }
    __syncthreads();
    const int row = lane & 15;   // each half of a warp reads the (at most) sixteen rows
    const bool in = row < nv;
#pragma unroll
    for (int m = 0; m < MS; ++m) {
        double v = in ? b[row * kSolveRed + m] : 0.0;
#pragma unroll
        for (int o = 8; o; o >>= 1) v += __shfl_xor_sync(kFull, v, o);
        s[m] = v;
    }
    double v = in ? b[row * kSolveRed + kSolveRed - 1] : -CUDART_INF;
#pragma unroll
    for (int o = 8; o; o >>= 1) v = fmax(v, __shfl_xor_sync(kFull, v, o));
    mx = v;
}

// Sums of the conjugate-gradient step over the block, in fp32 (the iteration corrects itself: the residual is updated
// with the step actually taken): s[0..MS) are added, mx is maximised, the three low bits of flags are OR-ed.  Only the
// first nv <= 16 warps hold data; they receive everything, the other warps the flags only (loop control).  One
// barrier; both levels are warp shuffles in a fixed order; the scratch alternates between calls.
constexpr int kCgRow = 8;   // floats per warp row of the scratch
template <int MS>
__device__ __forceinline__ void cg_reduce(float (&s)[MS], float &mx, int &flags, float *buf, int &tog, int nv) {
    static_assert(MS + 2 <= kCgRow, "scratch row too short");
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    float *b = buf + tog * (kMasterWarps * kCgRow);
    tog ^= 1;
    if (warp < nv) {
#pragma unroll
        for (int o = 16; o; o >>= 1) {
#pragma unroll
            for (int m = 0; m < MS; ++m) s[m] += __shfl_xor_sync(kFull, s[m], o);
            mx = fmaxf(mx, __shfl_xor_sync(kFull, mx, o));
        }
        const int f = __reduce_or_sync(kFull, flags & 7);
        if (lane == 0) {
#pragma unroll
            for (int m = 0; m < MS; ++m) b[warp * kCgRow + m] = s[m];
            b[warp * kCgRow + MS] = mx;
            b[warp * kCgRow + MS + 1] = __int_as_float(f);
        }
    }
    __syncthreads();
    const int row = lane & 15;   // each half of a warp reads the (at most) sixteen rows
    const bool in = row < nv;
    flags = __reduce_or_sync(kFull, in ? __float_as_int(b[row * kCgRow + MS + 1]) : 0);
    if (warp < nv) {
        float v[MS], m2 = in ? b[row * kCgRow + MS] : -CUDART_INF_F;
#pragma unroll
        for (int m = 0; m < MS; ++m) v[m] = in ? b[row * kCgRow + m] : 0.f;
#pragma unroll
        for (int o = 8; o; o >>= 1) {
#pragma unroll
            for (int m = 0; m < MS; ++m) v[m] += __shfl_xor_sync(kFull, v[m], o);
            m2 = fmaxf(m2, __shfl_xor_sync(kFull, m2, o));
        }
#pragma unroll
        for (int m = 0; m < MS; ++m) s[m] = v[m];
        mx = m2;
    }
}

__device__ void newton_solver(const MasterArgs &a, float4 *smem_raw, unsigned long long ebase, unsigned long long abase) {
    const int N = a.N, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    __shared__ int sK, s_timeout;
    int *timed_out = &s_timeout;
    if (tid == 0) s_timeout = 0;
    // vectors over the beams (fp64), then the matrix (fp32, K x Kp, Kp / 4 odd: rows 16-byte aligned and conflict free
    // for one thread per row), then the maps
    double *vy = reinterpret_cast<double *>(smem_raw);
    double *vg = vy + N, *yc = vg + N, *vd = yc + N, *vyn = vd + N;
    double *vgn = vyn + N, *vp = vgn + N, *linf = vp + N, *rdt = linf + N, *Minv = rdt + N, *dGb = Minv + N;
    double *redb = dGb + N;                                  // 2 x kMasterWarps x kSolveRed
    int *sk = reinterpret_cast<int *>(redb + 2 * kMasterWarps * kSolveRed), *ik = sk + N;
    int *nxl = ik + N, *pvl = nxl + N;   // neighbours of beam k in Eq. 2 (as in master_setup)
    int *pk = pvl + N;                   // row / column of beam k in H32 (the free beams of a Newton step: see its loop), else -1
    int *pp = pk + N;                    // the beam of row p
    float *dc = reinterpret_cast<float *>((reinterpret_cast<uintptr_t>(pp + N) + 15) & ~(uintptr_t)15);   // direction, in H32's order
    const int Np = ((N + 3) / 4) | 1;                        // float4s per row at K = N
    float *cgb = dc + 4 * Np;                                // 2 x kMasterWarps x kCgRow floats: scratch of cg_reduce
    float *hpart = cgb + 2 * kMasterWarps * kCgRow;                     // the product with the matrix, and the part of its second half
    float *hpart2 = hpart + kMasterThreads / 2;
    float *H32 = hpart2 + kMasterThreads / 2;                // Kp x Kp floats, Kp = 4 Kp4 >= K
    // occupied beams, ascending
    if (tid < 32) {
        int base = 0;
        for (int k0 = 0; k0 < N; k0 += 32) {
            const int k = k0 + tid;
            const bool f = k < N && a.occ[k];
            const unsigned m = __ballot_sync(kFull, f);
            if (f) sk[base + __popc(m & ((1u << tid) - 1u))] = k;
            if (k < N) ik[k] = f ? base + __popc(m & ((1u << tid) - 1u)) : -1;
            base += __popc(m);
        }
        if (tid == 0) sK = base;
    }
    const double lb = a.lb, ub = a.ub;
    const bool has_ub = ub < CUDART_INF;
    auto at_bound = [lb, ub](double yk, double g) { return (yk <= lb && g >= 0.0) || (yk >= ub && g <= 0.0); };
    double l1l = 0.0;
    for (int k = tid; k < N; k += kMasterThreads) {
        double yk = a.y[k];
        const bool on = a.occ[k] != 0;
        if (!on) yk = 0.0;
        else if (!(yk > lb)) yk = lb;
        else if (yk > ub) yk = ub;
        vy[k] = yk;
        vd[k] = 0.0;
        int nxk = k + 1 < N ? k + 1 : -1, pvk = k - 1;
        if (a.occ_only) {
            if (!on) nxk = pvk = -1;
            else {
                while (nxk >= 0 && !a.occ[nxk]) nxk = nxk + 1 < N ? nxk + 1 : -1;
                while (pvk >= 0 && !a.occ[pvk]) --pvk;
            }
        }
        nxl[k] = nxk;
        pvl[k] = pvk;
        rdt[k] = nxk >= 0 ? 1.0 / (a.theta[nxk] - a.theta[k]) : 0.0;
        double lf = 0.0;
        if (on) {
            const ColStat cs = a.colstat[k];
            lf = (double)cs.linf * a.fx_inv * 1.000001;
            l1l = fmax(l1l, (double)cs.l1 * a.fx_inv * 1.000001);
        }
        linf[k] = lf;
    }
    int tog = 0;
    const int nvs = (N + 31) / 32;   // warps that hold beams (one per thread)
    double none[1] = {0.0};
    solver_reduce<1>(none, l1l, redb, tog, nvs);   // its barrier also publishes sk, ik, vy, rdt, linf
    const double l1max = l1l;
    const int K = sK;
    const int Kp4 = ((K + 3) / 4) | 1, Kp = 4 * Kp4;
    const double Tm = (double)a.Tmax, ab = (double)a.abmax, Spd = (double)a.Sp;
    const double c1a = 1e-4, noise = 2e-7;
    int bad = 0, inner = 0, backtracks = 0, stop = 0, stall = 0, cur = 0;
    unsigned ph = a.phase[0];
    const unsigned ph_entry = ph;
    const int recn = 2 * N + 2;
    unsigned long long epub = ebase, npass = 0;
    Mail *mail = a.mail;
    float *mcoef = reinterpret_cast<float *>(mail + 1);
    double scF = 1.0, iF = 1.0, scG = 1.0, iG = 1.0;
    long long clk_wait = 0, clk_load = 0, clk_cg = 0, cg_steps = 0;   // bookkeeping (thread 0): where the solver's time goes

    // G(v) and dG/dv (Eq. 2; S2, S3), and the dose bound sum_k |v_k| max|d_k|
    auto smooth_of = [&](const double *v, double &G, double &zb) {
        double s[2] = {0.0, 0.0}, mx = 0.0;
        for (int k = tid; k < N; k += kMasterThreads) {
            const int nx = nxl[k], pv = pvl[k];
            const double e1 = nx >= 0 ? (v[nx] - v[k]) * rdt[k] : 0.0;
            const double e0 = pv >= 0 ? (v[k] - v[pv]) * rdt[pv] : 0.0;
            if (nx >= 0) s[0] += (v[nx] - v[k]) * e1;
            dGb[k] = 2.0 * (e0 - e1);
            s[1] += fabs(v[k]) * linf[k];
        }
        solver_reduce<2>(s, mx, redb, tog, nvs);
        G = s[0];
        zb = s[1];
    };
    // tell the workers what to do next: evaluate at v (into buffer pair dst), or finish
    auto send = [&](int state, int dst, const double *v, double zb) {
        const double dev = Tm + zb;
        const FxScale sF = fx_scale_for(1.01 * Spd * ab * dev * dev, bad);
        const FxScale sG = fx_scale_for(2.02 * ab * dev * l1max, bad);
        scF = sF.scale, iF = sF.inv, scG = sG.scale, iG = sG.inv;
        if (bad) state = kFinish;
        if (v)
            for (int k = tid; k < N; k += kMasterThreads) mcoef[k] = (float)v[k];
        if (tid == 0) {
            mail->scF = scF;
            mail->scG = scG;
            mail->state = state;
            mail->dst = dst;
            mail->cur = cur;
        }
        __syncthreads();
        ++epub;
        if (tid == 0) {
            __threadfence();
            st_release_u64(a.sync + 1, epub);
        }
        return state;
    };
    // wait for the pass the last message asked for; F and the F-part of the gradient at its point -> Fv, gout
    auto receive = [&](double &Fv, double *gout) {
        ++npass;
        const long long c0 = clock64();
        if (tid == 0 && !spin_until(a.sync, abase + (unsigned long long)a.nblk * npass)) *timed_out = 1;
        __syncthreads();
        clk_wait += clock64() - c0;
        const long long *rec = a.accbuf + (size_t)(ph % 3) * kSumGroups * recn;
        ++ph;
        if (s_timeout) bad = 1;
        Fv = (double)__ldcg(rec) * iF + a.F_out;
        for (int k = tid; k < N; k += kMasterThreads) {
            const int i = ik[k];
            gout[k] = i >= 0 ? (double)__ldcg(rec + 2 + i) * iG + a.gamma * dGb[k] : 0.0;
        }
        __syncthreads();
    };

    // ---- the incoming point -----------------------------------------------------------------------------
    double F = 0.0, Gs = 0.0, Phi = 0.0, zb = 0.0, pgmax = 0.0, pg_entry = 0.0, tol = 0.0, Phi0 = 0.0;
    smooth_of(vy, Gs, zb);
    // Warm entry (inside vmat_solve): the solve before this one left z, w, F and d_k . w of its beams current, the one
    // beam the leaf search has occupied since enters at y = 0 (so the dose has not moved) with the price the search formed
    // as its gradient, and k_column_finish has entered its column into H_F: no pass is needed before the first step.
    const bool warm = a.warm && a.lb == 0.0 && a.gflag[0] == 1 && a.sel->beam >= 0 && a.hvalid[a.sel->beam];
    int state = kRunTrial;
    if (warm) {
        const int knew = a.sel->beam;
        const double pnew = a.sel->price;
        for (int k = tid; k < N; k += kMasterThreads)
            vg[k] = ik[k] < 0 ? 0.0 : (k == knew ? pnew : a.gsave[k] + a.gamma * dGb[k]);
        F = a.cost3[0];
        __syncthreads();
    } else {
        state = send(kRunTrial, 0, vy, zb);
        if (state != kFinish) receive(F, vg);
    }
    if (state != kFinish) {
        Phi = F + a.gamma * Gs;
        Phi0 = Phi;
        double pgl = 0.0;
        for (int k = tid; k < N; k += kMasterThreads)
            if (ik[k] >= 0 && !at_bound(vy[k], vg[k])) pgl = fmax(pgl, fabs(vg[k]));
        solver_reduce<1>(none, pgl, redb, tog, nvs);
        pgmax = pg_entry = pgl;
        tol = a.eps * fmax(1.0, pgmax);
        if (a.max_inner <= 0 && pgmax > tol) stop = 1;
    }
    auto stall_threshold = [&](double Phin) {
        return (Phi0 - Phin <= 1e-2 * fabs(Phin)) ? a.stall_rel : 1e-2 * a.stall_rel;
    };

    // ---- Newton iterations ------------------------------------------------------------------------------
    while (state != kFinish && !stop && pgmax > tol) {
        // The face of this Newton step: the occupied beams that are not at a bound with the gradient pointing outwards.
        // The model is solved on it (a beam that reaches a bound on the way stays there; a held beam is released, if
        // the TRUE gradient says so, when the next step forms its face), so only the free beams take part: H32 = H_F
        // over the free beams, in ascending order (about half of an arc's beams sit at y = 0 and are left out).
        const long long c0 = clock64();
        __shared__ int s_nF, s_cF[kMasterWarps];
        {
            const int k = tid;                               // one beam per thread (N <= kMasterThreads)
            const bool fre = k < N && ik[k] >= 0 && !at_bound(vy[k], vg[k]);
            const unsigned mF = __ballot_sync(kFull, fre);
            if (lane == 0) s_cF[warp] = __popc(mF);
            __syncthreads();
            int bF = 0, nFt = 0;
#pragma unroll
            for (int w2 = 0; w2 < kMasterWarps; ++w2) {
                const int cf = s_cF[w2];
                if (w2 < warp) bF += cf;
                nFt += cf;
            }
            const int p = fre ? bF + __popc(mF & ((1u << lane) - 1u)) : -1;
            if (k < N) pk[k] = p;                            // row / column of beam k in H32, -1 if it is not free
            if (fre) pp[p] = k;                              // and the beam of row p
            if (tid == 0) s_nF = nFt;
        }
        __syncthreads();
        const int nF = s_nF, nF4 = (nF + 3) / 4;
        {
            const int npair = nF * (nF + 1) / 2;
            for (int e0 = 0; e0 < npair; e0 += 8 * kMasterThreads) {
                long long v[8];
                int ri[8], ci[8];
#pragma unroll
                for (int u = 0; u < 8; ++u) {
                    const int e = e0 + u * kMasterThreads + tid;
                    ri[u] = -1;
                    v[u] = 0;
                    if (e < npair) {   // row i of the upper triangle starts at i nF - i (i - 1) / 2
                        int i = (int)((2.0f * nF + 1.0f - sqrtf((2.0f * nF + 1.0f) * (2.0f * nF + 1.0f) - 8.0f * (float)e)) * 0.5f);
                        while (i > 0 && i * nF - i * (i - 1) / 2 > e) --i;
                        while ((i + 1) * nF - (i + 1) * i / 2 <= e) ++i;
                        ri[u] = i;
                        ci[u] = i + e - (i * nF - i * (i - 1) / 2);
                        v[u] = __ldcg(a.hess + (size_t)pp[i] * N + pp[ci[u]]);   // pp ascending: the upper triangle
                    }
                }
#pragma unroll
                for (int u = 0; u < 8; ++u)
                    if (ri[u] >= 0) {
                        const float f = (float)((double)v[u] * a.hinv);
                        H32[ri[u] * Kp + ci[u]] = f;
                        H32[ci[u] * Kp + ri[u]] = f;
                    }
            }
        }
        for (int e = tid; e < (4 * nF4 - nF) * Kp; e += kMasterThreads) H32[(size_t)nF * Kp + e] = 0.f;   // rows nF..4 nF4 - 1 (read with d = 0)
        for (int k = tid; k < N; k += kMasterThreads) {
            yc[k] = vy[k];
            vd[k] = 0.0;
        }
        for (int i = tid; i < Kp; i += kMasterThreads) dc[i] = 0.f;
        __syncthreads();
        for (int k = tid; k < N; k += kMasterThreads) {
            const int i = pk[k];
            double m = 0.0;
            if (i >= 0) m = 2.0 * (double)H32[i * Kp + i] + 2.0 * a.gamma * ((pvl[k] >= 0 ? rdt[pvl[k]] : 0.0) + rdt[k]);
            Minv[k] = m > 0.0 ? 1.0 / m : 1.0;
        }
        const long long c1 = clock64();
        clk_load += c1 - c0;
        // Conjugate gradients on that face of the box for the quadratic model at (vy, vg), and on its sub-faces as beams
        // reach a bound: one beam per thread (the first nv warps), all warps on the product with the matrix.  One sum over the beams per step: with the
        // residual r, the preconditioner M, the direction d and H d at hand, A = sum M r^2, B = sum M r (H d) and
        // C = sum M (H d)^2 over the face give the Polak-Ribiere numerator of the NEXT residual r + t H d without a
        // second sum, (r+ - r) M r+ = t (B + t C), and its denominator is A.  Whether the face changed, whether any
        // entry of the new projected residual is still above the tolerance and whether to give up travel as three bits
        // OR-ed into a shared word.  Step lengths, the sums and the ratios to the bounds are fp32: the iteration
        // corrects itself (the residual is updated with the step actually taken) and a beam that reaches its bound is
        // set on it explicitly.
        const double qtol = fmax(0.5 * tol, 0.05 * pgmax);
        const int k = tid;                                   // this thread's beam (k < N: checked on the host)
        const bool mine = k < N && pk[k] >= 0;               // a beam of the face
        const int myp = mine ? pk[k] : 0;                    // its row and column of H32
        const int nv = (N + 31) / 32;                        // warps that hold beams
        auto ratio = [](double num, double den) { return (double)__fdividef((float)num, (float)den); };
        __shared__ int s_fl[2];
        int tf = 0, togc = 0;
        auto any_flags = [&](int bits) {                     // OR of the bits over the block; one barrier
            const int wb = __reduce_or_sync(kFull, bits);
            if (lane == 0 && wb) atomicOr(&s_fl[tf], wb);
            __syncthreads();
            const int r = s_fl[tf];
            tf ^= 1;
            if (tid == 0) s_fl[tf] = 0;                      // the word of the next call; nobody touches it before another barrier
            return r;
        };
        if (tid < 2) s_fl[tid] = 0;
        __syncthreads();
        // state of this thread's beam
        double yk = mine ? vy[k] : 0.0, rk = mine ? vg[k] : 0.0, beta = 0.0;
        const double mk = mine ? Minv[k] : 1.0;
        int fr = mine;                                       // still free (a beam that reaches a bound leaves the face for good)
        double prk = fr ? rk : 0.0, dk = -mk * prk;
        bool halt = false;
        const int maxcg = 4 * nF + 20;
        int it = 0;
        int fl = any_flags(fabs(prk) > qtol ? 2 : 0);
        while ((fl & 2) && !(fl & 4) && it < maxcg) {
            if (k < N) vd[k] = dk;
            if (mine) dc[myp] = (float)dk;
            __syncthreads();
            ++cg_steps;
            ++it;
            // H32 d, fp32.  The matrix is symmetric: thread (r, h) sums H[c][r] d_c over the columns c of its half h, so
            // that the lanes of a warp read consecutive words of row c (no bank conflict, 128 bytes per request) and
            // d_c is the same word for the whole warp.  Two halves: threads 0..255 and 256..511.
            {
                const int r = tid & (kMasterThreads / 2 - 1), h = tid / (kMasterThreads / 2);
                const int q0 = h * ((nF4 + 1) / 2), q1 = min(nF4, q0 + (nF4 + 1) / 2);   // float4s of d of this half
                float acc0 = 0.f, acc1 = 0.f;
                if (r < nF) {
                    const float4 *d4 = reinterpret_cast<const float4 *>(dc);
                    const float *hc = H32 + r;
                    for (int q = q0; q < q1; ++q) {
                        const float4 dv = d4[q];
                        const float *h4 = hc + (size_t)(4 * q) * Kp;
                        acc0 = fmaf(h4[0], dv.x, acc0);
                        acc1 = fmaf(h4[Kp], dv.y, acc1);
                        acc0 = fmaf(h4[2 * Kp], dv.z, acc0);
                        acc1 = fmaf(h4[3 * Kp], dv.w, acc1);
                    }
                }
                if (h == 1 && r < nF) hpart2[r] = acc0 + acc1;
                __syncthreads();
                if (h == 0 && r < nF) hpart[r] = (acc0 + acc1) + hpart2[r];
            }
            __syncthreads();
            double hdk = 0.0;
            float s5[5] = {0.f, 0.f, 0.f, 0.f, 0.f}, ntl = -CUDART_INF_F;
            if (mine) {
                const int nx = nxl[k], pv = pvl[k];
                const double e1 = nx >= 0 ? (vd[nx] - dk) * rdt[k] : 0.0;
                const double e0 = pv >= 0 ? (dk - vd[pv]) * rdt[pv] : 0.0;
                hdk = 2.0 * (double)hpart[myp] + 2.0 * a.gamma * (e0 - e1);
                s5[0] = (float)(dk * hdk);
                s5[1] = (float)(rk * dk);
                if (fr) {
                    const double mr = mk * rk;
                    s5[2] = (float)(mr * rk);
                    s5[3] = (float)(mr * hdk);
                    s5[4] = (float)(mk * hdk * hdk);
                }
                if (dk < 0.0) ntl = -(float)ratio(yk - lb, -dk);
                if (has_ub && dk > 0.0) ntl = -(float)ratio(ub - yk, dk);
            }
            int nofl = 0;
            cg_reduce<5>(s5, ntl, nofl, cgb, togc, nv);
            const float tmaxf = -ntl;                            // fp32: the same bits wherever the ratio is formed
            const double tmax = (double)tmaxf;
            bool hit = false;
            double t = 0.0;
            if (warp >= nv) {            // no beams, and no sums either: this warp only follows the flags
            } else if (!(s5[1] < 0.f)) { // not a descent direction of the model: open steepest descent again, or give up
                if (beta == 0.0) halt = true;
            } else {
                t = s5[0] > 0.f ? (double)__fdividef(-s5[1], s5[0]) : tmax;
                if (!(t < CUDART_INF)) {
                    halt = true;
                    t = 0.0;
                } else {
                    hit = t >= tmax;
                    if (hit) t = tmax;
                    if (mine) {
                        double v = yk + t * dk;
                        if (v < lb || (hit && dk < 0.0 && (float)ratio(yk - lb, -dk) <= tmaxf)) v = lb;
                        else if (has_ub && (v > ub || (hit && dk > 0.0 && (float)ratio(ub - yk, dk) <= tmaxf))) v = ub;
                        yk = v;
                        rk += t * hdk;
                    }
                }
            }
            const int fn = fr && !at_bound(yk, rk);
            prk = fn ? rk : 0.0;
            fl = any_flags(warp >= nv ? 0 : (fn != fr || hit || t == 0.0 ? 1 : 0) | (fabs(prk) > qtol ? 2 : 0) | (halt ? 4 : 0));
            // (only the warps that hold beams know the sums; `halt` and the rest of the loop control travel as flags)
            beta = (fl & 1) || !(s5[2] > 0.f) ? 0.0 : (double)fmaxf(0.f, __fdividef((float)t * (s5[3] + (float)t * s5[4]), s5[2]));
            dk = fn ? -mk * prk + beta * dk : 0.0;
            fr = fn;
        }
        if (mine) yc[k] = yk;
        __syncthreads();
        clk_cg += clock64() - c1;
        // the step and its slope on the true gradient
        double sl[1] = {0.0}, mxp = 0.0;
        if (tid < N) {
            const double pk = yc[tid] - vy[tid];
            vp[tid] = pk;
            sl[0] = vg[tid] * pk;
            mxp = fabs(pk);
        }
        solver_reduce<1>(sl, mxp, redb, tog, nvs);
        const double slope = sl[0];
        if (!(slope < 0.0) || !(mxp > 0.0)) {
            stop = 2;
            break;
        }
        // back-tracking on the true cost, from the full step
        double t = 1.0;
        int half = 0;
        for (;;) {
            if (tid < N) vyn[tid] = half == 0 ? yc[tid] : fmin(fmax(vy[tid] + t * vp[tid], ik[tid] >= 0 ? lb : 0.0), ik[tid] >= 0 ? ub : 0.0);
            __syncthreads();
            double Gn, zbn, Fn;
            smooth_of(vyn, Gn, zbn);
            state = send(kRunTrial, cur ^ 1, vyn, zbn);
            if (state == kFinish) break;
            receive(Fn, vgn);
            const double Phin = Fn + a.gamma * Gn;
            double sn[1] = {0.0}, pgm = 0.0;
            if (tid < N) {
                sn[0] = vgn[tid] * vp[tid];
                if (ik[tid] >= 0 && !at_bound(vyn[tid], vgn[tid])) pgm = fabs(vgn[tid]);
            }
            solver_reduce<1>(sn, pgm, redb, tog, nvs);
            const bool accepted = Phin <= Phi + c1a * t * slope ||
                                  (Phin <= Phi + noise * fabs(Phi) && fabs(sn[0]) <= 0.9 * fabs(slope));
            if (accepted) {
                stall = (Phi - Phin <= stall_threshold(Phin) * fabs(Phi)) ? stall + 1 : 0;
                cur ^= 1;
                if (tid < N) {
                    vy[tid] = vyn[tid];
                    vg[tid] = vgn[tid];
                }
                F = Fn;
                Gs = Gn;
                Phi = Phin;
                pgmax = pgm;
                ++inner;
                __syncthreads();
                break;
            }
            t *= 0.5;
            ++backtracks;
            if (-t * slope <= stall_threshold(Phi) * fabs(Phi)) {   // no shorter step can lower the cost by more than fp32 resolves
                stop = 4;
                break;
            }
            if (++half >= 40) {
                stop = 3;
                break;
            }
        }
        if (stop || state == kFinish) break;
        if (stall >= a.stall_count) stop = 4;
        else if (inner >= a.max_inner) stop = 1;
    }
    if (bad) stop = 5;
    if (s_timeout) stop = 6;
    if (state != kFinish) send(kFinish, 0, nullptr, 0.0);
    // results; d_k . w at the point the solve leaves, for the warm entry of the next one
    const bool evaluated = npass > 0 && !bad && !s_timeout;   // z, w, F and vg belong to vy
    {
        double Gx, zbx;
        smooth_of(vy, Gx, zbx);   // dG/dy at vy (the last point sent may have been a rejected trial)
    }
    for (int k = tid; k < N; k += kMasterThreads) {
        a.y[k] = vy[k];
        if (a.occ[k] && npass > 0) a.hvalid[k] = 1;   // every occupied beam is in the matrix now (the first pass saw to it)
        if (evaluated || warm) a.gsave[k] = ik[k] >= 0 ? vg[k] - a.gamma * dGb[k] : 0.0;
    }
    if (tid == 0) {
        a.phase[0] = ph % 3;
        a.sync[2] = epub;
        a.sync[3] = abase + (unsigned long long)a.nblk * npass;
        a.gflag[0] = (evaluated || warm) ? 1 : 0;
        if (npass > 0) a.hlive[0] = 1;
        atomicAdd(a.mcount + 1, (unsigned long long)(ph - ph_entry));
        a.mcount[2] += (unsigned long long)cg_steps;
        a.mcount[3] += (unsigned long long)clk_cg;
        a.mcount[4] += (unsigned long long)clk_wait;
        a.mcount[5] += (unsigned long long)clk_load;
        MasterOut o;
        o.inner = inner;
        o.backtracks = backtracks;
        o.stop_reason = stop;
        o.pad = (int)(ph - ph_entry);
        o.pg_entry = pg_entry;
        o.pg_exit = pgmax;
        o.F = F;
        o.G = Gs;
        o.cost = Phi;
        *a.out = o;
        a.cost3[0] = F;
        a.cost3[1] = Gs;
        a.cost3[2] = Phi;
        if (a.trace_it >= 0) {
            a.trF[a.trace_it] = F;
            a.trG[a.trace_it] = Gs;
            a.trC[a.trace_it] = Phi;
            a.trInner[a.trace_it] = inner;
        }
    }
}

__global__ void __launch_bounds__(kMasterThreads, 1) k_newton(const MasterArgs a) {
    extern __shared__ float4 smem_raw[];
    const int tid = threadIdx.x;
    const unsigned long long ebase = a.sync[2];   // written by the launch before this one: stream ordered
    const unsigned long long abase = a.sync[3];
    if ((int)blockIdx.x == a.nblk) {
        newton_solver(a, smem_raw, ebase, abase);
        return;
    }
    Smem sm;
    const Setup su = master_setup<true>(a, sm, smem_raw);
    const int K = su.K, Ku = su.Ku, ngroups = su.ngroups;
    // T, alpha, beta of the block's own slots are read once
    if (a.rslots > 0) {
        for (int ls = tid; ls < a.rslots; ls += kMasterThreads) {
            const int c = (int)blockIdx.x + (ls >> 7) * a.nblk;
            const bool in = c < a.nchunks;
            const size_t s = (size_t)c * kChunk + (ls & (kChunk - 1));
            sm.rT[ls] = in ? a.T[s] : 0.f;
            sm.ral[ls] = in ? a.alpha[s] : 0.f;
            sm.rbe[ls] = in ? a.beta[s] : 0.f;
            sm.rom[ls] = in ? a.omref[s] : 0.f;
        }
    }
    // which occupied columns are in H_F already: fresh = the one that is not (-1: none, -2: several)
    __shared__ int s_fresh;
    if (tid == 0) s_fresh = INT_MAX;
    __syncthreads();
    int missing = 0;
    for (int i = tid; i < K; i += kMasterThreads) {
        const int v = a.hvalid[sm.sk[i]] != 0;
        sm.hv[i] = v;
        if (!v) {
            ++missing;
            atomicMin(&s_fresh, i);
        }
    }
    missing = __syncthreads_count(missing);   // (K <= kMasterThreads: at most one column per thread)
    int fresh = missing == 0 ? -1 : (missing == 1 ? s_fresh : -2);
    const int recn = 2 * a.N + 2;
    unsigned ph = a.phase[0];
    const unsigned ph_entry = ph;
    const Mail *mail = a.mail;
    const float *mcoef = reinterpret_cast<const float *>(mail + 1);
    unsigned long long e = ebase;
    int cur = 0;
    for (;;) {
        ++e;
        __shared__ int s_gone;
        if (tid == 0) s_gone = !spin_until(a.sync + 1, e);
        __syncthreads();
        // the whole message in one round trip to L2: header and this thread's coefficient are loaded before any is used
        const int mstate = __ldcg(&mail->state), dst = __ldcg(&mail->dst), mcur = __ldcg(&mail->cur);
        const double scF = __ldcg(&mail->scF), scG = __ldcg(&mail->scG);
        float cf = 0.f;
        if (tid < K) cf = __ldcg(mcoef + sm.sk[tid]);   // K <= kMasterThreads / 2
        const int state = s_gone ? kFinish : mstate;
        if (state == kFinish) {
            cur = s_gone ? 0 : mcur;
            break;
        }
        if (tid < K) sm.coef[tid] = cf;
        if (blockIdx.x == 0) {   // block 0 clears the record of the pass after this one
            long long *nx = a.accbuf + (size_t)((ph + 1) % 3) * kSumGroups * recn;
            for (int i = tid; i < kSumGroups * recn; i += kMasterThreads) nx[i] = 0;
        }
        long long *rec = a.accbuf + (size_t)(ph % 3) * kSumGroups * recn;
        ++ph;
        __syncthreads();
        newton_pass(a, sm, K, Ku, ngroups, dst ? a.zn : a.z, dst ? a.wn : a.w, rec, scF, scG, su.red, fresh);
        if (fresh != -1) {
            __syncthreads();
            for (int i = tid; i < K; i += kMasterThreads) sm.hv[i] = 1;
            fresh = -1;
        }
        __syncthreads();
        if (tid == 0) {
            __threadfence();
            atomicAdd(a.sync, 1ull);
        }
    }
    // the accepted point sits in the second buffer pair: bring the block's own slots home
    if (cur) {
        for (int g = 0; g < ngroups; ++g)
            for (int o = tid; o < kGroup * kChunk; o += kMasterThreads) {
                const int c = chunk_of(a, g, o >> 7);
                if (c < a.nchunks) {
                    const size_t s = (size_t)c * kChunk + (o & (kChunk - 1));
                    a.z[s] = a.zn[s];
                    a.w[s] = a.wn[s];
                }
            }
    }
    if (tid == 0) atomicAdd(a.mcount, (unsigned long long)su.segs * (unsigned long long)(ph - ph_entry));
}

// shared memory of k_newton's solving block (newton_solver's carve-up)
// for N beams of which at most K are occupied
size_t solver_smem_bytes(int64_t N, int64_t K) {
    const int64_t Np = ((N + 3) / 4) | 1, Kp = 4 * (((K + 3) / 4) | 1);
    return (size_t)(11 * N + 2 * kMasterWarps * kSolveRed) * 8 + (size_t)6 * N * 4 + 16 + (size_t)4 * Np * 4 +
           (size_t)(kMasterThreads + 2 * kMasterWarps * kCgRow) * 4 + (size_t)Kp * Kp * 4;
}

}  // namespace

size_t newton_solver_smem_bytes(int64_t N, int64_t K) { return solver_smem_bytes(N, K); }

size_t newton_mail_bytes(int64_t N) { return sizeof(Mail) + 4 * (size_t)N; }

// The attribute is a per-function, per-device setting shared by every plan of the process: it is set to the device's
// opt-in maximum (the same value from every vmat_create), never to one plan's own size, so that a plan created later
// cannot shrink it under a live one.  Each launch passes its own size <= optin.
int newton_prepare_kernel(vmat_plan *p, int optin) {
    cudaFuncAttributes fa;
    VMAT_CUDA(p, cudaFuncGetAttributes(&fa, k_newton));
    VMAT_CUDA(p, cudaFuncSetAttribute(k_newton, cudaFuncAttributeMaxDynamicSharedMemorySize, optin - (int)fa.sharedSizeBytes));
    return VMAT_OK;
}

int newton_blocks_per_sm(vmat_plan *p, size_t smem, int *per_sm) {
    VMAT_CUDA(p, cudaOccupancyMaxActiveBlocksPerMultiprocessor(per_sm, k_newton, kMasterThreads, smem));
    return VMAT_OK;
}

int newton_launch(vmat_plan *p, const MasterArgs &a, int grid, size_t smem) {
    MasterArgs copy = a;
    void *args[] = {&copy};
    VMAT_CUDA(p, cudaLaunchCooperativeKernel((const void *)k_newton, dim3((unsigned)grid), dim3(kMasterThreads), args, smem,
                                             p->stream));
    return VMAT_OK;
}

}  // namespace vmat
