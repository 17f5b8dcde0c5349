// vmat_master.cu — steps (a), (b) and (e): master mode 0 (k_master) and the host side of both master kernels
// (configuration, the Hessian's life cycle, the per-launch choice between k_master and k_newton).  The column build is
// in vmat_column.cu, mode 1 (k_newton) in vmat_newton.cu, what the two kernels share in vmat_master_common.cuh.
//
//   aperture-dose columns  d_k = sum_{i in A_k} D_i.        (the inner sum of PAPER.md:69 / :88)
//   dose                   z   = sum_k y_k d_k
//   penalty gradient       w_j = -2 alpha_j max(0,T_j-z_j) + 2 beta_j max(0,z_j-T_j)      (Eq. 1)
//   master problem         min_{y>=0} F(z(y)) + gamma G(y), gradient projection (Eq. 3)
//
// Layout: the columns are DENSE over the support of D, fp32, cut into chunks of 128 slots
// (one warp of float4) and stored CHUNK-MAJOR, Dd[chunk][k][128]: the segments of all columns for one chunk are
// neighbours in memory, so a block that walks a chunk's beams streams one contiguous region.  Each column carries the range of chunks it
// touches, so both products of one inner iteration — q = Dc^T d (per slot) and grad = Dc w (per
// beam) — skip the part of a row that is all zero.  Chunks are dealt to the blocks round-robin
// (the touched slots cluster in the slabs the apertures irradiate), a block works on groups of
// kGroup chunks at a time with the beam loop split over its warps, so every lane keeps kGroup
// independent 16-byte loads in flight.
//
// The whole master solve is ONE persistent cooperative kernel: the K-vectors (y, direction,
// gradient) live in every block's shared memory and all scalar decisions (step length, sufficient
// decrease, conjugacy, stop) are taken redundantly by every block from the same sums, so control
// flow is uniform with two grid barriers per inner iteration and no host round trip.  Sums over
// the grid (F, the curvature, the K gradient entries) are accumulated with 64-bit FIXED-POINT
// atomics whose scale every block derives from the same bound: integer addition is order free, so
// a solve is bit-reproducible from run to run although the blocks arrive in any order.
#include <cooperative_groups.h>

#include "vmat_master_common.cuh"

namespace cg = cooperative_groups;

namespace vmat {

namespace {

// max |T| and max(alpha, beta) over the support (bounds for the fixed-point scales of the master)
__global__ void k_voxel_bounds(const float *__restrict__ T, const float *__restrict__ alpha,
                               const float *__restrict__ beta, long long Sp, unsigned int *__restrict__ out2) {
    const long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    float t = 0.f, ab = 0.f;
    if (s < Sp) {
        t = fabsf(T[s]);
        ab = fmaxf(alpha[s], beta[s]);
    }
#pragma unroll
    for (int o = 16; o; o >>= 1) {
        t = fmaxf(t, __shfl_xor_sync(kFull, t, o));
        ab = fmaxf(ab, __shfl_xor_sync(kFull, ab, o));
    }
    if ((threadIdx.x & 31) == 0) {   // non-negative floats order like their bit patterns
        atomicMax(out2, __float_as_uint(t));
        atomicMax(out2 + 1, __float_as_uint(ab));
    }
}

// Mode 0: gradient projection with conjugate directions on the current face; two passes over the columns and two
// grid barriers per inner iteration (q = Dc^T d and the curvature, then the trial point).
__global__ void __launch_bounds__(kMasterThreads, 1) k_master(const MasterArgs a) {
    extern __shared__ float4 smem_raw[];   // 16-byte aligned: float4 tiles first, then doubles, floats, ints
    const int N = a.N, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    Smem sm;
    const Setup su = master_setup<false>(a, sm, smem_raw);
    const int K = su.K, Ku = su.Ku, ngroups = su.ngroups, sSegs = su.segs;
    const double l1max = su.l1max;
    double *red = su.red, *cred = su.cred;
    const double Tm = (double)a.Tmax, ab = (double)a.abmax, Spd = (double)a.Sp;

    const int recn = 2 * N + 2;
    unsigned ph = a.phase[0];      // rotation of the records; written by the previous launch, stream ordered
    const unsigned ph_entry = ph;
    float *zcur = a.z, *znext = a.zn;
    // resident slot data: T, alpha, beta of the block's own slots are read once, z and q never leave the SM
    const bool res = a.rslots > 0;
    float *rzcur = sm.rz0, *rznext = sm.rz1;
    if (res) {
        for (int ls = tid; ls < a.rslots; ls += kMasterThreads) {
            const int c = (int)blockIdx.x + (ls >> 7) * a.nblk;
            const bool in = c < a.nchunks;
            const size_t s = (size_t)c * kChunk + (ls & (kChunk - 1));
            sm.rT[ls] = in ? a.T[s] : 0.f;
            sm.ral[ls] = in ? a.alpha[s] : 0.f;
            sm.rbe[ls] = in ? a.beta[s] : 0.f;
        }
    }

    // start a pass: the record that collects its sums; block 0 clears the record of the next pass
    auto begin_pass = [&]() -> long long * {
        if (blockIdx.x == 0) {
            long long *nx = a.accbuf + (size_t)((ph + 1) % 3) * kSumGroups * recn;
            for (int i = tid; i < kSumGroups * recn; i += kMasterThreads) nx[i] = 0;
        }
        return a.accbuf + ((size_t)(ph % 3) * kSumGroups + blockIdx.x % kSumGroups) * recn;
    };

    // after the grid barrier: one round trip to L2 for the whole record, then the control warp works from smem
    auto fetch_record = [&](const long long *rec, int count) {
        // sum of the group records (integers: any order gives the same bits); rec is this block's own record
        const long long *r0 = rec - (size_t)(blockIdx.x % kSumGroups) * recn;
        for (int i = tid; i < count; i += kMasterThreads) {
            long long v = 0;
#pragma unroll
            for (int gq = 0; gq < kSumGroups; ++gq) v += __ldcg(r0 + (size_t)gq * recn + i);
            sm.recv[i] = v;
        }
        __syncthreads();
    };

    // ---- control group: the first nw warps of every block share the N-vector work (one entry per thread
    // for N <= 512); every thread of the group carries the same scalars, all blocks take the same decisions
    const int nw = min(kMasterWarps, (N + 31) / 32), CT = nw * 32;
    const bool ctl = warp < nw;
    int tog = 0;
    int bad = 0, inner = 0, backtracks = 0, stop = 0, stall = 0, hit = 0, half = 0;
    double F = 0.0, Gs = 0.0, Phi = 0.0, pgmax = 0.0, pg_entry = 0.0, tol = 0.0;
    double phi1 = 0.0, Gd = 0.0, tmax = 0.0, qb = 0.0, yb = 0.0, t = 0.0, Gn = 0.0;
    const double c1a = 1e-4, noise = 2e-7;
    // gradient projection on the box lb <= y_k <= ub (default: y_k >= 0): a beam at a bound whose gradient points
    // out of the box does not move (the same test with g = -d_k keeps a direction feasible)
    const double lb = a.lb, ub = a.ub;
    const bool has_ub = ub < CUDART_INF;   // the default box has no upper face: skip its divisions
    auto at_bound = [lb, ub](double yk, double g) { return (yk <= lb && g >= 0.0) || (yk >= ub && g <= 0.0); };
    // The stall rule (stop at the fp32 resolution of the cost) is calibrated for warm starts, where a step that
    // lowers the cost by <= stall_rel of it really is the end.  A solve that has already lowered the cost by more
    // than 1 % started far from the optimum: conjugate directions then pass through plateaus of tiny steps before
    // the next long one, so the rule is applied 100x more strictly there.
    double Phi0 = 0.0;
    auto stall_threshold = [&](double Phin) {
        return (Phi0 - Phin <= 1e-2 * fabs(Phin)) ? a.stall_rel : 1e-2 * a.stall_rel;
    };

    auto set_eval_scales = [&](double zb) {
        const double dev = Tm + zb;
        const FxScale sF = fx_scale_for(1.01 * Spd * ab * dev * dev, bad);
        const FxScale sG = fx_scale_for(2.02 * ab * dev * l1max, bad);
        if (tid == 0) {
            sm.ctl->scF = sF.scale;
            sm.ctl->iF = sF.inv;
            sm.ctl->scG = sG.scale;
            sm.ctl->iG = sG.inv;
        }
    };
    // everything the direction pass and the step rule need from (y, grad, d), in one sweep and one
    // batched reduction: slope phi1 = grad.d, the dose bounds qb, yb (sum_k |v_k| max|d_k| >=
    // max_j |sum_k v_k d_kj|), Gd = d^T L d = G(d), and the largest feasible step tmax
    auto direction_sums = [&]() {
        double s[4] = {0.0, 0.0, 0.0, 0.0}, ntl = -CUDART_INF;
        for (int k = tid; k < N; k += CT) {
            const double dk = sm.d[k], yk = sm.y[k], lf = sm.linf[k];
            s[0] += sm.grad[k] * dk;
            s[1] += fabs(dk) * lf;
            s[2] += fabs(yk) * lf;
            if (sm.nx[k] >= 0) {
                const double dv = sm.d[sm.nx[k]] - dk;
                s[3] += dv * dv * sm.rdt[k];
            }
            if (dk < 0.0) ntl = fmax(ntl, -((yk - lb) / (-dk)));
            if (has_ub && dk > 0.0) ntl = fmax(ntl, -((ub - yk) / dk));
        }
        ctl_reduce<4>(s, ntl, cred, tog, nw, CT);
        phi1 = s[0];
        qb = s[1];
        yb = s[2];
        Gd = s[3];
        tmax = -ntl;
    };
    // slope along d (steepest descent if d does not descend) and the coefficients / scale of the
    // direction pass.  Returns false (stop set) if no descent is possible.
    auto prepare_direction = [&]() {
        direction_sums();
        if (!(phi1 < 0.0)) {
            for (int k = tid; k < N; k += CT) sm.d[k] = -sm.pg[k];
            ctl_sync(CT);
            direction_sums();
            if (!(phi1 < 0.0)) {
                stop = 2;
                return false;
            }
        }
        const FxScale sC = fx_scale_for(1.01 * Spd * ab * qb * qb, bad);
        for (int i = tid; i < K; i += CT) sm.coef[i] = (float)sm.d[sm.sk[i]];
        if (tid == 0) {
            sm.ctl->scC = sC.scale;
            sm.ctl->iC = sC.inv;
        }
        return !bad;
    };
    // trial point y + t d (clamped), G and dG there
    auto prepare_trial = [&]() {
        for (int k = tid; k < N; k += CT) {
            const double yk = sm.y[k], dk = sm.d[k];
            double v = yk + t * dk;
            if (sm.ik[k] >= 0) {
                if (v < lb || (hit && dk < 0.0 && (yk - lb) / (-dk) <= tmax)) v = lb;
                else if (has_ub && (v > ub || (hit && dk > 0.0 && (ub - yk) / dk <= tmax))) v = ub;
            }
            sm.yn[k] = v;
        }
        ctl_sync(CT);
        double sg[1] = {smooth_part(sm.yn, sm, N, CT, true)}, mx = 0.0;
        ctl_reduce<1>(sg, mx, cred, tog, nw, CT);
        Gn = sg[0];
        if (tid == 0) sm.ctl->tf = (float)t;
    };

    // objective and gradient at the incoming y
    if (ctl) {
        double s[2] = {0.0, smooth_part(sm.y, sm, N, CT, true)}, mx = 0.0;
        for (int k = tid; k < N; k += CT) s[0] += fabs(sm.y[k]) * sm.linf[k];
        ctl_reduce<2>(s, mx, cred, tog, nw, CT);
        set_eval_scales(s[0]);
        yb = s[0];
        Gs = s[1];
    }
    __syncthreads();
    // Warm entry: the previous solve left z, w, F and d_k . w of its beams current, and the one beam the leaf search
    // has occupied since enters at y = 0, so the dose has not moved; its own d_k . w is the price the search formed
    // minus the smoothing term.  The evaluation pass (and its grid barrier) is then not needed.  With a lower bound
    // y_min > 0 (vmat_set_dose_rate_bounds) the new beam enters at y_min and the dose does move: no warm entry.
    const bool warm = a.warm && a.lb == 0.0 && a.gflag[0] == 1 && a.sel->beam >= 0;
    long long *rec = nullptr;
    if (!warm) {
        rec = begin_pass();
        eval_pass<true>(a, sm, K, Ku, ngroups, nullptr, zcur, nullptr, rzcur, 0.f, rec, sm.ctl->scF, sm.ctl->scG, red);
        cg::this_grid().sync();
        ++ph;
        fetch_record(rec, K + 2);
    } else if (res) {
        for (int ls = tid; ls < a.rslots; ls += kMasterThreads) {
            const int c = (int)blockIdx.x + (ls >> 7) * a.nblk;
            rzcur[ls] = c < a.nchunks ? a.z[(size_t)c * kChunk + (ls & (kChunk - 1))] : 0.f;
        }
    }
    if (ctl) {
        const double iG = sm.ctl->iG;
        const int knew = warm ? a.sel->beam : -1;
        const double pnew = warm ? a.sel->price : 0.0;
        double pgl = 0.0;
        for (int k = tid; k < N; k += CT) {
            const int i = sm.ik[k];
            double gk = 0.0;
            if (i >= 0) {
                if (!warm) gk = (double)sm.recv[2 + i] * iG + a.gamma * sm.dG[k];
                else if (k == knew) gk = pnew;   // = 2^-30 total + gamma dG/dy_k, the reduced cost itself
                else gk = a.gsave[k] + a.gamma * sm.dG[k];
            }
            const double p = (i < 0 || at_bound(sm.y[k], gk)) ? 0.0 : gk;
            sm.grad[k] = gk;
            sm.pg[k] = p;
            sm.d[k] = -p;
            pgl = fmax(pgl, fabs(p));
        }
        double s0[1] = {0.0};
        ctl_reduce<1>(s0, pgl, cred, tog, nw, CT);   // its barrier also publishes grad, pg, d to the group
        F = warm ? a.cost3[0] : (double)sm.recv[0] * sm.ctl->iF + a.F_out;
        Phi = F + a.gamma * Gs;
        pgmax = pgl;
        pg_entry = pgmax;
        Phi0 = Phi;
        tol = a.eps * fmax(1.0, pgmax);
        int state = kRunDirection;
        if (!(pgmax > tol) || bad) state = kFinish;
        else if (a.max_inner <= 0) {
            stop = 1;
            state = kFinish;
        } else if (!prepare_direction()) state = kFinish;
        if (tid == 0) {
            sm.ctl->state = state;
            sm.ctl->accepted = 0;
        }
    }
    __syncthreads();

    while (sm.ctl->state != kFinish) {
        // ---- q = Dc^T d and the curvature of the quadratic piece at t = 0 ------------------------------
        rec = begin_pass();
        double curv = 0.0;
        for (int g = 0; g < ngroups; ++g) {
            float qv[kOutPerThread];
            combine_group(a, sm, Ku, g, qv);
#pragma unroll
            for (int r = 0; r < kOutPerThread; ++r) {
                const int o = tid + r * kMasterThreads, c = chunk_of(a, g, o >> 7);
                if (c < a.nchunks) {
                    const size_t sl = (size_t)c * kChunk + (o & (kChunk - 1));
                    const int ls = g * (kGroup * kChunk) + o;
                    float zv, Tv, al, be;
                    if (res) {
                        zv = rzcur[ls], Tv = sm.rT[ls], al = sm.ral[ls], be = sm.rbe[ls];
                        sm.rq[ls] = qv[r];
                    } else {
                        zv = zcur[sl], Tv = a.T[sl], al = a.alpha[sl], be = a.beta[sl];
                        a.q[sl] = qv[r];
                    }
                    const float om = zv < Tv ? al : (zv > Tv ? be : 0.f);
                    curv += (double)om * (double)qv[r] * (double)qv[r];
                }
            }
            __syncthreads();
        }
        curv = block_sum(curv, red);
        if (tid == 0) fx_add(rec + 1, curv, sm.ctl->scC);
        cg::this_grid().sync();
        ++ph;
        fetch_record(rec, K + 2);
        if (ctl) {
            const double curvF = (double)sm.recv[1] * sm.ctl->iC;
            const double phi2 = 2.0 * curvF + 2.0 * a.gamma * Gd;
            t = phi2 > 0.0 ? -phi1 / phi2 : (isfinite(tmax) ? tmax : 1.0);
            hit = 0;
            if (t >= tmax) {
                t = tmax;
                hit = 1;
            }
            half = 0;
            set_eval_scales(yb + t * qb);   // |z + t q| <= sum_k (|y_k| + t |d_k|) max|d_k|; t only shrinks below
            prepare_trial();
            if (tid == 0) sm.ctl->state = bad ? kFinish : kRunTrial;
        }
        __syncthreads();
        // ---- backtracking on the true cost ----------------------------------------------------------------
        while (sm.ctl->state == kRunTrial) {
            rec = begin_pass();
            eval_pass<false>(a, sm, K, Ku, ngroups, zcur, znext, rzcur, rznext, sm.ctl->tf, rec, sm.ctl->scF,
                             sm.ctl->scG, red);
            cg::this_grid().sync();
            ++ph;
            fetch_record(rec, K + 2);
            if (ctl) {
                // gn = Dc w + gamma dG at the trial point, and the sums of the acceptance test and of the
                // Polak-Ribiere+ update, in one sweep and one batched reduction
                const double iG = sm.ctl->iG;
                const double Fn = (double)sm.recv[0] * sm.ctl->iF + a.F_out;
                // The working direction lives on the FACE of the beams that are off their bounds: a beam at a bound is
                // held there (its entry of the working gradient pf is 0) even if its gradient points inwards, until the
                // gradient on the face is small against the held inward part (s[4] <= eta^2 s[5]); then the held
                // beams are released and the conjugate directions restart.  Releasing at once, as the textbook rule
                // does, made beams near y = 0 enter and leave the face from one step to the next: over a third of all
                // steps of a configs[1] plan were restarts.  Convergence is still judged on the true projected gradient.
                double s[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0}, pgm = 0.0;
                for (int k = tid; k < N; k += CT) {
                    const int i = sm.ik[k];
                    const double gk = i >= 0 ? (double)sm.recv[2 + i] * iG + a.gamma * sm.dG[k] : 0.0;
                    const double yk = sm.yn[k], po = sm.pg[k];
                    const double pn = (i < 0 || at_bound(yk, gk)) ? 0.0 : gk;
                    const bool atb = yk <= lb || (has_ub && yk >= ub);
                    const double pf = (i < 0 || atb) ? 0.0 : gk;
                    sm.gn[k] = gk;
                    s[3] += ((pf == 0.0) != (po == 0.0)) ? 1.0 : 0.0;   // entries entering / leaving the face
                    s[0] += pf * (pf - po);
                    s[1] += po * po;
                    s[2] += gk * sm.d[k];
                    s[4] += pf * pf;
                    if (atb) s[5] += pn * pn;                            // held, but the gradient points inwards
                    pgm = fmax(pgm, fabs(pn));
                }
                ctl_reduce<6>(s, pgm, cred, tog, nw, CT);
                bool release = s[5] > 0.0 && s[4] <= kReleaseEta2 * s[5];
                                const double Phin = Fn + a.gamma * Gn;
                // sufficient decrease; below the resolution of Phi accept on the slope instead
                const bool accepted = Phin <= Phi + c1a * t * phi1 ||
                                      (Phin <= Phi + noise * fabs(Phi) && fabs(s[2]) <= 0.9 * fabs(phi1));
                int state;
                if (accepted) {
                    // take the step; Polak-Ribiere+ direction on the current face, restart when the active set changes
                    stall = (Phi - Phin <= stall_threshold(Phin) * fabs(Phi)) ? stall + 1 : 0;
                    if (stall >= a.stall_count && s[5] > 0.0 && !release) {
                        release = true;   // never stop on a face while held beams want in: release them and go on
                        stall = 0;
                    }
                    const bool changed = hit || release || s[3] > 0.0;
                    F = Fn;
                    Gs = Gn;
                    Phi = Phin;
                    pgmax = pgm;
                    const double bpr = (changed || !(s[1] > 0.0) || s[0] <= 0.0) ? 0.0 : s[0] / s[1];
                    for (int k = tid; k < N; k += CT) {
                        const double yk = sm.yn[k], gk = sm.gn[k];
                        const bool off = sm.ik[k] < 0;
                        const bool atb = yk <= lb || (has_ub && yk >= ub);
                        const double pn = (off || (release ? at_bound(yk, gk) : atb)) ? 0.0 : gk;   // working gradient
                        double dk = -pn + bpr * sm.d[k];
                        if (off || at_bound(yk, -dk)) dk = 0.0;   // stay feasible
                        sm.y[k] = yk;
                        sm.grad[k] = gk;
                        sm.pg[k] = pn;
                        sm.d[k] = dk;
                    }
                    ctl_sync(CT);
                                        ++inner;
                    state = kRunDirection;
                    if (!(pgmax > tol)) state = kFinish;
                    else if (stall >= a.stall_count) {
                        stop = 4;
                        state = kFinish;
                    } else if (inner >= a.max_inner) {
                        stop = 1;
                        state = kFinish;
                    } else if (!prepare_direction()) state = kFinish;
                } else {
                    t *= 0.5;
                    hit = 0;
                    ++backtracks;
                    state = kRunTrial;
                    if (-t * phi1 <= stall_threshold(Phi) * fabs(Phi)) {
                        // whatever shorter step might pass the test, it cannot lower the cost by more than -t phi'(0),
                        // which is below what fp32 dose arithmetic resolves: the solve has ended (measured on configs[4]:
                        // without this, late solves spent 35 halvings per step on a slope lost in the noise of the cost)
                        stop = 4;
                        state = kFinish;
                    } else if (++half >= 60) {
                        stop = 3;
                        state = kFinish;
                    } else prepare_trial();
                }
                                if (tid == 0) {
                    sm.ctl->state = state;
                    sm.ctl->accepted = accepted ? 1 : 0;
                }
            }
            __syncthreads();
            if (sm.ctl->accepted) {
                float *tmpz = zcur;
                zcur = znext;
                znext = tmpz;
                tmpz = rzcur;
                rzcur = rznext;
                rznext = tmpz;
            }
        }
    }

    // z, w and the cost from the final y (no drift from the z += t q updates)
    __syncthreads();
    if (ctl) {
        if (bad) stop = 5;
        const int redo = (inner > 0 || zcur != a.z) && !bad;
        if (redo) {
            double s[2] = {0.0, smooth_part(sm.y, sm, N, CT, true)}, mx = 0.0;
            for (int k = tid; k < N; k += CT) s[0] += fabs(sm.y[k]) * sm.linf[k];
            ctl_reduce<2>(s, mx, cred, tog, nw, CT);
            set_eval_scales(s[0]);
            Gs = s[1];
            for (int i = tid; i < K; i += CT) sm.coef[i] = (float)sm.y[sm.sk[i]];
        }
        if (tid == 0) sm.ctl->accepted = redo;
    }
    __syncthreads();
    if (sm.ctl->accepted) {
        rec = begin_pass();
        eval_pass<true>(a, sm, K, Ku, ngroups, nullptr, a.z, nullptr, rzcur, 0.f, rec, sm.ctl->scF, sm.ctl->scG, red);
        cg::this_grid().sync();
        ++ph;
        fetch_record(rec, K + 2);
        if (ctl) {
            F = (double)sm.recv[0] * sm.ctl->iF + a.F_out;
            Phi = F + a.gamma * Gs;
            if (blockIdx.x == 0) {   // d_k . w at the final y, for the warm entry of the next solve
                const double iG = sm.ctl->iG;
                for (int k = tid; k < N; k += CT) {
                    const int i = sm.ik[k];
                    a.gsave[k] = i >= 0 ? (double)sm.recv[2 + i] * iG : 0.0;
                }
            }
        }
    }
    if (blockIdx.x == 0 && tid == 0) a.gflag[0] = sm.ctl->accepted ? 1 : 0;   // no final pass: nothing saved
    if (tid == 0) {
        atomicAdd(a.mcount, (unsigned long long)sSegs * (unsigned long long)(ph - ph_entry));
        if (blockIdx.x == 0) atomicAdd(a.mcount + 1, (unsigned long long)(ph - ph_entry));
    }
    if (blockIdx.x == 0 && warp == 0) {
        for (int k = lane; k < N; k += 32) a.y[k] = sm.y[k];
        if (lane == 0) {
            a.phase[0] = ph % 3;
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
}


}  // namespace

// launch shape of one of the two master kernels for this plan; cfg->grid stays 0 if it does not fit
static int configure_kernel(vmat_plan *p, bool newton, size_t budget, vmat_plan::MasterCfg *cfg) {
    const int64_t nchunks = p->Sp / kChunk;
    *cfg = vmat_plan::MasterCfg();
    int64_t grid = p->sm_count - (newton ? 1 : 0);    // one block per SM, chunks dealt round-robin
    if (grid > nchunks) grid = nchunks;
    if (grid < 1) grid = 1;
    // resident slot data (z, z trial, q, T, alpha, beta of a block's own slots) if it fits in 128 KB: on a large
    // support the tile holds a few per cent of the columns whatever its size, while slot data read from L2 / HBM
    // costs every group of every pass a round trip
    const int64_t ngroups = (nchunks + grid * kGroup - 1) / (grid * kGroup);
    int64_t rslots = ngroups * kGroup * kChunk;
    if (rslots * (newton ? 7 : 6) * 4 > 128 * 1024) rslots = 0;
    // per-chunk lists of the unstaged beams (one entry per column and local chunk at most) if they fit in 64 KB
    int64_t ul_cap = p->N * ngroups * kGroup;
    if (ul_cap * 2 > 64 * 1024 || p->N > 65535) ul_cap = 0;
    if (!p->opt.master_unstaged_lists) ul_cap = 0;         // option: force the fallback path (tests)
    size_t fixed = master_smem_bytes(p->N, rslots, 0, ngroups, newton, ul_cap);
    if (fixed > budget) {
        rslots = 0;
        fixed = master_smem_bytes(p->N, 0, 0, ngroups, newton, ul_cap);
    }
    if (fixed > budget) {
        ul_cap = 0;
        fixed = master_smem_bytes(p->N, 0, 0, ngroups, newton, 0);
    }
    if (fixed > budget) return VMAT_OK;
    // what is left of the SM's opt-in shared memory (minus static use and room for L1) holds the tile of Dd
    int64_t cache_segs = (int64_t)((budget - fixed) / seg_bytes(newton));
    if (cache_segs > 65535 || ngroups * kGroup > 32767) cache_segs = 0;   // 16-bit fields of the lists
    cfg->smem = master_smem_bytes(p->N, rslots, cache_segs, ngroups, newton, ul_cap);
    int per_sm = 0;
    if (newton) {
        int rc = newton_blocks_per_sm(p, cfg->smem, &per_sm);
        if (rc) return rc;
    } else VMAT_CUDA(p, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_master, kMasterThreads, cfg->smem));
    if (per_sm < 1) return VMAT_OK;
    cfg->nblk = (int)grid;
    cfg->grid = (int)grid + (newton ? 1 : 0);
    cfg->rslots = (int)rslots;
    cfg->ul_cap = (int)ul_cap;
    cfg->cache_segs = (int)cache_segs;
    return VMAT_OK;
}

int master_configure(vmat_plan *p) {
    const int64_t nchunks = p->Sp / kChunk;
    int optin = 0;
    VMAT_CUDA(p, cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, p->device));
    const size_t budget = (size_t)optin > 8 * 1024 ? (size_t)optin - 8 * 1024 : 0;
    // The attribute is a per-function, per-device setting shared by every plan of the process: it is set to the
    // device's opt-in maximum (the same value from every vmat_create), never to this plan's own size, so that a plan
    // created later cannot shrink it under a live one.  Each launch passes its own size <= optin.
    cudaFuncAttributes fa0;
    VMAT_CUDA(p, cudaFuncGetAttributes(&fa0, k_master));
    VMAT_CUDA(p, cudaFuncSetAttribute(k_master, cudaFuncAttributeMaxDynamicSharedMemorySize, optin - (int)fa0.sharedSizeBytes));
    int rc;
    if ((rc = newton_prepare_kernel(p, optin))) return rc;
    if ((rc = configure_kernel(p, false, budget, &p->mcfg[0]))) return rc;
    if (p->mcfg[0].grid == 0) return fail(p, VMAT_EINVAL, "n_beams too large for the master kernel's shared memory");
    // mode 1 (k_newton) gives one block of the grid to the reduced problems: its vectors take one thread per beam, the
    // product with its matrix one thread per occupied beam and half of the columns, and the matrix must fit that
    // block's shared memory.  The last two bound the number of OCCUPIED beams: a launch with more of them runs k_master.
    p->newton_kmax = 0;
    p->newton_retired = false;
    if (p->opt.master_mode == 1 && p->sm_count >= 2 && p->N <= kMasterThreads) {
        if ((rc = configure_kernel(p, true, budget, &p->mcfg[1]))) return rc;
        if (p->mcfg[1].grid > 0) {
            int64_t kmax = p->N < kMasterThreads / 2 ? p->N : kMasterThreads / 2;
            while (kmax > 0 && newton_solver_smem_bytes(p->N, kmax) > budget) --kmax;
            if (p->opt.master_newton_max_beams > 0 && kmax > p->opt.master_newton_max_beams) kmax = p->opt.master_newton_max_beams;
            p->newton_kmax = (int)kmax;
        }
    }
    const bool newton = p->newton_kmax > 0;
    p->master_newton = newton;
    if ((rc = dev_alloc(p, &p->accbuf, 3 * kSumGroups * (2 * p->N + 2)))) return rc;
    if ((rc = dev_alloc(p, &p->phase, 2))) return rc;
    if ((rc = dev_alloc(p, &p->mcount, 16))) return rc;
    if ((rc = dev_alloc(p, &p->gsave, p->N))) return rc;
    if ((rc = dev_alloc(p, &p->gflag, 1))) return rc;
    VMAT_CUDA(p, cudaMemsetAsync(p->gflag, 0, 4, p->stream));
    VMAT_CUDA(p, cudaMemsetAsync(p->mcount, 0, 128, p->stream));
    if ((rc = dev_alloc(p, &p->colstat, p->N))) return rc;
    p->touch_words = (int)((nchunks + 31) / 32);
    if ((rc = dev_alloc(p, &p->col_touch, p->N * p->touch_words))) return rc;
    VMAT_CUDA(p, cudaMemsetAsync(p->col_touch, 0, (size_t)p->N * p->touch_words * 4, p->stream));
    if ((rc = dev_alloc(p, &p->vbounds, 2))) return rc;
    if (newton) {
        if ((rc = dev_alloc(p, &p->hess, p->N * p->N))) return rc;
        if ((rc = dev_alloc(p, &p->omref, p->Sp))) return rc;
        if ((rc = dev_alloc(p, &p->hvalid, p->N))) return rc;
        if ((rc = dev_alloc(p, &p->hlive, 1))) return rc;
        if ((rc = dev_alloc(p, &p->wn_s, p->Sp))) return rc;
        if ((rc = dev_alloc(p, (char **)&p->mail, (int64_t)newton_mail_bytes(p->N)))) return rc;
        if ((rc = dev_alloc(p, &p->nsync, 4))) return rc;
        VMAT_CUDA(p, cudaMemsetAsync(p->wn_s, 0, (size_t)p->Sp * 4, p->stream));
        VMAT_CUDA(p, cudaMemsetAsync(p->mail, 0, newton_mail_bytes(p->N), p->stream));
        VMAT_CUDA(p, cudaMemsetAsync(p->nsync, 0, 32, p->stream));
        if ((rc = reset_hessian(p))) return rc;
    }
    VMAT_CUDA(p, cudaMemsetAsync(p->accbuf, 0, (size_t)3 * kSumGroups * (2 * p->N + 2) * 8, p->stream));
    VMAT_CUDA(p, cudaMemsetAsync(p->phase, 0, 8, p->stream));
    VMAT_CUDA(p, cudaMemsetAsync(p->colstat, 0, (size_t)p->N * sizeof(ColStat), p->stream));
    VMAT_CUDA(p, cudaMemsetAsync(p->vbounds, 0, 8, p->stream));
    k_voxel_bounds<<<(unsigned)((p->Sp + 255) / 256), 256, 0, p->stream>>>(p->T_s, p->alpha_s, p->beta_s,
                                                                         (long long)p->Sp, p->vbounds);
    VMAT_CUDA(p, cudaGetLastError());
    float hb[2];
    VMAT_CUDA(p, cudaMemcpyAsync(hb, p->vbounds, 8, cudaMemcpyDeviceToHost, p->stream));
    VMAT_CUDA(p, cudaStreamSynchronize(p->stream));
    p->Tmax = hb[0];
    p->abmax = hb[1];
    // fixed-point scale of H_F: |sum_s omega_s d_k[s] d_k'[s]| <= max(alpha, beta) Sp (R C max|D|)^2 < 2^e
    // (p->fx_inv = 2^(e2 - 40) with max|D| < 2^e2: vmat_layout.cu)
    {
        int e2 = 0, eab = 0, esp = 0, erc = 0;
        std::frexp(p->fx_inv, &e2);   // fx_inv = 2^(e2' - 40) = 0.5 * 2^(e2' - 39): frexp exponent = e2' - 39
        e2 += 39;
        std::frexp((double)(p->abmax > 0.f ? p->abmax : 1.f), &eab);
        std::frexp((double)p->Sp, &esp);
        std::frexp((double)p->RC, &erc);
        const int e = eab + esp + 2 * (erc + e2);
        p->hscale = std::ldexp(1.0, 60 - e);
        p->hinv = std::ldexp(1.0, e - 60);
    }
    return VMAT_OK;
}

// H_F, the omega it was built with and the flags of its columns back to "empty" (after vmat_set_plan: the apertures
// behind the columns may all have changed)
int reset_hessian(vmat_plan *p) {
    if (!p->master_newton) return VMAT_OK;
    p->newton_retired = false;
    VMAT_CUDA(p, cudaMemsetAsync(p->hess, 0, (size_t)p->N * p->N * 8, p->stream));
    VMAT_CUDA(p, cudaMemsetAsync(p->omref, 0, (size_t)p->Sp * 4, p->stream));
    VMAT_CUDA(p, cudaMemsetAsync(p->hvalid, 0, (size_t)p->N, p->stream));
    VMAT_CUDA(p, cudaMemsetAsync(p->hlive, 0, 4, p->stream));
    return VMAT_OK;
}

static int launch_master_impl(vmat_plan *p, int max_inner, int trace_it, int warm, int k_occ) {
    // which kernel: k_newton while the occupied beams (k_occ: an upper bound) fit its solving block.  Past that the
    // plan runs k_master; H_F is then no longer kept up, so k_column_finish is told to stop adding rows to it.
    bool newton = p->master_newton && k_occ <= p->newton_kmax;
    if (p->master_newton && !newton && !p->newton_retired) {
        VMAT_CUDA(p, cudaMemsetAsync(p->hlive, 0, 4, p->stream));
        VMAT_CUDA(p, cudaMemsetAsync(p->hvalid, 0, (size_t)p->N, p->stream));
        p->newton_retired = true;
    } else if (newton && p->newton_retired) {
        int rc = reset_hessian(p);   // back under the bound (apertures were removed): the matrix is rebuilt from empty
        if (rc) return rc;
    }
    const vmat_plan::MasterCfg &cfg = p->mcfg[newton ? 1 : 0];
    MasterArgs a;
    a.warm = warm;
    a.sel = p->sel;
    a.gsave = p->gsave;
    a.gflag = p->gflag;
    a.Dd = p->Dd;
    a.Sp = (long long)p->Sp;
    a.nchunks = (int)(p->Sp / kChunk);
    a.T = p->T_s;
    a.alpha = p->alpha_s;
    a.beta = p->beta_s;
    a.z = p->z_s;
    a.zn = p->zn_s;
    a.q = p->q_s;
    a.q2 = p->q2_s;
    a.w = p->w_s;
    a.occ = p->occ;
    a.y = p->y;
    a.theta = p->theta;
    a.N = (int)p->N;
    a.gamma = p->gamma;
    a.F_out = p->F_out;
    a.eps = p->opt.master_eps;
    a.stall_rel = p->opt.master_stall_rel;
    a.stall_count = p->opt.master_stall_count;
    a.occ_only = p->opt.occupied_only_G ? 1 : 0;
    a.lb = p->y_min;
    a.ub = p->y_max;
    a.max_inner = max_inner;
    a.rslots = cfg.rslots;
    a.cache_segs = cfg.cache_segs;
    a.ul_cap = cfg.ul_cap;
    a.colstat = p->colstat;
    a.touch = p->col_touch;
    a.touch_words = p->touch_words;
    a.fx_inv = p->fx_inv;
    a.Tmax = p->Tmax;
    a.abmax = p->abmax;
    a.accbuf = p->accbuf;
    a.phase = p->phase;
    a.mcount = p->mcount;
    a.out = p->mout;
    a.cost3 = p->cost3;
    a.trF = p->tr_F;
    a.trG = p->tr_G;
    a.trC = p->tr_cost;
    a.trInner = p->tr_inner;
    a.trace_it = trace_it;
    a.nblk = cfg.nblk;
    a.hess = p->hess;
    a.omref = p->omref;
    a.hvalid = p->hvalid;
    a.hlive = p->hlive;
    a.hscale = p->hscale;
    a.hinv = p->hinv;
    a.wn = p->wn_s;
    a.mail = (Mail *)p->mail;
    a.sync = p->nsync;
    if (newton) {
        size_t smem = cfg.smem;
        if (newton_solver_smem_bytes(p->N, k_occ) > smem) smem = newton_solver_smem_bytes(p->N, k_occ);
        int rc = newton_launch(p, a, cfg.grid, smem);
        if (rc) return rc;
    } else {
        void *args[] = {&a};
        VMAT_CUDA(p, cudaLaunchCooperativeKernel((const void *)k_master, dim3((unsigned)cfg.grid), dim3(kMasterThreads), args,
                                                 cfg.smem, p->stream));
    }
    ++p->launches;
    return VMAT_OK;
}

int launch_master(vmat_plan *p, int trace_it, int warm, int k_occ) {
    return launch_master_impl(p, p->opt.master_max_inner, trace_it, warm, k_occ);
}

}  // namespace vmat
