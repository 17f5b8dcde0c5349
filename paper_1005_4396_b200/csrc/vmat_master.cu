// vmat_master.cu — steps (a), (b) and (e).
//
//   aperture-dose columns  d_k = sum_{i in A_k} D_i.        (the inner sum of PAPER.md:69 / :88)
//   dose                   z   = sum_k y_k d_k
//   penalty gradient       w_j = -2 alpha_j max(0,T_j-z_j) + 2 beta_j max(0,z_j-T_j)      (Eq. 1)
//   master problem         min_{y>=0} F(z(y)) + gamma G(y), gradient projection (Eq. 3)
//
// Layout: the columns are DENSE rows over the support of D, Dd[k][slot], fp32.
// Both products of one inner iteration — q = Dc^T d (per slot) and grad = Dc w (per beam) — stream
// the same rows with coalesced float4 loads, both are tiled over chunks of 128 slots, and every
// reduction runs in a fixed order, so a solve is bit-reproducible from run to run.
//
// The whole master solve is ONE persistent cooperative kernel: blocks own fixed slot ranges, the
// K-vectors (y, direction, gradient) live in every block's shared memory and all scalar decisions
// (step length, sufficient decrease, conjugacy, stop) are taken redundantly by every block from
// the same partial sums in the same order, so control flow is uniform with two grid barriers per
// inner iteration and no host round trip.
#include <cooperative_groups.h>
#include <math_constants.h>

#include "vmat_internal.cuh"

namespace cg = cooperative_groups;

namespace vmat {

namespace {

constexpr unsigned kFull = 0xffffffffu;

// ------------------------------------------------------------------------------------------------
// aperture-dose column of one beam: fixed-point scatter (order free, hence reproducible) + convert
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_column_scatter(const uint32_t *__restrict__ rowq, const float4 *__restrict__ val4, const int4 *__restrict__ col4,
                 const Sel *__restrict__ sel, int beam, const int32_t *__restrict__ left,
                 const int32_t *__restrict__ right, int R, int C, double fx_scale, unsigned long long *__restrict__ acc) {
    const int k = sel ? sel->beam : beam;
    if (k < 0) return;
    const int lane = threadIdx.x & 31;
    const int idx = blockIdx.x * 8 + (threadIdx.x >> 5);
    if (idx >= R * C) return;
    const int r = idx / C, c = idx - r * C;
    if (c < left[k * R + r] || c >= right[k * R + r]) return;   // beamlet not exposed (A_k)
    const long long row = ((long long)k * R + r) * C + c;
    const uint32_t a = rowq[row], b = rowq[row + 1];
    for (uint32_t q = a + lane; q < b; q += 32) {
        const float4 v = __ldg(val4 + q);
        const int4 s = __ldg(col4 + q);
        if (v.x != 0.f) atomicAdd(acc + s.x, (unsigned long long)__double2ll_rn((double)v.x * fx_scale));
        if (v.y != 0.f) atomicAdd(acc + s.y, (unsigned long long)__double2ll_rn((double)v.y * fx_scale));
        if (v.z != 0.f) atomicAdd(acc + s.z, (unsigned long long)__double2ll_rn((double)v.z * fx_scale));
        if (v.w != 0.f) atomicAdd(acc + s.w, (unsigned long long)__double2ll_rn((double)v.w * fx_scale));
    }
}

__global__ void __launch_bounds__(256)
k_column_finish(unsigned long long *__restrict__ acc, long long Sp, const Sel *__restrict__ sel, int beam,
                double fx_inv, float *__restrict__ Dd) {
    const int k = sel ? sel->beam : beam;
    if (k < 0) return;
    const long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= Sp) return;
    const long long v = (long long)acc[s];
    Dd[(size_t)k * Sp + s] = (float)((double)v * fx_inv);
    acc[s] = 0ull;
}

// ------------------------------------------------------------------------------------------------
// slot space <-> voxel space
// ------------------------------------------------------------------------------------------------
__global__ void k_expand(const float *__restrict__ src_s, const int32_t *__restrict__ slot_of,
                         const float *__restrict__ T, const float *__restrict__ alpha, const float *__restrict__ beta,
                         long long V, int what, float *__restrict__ dst) {
    const long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= V) return;
    const int s = slot_of[j];
    float v;
    if (s >= 0) v = src_s[s];
    else if (what == 0) v = 0.f;                                   // no beamlet reaches j: z_j = 0
    else {
        const float t = T[j];
        v = -2.f * alpha[j] * fmaxf(0.f, t) + 2.f * beta[j] * fmaxf(0.f, -t);   // Eq. 1 at z_j = 0
    }
    dst[j] = v;
}

__global__ void k_compress(const float *__restrict__ src_V, const int32_t *__restrict__ voxel_of, long long S,
                           long long Sp, float *__restrict__ dst_s) {
    const long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= Sp) return;
    dst_s[s] = s < S ? src_V[voxel_of[s]] : 0.f;
}

// ------------------------------------------------------------------------------------------------
// the master kernel
// ------------------------------------------------------------------------------------------------
struct MasterArgs {
    const float *Dd;
    long long Sp;
    int nchunks;
    const float *T, *alpha, *beta;
    float *z, *zn, *q, *w;
    const uint8_t *occ;
    double *y;
    const double *theta;
    int N;
    double gamma, F_out, eps;
    int max_inner;
    double *partA, *partF, *partG;
    MasterOut *out;
    double *cost3;
    double *trF, *trG, *trC;
    int32_t *trInner;
    int trace_it;
};

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(kFull, v, o);
    return v;
}
// every thread receives the same total, summed in a fixed order
__device__ __forceinline__ double block_sum(double v, double *red) {
    v = warp_sum(v);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
    __syncthreads();
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < kMasterWarps; ++i) s += red[i];
    __syncthreads();
    return s;
}
__device__ __forceinline__ double block_max(double v, double *red) {
#pragma unroll
    for (int o = 16; o; o >>= 1) v = fmax(v, __shfl_xor_sync(kFull, v, o));
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
    __syncthreads();
    double s = red[0];
#pragma unroll
    for (int i = 1; i < kMasterWarps; ++i) s = fmax(s, red[i]);
    __syncthreads();
    return s;
}
__device__ __forceinline__ double block_min(double v, double *red) { return -block_max(-v, red); }

struct Smem {
    double *y, *d, *grad, *pg, *yn, *gn, *dG, *dt, *gacc, *red;
    float *part, *wchunk, *coef;
    int *sk;
};

// value[slot] = sum_i coef[i] * Dd[sk[i]][slot] for the 128 slots of chunk c; the beam loop is split
// over the warps, partials meet in shared memory and are added in warp order.  Result valid for
// tid < 128 (slot = c*128 + tid).  Ends with the block in sync.
__device__ __forceinline__ float combine_chunk(const MasterArgs &a, const Smem &sm, int K, int c) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const float4 *base = reinterpret_cast<const float4 *>(a.Dd + (size_t)c * kChunk) + lane;
    const size_t stride4 = (size_t)a.Sp / 4;
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll 4
    for (int i = warp; i < K; i += kMasterWarps) {
        const float cf = sm.coef[i];
        if (cf != 0.f) {
            const float4 v = __ldg(base + (size_t)sm.sk[i] * stride4);
            acc.x = fmaf(cf, v.x, acc.x);
            acc.y = fmaf(cf, v.y, acc.y);
            acc.z = fmaf(cf, v.z, acc.z);
            acc.w = fmaf(cf, v.w, acc.w);
        }
    }
    reinterpret_cast<float4 *>(sm.part)[warp * 32 + lane] = acc;
    __syncthreads();
    float r = 0.f;
    if (tid < kChunk) {
#pragma unroll
        for (int wv = 0; wv < kMasterWarps; ++wv) r += sm.part[wv * kChunk + tid];
    }
    return r;
}

__device__ __forceinline__ void penalty(float z, float T, float al, float be, float &w, double &F) {
    const float under = fmaxf(0.f, T - z), over = fmaxf(0.f, z - T);
    w = -2.f * al * under + 2.f * be * over;                                       // Eq. 1, derivative
    F = (double)al * (double)under * (double)under + (double)be * (double)over * (double)over;
}

// One pass over the block's chunks that evaluates the objective at a new dose:
//   from_y:  z_new = sum_k y_k d_k            (coef must hold y)             -> stored to zdst, w to a.w
//   else:    z_new = zsrc + t q               (line-search trial)            -> stored to zdst
// and in the same pass F (partial, fp64) and the block's share of grad = Dc w_new.
__device__ __forceinline__ void eval_pass(const MasterArgs &a, const Smem &sm, int K, int c0, int c1, bool from_y,
                                          const float *zsrc, float *zdst, float tf, double *partF, double *partG) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const size_t stride4 = (size_t)a.Sp / 4;
    for (int i = tid; i < K; i += kMasterThreads) sm.gacc[i] = 0.0;
    double F = 0.0;
    __syncthreads();
    for (int c = c0; c < c1; ++c) {
        float zv = 0.f;
        if (from_y) zv = combine_chunk(a, sm, K, c);
        if (tid < kChunk) {
            const size_t s = (size_t)c * kChunk + tid;
            if (!from_y) zv = fmaf(tf, a.q[s], zsrc[s]);
            float wv;
            double f;
            penalty(zv, a.T[s], a.alpha[s], a.beta[s], wv, f);
            F += f;
            zdst[s] = zv;
            if (from_y) a.w[s] = wv;
            sm.wchunk[tid] = wv;
        }
        __syncthreads();
        const float4 w4 = reinterpret_cast<const float4 *>(sm.wchunk)[lane];
        const float4 *base = reinterpret_cast<const float4 *>(a.Dd + (size_t)c * kChunk) + lane;
#pragma unroll 4
        for (int i = warp; i < K; i += kMasterWarps) {
            const float4 v = __ldg(base + (size_t)sm.sk[i] * stride4);
            double dot = (double)(v.x * w4.x + v.y * w4.y) + (double)(v.z * w4.z + v.w * w4.w);
            dot = warp_sum(dot);
            if (lane == 0) sm.gacc[i] += dot;   // index i is owned by this warp
        }
        __syncthreads();
    }
    F = block_sum(F, sm.red);
    if (tid == 0) partF[blockIdx.x] = F;
    for (int i = tid; i < K; i += kMasterThreads) partG[(size_t)blockIdx.x * a.N + i] = sm.gacc[i];
}

// G(v) = sum_k (v_{k+1}-v_k)^2 / (theta_{k+1}-theta_k)   (Eq. 2; S2, S3)
__device__ __forceinline__ double smooth_G(const double *v, const Smem &sm, int N) {
    double s = 0.0;
    for (int k = threadIdx.x; k + 1 < N; k += kMasterThreads) {
        const double dv = v[k + 1] - v[k];
        s += dv * dv / sm.dt[k];
    }
    return block_sum(s, sm.red);
}
__device__ __forceinline__ void smooth_dG(const double *v, const Smem &sm, int N) {
    for (int k = threadIdx.x; k < N; k += kMasterThreads) {
        double s = 0.0;
        if (k > 0) s += 2.0 * (v[k] - v[k - 1]) / sm.dt[k - 1];
        if (k + 1 < N) s -= 2.0 * (v[k + 1] - v[k]) / sm.dt[k];
        sm.dG[k] = s;
    }
    __syncthreads();
}

__global__ void __launch_bounds__(kMasterThreads) k_master(const MasterArgs a) {
    cg::grid_group grid = cg::this_grid();
    extern __shared__ float4 smem_raw[];   // 16-byte aligned: float4 tiles first, then doubles, floats, ints
    const int N = a.N, tid = threadIdx.x;
    Smem sm;
    sm.part = reinterpret_cast<float *>(smem_raw);
    sm.wchunk = sm.part + kMasterWarps * kChunk;
    sm.y = reinterpret_cast<double *>(sm.wchunk + kChunk);
    sm.d = sm.y + N;
    sm.grad = sm.d + N;
    sm.pg = sm.grad + N;
    sm.yn = sm.pg + N;
    sm.gn = sm.yn + N;
    sm.dG = sm.gn + N;
    sm.dt = sm.dG + N;
    sm.gacc = sm.dt + N;
    sm.red = sm.gacc + N;
    sm.coef = reinterpret_cast<float *>(sm.red + kMasterWarps);
    sm.sk = reinterpret_cast<int *>(sm.coef + N);
    __shared__ int sK;

    // occupied beams in ascending order
    if (tid < 32) {
        int base = 0;
        for (int k0 = 0; k0 < N; k0 += 32) {
            const int k = k0 + tid;
            const bool f = k < N && a.occ[k];
            const unsigned m = __ballot_sync(kFull, f);
            if (f) sm.sk[base + __popc(m & ((1u << tid) - 1u))] = k;
            base += __popc(m);
        }
        if (tid == 0) sK = base;
    }
    for (int k = tid; k < N; k += kMasterThreads) {
        double yk = a.y[k];
        if (!a.occ[k] || !(yk > 0.0)) yk = 0.0;
        sm.y[k] = yk;
        sm.d[k] = 0.0;
        sm.dt[k] = k + 1 < N ? a.theta[k + 1] - a.theta[k] : 1.0;
    }
    __syncthreads();
    const int K = sK;

    // this block's chunks
    const int G = gridDim.x;
    const int per = (a.nchunks + G - 1) / G;
    const int c0 = min(a.nchunks, (int)blockIdx.x * per), c1 = min(a.nchunks, c0 + per);
    const int nb = (a.nchunks + per - 1) / per;   // blocks that own chunks
    double *partF[2] = {a.partF, a.partF + G};
    double *partG[2] = {a.partG, a.partG + (size_t)G * N};
    int buf = 0;

    auto reduce_eval = [&](int b, const double *yv, double &F, double &Gv) {
        // F, and gn = Dc w + gamma dG(yv) at occupied beams (0 elsewhere)
        double s = 0.0;
        for (int i = tid; i < nb; i += kMasterThreads) s += __ldcg(partF[b] + i);
        F = block_sum(s, sm.red) + a.F_out;
        Gv = smooth_G(yv, sm, N);
        smooth_dG(yv, sm, N);
        for (int k = tid; k < N; k += kMasterThreads) sm.gn[k] = 0.0;
        __syncthreads();
        for (int i = tid; i < K; i += kMasterThreads) {
            double g = 0.0;
            for (int bb = 0; bb < nb; ++bb) g += __ldcg(partG[b] + (size_t)bb * N + i);
            const int k = sm.sk[i];
            sm.gn[k] = g + a.gamma * sm.dG[k];
        }
        __syncthreads();
    };

    float *zcur = a.z, *znext = a.zn;

    // objective and gradient at the incoming y
    for (int i = tid; i < K; i += kMasterThreads) sm.coef[i] = (float)sm.y[sm.sk[i]];
    __syncthreads();
    eval_pass(a, sm, K, c0, c1, true, nullptr, zcur, 0.f, partF[buf], partG[buf]);
    grid.sync();
    double F, Gs;
    reduce_eval(buf, sm.y, F, Gs);
    buf ^= 1;
    double Phi = F + a.gamma * Gs;

    double pgl = 0.0;
    for (int k = tid; k < N; k += kMasterThreads) {
        const double gk = sm.gn[k];
        const double p = (!a.occ[k] || (sm.y[k] <= 0.0 && gk >= 0.0)) ? 0.0 : gk;
        sm.grad[k] = gk;
        sm.pg[k] = p;
        sm.d[k] = -p;
        pgl = fmax(pgl, fabs(p));
    }
    double pgmax = block_max(pgl, sm.red);
    const double pg_entry = pgmax;
    const double tol = a.eps * fmax(1.0, pgmax);
    const double c1a = 1e-4, noise = 2e-7;
    int inner = 0, backtracks = 0, stop = 0, stall = 0;

    while (pgmax > tol) {
        if (inner >= a.max_inner) {
            stop = 1;
            break;
        }
        // slope along d; fall back to steepest descent if d is not a descent direction
        double s = 0.0;
        for (int k = tid; k < N; k += kMasterThreads) s += sm.grad[k] * sm.d[k];
        double phi1 = block_sum(s, sm.red);
        if (!(phi1 < 0.0)) {
            s = 0.0;
            for (int k = tid; k < N; k += kMasterThreads) {
                sm.d[k] = -sm.pg[k];
                s += sm.grad[k] * sm.d[k];
            }
            phi1 = block_sum(s, sm.red);
            if (!(phi1 < 0.0)) {
                stop = 2;
                break;
            }
        }
        // q = Dc^T d and the curvature of the quadratic piece at t = 0
        for (int i = tid; i < K; i += kMasterThreads) sm.coef[i] = (float)sm.d[sm.sk[i]];
        __syncthreads();
        double curv = 0.0;
        for (int c = c0; c < c1; ++c) {
            const float qv = combine_chunk(a, sm, K, c);
            if (tid < kChunk) {
                const size_t sl = (size_t)c * kChunk + tid;
                const float zv = zcur[sl], Tv = a.T[sl];
                const float om = zv < Tv ? a.alpha[sl] : (zv > Tv ? a.beta[sl] : 0.f);
                curv += (double)om * (double)qv * (double)qv;
                a.q[sl] = qv;
            }
            __syncthreads();
        }
        curv = block_sum(curv, sm.red);
        if (tid == 0) a.partA[blockIdx.x] = curv;
        grid.sync();
        s = 0.0;
        for (int i = tid; i < nb; i += kMasterThreads) s += __ldcg(a.partA + i);
        const double curvF = block_sum(s, sm.red);
        const double phi2 = 2.0 * curvF + 2.0 * a.gamma * smooth_G(sm.d, sm, N);   // d^T L d = G(d)
        double tl = CUDART_INF;
        for (int k = tid; k < N; k += kMasterThreads)
            if (sm.d[k] < 0.0) tl = fmin(tl, sm.y[k] / (-sm.d[k]));
        const double tmax = block_min(tl, sm.red);
        double t = phi2 > 0.0 ? -phi1 / phi2 : (isfinite(tmax) ? tmax : 1.0);
        int hit = 0;
        if (t >= tmax) {
            t = tmax;
            hit = 1;
        }
        // backtracking on the true cost
        bool accepted = false;
        double Fn = 0.0, Gn = 0.0, Phin = 0.0;
        for (int half = 0; half < 60; ++half) {
            for (int k = tid; k < N; k += kMasterThreads) {
                double v = sm.y[k] + t * sm.d[k];
                if (v < 0.0 || (hit && sm.d[k] < 0.0 && sm.y[k] / (-sm.d[k]) <= tmax)) v = 0.0;
                sm.yn[k] = v;
            }
            __syncthreads();
            eval_pass(a, sm, K, c0, c1, false, zcur, znext, (float)t, partF[buf], partG[buf]);
            grid.sync();
            reduce_eval(buf, sm.yn, Fn, Gn);
            buf ^= 1;
            Phin = Fn + a.gamma * Gn;
            if (Phin <= Phi + c1a * t * phi1) accepted = true;
            else if (Phin <= Phi + noise * fabs(Phi)) {
                // below the resolution of Phi: accept on the slope instead
                s = 0.0;
                for (int k = tid; k < N; k += kMasterThreads) s += sm.gn[k] * sm.d[k];
                const double phi1n = block_sum(s, sm.red);
                if (fabs(phi1n) <= 0.9 * fabs(phi1)) accepted = true;
            }
            if (accepted) break;
            t *= 0.5;
            hit = 0;
            ++backtracks;
        }
        if (!accepted) {
            stop = 3;
            break;
        }
        // take the step
        stall = (Phi - Phin <= 1e-8 * fabs(Phi)) ? stall + 1 : 0;
        float *tmpz = zcur;
        zcur = znext;
        znext = tmpz;
        F = Fn;
        Gs = Gn;
        Phi = Phin;
        // Polak-Ribiere+ direction on the current face, restart when the active set changes
        double num = 0.0, den = 0.0, pgm = 0.0;
        int changed = hit;
        for (int k = tid; k < N; k += kMasterThreads) {
            const double yk = sm.yn[k], gk = sm.gn[k];
            const double pn = (!a.occ[k] || (yk <= 0.0 && gk >= 0.0)) ? 0.0 : gk;
            const double po = sm.pg[k];
            if ((pn == 0.0) != (po == 0.0)) changed = 1;
            num += pn * (pn - po);
            den += po * po;
            pgm = fmax(pgm, fabs(pn));
            sm.y[k] = yk;
            sm.grad[k] = gk;
            sm.pg[k] = pn;
        }
        changed = __syncthreads_or(changed);
        num = block_sum(num, sm.red);
        den = block_sum(den, sm.red);
        pgmax = block_max(pgm, sm.red);
        const double bpr = (changed || !(den > 0.0) || num <= 0.0) ? 0.0 : num / den;
        for (int k = tid; k < N; k += kMasterThreads) {
            double dk = -sm.pg[k] + bpr * sm.d[k];
            if (!a.occ[k] || (sm.y[k] <= 0.0 && dk < 0.0)) dk = 0.0;   // stay feasible
            sm.d[k] = dk;
        }
        __syncthreads();
        ++inner;
        if (stall >= 3 && pgmax > tol) {
            stop = 4;
            break;
        }
    }

    // z, w and the cost from the final y (no drift from the z += t q updates)
    if (inner > 0 || zcur != a.z) {
        for (int i = tid; i < K; i += kMasterThreads) sm.coef[i] = (float)sm.y[sm.sk[i]];
        __syncthreads();
        eval_pass(a, sm, K, c0, c1, true, nullptr, a.z, 0.f, partF[buf], partG[buf]);
        grid.sync();
        reduce_eval(buf, sm.y, F, Gs);
        Phi = F + a.gamma * Gs;
    }
    if (blockIdx.x == 0) {
        for (int k = tid; k < N; k += kMasterThreads) a.y[k] = sm.y[k];
        if (tid == 0) {
            MasterOut o;
            o.inner = inner;
            o.backtracks = backtracks;
            o.stop_reason = stop;
            o.pad = 0;
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

size_t master_smem_bytes(int64_t N) {
    return (size_t)(9 * N + kMasterWarps) * 8 + (size_t)(kMasterWarps * kChunk + kChunk + N) * 4 + (size_t)N * 4;
}

}  // namespace

int master_configure(vmat_plan *p) {
    p->master_smem = master_smem_bytes(p->N);
    if (p->master_smem > 200 * 1024) return fail(p, VMAT_EINVAL, "n_beams too large for the master kernel's shared memory");
    VMAT_CUDA(p, cudaFuncSetAttribute(k_master, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p->master_smem));
    int per_sm = 0;
    VMAT_CUDA(p, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_master, kMasterThreads, p->master_smem));
    if (per_sm < 1) return fail(p, VMAT_ECUDA, "master kernel does not fit on an SM");
    if (per_sm > 2) per_sm = 2;
    const int64_t nchunks = p->Sp / kChunk;
    int64_t grid = (int64_t)per_sm * p->sm_count;
    if (grid > nchunks) grid = nchunks;
    if (grid < 1) grid = 1;
    p->master_grid = (int)grid;
    int rc;
    if ((rc = dev_alloc(p, &p->partA, grid))) return rc;
    if ((rc = dev_alloc(p, &p->partF, 2 * grid))) return rc;
    if ((rc = dev_alloc(p, &p->partG, 2 * grid * p->N))) return rc;
    return VMAT_OK;
}

int launch_column_build(vmat_plan *p, int beam) {
    const Sel *sel = beam < 0 ? p->sel : nullptr;
    const unsigned blocks = (unsigned)((p->RC + 7) / 8);
    k_column_scatter<<<blocks, 256, 0, p->stream>>>(p->rowq, p->val4, p->col4, sel, beam, p->left, p->right, (int)p->R,
                                                   (int)p->C, p->fx_scale, p->acc);
    k_column_finish<<<(unsigned)((p->Sp + 255) / 256), 256, 0, p->stream>>>(p->acc, (long long)p->Sp, sel, beam,
                                                                          p->fx_inv, p->Dd);
    p->launches += 2;
    VMAT_CUDA(p, cudaGetLastError());
    return VMAT_OK;
}

static int launch_master_impl(vmat_plan *p, int max_inner, int trace_it) {
    MasterArgs a;
    a.Dd = p->Dd;
    a.Sp = (long long)p->Sp;
    a.nchunks = (int)(p->Sp / kChunk);
    a.T = p->T_s;
    a.alpha = p->alpha_s;
    a.beta = p->beta_s;
    a.z = p->z_s;
    a.zn = p->zn_s;
    a.q = p->q_s;
    a.w = p->w_s;
    a.occ = p->occ;
    a.y = p->y;
    a.theta = p->theta;
    a.N = (int)p->N;
    a.gamma = p->gamma;
    a.F_out = p->F_out;
    a.eps = p->opt.master_eps;
    a.max_inner = max_inner;
    a.partA = p->partA;
    a.partF = p->partF;
    a.partG = p->partG;
    a.out = p->mout;
    a.cost3 = p->cost3;
    a.trF = p->tr_F;
    a.trG = p->tr_G;
    a.trC = p->tr_cost;
    a.trInner = p->tr_inner;
    a.trace_it = trace_it;
    void *args[] = {&a};
    VMAT_CUDA(p, cudaLaunchCooperativeKernel((void *)k_master, dim3((unsigned)p->master_grid), dim3(kMasterThreads), args,
                                             p->master_smem, p->stream));
    ++p->launches;
    return VMAT_OK;
}

int launch_master(vmat_plan *p, int trace_it) { return launch_master_impl(p, p->opt.master_max_inner, trace_it); }

// steps (a)+(b) alone: the master kernel's evaluation pass with no iteration allowed
int launch_dose_grad(vmat_plan *p) { return launch_master_impl(p, 0, -1); }

int launch_expand(vmat_plan *p, const float *src_s, float *dst_V, int what) {
    if (p->V == 0) return VMAT_OK;
    k_expand<<<(unsigned)((p->V + 255) / 256), 256, 0, p->stream>>>(src_s, p->slot_of, p->T_V, p->alpha_V, p->beta_V,
                                                                   (long long)p->V, what, dst_V);
    ++p->launches;
    VMAT_CUDA(p, cudaGetLastError());
    return VMAT_OK;
}

int launch_compress(vmat_plan *p, const float *src_V, float *dst_s) {
    k_compress<<<(unsigned)((p->Sp + 255) / 256), 256, 0, p->stream>>>(src_V, p->voxel_of, (long long)p->S,
                                                                      (long long)p->Sp, dst_s);
    ++p->launches;
    VMAT_CUDA(p, cudaGetLastError());
    return VMAT_OK;
}

int launch_direct_dose(vmat_plan *p) { return fail(p, VMAT_ESTATE, "direct dose path not built"); }

}  // namespace vmat
