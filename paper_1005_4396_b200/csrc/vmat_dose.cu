// vmat_dose.cu — steps (a)+(b) straight from D: the fused dose + penalty-gradient pass over the
// beamlet-major CSR (BASELINE.json north_star: "beamlet-major CSR, plus a voxel-major copy or an
// atomics path for dose, chosen by measurement"; this is the atomics path).
//
//   z_j = sum_k y_k sum_{i in A_k} D_ij
//   w_j = -2 alpha_j max(0,T_j-z_j) + 2 beta_j max(0,z_j-T_j),  F = sum_j F(z_j)   (Eq. 1)
//   G   = sum_k (y_{k+1}-y_k)^2 / (theta_{k+1}-theta_k)                            (Eq. 2)
//
// Only the rows of exposed beamlets are streamed (8 bytes per stored entry, 16 lanes per beamlet, one
// entry per lane and step); every product y_k D_ij is added to its voxel's 64-bit FIXED-POINT accumulator, so
// the sum does not depend on the order in which the atomics land and the dose is bit-reproducible.
// A second pass over the support turns the accumulator into z and w, clears it and sums F in a
// fixed order.  vmat_dose uses this path when vmat_options.dose_path = 1; the default (0) forms
// z = sum_k y_k d_k from the aperture-dose columns the master problem keeps anyway (vmat_master.cu).
// bench.py times both (DESIGN.md section 6 has the numbers behind the default).
#include <math_constants.h>

#include "vmat_internal.cuh"

namespace vmat {

namespace {

constexpr unsigned kFull = 0xffffffffu;
constexpr int kDoseThreads = 256;
constexpr int kDoseLanes = 16;    // lanes per beamlet
constexpr int kDoseEntries = 8;   // 4-byte loads of values and of indices in flight per lane

// this thread's share of Eq. 2: the pairs (k, next(k)) for k = first, first + stride, ..; next(k) = k + 1 with
// y = 0 at un-occupied beams (S2), or the next occupied beam (the other reading, occ_only)
__device__ __forceinline__ double smooth_share(const uint8_t *occ, const double *y, const double *theta, int N, int occ_only,
                                               int first, int stride) {
    double g = 0.0;
    for (int k = first; k + 1 < N; k += stride) {
        if (occ_only && !occ[k]) continue;
        int n = k + 1;
        if (occ_only)
            while (n < N && !occ[n]) ++n;
        if (n >= N) continue;
        const double y0 = occ[k] ? y[k] : 0.0, y1 = occ[n] ? y[n] : 0.0, dv = y1 - y0;
        g += dv * dv / (theta[n] - theta[k]);
    }
    return g;
}

struct DoseScale {
    double scale, inv;            // fixed-point scale of y_k * D_ij and its inverse (powers of two)
    double G;                     // Eq. 2
    unsigned int count;           // exposed beamlets listed by k_dose_prepare (reset by k_dose_finish)
    unsigned int ticket;          // blocks of k_dose_finish that are done (reset by the last one)
    unsigned int ticket2;         // the same for k_dose_columns
};

// First launch of the pass.  Every block lists the exposed beamlets of 256 leaf rows (k, r) of occupied beams (PAPER.md:69,
// the sets A_k) in exp_list (any order: what each adds to the accumulator is an integer); block 0 also forms the scale
// from max y (|y_k D_ij| * scale < 2^40 given |D_ij| * fx_scale <= 2^40) and G(y).
__global__ void __launch_bounds__(kDoseThreads)
k_dose_prepare(const uint8_t *__restrict__ occ, const int32_t *__restrict__ left, const int32_t *__restrict__ right,
               const double *__restrict__ y, const double *__restrict__ theta, int N, int R, int C, double fx_scale,
               int occ_only, DoseScale *__restrict__ out, int32_t *__restrict__ exp_list) {
    pdl_trigger();   // the scatter may be scheduled; it waits for the list and the scale itself
    __shared__ double s_max[kDoseThreads / 32], s_sum[kDoseThreads / 32];
    __shared__ int s_cnt[kDoseThreads / 32];
    __shared__ unsigned s_base;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    // exposed beamlets of this thread's leaf row
    const int kr = blockIdx.x * kDoseThreads + threadIdx.x;
    int n = 0, l = 0;
    if (kr < N * R && occ[kr / R] && y[kr / R] != 0.0) {
        l = left[kr];
        n = max(0, right[kr] - l);
    }
    int incl = n;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int v = __shfl_up_sync(kFull, incl, o);
        if (lane >= o) incl += v;
    }
    if (lane == 31) s_cnt[warp] = incl;
    __syncthreads();
    int before = 0, total = 0;
    for (int w2 = 0; w2 < kDoseThreads / 32; ++w2) {
        if (w2 < warp) before += s_cnt[w2];
        total += s_cnt[w2];
    }
    if (threadIdx.x == 0) s_base = total ? atomicAdd(&out->count, (unsigned)total) : 0u;
    __syncthreads();
    int32_t *dst = exp_list + s_base + before + incl - n;
    for (int c = 0; c < n; ++c) dst[c] = kr * C + l + c;
    if (blockIdx.x != 0) return;
    double mx = 0.0, g = smooth_share(occ, y, theta, N, occ_only, threadIdx.x, kDoseThreads);
    for (int k = threadIdx.x; k < N; k += kDoseThreads) mx = fmax(mx, occ[k] ? fabs(y[k]) : 0.0);
#pragma unroll
    for (int o = 16; o; o >>= 1) {
        mx = fmax(mx, __shfl_xor_sync(kFull, mx, o));
        g += __shfl_xor_sync(kFull, g, o);
    }
    if (lane == 0) {
        s_max[warp] = mx;
        s_sum[warp] = g;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int i = 1; i < kDoseThreads / 32; ++i) {
            mx = fmax(mx, s_max[i]);
            g += s_sum[i];
        }
        int e = 0;
        frexp(fmax(mx, 1e-300), &e);   // mx < 2^e
        if (e < -200) e = -200;
        out->scale = ldexp(fx_scale, -e);
        out->inv = 1.0 / out->scale;
        out->G = g;
    }
}

// kDoseLanes lanes per exposed beamlet, the listed beamlets dealt to the lane groups of a fixed grid
__global__ void __launch_bounds__(kDoseThreads)
k_dose_scatter(const uint32_t *__restrict__ rowq, const float4 *__restrict__ val4, const int4 *__restrict__ col4,
               const double *__restrict__ y, int RC, const DoseScale *__restrict__ ds,
               const int32_t *__restrict__ exp_list, unsigned long long *__restrict__ acc) {
    pdl_wait();
    pdl_trigger();
    const int lane = threadIdx.x & (kDoseLanes - 1);
    const unsigned count = ds->count, ngroups = gridDim.x * (kDoseThreads / kDoseLanes);
    const double scale = ds->scale;
    // One ENTRY per lane and step: the lanes of a beamlet then hold consecutive entries of the row, whose voxel
    // ids come in runs of consecutive slots (a beamlet's lateral support), so one warp-wide reduction instruction
    // lands several of its 64-bit adds in the same 32-byte sector of the accumulator and the L2 merges them.
    // (With one quad per lane the four adds of a run went out as four instructions: 1.8 adds per sector op
    // measured, and the pass ran at the L2 reduction rate, not at the HBM rate.)
    const float *__restrict__ val = reinterpret_cast<const float *>(val4);
    const int *__restrict__ col = reinterpret_cast<const int *>(col4);
    for (unsigned i = blockIdx.x * (kDoseThreads / kDoseLanes) + threadIdx.x / kDoseLanes; i < count; i += ngroups) {
        const long long row = exp_list[i];
        const double f = y[row / RC] * scale;
        const uint64_t a = (uint64_t)rowq[row] * 4u, b = (uint64_t)rowq[row + 1] * 4u;   // entries: past 2^32 from 2^30 quads on
        for (uint64_t e = a + lane; e < b; e += kDoseLanes * kDoseEntries) {
            float v[kDoseEntries];
            int s[kDoseEntries];
#pragma unroll
            for (int u = 0; u < kDoseEntries; ++u) {
                const bool in = e + kDoseLanes * u < b;
                v[u] = in ? __ldg(val + e + kDoseLanes * u) : 0.f;
                s[u] = in ? __ldg(col + e + kDoseLanes * u) : 0;
            }
#pragma unroll
            for (int u = 0; u < kDoseEntries; ++u)
                if (v[u] != 0.f) atomicAdd(acc + s[u], (unsigned long long)__double2ll_rn((double)v[u] * f));
        }
    }
}

// accumulator -> z, w; clears the accumulator; per-block partial of F (fixed order within the block); the block that
// finishes last adds the partials in index order: cost3 = {F, G, F + gamma G}
__global__ void __launch_bounds__(kDoseThreads)
k_dose_finish(unsigned long long *__restrict__ acc, long long Sp, DoseScale *__restrict__ ds,
              const float *__restrict__ T, const float *__restrict__ alpha, const float *__restrict__ beta,
              float *__restrict__ z, float *__restrict__ w, double *__restrict__ partF, double F_out, double gamma,
              double *__restrict__ cost3) {
    pdl_wait();
    __shared__ double s_sum[kDoseThreads];
    __shared__ int s_last;
    const long long s = (long long)blockIdx.x * kDoseThreads + threadIdx.x;
    double F = 0.0;
    if (s < Sp) {
        const long long v = (long long)acc[s];
        acc[s] = 0ull;
        const float zv = (float)((double)v * ds->inv);
        const float t = T[s], al = alpha[s], be = beta[s];
        const float under = fmaxf(0.f, t - zv), over = fmaxf(0.f, zv - t);
        z[s] = zv;
        w[s] = -2.f * al * under + 2.f * be * over;                                    // Eq. 1, derivative
        F = (double)al * (double)under * (double)under + (double)be * (double)over * (double)over;
    }
#pragma unroll
    for (int o = 16; o; o >>= 1) F += __shfl_xor_sync(kFull, F, o);
    if ((threadIdx.x & 31) == 0) s_sum[threadIdx.x >> 5] = F;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int i = 1; i < kDoseThreads / 32; ++i) F += s_sum[i];
        partF[blockIdx.x] = F;
        __threadfence();
        s_last = atomicAdd(&ds->ticket, 1u) == gridDim.x - 1u;
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    double f = 0.0;
    for (int i = threadIdx.x; i < (int)gridDim.x; i += kDoseThreads) f += __ldcg(partF + i);
    s_sum[threadIdx.x] = f;
    __syncthreads();
    for (int o = kDoseThreads / 2; o; o >>= 1) {
        if (threadIdx.x < o) s_sum[threadIdx.x] += s_sum[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        const double Ft = s_sum[0] + F_out;
        cost3[0] = Ft;
        cost3[1] = ds->G;
        cost3[2] = Ft + gamma * ds->G;
        ds->ticket = 0u;   // ready for the next pass
        ds->count = 0u;
    }
}


// ------------------------------------------------------------------------------------------------
// steps (a)+(b) from the aperture-dose columns: z = sum_k y_k d_k, no atomics
// ------------------------------------------------------------------------------------------------
// One block per chunk of 128 slots: the occupied beams whose column holds a non-zero entry in the chunk are listed
// (ascending), the eight warps take every eighth of them (one float4 of the column's 512-byte segment per lane, all
// loads of a warp in flight at once), the eight partial sums meet in shared memory in warp order (a fixed order: the
// pass is bit-reproducible), then w, F.  The block that finishes last adds the per-chunk F in chunk order and G.
constexpr int kColWarps = 8;

__global__ void __launch_bounds__(kColWarps * 32)
k_dose_columns(const float *__restrict__ Dd, int N, int nchunks, const uint8_t *__restrict__ occ,
               const double *__restrict__ y, const double *__restrict__ theta, const uint32_t *__restrict__ touch,
               int touch_words, const float *__restrict__ T, const float *__restrict__ alpha,
               const float *__restrict__ beta, float *__restrict__ z, float *__restrict__ w, double *__restrict__ partF,
               unsigned int *__restrict__ ticket, double F_out, double gamma, int occ_only, double *__restrict__ cost3) {
    __shared__ int s_list[2048];           // vmat_create: N <= 2048
    __shared__ float s_coef[2048];
    __shared__ int s_wcnt[kColWarps], s_n;
    __shared__ float4 s_part[kColWarps][32];
    __shared__ double s_f[kDoseThreads];
    __shared__ int s_last;
    const int c = blockIdx.x, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    // occupied beams with a non-zero dose rate that touch the chunk, ascending
    int run = 0;
    for (int k0 = 0; k0 < N; k0 += kColWarps * 32) {
        const int k = k0 + threadIdx.x;
        double yk = 0.0;
        const bool f = k < N && occ[k] && (yk = y[k]) != 0.0 && ((touch[(size_t)k * touch_words + (c >> 5)] >> (c & 31)) & 1u);
        const unsigned m = __ballot_sync(kFull, f);
        if (lane == 0) s_wcnt[warp] = __popc(m);
        __syncthreads();
        int before = run;
        for (int x = 0; x < warp; ++x) before += s_wcnt[x];
        if (f) {
            const int pos = before + __popc(m & ((1u << lane) - 1u));
            s_list[pos] = k;
            s_coef[pos] = (float)yk;
        }
        for (int x = 0; x < kColWarps; ++x) run += s_wcnt[x];
        __syncthreads();
    }
    const int n = run;
    const float4 *seg = reinterpret_cast<const float4 *>(Dd + (size_t)c * N * kChunk) + lane;
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int i0 = warp; i0 < n; i0 += kColWarps * 8) {
        float4 v[8];
        float cf[8];
#pragma unroll
        for (int x = 0; x < 8; ++x) {
            const int i = i0 + kColWarps * x;
            cf[x] = 0.f;
            v[x] = make_float4(0.f, 0.f, 0.f, 0.f);
            if (i < n) {
                cf[x] = s_coef[i];
                v[x] = __ldg(seg + (size_t)s_list[i] * (kChunk / 4));
            }
        }
#pragma unroll
        for (int x = 0; x < 8; ++x) {
            acc.x = fmaf(cf[x], v[x].x, acc.x);
            acc.y = fmaf(cf[x], v[x].y, acc.y);
            acc.z = fmaf(cf[x], v[x].z, acc.z);
            acc.w = fmaf(cf[x], v[x].w, acc.w);
        }
    }
    s_part[warp][lane] = acc;
    __syncthreads();
    double F = 0.0;
    if (threadIdx.x < kChunk) {
        const int sl = threadIdx.x;
        float zv = 0.f;
#pragma unroll
        for (int x = 0; x < kColWarps; ++x) zv += reinterpret_cast<const float *>(s_part[x])[sl];
        const size_t s = (size_t)c * kChunk + sl;
        const float t = T[s], al = alpha[s], be = beta[s];
        const float under = fmaxf(0.f, t - zv), over = fmaxf(0.f, zv - t);
        z[s] = zv;
        w[s] = -2.f * al * under + 2.f * be * over;                                    // Eq. 1, derivative
        F = (double)al * (double)under * (double)under + (double)be * (double)over * (double)over;
    }
    s_f[threadIdx.x] = F;
    __syncthreads();
    for (int o = kDoseThreads / 2; o; o >>= 1) {
        if ((int)threadIdx.x < o) s_f[threadIdx.x] += s_f[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        partF[c] = s_f[0];
        __threadfence();
        s_last = atomicAdd(ticket, 1u) == gridDim.x - 1u;
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    double f = 0.0;
    for (int i = threadIdx.x; i < nchunks; i += kDoseThreads) f += __ldcg(partF + i);
    const double g = smooth_share(occ, y, theta, N, occ_only, threadIdx.x, kDoseThreads);
    __shared__ double s_g[kDoseThreads];
    s_f[threadIdx.x] = f;
    s_g[threadIdx.x] = g;
    __syncthreads();
    for (int o = kDoseThreads / 2; o; o >>= 1) {
        if ((int)threadIdx.x < o) {
            s_f[threadIdx.x] += s_f[threadIdx.x + o];
            s_g[threadIdx.x] += s_g[threadIdx.x + o];
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        const double Ft = s_f[0] + F_out;
        cost3[0] = Ft;
        cost3[1] = s_g[0];
        cost3[2] = Ft + gamma * s_g[0];
        *ticket = 0u;
    }
}

}  // namespace

int dose_configure(vmat_plan *p) {
    p->dose_blocks = (int)((p->Sp + kDoseThreads - 1) / kDoseThreads);
    int rc;
    if ((rc = dev_alloc(p, &p->part_dose, p->dose_blocks))) return rc;
    if ((rc = dev_alloc(p, &p->part_dose2, p->Sp / kChunk))) return rc;
    if ((rc = dev_alloc(p, (DoseScale **)&p->dose_scale, 1))) return rc;
    if ((rc = dev_alloc(p, &p->dose_list, p->B))) return rc;
    VMAT_CUDA(p, cudaMemsetAsync(p->dose_scale, 0, sizeof(DoseScale), p->stream));
    return VMAT_OK;
}

// z_s, w_s, cost3 for the plan's (occ, leaves, y) from the aperture-dose columns of the occupied beams (which the caller
// has brought up to date): one launch
int launch_columns_dose(vmat_plan *p) {
    static_assert(kColWarps * 32 == kDoseThreads, "k_dose_columns is written for blocks of kDoseThreads");
    DoseScale *ds = (DoseScale *)p->dose_scale;
    const int nchunks = (int)(p->Sp / kChunk);
    k_dose_columns<<<(unsigned)nchunks, kDoseThreads, 0, p->stream>>>(p->Dd, (int)p->N, nchunks, p->occ, p->y, p->theta,
                                                                     p->col_touch, p->touch_words, p->T_s, p->alpha_s,
                                                                     p->beta_s, p->z_s, p->w_s, p->part_dose2, &ds->ticket2,
                                                                     p->F_out, p->gamma, p->opt.occupied_only_G ? 1 : 0,
                                                                     p->cost3);
    ++p->launches;
    VMAT_CUDA(p, cudaGetLastError());
    return VMAT_OK;
}

// z_s, w_s, cost3 for the plan's (occ, leaves, y) straight from D; p->acc must be all zero (it is between uses).
// Three launches chained by programmatic dependent launch: list the exposed beamlets (+ scale, G), scatter, finish (+ cost).
int launch_direct_dose(vmat_plan *p) {
    DoseScale *ds = (DoseScale *)p->dose_scale;
    const unsigned pblocks = (unsigned)((p->N * p->R + kDoseThreads - 1) / kDoseThreads);
    k_dose_prepare<<<pblocks, kDoseThreads, 0, p->stream>>>(p->occ, p->left, p->right, p->y, p->theta, (int)p->N, (int)p->R,
                                                            (int)p->C, p->fx_scale, p->opt.occupied_only_G ? 1 : 0, ds,
                                                            p->dose_list);
    if (p->B > 0) {
        // a fixed grid (a few blocks per SM) walks the list: its length is known on the device only
        const unsigned blocks = (unsigned)(p->sm_count * 6);   // (16 per SM measured the same: the reductions bound the pass)
        VMAT_CUDA(p, launch_pdl(k_dose_scatter, dim3(blocks), dim3(kDoseThreads), p->stream, p->rowq, p->val4, p->col4, p->y,
                                (int)p->RC, ds, p->dose_list, p->acc));
    }
    VMAT_CUDA(p, launch_pdl(k_dose_finish, dim3((unsigned)p->dose_blocks), dim3(kDoseThreads), p->stream, p->acc,
                            (long long)p->Sp, ds, p->T_s, p->alpha_s, p->beta_s, p->z_s, p->w_s, p->part_dose, p->F_out,
                            p->gamma, p->cost3));
    p->launches += 3;
    VMAT_CUDA(p, cudaGetLastError());
    return VMAT_OK;
}

}  // namespace vmat
