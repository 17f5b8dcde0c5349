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

struct DoseScale {
    double scale, inv;            // fixed-point scale of y_k * D_ij and its inverse (powers of two)
    double G;                     // Eq. 2
};

// one block: the scale from max y (|y_k D_ij| * scale < 2^40 given |D_ij| * fx_scale <= 2^40), and G(y)
__global__ void __launch_bounds__(kDoseThreads)
k_dose_prepare(const uint8_t *__restrict__ occ, const double *__restrict__ y, const double *__restrict__ theta, int N,
               double fx_scale, DoseScale *__restrict__ out) {
    pdl_trigger();   // the scatter may be scheduled; it waits for the scale itself
    __shared__ double s_max[kDoseThreads / 32], s_sum[kDoseThreads / 32];
    double mx = 0.0, g = 0.0;
    for (int k = threadIdx.x; k < N; k += kDoseThreads) {
        const double yk = occ[k] ? y[k] : 0.0;
        mx = fmax(mx, fabs(yk));
        if (k + 1 < N) {
            const double yn = occ[k + 1] ? y[k + 1] : 0.0, dv = yn - yk;
            g += dv * dv / (theta[k + 1] - theta[k]);
        }
    }
#pragma unroll
    for (int o = 16; o; o >>= 1) {
        mx = fmax(mx, __shfl_xor_sync(kFull, mx, o));
        g += __shfl_xor_sync(kFull, g, o);
    }
    if ((threadIdx.x & 31) == 0) {
        s_max[threadIdx.x >> 5] = mx;
        s_sum[threadIdx.x >> 5] = g;
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
        DoseScale d;
        d.scale = ldexp(fx_scale, -e);
        d.inv = 1.0 / d.scale;
        d.G = g;
        *out = d;
    }
}

// kDoseLanes lanes per beamlet; beamlets that are not exposed leave at once
__global__ void __launch_bounds__(kDoseThreads)
k_dose_scatter(const uint32_t *__restrict__ rowq, const float4 *__restrict__ val4, const int4 *__restrict__ col4,
               const uint8_t *__restrict__ occ, const int32_t *__restrict__ left, const int32_t *__restrict__ right,
               const double *__restrict__ y, int R, int C, long long B, const DoseScale *__restrict__ ds,
               unsigned long long *__restrict__ acc) {
    pdl_wait();
    pdl_trigger();
    const int lane = threadIdx.x & (kDoseLanes - 1);
    const long long row = (long long)blockIdx.x * (kDoseThreads / kDoseLanes) + threadIdx.x / kDoseLanes;
    if (row >= B) return;
    const int c = (int)(row % C);
    const long long kr = row / C;
    const int k = (int)(kr / R);
    if (!occ[k] || c < left[kr] || c >= right[kr]) return;     // beamlet not in A_k
    const double f = y[k] * ds->scale;
    if (f == 0.0) return;
    // One ENTRY per lane and step: the lanes of a beamlet then hold consecutive entries of the row, whose voxel
    // ids come in runs of consecutive slots (a beamlet's lateral support), so one warp-wide reduction instruction
    // lands several of its 64-bit adds in the same 32-byte sector of the accumulator and the L2 merges them.
    // (With one quad per lane the four adds of a run went out as four instructions: 1.8 adds per sector op
    // measured, and the pass ran at the L2 reduction rate, not at the HBM rate.)
    const float *__restrict__ val = reinterpret_cast<const float *>(val4);
    const int *__restrict__ col = reinterpret_cast<const int *>(col4);
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

// accumulator -> z, w; clears the accumulator; per-block partial of F (fixed order within the block)
__global__ void __launch_bounds__(kDoseThreads)
k_dose_finish(unsigned long long *__restrict__ acc, long long Sp, const DoseScale *__restrict__ ds,
              const float *__restrict__ T, const float *__restrict__ alpha, const float *__restrict__ beta,
              float *__restrict__ z, float *__restrict__ w, double *__restrict__ partF) {
    pdl_wait();
    pdl_trigger();
    __shared__ double s_sum[kDoseThreads / 32];
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
    }
}

// one block: F = F_out + sum of the partials in index order; cost3 = {F, G, F + gamma G}
__global__ void __launch_bounds__(kDoseThreads)
k_dose_cost(const double *__restrict__ partF, int nblocks, double F_out, double gamma, const DoseScale *__restrict__ ds,
            double *__restrict__ cost3) {
    pdl_wait();
    __shared__ double s_sum[kDoseThreads];
    double f = 0.0;
    for (int i = threadIdx.x; i < nblocks; i += kDoseThreads) f += partF[i];
    s_sum[threadIdx.x] = f;
    __syncthreads();
    for (int o = kDoseThreads / 2; o; o >>= 1) {
        if (threadIdx.x < o) s_sum[threadIdx.x] += s_sum[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        const double F = s_sum[0] + F_out;
        cost3[0] = F;
        cost3[1] = ds->G;
        cost3[2] = F + gamma * ds->G;
    }
}

}  // namespace

int dose_configure(vmat_plan *p) {
    p->dose_blocks = (int)((p->Sp + kDoseThreads - 1) / kDoseThreads);
    int rc;
    if ((rc = dev_alloc(p, &p->part_dose, p->dose_blocks))) return rc;
    if ((rc = dev_alloc(p, (DoseScale **)&p->dose_scale, 1))) return rc;
    return VMAT_OK;
}

// z_s, w_s, cost3 for the plan's (occ, leaves, y) straight from D; p->acc must be all zero (it is between uses)
int launch_direct_dose(vmat_plan *p) {
    DoseScale *ds = (DoseScale *)p->dose_scale;
    k_dose_prepare<<<1, kDoseThreads, 0, p->stream>>>(p->occ, p->y, p->theta, (int)p->N, p->fx_scale, ds);
    if (p->B > 0) {
        const int rows_per_block = kDoseThreads / kDoseLanes;
        const unsigned blocks = (unsigned)((p->B + rows_per_block - 1) / rows_per_block);
        VMAT_CUDA(p, launch_pdl(k_dose_scatter, dim3(blocks), dim3(kDoseThreads), p->stream, p->rowq, p->val4, p->col4, p->occ,
                                p->left, p->right, p->y, (int)p->R, (int)p->C, (long long)p->B, ds, p->acc));
    }
    VMAT_CUDA(p, launch_pdl(k_dose_finish, dim3((unsigned)p->dose_blocks), dim3(kDoseThreads), p->stream, p->acc,
                            (long long)p->Sp, ds, p->T_s, p->alpha_s, p->beta_s, p->z_s, p->w_s, p->part_dose));
    VMAT_CUDA(p, launch_pdl(k_dose_cost, dim3(1), dim3(kDoseThreads), p->stream, p->part_dose, p->dose_blocks, p->F_out,
                            p->gamma, ds, p->cost3));
    p->launches += 4;
    VMAT_CUDA(p, cudaGetLastError());
    return VMAT_OK;
}

}  // namespace vmat
