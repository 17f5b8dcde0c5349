// vmat_column.cu — the aperture-dose column of a newly committed aperture, d_k = sum_{i in A_k} D_i. (the inner sum of
// PAPER.md:69 / :88), its row of the reduced Hessian of master mode 1, the maps between slot space and voxel space, and
// the dose-rate feasibility test.
//
// Layout: the columns are DENSE over the support of D, fp32, cut into chunks of 128 slots
// (one warp of float4) and stored CHUNK-MAJOR, Dd[chunk][k][128]: the segments of all columns for one chunk are
// neighbours in memory, so a block that walks a chunk's beams streams one contiguous region.
#include "vmat_master_common.cuh"

namespace vmat {

namespace {

// ------------------------------------------------------------------------------------------------
// aperture-dose column of one beam: fixed-point scatter (order free, hence reproducible) + convert
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_column_scatter(const uint32_t *__restrict__ rowq, const float4 *__restrict__ val4, const int4 *__restrict__ col4,
                 const Sel *__restrict__ sel, int beam, const int32_t *__restrict__ left,
                 const int32_t *__restrict__ right, int R, int C, double fx_scale, unsigned long long *__restrict__ acc,
                 ColStat *__restrict__ colstat, uint32_t *__restrict__ touch, int touch_words) {
    pdl_wait();      // the leaf search's choice
    pdl_trigger();   // k_column_finish may be scheduled; it waits for the accumulator itself
    const int k = sel ? sel->beam : beam;
    if (k < 0) return;
    if (blockIdx.x == 0) {   // statistics and touched-chunk bitmap of the column, filled by k_column_finish
        if (threadIdx.x == 0) {
            ColStat cs;
            cs.l1 = 0ull;
            cs.linf = 0ull;
            cs.clo = INT_MAX;
            cs.chi = -1;
            colstat[k] = cs;
        }
        for (int w = threadIdx.x; w < touch_words; w += blockDim.x) touch[(size_t)k * touch_words + w] = 0u;
    }
    const int lane = threadIdx.x & 31;
    const int idx = blockIdx.x * 8 + (threadIdx.x >> 5);
    if (idx >= R * C) return;
    const int r = idx / C, c = idx - r * C;
    if (c < left[k * R + r] || c >= right[k * R + r]) return;   // beamlet not exposed (A_k)
    const long long row = ((long long)k * R + r) * C + c;
    const uint32_t a = rowq[row], b = rowq[row + 1];
    // four quads per lane in flight before the first atomic (a row is ~100 quads: one round trip, not four)
    for (uint32_t q = a + lane; q < b; q += 32 * 4) {
        float4 v[4];
        int4 s[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            if (q + 32 * u < b) {
                v[u] = __ldg(val4 + q + 32 * u);
                s[u] = __ldg(col4 + q + 32 * u);
            } else {
                v[u] = make_float4(0.f, 0.f, 0.f, 0.f);
                s[u] = make_int4(0, 0, 0, 0);
            }
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            if (v[u].x != 0.f) atomicAdd(acc + s[u].x, (unsigned long long)__double2ll_rn((double)v[u].x * fx_scale));
            if (v[u].y != 0.f) atomicAdd(acc + s[u].y, (unsigned long long)__double2ll_rn((double)v[u].y * fx_scale));
            if (v[u].z != 0.f) atomicAdd(acc + s[u].z, (unsigned long long)__double2ll_rn((double)v[u].z * fx_scale));
            if (v[u].w != 0.f) atomicAdd(acc + s[u].w, (unsigned long long)__double2ll_rn((double)v[u].w * fx_scale));
        }
    }
}

// What k_column_finish needs to enter the new column into the Hessian of mode 1 (k_newton); hess == nullptr otherwise.
struct HessRowArgs {
    long long *hess;          // N x N fixed point, upper triangle
    const float *omref;       // Sp: the omega the matrix was built with
    const uint8_t *occ;       // N
    uint8_t *hvalid;          // N: column i is in the matrix
    const int *hlive;         // the matrix is built (a master solve has run since it was last reset)
    double hscale;
};

// Dd[k][.] = fixed-point accumulator as fp32; clears the accumulator; gathers the column's
// statistics (exact integer sums / extrema, hence order free): sum and max of |d_k|, first and
// last chunk with a non-zero entry.  One block = 256 slots = 2 chunks.
// Mode 1 of the master: the block also adds its two chunks' share of the new column's row of the Hessian,
// H_F[k][i] = sum_s omega_s d_k[s] d_i[s] over the columns i already in the matrix, so that the next master solve needs
// no pass of its own for it (and none at all before its first Newton step).
__global__ void __launch_bounds__(256)
k_column_finish(unsigned long long *__restrict__ acc, long long Sp, const Sel *__restrict__ sel, int beam,
                double fx_inv, float *__restrict__ Dd, int N, ColStat *__restrict__ colstat,
                uint32_t *__restrict__ touch, int touch_words, const HessRowArgs hr) {
    pdl_wait();      // the scatter's adds
    const int k = sel ? sel->beam : beam;
    if (k < 0) return;
    __shared__ unsigned long long s_sum[8], s_max[8];
    __shared__ int s_lo[8], s_hi[8];
    const long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    unsigned long long mag = 0ull;
    float dk = 0.f;
    if (s < Sp) {
        const long long v = (long long)acc[s];
        dk = (float)((double)v * fx_inv);
        Dd[((size_t)(s / kChunk) * N + k) * kChunk + (s & (kChunk - 1))] = dk;   // chunk-major
        acc[s] = 0ull;
        mag = (unsigned long long)(v < 0 ? -v : v);
    }
    const int chunk = (int)(s / kChunk);   // the same for the whole warp
    if (__any_sync(kFull, mag != 0ull) && (threadIdx.x & 31) == 0)
        atomicOr(touch + (size_t)k * touch_words + (chunk >> 5), 1u << (chunk & 31));
    unsigned long long sum = mag, mx = mag;
    int lo = mag ? chunk : INT_MAX, hi = mag ? chunk : -1;
#pragma unroll
    for (int o = 16; o; o >>= 1) {
        sum += __shfl_xor_sync(kFull, sum, o);
        const unsigned long long om = __shfl_xor_sync(kFull, mx, o);
        mx = om > mx ? om : mx;
        lo = min(lo, __shfl_xor_sync(kFull, lo, o));
        hi = max(hi, __shfl_xor_sync(kFull, hi, o));
    }
    const int warp = threadIdx.x >> 5;
    if ((threadIdx.x & 31) == 0) {
        s_sum[warp] = sum;
        s_max[warp] = mx;
        s_lo[warp] = lo;
        s_hi[warp] = hi;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int i = 1; i < 8; ++i) {
            sum += s_sum[i];
            mx = s_max[i] > mx ? s_max[i] : mx;
            lo = min(lo, s_lo[i]);
            hi = max(hi, s_hi[i]);
        }
        if (mx) {
            atomicAdd(&colstat[k].l1, sum);
            atomicMax(&colstat[k].linf, mx);
            atomicMin(&colstat[k].clo, lo);
            atomicMax(&colstat[k].chi, hi);
        }
    }
    // ---- the new column's row of the Hessian (mode 1) ------------------------------------------------
    if (hr.hess == nullptr || !*hr.hlive || N > kMasterThreads) return;   // the same for the whole grid
    if (blockIdx.x == 0 && threadIdx.x == 0) hr.hvalid[k] = 1;   // (no block reads the flag of k itself)
    __shared__ int s_live[2], s_cnt[2], s_list[2][kMasterThreads];
    __shared__ float4 s_u[2][kChunk / 4], s_d[2][kChunk / 4];
    const int lane = threadIdx.x & 31, half = threadIdx.x >> 7;   // warps 0-3: the block's first chunk, 4-7: its second
    const int sl = threadIdx.x & (kChunk - 1);
    const float u = s < Sp ? hr.omref[s] * dk : 0.f;
    reinterpret_cast<float *>(s_u[half])[sl] = u;
    reinterpret_cast<float *>(s_d[half])[sl] = dk;
    if (threadIdx.x < 2) s_live[threadIdx.x] = s_cnt[threadIdx.x] = 0;
    __syncthreads();
    if (__any_sync(kFull, u != 0.f) && lane == 0) s_live[half] = 1;
    __syncthreads();
    // the columns in the matrix that touch the chunk (any order: what each adds is an integer)
    for (int i = threadIdx.x; i < N; i += 256) {
        if (i == k || !hr.occ[i] || !hr.hvalid[i]) continue;
        const uint32_t *tw = touch + (size_t)i * touch_words;
        for (int h = 0; h < 2; ++h) {
            const int c = 2 * (int)blockIdx.x + h;
            if (s_live[h] && (long long)c * kChunk < Sp && ((tw[c >> 5] >> (c & 31)) & 1u)) s_list[h][atomicAdd(&s_cnt[h], 1)] = i;
        }
    }
    __syncthreads();
    if (!s_live[half]) return;
    // every warp of the chunk takes every fourth column of the list, eight at a time: one float4 of the column's
    // 512-byte segment per lane (all eight loads in flight), the eight sums over the warp by one butterfly
    const int c = 2 * (int)blockIdx.x + half, wq = (threadIdx.x >> 5) & 3, n1 = s_cnt[half];
    const float4 u4 = s_u[half][lane];
    const float4 *seg = reinterpret_cast<const float4 *>(Dd + (size_t)c * N * kChunk) + lane;
    const int slot8 = ((lane >> 4) & 1) * 4 + ((lane >> 3) & 1) * 2 + ((lane >> 2) & 1);   // warp_sum8's layout
    for (int n = wq; n < n1; n += 32) {
        double v[8];
        int id[8];
#pragma unroll
        for (int x = 0; x < 8; ++x) {
            id[x] = n + 4 * x < n1 ? s_list[half][n + 4 * x] : -1;
            float4 d4 = make_float4(0.f, 0.f, 0.f, 0.f);
            if (id[x] >= 0) d4 = __ldg(seg + (size_t)id[x] * (kChunk / 4));
            v[x] = (double)((u4.x * d4.x + u4.y * d4.y) + (u4.z * d4.z + u4.w * d4.w));
        }
        const double r = warp_sum8(v, lane);
        int mine = -1;
#pragma unroll
        for (int x = 0; x < 8; ++x)
            if (x == slot8) mine = id[x];
        if ((lane & 3) == 0 && mine >= 0 && r != 0.0)
            atomicAdd(reinterpret_cast<unsigned long long *>(hr.hess) + (size_t)min(mine, k) * N + max(mine, k),
                      (unsigned long long)__double2ll_rn(r * hr.hscale));
    }
    if (wq == 0) {   // the diagonal entry
        const float4 d4 = s_d[half][lane];
        double dg = (double)((u4.x * d4.x + u4.y * d4.y) + (u4.z * d4.z + u4.w * d4.w));
#pragma unroll
        for (int o = 16; o; o >>= 1) dg += __shfl_xor_sync(kFull, dg, o);
        if (lane == 0 && dg != 0.0)
            atomicAdd(reinterpret_cast<unsigned long long *>(hr.hess) + (size_t)k * N + k, (unsigned long long)__double2ll_rn(dg * hr.hscale));
    }
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

// dose-rate feasibility test: ratio = max_k |y_{k+1} - y_k| / (rho (theta_{k+1} - theta_k)),
// y = 0 at un-occupied beams (S2); one block, maximum taken in a fixed order
__global__ void __launch_bounds__(256)
k_rate_ratio(const uint8_t *__restrict__ occ, const double *__restrict__ y, const double *__restrict__ theta, int N,
             double rho, double *__restrict__ out) {
    __shared__ double s_max[8];
    double r = 0.0;
    for (int k = threadIdx.x; k + 1 < N; k += 256) {
        const double y0 = occ[k] ? y[k] : 0.0, y1 = occ[k + 1] ? y[k + 1] : 0.0;
        r = fmax(r, fabs(y1 - y0) / (rho * (theta[k + 1] - theta[k])));
    }
#pragma unroll
    for (int o = 16; o; o >>= 1) r = fmax(r, __shfl_xor_sync(kFull, r, o));
    if ((threadIdx.x & 31) == 0) s_max[threadIdx.x >> 5] = r;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int i = 1; i < 8; ++i) r = fmax(r, s_max[i]);
        *out = r;
    }
}


}  // namespace

int launch_column_build(vmat_plan *p, int beam) {
    const Sel *sel = beam < 0 ? p->sel : nullptr;
    const unsigned blocks = (unsigned)((p->RC + 7) / 8);
    VMAT_CUDA(p, launch_pdl(k_column_scatter, dim3(blocks), dim3(256), p->stream, p->rowq, p->val4, p->col4, sel, beam, p->left,
                            p->right, (int)p->R, (int)p->C, p->fx_scale, p->acc, p->colstat, p->col_touch, p->touch_words));
    HessRowArgs hr;
    hr.hess = p->master_newton ? p->hess : nullptr;
    hr.omref = p->omref;
    hr.occ = p->occ;
    hr.hvalid = p->hvalid;
    hr.hlive = p->hlive;
    hr.hscale = p->hscale;
    VMAT_CUDA(p, launch_pdl(k_column_finish, dim3((unsigned)((p->Sp + 255) / 256)), dim3(256), p->stream, p->acc,
                            (long long)p->Sp, sel, beam, p->fx_inv, p->Dd, (int)p->N, p->colstat, p->col_touch,
                            p->touch_words, hr));
    p->launches += 2;
    VMAT_CUDA(p, cudaGetLastError());
    return VMAT_OK;
}

int launch_rate_ratio(vmat_plan *p, double rho, double *ratio_dev) {
    k_rate_ratio<<<1, 256, 0, p->stream>>>(p->occ, p->y, p->theta, (int)p->N, rho, ratio_dev);
    ++p->launches;
    VMAT_CUDA(p, cudaGetLastError());
    return VMAT_OK;
}

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

}  // namespace vmat
