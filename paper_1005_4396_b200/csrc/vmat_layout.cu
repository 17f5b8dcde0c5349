// vmat_layout.cu — vmat_create's device work: validate the problem, find the support of D,
// re-lay-out D as a padded beamlet-major CSR in slot space.
// Set-up code (runs once per plan).
#include <cmath>
#include <cstring>

#include "vmat_internal.cuh"

namespace vmat {

namespace {

enum : unsigned {
    kBadRowPtr = 1u,
    kBadCol = 2u,
    kBadOrder = 4u,
    kBadVal = 8u,
    kBadVoxel = 16u,
};

__global__ void k_check_row_ptr(const int64_t *__restrict__ row_ptr, int64_t B, int64_t nnz, unsigned *flags) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i > B) return;
    const int64_t a = row_ptr[i];
    bool bad = a < 0 || a > nnz;
    if (i == 0 && a != 0) bad = true;
    if (i == B && a != nnz) bad = true;
    if (i < B && row_ptr[i + 1] < a) bad = true;
    if (bad) atomicOr(flags, kBadRowPtr);
}

// one warp per row: column range, strict order, finite values; marks the support
__global__ void k_check_rows(const int64_t *__restrict__ row_ptr, const int32_t *__restrict__ col,
                             const float *__restrict__ val, int64_t B, int64_t V, int validate,
                             int32_t *__restrict__ reach, unsigned *flags, unsigned *maxabs_bits) {
    const int lane = threadIdx.x & 31;
    const int64_t row = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (row >= B) return;
    const int64_t a = row_ptr[row], b = row_ptr[row + 1];
    unsigned bad = 0, mx = 0;
    for (int64_t e = a + lane; e < b; e += 32) {
        const int32_t c = col[e];
        const float v = val[e];
        if (c < 0 || c >= V) {
            bad |= kBadCol;
            continue;
        }
        if (validate) {
            if (e > a && col[e - 1] >= c) bad |= kBadOrder;
            if (!isfinite(v)) bad |= kBadVal;
        }
        reach[c] = 1;
        const unsigned bits = __float_as_uint(fabsf(v));
        mx = bits > mx ? bits : mx;
    }
    if (bad) atomicOr(flags, bad);
    for (int o = 16; o; o >>= 1) {
        const unsigned other = __shfl_xor_sync(0xffffffffu, mx, o);
        mx = other > mx ? other : mx;
    }
    if (lane == 0 && mx) atomicMax(maxabs_bits, mx);
}

__global__ void k_check_voxels(const float *__restrict__ T, const float *__restrict__ alpha,
                               const float *__restrict__ beta, int64_t V, unsigned *flags) {
    const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= V) return;
    const float t = T[j], a = alpha[j], b = beta[j];
    if (!isfinite(t) || !isfinite(a) || !isfinite(b) || a < 0.f || b < 0.f) atomicOr(flags, kBadVoxel);
}

__global__ void k_row_quads(const int64_t *__restrict__ row_ptr, int64_t B, uint32_t *__restrict__ cnt) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i > B) return;
    cnt[i] = i < B ? (uint32_t)((row_ptr[i + 1] - row_ptr[i] + 3) >> 2) : 0u;
}

// slot_of[j] = exclusive count if reachable else -1; voxel_of[slot] = j; slot-space T/alpha/beta;
// per-block partial of the constant cost of the voxels outside the support (z_j = 0 there)
__global__ void k_slots(const int32_t *__restrict__ reach, const int32_t *__restrict__ excl, int64_t V,
                        const float *__restrict__ T, const float *__restrict__ alpha, const float *__restrict__ beta,
                        int32_t *__restrict__ slot_of, int32_t *__restrict__ voxel_of, float *__restrict__ T_s,
                        float *__restrict__ alpha_s, float *__restrict__ beta_s, double *__restrict__ part) {
    __shared__ double red[256];
    const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    double f = 0.0;
    if (j < V) {
        if (reach[j]) {
            const int32_t s = excl[j];
            slot_of[j] = s;
            voxel_of[s] = (int32_t)j;
            T_s[s] = T[j];
            alpha_s[s] = alpha[j];
            beta_s[s] = beta[j];
        } else {
            slot_of[j] = -1;
            const double t = (double)T[j];
            const double under = fmax(0.0, t), over = fmax(0.0, -t);   // Eq. 1 at z_j = 0
            f = (double)alpha[j] * under * under + (double)beta[j] * over * over;
        }
    }
    red[threadIdx.x] = f;
    __syncthreads();
    for (int o = 128; o; o >>= 1) {
        if (threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) part[blockIdx.x] = red[0];
}

// one warp per row: copy into the padded layout, voxel ids -> slots.  Padding entries repeat the
// row's last slot with value 0 so that every quad is a valid 16-byte load + 4 valid gathers.
__global__ void k_fill_padded(const int64_t *__restrict__ row_ptr, const int32_t *__restrict__ col,
                              const float *__restrict__ val, const int32_t *__restrict__ slot_of,
                              const uint32_t *__restrict__ rowq, int64_t B, float *__restrict__ val_out,
                              int32_t *__restrict__ col_out) {
    const int lane = threadIdx.x & 31;
    const int64_t row = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (row >= B) return;
    const int64_t a = row_ptr[row], len = row_ptr[row + 1] - a;
    const int64_t o = (int64_t)rowq[row] * 4, plen = (int64_t)(rowq[row + 1] - rowq[row]) * 4;
    for (int64_t e = lane; e < plen; e += 32) {
        const int64_t src = e < len ? e : len - 1;
        col_out[o + e] = slot_of[col[a + src]];
        val_out[o + e] = e < len ? val[a + src] : 0.f;
    }
}

// ---- exclusive prefix sum (the two scans of the set-up: support flags -> slots, row quads -> row starts) --------
// Three short kernels: every block scans kScanTile elements and records its total, one block scans the totals,
// every block adds the sum of the blocks before it.  In place is allowed (in == out).
constexpr int kScanThreads = 256, kScanPer = 4, kScanTile = kScanThreads * kScanPer;

template <typename T>
__device__ __forceinline__ T block_exclusive_scan(T v, T *warp_tot, T &total) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    T incl = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const T n = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += n;
    }
    if (lane == 31) warp_tot[warp] = incl;
    __syncthreads();
    T base = 0, tot = 0;
    for (int w = 0; w < (int)(blockDim.x >> 5); ++w) {
        const T t = warp_tot[w];
        if (w < warp) base += t;
        tot += t;
    }
    __syncthreads();
    total = tot;
    return base + incl - v;
}

template <typename T>
__global__ void __launch_bounds__(kScanThreads) k_scan_tiles(const T *__restrict__ in, T *__restrict__ out, int64_t n,
                                                             T *__restrict__ tile_sums) {
    __shared__ T warp_tot[kScanThreads / 32];
    const int64_t i0 = ((int64_t)blockIdx.x * kScanThreads + threadIdx.x) * kScanPer;
    T v[kScanPer], sum = 0;
#pragma unroll
    for (int u = 0; u < kScanPer; ++u) {
        v[u] = i0 + u < n ? in[i0 + u] : (T)0;
        sum += v[u];
    }
    T total;
    T run = block_exclusive_scan(sum, warp_tot, total);
#pragma unroll
    for (int u = 0; u < kScanPer; ++u) {
        if (i0 + u < n) out[i0 + u] = run;
        run += v[u];
    }
    if (threadIdx.x == 0) tile_sums[blockIdx.x] = total;
}

template <typename T>
__global__ void __launch_bounds__(kScanThreads) k_scan_sums(T *__restrict__ tile_sums, int64_t ntiles) {
    __shared__ T warp_tot[kScanThreads / 32];
    T carry = 0;
    for (int64_t b0 = 0; b0 < ntiles; b0 += kScanThreads) {
        const int64_t b = b0 + threadIdx.x;
        const T v = b < ntiles ? tile_sums[b] : (T)0;
        T total;
        const T ex = block_exclusive_scan(v, warp_tot, total);
        if (b < ntiles) tile_sums[b] = carry + ex;
        carry += total;
    }
}

template <typename T>
__global__ void __launch_bounds__(kScanThreads) k_scan_add(T *__restrict__ out, int64_t n, const T *__restrict__ tile_sums) {
    const int64_t i0 = ((int64_t)blockIdx.x * kScanThreads + threadIdx.x) * kScanPer;
    const T base = tile_sums[blockIdx.x];
#pragma unroll
    for (int u = 0; u < kScanPer; ++u)
        if (i0 + u < n) out[i0 + u] += base;
}

template <typename T>
cudaError_t exclusive_scan(const T *in, T *out, int64_t n, T *tile_sums, cudaStream_t st) {
    if (n <= 0) return cudaSuccess;
    const int64_t ntiles = (n + kScanTile - 1) / kScanTile;
    k_scan_tiles<T><<<(unsigned)ntiles, kScanThreads, 0, st>>>(in, out, n, tile_sums);
    k_scan_sums<T><<<1, kScanThreads, 0, st>>>(tile_sums, ntiles);
    k_scan_add<T><<<(unsigned)ntiles, kScanThreads, 0, st>>>(out, n, tile_sums);
    return cudaGetLastError();
}


// ---- d_format 1: a second copy of D for the pricing product in aligned slot PAIRS with 16-bit ids ---------------
// The slot ids of a row of D come in runs of consecutive slots (a beamlet's lateral support along a voxel row): a
// UNIT is the aligned pair of slots (2m, 2m+1) with the row's two values there (0 where the row has no entry), so one
// 8-byte gather of w serves up to two entries (0.62 / 0.57 units per entry on configs[1] / [2]).  The pair ids are
// cut into panels of 65536 pairs; a row's units fall into one run per panel, padded to whole GROUPS of four units
// (values 0, the run's last id repeated).  A group carries two float4 of values (arrays va, vb: units 0-1 and 2-3),
// four 16-bit pair ids relative to its panel (array ix) and one byte with the panel (array pan): 41 bytes per group,
// 6.35 / 5.86 bytes per entry of D against 8.  rowo[i] = first group of row i.
constexpr int kPanelBits = 16;

// Within a run the units are dealt to the groups in blocks of 16 groups (one per lane of the pricing kernel): unit t
// of a block of n <= 16 groups sits in group t mod n at position t div n, so that the gather of position u reads n
// CONSECUTIVE units across the lanes (consecutive pairs of w: a few cache lines instead of one per lane).
__device__ __forceinline__ void unit_place(int u, int Gp, int &group, int &pos) {
    const int k = u >> 6, n = min(16, Gp - 16 * k), t = u - 64 * k;
    group = 16 * k + t % n;
    pos = t / n;
}

// one warp per row.  FILL = false: cnt[row] = groups the row needs; FILL = true: write the row's groups.
template <bool FILL>
__global__ void k_pairs_build(const uint32_t *__restrict__ rowq, const float4 *__restrict__ val4,
                              const int4 *__restrict__ col4, int64_t B, uint32_t *__restrict__ cnt,
                              const uint32_t *__restrict__ rowo, float *__restrict__ va, float *__restrict__ vb,
                              uint16_t *__restrict__ ix, uint8_t *__restrict__ pan) {
    const int lane = threadIdx.x & 31;
    const int64_t row = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (row > B) return;
    if (row == B) {
        if (!FILL && lane == 0) cnt[B] = 0u;
        return;
    }
    const int32_t *col = reinterpret_cast<const int32_t *>(col4);
    const float *val = reinterpret_cast<const float *>(val4);
    const int64_t a = (int64_t)rowq[row] * 4, b = (int64_t)rowq[row + 1] * 4;
    uint32_t groups = 0;
    if (b > a) {
        int64_t grp = FILL ? (int64_t)rowo[row] : 0;   // first group of the current run
        const int p1 = (col[b - 1] >> 1) >> kPanelBits;
        for (int pn = (col[a] >> 1) >> kPanelBits; pn <= p1; ++pn) {
            // units of the row in this panel: entries ascend, a pair id different from the entry before opens a unit
            int U = 0, lastp = -1;
            for (int64_t e0 = a; e0 < b; e0 += 32) {
                const int64_t e = e0 + lane;
                const bool in = e < b;
                const int pair = in ? col[e] >> 1 : -2;
                int before = __shfl_up_sync(0xffffffffu, pair, 1);
                if (lane == 0) before = e0 == a ? -1 : lastp;
                const bool mine = in && (pair >> kPanelBits) == pn;
                U += __popc(__ballot_sync(0xffffffffu, mine && pair != before));
                const unsigned inmask = __ballot_sync(0xffffffffu, in);
                lastp = __shfl_sync(0xffffffffu, pair, 31 - __clz(inmask));
            }
            if (U == 0) continue;
            const int Gp = (U + 3) >> 2;
            if (FILL) {
                int done = 0, endpair = 0;
                lastp = -1;
                for (int64_t e0 = a; e0 < b; e0 += 32) {
                    const int64_t e = e0 + lane;
                    const bool in = e < b;
                    const int sl = in ? col[e] : -4, pair = sl >> 1;
                    int before = __shfl_up_sync(0xffffffffu, pair, 1);
                    if (lane == 0) before = e0 == a ? -1 : lastp;
                    const bool mine = in && (pair >> kPanelBits) == pn, isnew = mine && pair != before;
                    const unsigned mnew = __ballot_sync(0xffffffffu, isnew), mm = __ballot_sync(0xffffffffu, mine);
                    if (mine) {
                        const int u = done + __popc(mnew & (0xffffffffu >> (31 - lane))) - 1;   // this entry's unit
                        int g, pos;
                        unit_place(u, Gp, g, pos);
                        const float v = val[e];   // one entry per slot: a plain store; the zero padding of the CSR rows
                        if (v != 0.f) ((pos & 2) ? vb : va)[(grp + g) * 4 + 2 * (pos & 1) + (sl & 1)] = v;   // must not write
                        if (isnew) ix[(grp + g) * 4 + pos] = (uint16_t)(pair & 0xffff);
                    }
                    done += __popc(mnew);
                    if (mm) endpair = __shfl_sync(0xffffffffu, pair, 31 - __clz(mm));
                    const unsigned inmask = __ballot_sync(0xffffffffu, in);
                    lastp = __shfl_sync(0xffffffffu, pair, 31 - __clz(inmask));
                }
                for (int u = U + lane; u < 4 * Gp; u += 32) {   // padding units: value 0 (the arrays start zeroed)
                    int g, pos;
                    unit_place(u, Gp, g, pos);
                    ix[(grp + g) * 4 + pos] = (uint16_t)(endpair & 0xffff);
                }
                for (int g = lane; g < Gp; g += 32) pan[grp + g] = (uint8_t)pn;
            }
            grp += Gp;
            groups += (uint32_t)Gp;
        }
    }
    if (!FILL && lane == 0) cnt[row] = groups;
}

}  // namespace

// d_format 1: build the pair copy of D from the padded layout (p->rowq, val4, col4 must be in place)
int build_pairs(vmat_plan *p) {
    const int64_t B = p->B;
    cudaStream_t st = p->stream;
    if (((p->Sp >> 1) >> kPanelBits) >= 256) return fail(p, VMAT_EINVAL, "d_format 1 needs a support below 2^25 voxels");
    int rc;
    uint32_t *cnt = nullptr;
    void *tiles = nullptr;
    const int64_t scan_tiles = (B + 1 + kScanTile - 1) / kScanTile;
    cudaError_t e;
    if ((e = pool_alloc((void **)&cnt, (size_t)(B + 1) * 4, p->device, st)) != cudaSuccess ||
        (e = pool_alloc(&tiles, (size_t)scan_tiles * 4, p->device, st)) != cudaSuccess) {
        cudaGetLastError();
        pool_free(cnt, p->device, st);
        return fail(p, VMAT_ENOMEM, std::string("device allocation (scratch) failed: ") + cudaGetErrorString(e));
    }
    auto done = [&](int code) {
        pool_free(cnt, p->device, st);
        pool_free(tiles, p->device, st);
        return code;
    };
    k_pairs_build<false><<<(unsigned)((B + 1 + 7) / 8), 256, 0, st>>>(p->rowq, p->val4, p->col4, B, cnt, nullptr, nullptr,
                                                                   nullptr, nullptr, nullptr);
    if ((rc = dev_alloc(p, &p->pr_rowo, B + 1))) return done(rc);
    if ((e = exclusive_scan<uint32_t>(cnt, p->pr_rowo, B + 1, (uint32_t *)tiles, st)) != cudaSuccess)
        return done(cuda_fail(p, e, "exclusive_scan"));
    uint32_t ng = 0;
    if ((e = cudaMemcpyAsync(&ng, p->pr_rowo + B, 4, cudaMemcpyDeviceToHost, st)) != cudaSuccess ||
        (e = cudaStreamSynchronize(st)) != cudaSuccess)
        return done(cuda_fail(p, e, "cudaMemcpyAsync"));
    p->pr_groups = ng;
    if ((rc = dev_alloc(p, &p->pr_va, (int64_t)ng))) return done(rc);
    if ((rc = dev_alloc(p, &p->pr_vb, (int64_t)ng))) return done(rc);
    if ((rc = dev_alloc(p, &p->pr_ix, (int64_t)ng))) return done(rc);
    if ((rc = dev_alloc(p, &p->pr_pan, (int64_t)ng))) return done(rc);
    if ((e = cudaMemsetAsync(p->pr_va, 0, (size_t)ng * 16, st)) != cudaSuccess ||
        (e = cudaMemsetAsync(p->pr_vb, 0, (size_t)ng * 16, st)) != cudaSuccess)
        return done(cuda_fail(p, e, "cudaMemsetAsync"));
    k_pairs_build<true><<<(unsigned)((B + 7) / 8), 256, 0, st>>>(p->rowq, p->val4, p->col4, B, nullptr, p->pr_rowo,
                                                              (float *)p->pr_va, (float *)p->pr_vb, (uint16_t *)p->pr_ix,
                                                              p->pr_pan);
    if ((e = cudaGetLastError()) != cudaSuccess) return done(cuda_fail(p, e, "k_pairs_build"));
    return done(VMAT_OK);
}

namespace {
}  // namespace

template <typename T>
static int stage_in(vmat_plan *p, const T *src, int64_t count, int mem_space, const T **dev, std::vector<void *> &tmp) {
    if (mem_space == VMAT_DEVICE) {
        *dev = src;
        return VMAT_OK;
    }
    void *d = nullptr;
    cudaError_t e = pool_alloc(&d, (size_t)(count > 0 ? count : 1) * sizeof(T), p->device, p->stream);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return fail(p, VMAT_ENOMEM, std::string("device allocation (staging) failed: ") + cudaGetErrorString(e));
    }
    tmp.push_back(d);
    VMAT_CUDA(p, cudaMemcpyAsync(d, src, (size_t)count * sizeof(T), cudaMemcpyHostToDevice, p->stream));
    *dev = (const T *)d;
    return VMAT_OK;
}

static int build_layout_impl(vmat_plan *p, const vmat_problem *pb, std::vector<void *> &tmp) {
    const int64_t B = p->B, V = p->V;
    cudaStream_t st = p->stream;
    int rc;

    // nnz = row_ptr[B]
    int64_t nnz = 0;
    if (pb->mem_space == VMAT_DEVICE) {
        VMAT_CUDA(p, cudaMemcpyAsync(&nnz, pb->row_ptr + B, sizeof(int64_t), cudaMemcpyDeviceToHost, st));
        VMAT_CUDA(p, cudaStreamSynchronize(st));
    } else {
        nnz = pb->row_ptr[B];
    }
    if (nnz < 0) return fail(p, VMAT_EINVAL, "row_ptr[B] is negative");
    if ((nnz + 3) / 4 + B >= (int64_t)0xffffffffll) return fail(p, VMAT_EINVAL, "D too large: padded quads exceed 2^32");
    p->nnz = nnz;

    const int64_t *d_row_ptr;
    const int32_t *d_col;
    const float *d_val, *d_T, *d_alpha, *d_beta;
    if ((rc = stage_in(p, pb->row_ptr, B + 1, pb->mem_space, &d_row_ptr, tmp))) return rc;
    if ((rc = stage_in(p, pb->col_idx, nnz, pb->mem_space, &d_col, tmp))) return rc;
    if ((rc = stage_in(p, pb->val, nnz, pb->mem_space, &d_val, tmp))) return rc;
    if ((rc = stage_in(p, pb->T, V, pb->mem_space, &d_T, tmp))) return rc;
    if ((rc = stage_in(p, pb->alpha, V, pb->mem_space, &d_alpha, tmp))) return rc;
    if ((rc = stage_in(p, pb->beta, V, pb->mem_space, &d_beta, tmp))) return rc;

    // scratch: flags (2 words), reach[V], excl[V], cnt[B+1]
    unsigned *d_flags;
    int32_t *d_reach, *d_excl;
    uint32_t *d_cnt;
    auto tmp_alloc = [&](void **ptr, size_t bytes) -> int {
        cudaError_t e = pool_alloc(ptr, bytes ? bytes : 1, p->device, p->stream);
        if (e != cudaSuccess) {
            cudaGetLastError();
            return fail(p, VMAT_ENOMEM, std::string("device allocation (scratch) failed: ") + cudaGetErrorString(e));
        }
        tmp.push_back(*ptr);
        return VMAT_OK;
    };
    if ((rc = tmp_alloc((void **)&d_flags, 2 * sizeof(unsigned)))) return rc;
    if ((rc = tmp_alloc((void **)&d_reach, (size_t)V * 4))) return rc;
    if ((rc = tmp_alloc((void **)&d_excl, (size_t)V * 4))) return rc;
    if ((rc = tmp_alloc((void **)&d_cnt, (size_t)(B + 1) * 4))) return rc;
    VMAT_CUDA(p, cudaMemsetAsync(d_flags, 0, 2 * sizeof(unsigned), st));
    VMAT_CUDA(p, cudaMemsetAsync(d_reach, 0, (size_t)V * 4, st));

    // row_ptr must be sane before any kernel walks the rows
    k_check_row_ptr<<<(unsigned)((B + 1 + 255) / 256), 256, 0, st>>>(d_row_ptr, B, nnz, d_flags);
    unsigned h_flags[2] = {0, 0};
    VMAT_CUDA(p, cudaMemcpyAsync(h_flags, d_flags, sizeof(h_flags), cudaMemcpyDeviceToHost, st));
    VMAT_CUDA(p, cudaStreamSynchronize(st));
    if (h_flags[0] & kBadRowPtr) return fail(p, VMAT_EINVAL, "row_ptr must start at 0, be non-decreasing and end at nnz");

    k_check_rows<<<(unsigned)((B + 7) / 8), 256, 0, st>>>(d_row_ptr, d_col, d_val, B, V, p->opt.validate, d_reach,
                                                         d_flags, d_flags + 1);
    if (p->opt.validate) k_check_voxels<<<(unsigned)((V + 255) / 256), 256, 0, st>>>(d_T, d_alpha, d_beta, V, d_flags);
    VMAT_CUDA(p, cudaMemcpyAsync(h_flags, d_flags, sizeof(h_flags), cudaMemcpyDeviceToHost, st));
    VMAT_CUDA(p, cudaStreamSynchronize(st));
    VMAT_CUDA(p, cudaGetLastError());
    if (h_flags[0] & kBadCol) return fail(p, VMAT_EINVAL, "col_idx has a voxel id outside [0, n_voxels)");
    if (h_flags[0] & kBadOrder) return fail(p, VMAT_EINVAL, "col_idx must be strictly ascending within a row");
    if (h_flags[0] & kBadVal) return fail(p, VMAT_EINVAL, "val has a NaN or Inf");
    if (h_flags[0] & kBadVoxel) return fail(p, VMAT_EINVAL, "T/alpha/beta must be finite with alpha, beta >= 0");

    // fixed-point scale of the aperture-column accumulator: |val| * fx_scale <= 2^40
    float maxabs;
    std::memcpy(&maxabs, &h_flags[1], 4);
    int e2 = 0;
    if (maxabs > 0.f) std::frexp((double)maxabs, &e2);   // maxabs < 2^e2
    p->fx_scale = std::ldexp(1.0, 40 - e2);
    p->fx_inv = std::ldexp(1.0, e2 - 40);

    // support: exclusive scan of the reach flags
    const int64_t scan_tiles = ((V > B + 1 ? V : B + 1) + kScanTile - 1) / kScanTile;
    void *d_tiles;
    if ((rc = tmp_alloc(&d_tiles, (size_t)scan_tiles * 4))) return rc;
    VMAT_CUDA(p, exclusive_scan<int32_t>(d_reach, d_excl, V, (int32_t *)d_tiles, st));
    int32_t last_excl = 0, last_flag = 0;
    if (V > 0) {
        VMAT_CUDA(p, cudaMemcpyAsync(&last_excl, d_excl + V - 1, 4, cudaMemcpyDeviceToHost, st));
        VMAT_CUDA(p, cudaMemcpyAsync(&last_flag, d_reach + V - 1, 4, cudaMemcpyDeviceToHost, st));
    }
    // row starts in quads
    k_row_quads<<<(unsigned)((B + 1 + 255) / 256), 256, 0, st>>>(d_row_ptr, B, d_cnt);
    if ((rc = dev_alloc(p, &p->rowq, B + 1))) return rc;
    VMAT_CUDA(p, exclusive_scan<uint32_t>(d_cnt, p->rowq, B + 1, (uint32_t *)d_tiles, st));
    uint32_t nq = 0;
    VMAT_CUDA(p, cudaMemcpyAsync(&nq, p->rowq + B, 4, cudaMemcpyDeviceToHost, st));
    VMAT_CUDA(p, cudaStreamSynchronize(st));
    p->S = (int64_t)last_excl + last_flag;
    p->Sp = ((p->S + kChunk - 1) / kChunk) * kChunk;
    if (p->Sp < kChunk) p->Sp = kChunk;
    p->nq = nq;

    // slot maps and slot-space voxel parameters
    if ((rc = dev_alloc(p, &p->T_V, V))) return rc;
    if ((rc = dev_alloc(p, &p->alpha_V, V))) return rc;
    if ((rc = dev_alloc(p, &p->beta_V, V))) return rc;
    VMAT_CUDA(p, cudaMemcpyAsync(p->T_V, d_T, (size_t)V * 4, cudaMemcpyDeviceToDevice, st));
    VMAT_CUDA(p, cudaMemcpyAsync(p->alpha_V, d_alpha, (size_t)V * 4, cudaMemcpyDeviceToDevice, st));
    VMAT_CUDA(p, cudaMemcpyAsync(p->beta_V, d_beta, (size_t)V * 4, cudaMemcpyDeviceToDevice, st));
    if ((rc = dev_alloc(p, &p->slot_of, V))) return rc;
    if ((rc = dev_alloc(p, &p->voxel_of, p->Sp))) return rc;
    if ((rc = dev_alloc(p, &p->T_s, p->Sp))) return rc;
    if ((rc = dev_alloc(p, &p->alpha_s, p->Sp))) return rc;
    if ((rc = dev_alloc(p, &p->beta_s, p->Sp))) return rc;
    VMAT_CUDA(p, cudaMemsetAsync(p->voxel_of, 0, (size_t)p->Sp * 4, st));
    VMAT_CUDA(p, cudaMemsetAsync(p->T_s, 0, (size_t)p->Sp * 4, st));
    VMAT_CUDA(p, cudaMemsetAsync(p->alpha_s, 0, (size_t)p->Sp * 4, st));
    VMAT_CUDA(p, cudaMemsetAsync(p->beta_s, 0, (size_t)p->Sp * 4, st));
    const unsigned vblocks = (unsigned)((V + 255) / 256);
    double *d_part;
    if ((rc = tmp_alloc((void **)&d_part, (size_t)vblocks * 8))) return rc;
    k_slots<<<vblocks, 256, 0, st>>>(d_reach, d_excl, V, d_T, d_alpha, d_beta, p->slot_of, p->voxel_of, p->T_s,
                                     p->alpha_s, p->beta_s, d_part);
    std::vector<double> h_part(vblocks);
    VMAT_CUDA(p, cudaMemcpyAsync(h_part.data(), d_part, (size_t)vblocks * 8, cudaMemcpyDeviceToHost, st));

    // padded CSR in slot space
    if ((rc = dev_alloc(p, &p->val4, p->nq))) return rc;
    if ((rc = dev_alloc(p, &p->col4, p->nq))) return rc;
    k_fill_padded<<<(unsigned)((B + 7) / 8), 256, 0, st>>>(d_row_ptr, d_col, d_val, p->slot_of, p->rowq, B,
                                                          (float *)p->val4, (int32_t *)p->col4);
    VMAT_CUDA(p, cudaStreamSynchronize(st));
    VMAT_CUDA(p, cudaGetLastError());
    double f_out = 0.0;
    for (unsigned b = 0; b < vblocks; ++b) f_out += h_part[b];
    p->F_out = f_out;

    return VMAT_OK;
}

int build_layout(vmat_plan *p, const vmat_problem *pb) {
    std::vector<void *> tmp;
    const int rc = build_layout_impl(p, pb, tmp);
    for (void *t : tmp) pool_free(t, p->device, p->stream);   // stream ordered: after the kernels that read them
    cudaStreamSynchronize(p->stream);
    return rc;
}

}  // namespace vmat
