// vmat_master.cu — steps (a), (b) and (e).
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
#include <math_constants.h>

#include <climits>
#include <cmath>

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

__device__ __forceinline__ double warp_sum8(double (&v)[8], int lane);

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

// ------------------------------------------------------------------------------------------------
// the master kernel
// ------------------------------------------------------------------------------------------------
struct Mail;
struct MasterArgs {
    const float *Dd;
    long long Sp;
    int nchunks;
    const float *T, *alpha, *beta;
    float *z, *zn, *q, *q2, *w;
    const uint8_t *occ;
    double *y;
    const double *theta;
    const ColStat *colstat;
    const uint32_t *touch;      // per column: bit c set iff chunk c holds a non-zero entry (touch_words words each)
    int touch_words;
    int N;
    double gamma, F_out, eps, fx_inv, stall_rel;
    double lb, ub;              // bounds on the dose rates of occupied beams (default 0, +inf)
    int occ_only;               // reading of Eq. 2: smoothing over successive occupied beams only (vmat_options.occupied_only_G)
    int stall_count;
    float Tmax, abmax;
    int max_inner;
    int rslots;                 // > 0: every block keeps z, q, T, alpha, beta of its own slots in shared memory
    int cache_segs;             // capacity of the shared-memory tile of Dd in 512-byte segments
    int ul_cap;                 // capacity of the per-chunk lists of unstaged beams (0: they do not fit, masked loops)
    int nblk;                   // blocks that own chunks: the whole grid (mode 0) or all but the last block (mode 1,
                                // whose last block solves the reduced problems)
    long long *accbuf;          // 3 rotating sets of kSumGroups records of (2N + 2) fixed-point sums: F, curvature,
                                // grad[0..K), and (fused mode) the Hessian-vector product [K..2K); a block adds
                                // to the record of its group (blockIdx mod kSumGroups)
    unsigned int *phase;        // rotation counter, persists from launch to launch
    unsigned long long *mcount; // bookkeeping: [0] += touched segments x passes (all blocks), [1] += passes
    // warm entry (inside vmat_solve): z, w and cost3 are current for the plan as it was before the leaf search
    // committed beam sel->beam at y = 0, and gsave holds the F-part of the gradient of the beams occupied then
    int warm;
    const Sel *sel;
    double *gsave;              // N: d_k . w at the y this kernel leaves (valid iff gflag[0] == 1)
    int *gflag;
    MasterOut *out;
    double *cost3;
    double *trF, *trG, *trC;
    int32_t *trInner;
    int trace_it;
    // mode 1 (k_newton)
    long long *hess;            // N x N (upper triangle used): H_F in fixed point, scale hscale
    float *omref;               // Sp: the omega H_F was built with
    uint8_t *hvalid;            // N: the column of beam k is in H_F
    int *hlive;                 // H_F is built: set by every k_newton launch, cleared when the matrix is reset
    double hscale, hinv;
    float *wn;                  // second buffer of w (the trial points write z, w to a.zn, a.wn)
    Mail *mail;                 // message of the solving block, followed by N floats
    unsigned long long *sync;   // [0] arrivals, [1] epoch published, [2], [3]: where both stand when a launch begins
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

// scale 2^(60-e) (and its inverse) for sums whose magnitude is bounded by `bound` < 2^e; flags a
// non-finite bound.  Powers of two built from the exponent field: conversions are exact.
struct FxScale {
    double scale, inv;
};
__device__ __forceinline__ FxScale fx_scale_for(double bound, int &bad) {
    if (!(bound < 1e300)) bad = 1;
    const double b = fmin(fmax(bound, 1e-18), 1e300);
    const int e = ((__double2hiint(b) >> 20) & 0x7ff) - 1022;   // b < 2^e
    FxScale r;
    r.scale = __hiloint2double((1023 + 60 - e) << 20, 0);
    r.inv = __hiloint2double((1023 - 60 + e) << 20, 0);
    return r;
}
__device__ __forceinline__ void fx_add(long long *dst, double v, double scale) {
    atomicAdd(reinterpret_cast<unsigned long long *>(dst), (unsigned long long)__double2ll_rn(v * scale));
}

// scalars every thread of the block needs, written by warp 0 (the block's control warp)
struct Ctl {
    double scF, scG, scC;   // fixed-point scales of the pass about to run
    double iF, iG, iC;      // and their inverses
    float tf;               // trial step of the line search
    int state;              // what the block does next (kRunDirection, ...)
    int accepted;           // the last trial was accepted: the z buffers swap roles
};
enum { kRunDirection = 0, kRunTrial = 1, kFinish = 2 };

constexpr int kRedSlots = 8;   // values per warp row of the control group's reduction scratch
// Records of grid-wide sums per rotation slot.  Measured: splitting the blocks into 16 groups with one record each
// (to spread same-address atomics) and a hand-rolled two-level barrier were both slower than one record and the
// cooperative-groups barrier (12.4 / 14.5 vs 11.7 us per inner iteration at K = 30), so there is one group.
constexpr int kSumGroups = 1;
constexpr int kKSplit = 8;     // beam-loop split of the passes; the two halves of the warps take alternate chunks
constexpr int kNoCache = INT_MIN;
constexpr double kReleaseEta2 = 0.0625;   // release the held beams when |g on the face|^2 <= this x |held inward g|^2
static_assert(kMasterWarps == 2 * kKSplit, "the passes split the warps in two chunk halves");

// 1-D bulk copies (TMA) global -> shared, completion counted in bytes on an mbarrier
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, unsigned bytes, uint64_t *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, unsigned parity) {
    asm volatile(
        "{\n.reg .pred p;\nWAIT_%=:\nmbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n@p bra DONE_%=;\nbra "
        "WAIT_%=;\nDONE_%=:\n}" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}


// Staged segments sit kSeg floats apart (128 used): with 544-byte strides two threads per segment, reading
// alternate float4s, touch eight distinct 16-byte bank groups per quarter warp, so the thread-per-segment
// gradient products below run free of bank conflicts.  The w / u buffers of a group use the same stride.
constexpr int kSeg = 136;
constexpr int kSeg4 = kSeg / 4;
static_assert(kMasterWarps == 2 * kGroup, "the staged products give every chunk of a group two warps");

struct Smem {
    double *y, *d, *grad, *pg, *yn, *gn, *dG, *rdt, *gacc, *linf;   // N each (control warp; gacc: 4N, all warps)
    double *gpart;            // 2 per staged segment: partial dots of its two threads with w
    float *part2, *wbuf, *coef;
    float *ombuf, *fl_dw;     // k_newton: omega of the group's slots; change of omega at each chunk's flipped slots
    float *ubuf;              // k_newton: omega d_new of the group's slots (d_new: the column that is new to H_F)
    double *gpartu, *gaccu;   // k_newton: like gpart, gacc for the products with ubuf
    long long *gfxu;          // k_newton: like gfx
    unsigned char *fl_slot;   // k_newton: the flipped slots of each chunk of the group (kGroup x kChunk), ascending
    int *fl_wc;               // k_newton: how many each of the four warps of a chunk found
    int *hm;                  // k_newton: members of the chunk whose Hessian part is being updated (segment | i << 16)
    int *hv;                  // k_newton: column i is in the Hessian already
    float *rz0, *rz1, *rq, *rT, *ral, *rbe;   // resident copies of the block's own slots (a.rslots each), or unused
    float *rom;               // k_newton: resident copy of a.omref (written through)
    float *tile;       // staged 512-byte segments of the block's part of Dd, kSeg floats apart
    int *nx, *pv;      // neighbours of beam k in Eq. 2 (-1: none): k + 1, k - 1, or the next / previous occupied beam
    int *sk, *lo, *hi, *ik;   // lo, hi: block-local range of chunks (j of b + jG) that may hold entries of column i
    int *nseg;         // how many of them really do
    unsigned long long *lmask;   // which: bit (j & 63) of word lmask[(j >> 6) * N + i]
    int *base;         // the touched chunks of column i are segments base[i], base[i] + 1, .. of the tile, in chunk
                       // order; kNoCache if column i is not staged
    int *coff;         // ngroups*kGroup + 1: entries [coff[j], coff[j+1]) of cseg belong to local chunk j
    int *cseg;         // staged segments chunk by chunk, beams ascending: segment | i << 16
    int *gseg;         // staged segments group by group, beams ascending, then chunks: segment | (j - g kGroup) << 16
    int *unc;          // beams that touch this block's chunks but are not staged, ascending
    int *wst;          // ngroups x (kGroup + 1): warps wst[g][cs] .. wst[g][cs+1]-1 share chunk cs of group g, in proportion to
                       // the work its lists hold (a staged entry counts 1, an unstaged one 4); fixed per solve
    int *uoff;         // (when a.ul_cap > 0) entries [uoff[j], uoff[j+1]) of ul: the unstaged beams that touch local chunk j
    unsigned short *ul;
    long long *gfx;    // (when a.ul_cap > 0) fixed-point gradient sums of the unstaged beams, N
    long long *recv;   // the pass's record of grid sums, fetched by the whole block after the barrier
    Ctl *ctl;
};

// chunk handled by this block as member `ch` of its group `g`: chunks are dealt round-robin
__device__ __forceinline__ int chunk_of(const MasterArgs &a, int g, int ch) { return (int)blockIdx.x + (g * kGroup + ch) * a.nblk; }

__device__ __forceinline__ bool touches(const Smem &sm, int N, int i, int j) {
    return (sm.lmask[(j >> 6) * N + i] >> (j & 63)) & 1ull;
}
// number of touched chunks of column i before local chunk j
__device__ __forceinline__ int seg_rank(const Smem &sm, int N, int i, int j) {
    int r = 0;
    for (int w = 0; w < (j >> 6); ++w) r += __popcll(sm.lmask[w * N + i]);
    return r + __popcll(sm.lmask[(j >> 6) * N + i] & ((1ull << (j & 63)) - 1ull));
}

// Columns that are NOT staged.  The four chunks (j = g*kGroup + chalf + 2h, h = 0..3) of column i that this
// warp's half of the group covers: v[h] = the lane's float4 of segment h, zero where the column does not touch
// the chunk; the four loads from L2 / HBM are independent.
__device__ __forceinline__ void load_half(const MasterArgs &a, const Smem &sm, int i, int g, int chalf, int lane,
                                          float4 (&v)[kGroup / 2]) {
    const unsigned m = ((unsigned)(sm.lmask[((g * kGroup) >> 6) * a.N + i] >> ((g * kGroup) & 63)) & 0xffu) >> chalf;
    const int j0 = g * kGroup + chalf, G = a.nblk;
    const float4 *row = reinterpret_cast<const float4 *>(a.Dd) +
                        ((size_t)((int)blockIdx.x + j0 * G) * a.N + sm.sk[i]) * (kChunk / 4) + lane;
#pragma unroll
    for (int h = 0; h < kGroup / 2; ++h)
        v[h] = (m >> (2 * h)) & 1u ? __ldg(row + (size_t)(2 * h * G) * a.N * (kChunk / 4)) : make_float4(0.f, 0.f, 0.f, 0.f);
}

// ---- columns that are not staged, walked through per-chunk lists (sm.ul) when the lists fit --------------
// Eight independent 16-byte loads per lane and step, every one of them a touched segment: the streaming part of
// a pass over a large problem is bound by bytes in flight, and the masked loops above keep only the touched
// fraction (a third) of theirs in flight.

// this warp's chunk cs of group g, its rank r among the c warps that share the chunk (c = 0: the warp is idle)
__device__ __forceinline__ void warp_share(const Smem &sm, int g, int warp, int &cs, int &r, int &c) {
    const int *w = sm.wst + g * (kGroup + 1);
    cs = 0;
    r = c = 0;
#pragma unroll
    for (int x = 0; x < kGroup; ++x)
        if (w[x] <= warp && warp < w[x + 1]) {
            cs = x;
            r = warp - w[x];
            c = w[x + 1] - w[x];
        }
}

// q-part of chunk j for rank r of the c warps that share the chunk's unstaged beams: adds into s1, s2
__device__ __forceinline__ void combine_unstaged_listed(const MasterArgs &a, const Smem &sm, int j, int r, int c, int lane,
                                                        float4 &s1, float4 &s2) {
    const float4 *Dd4 = reinterpret_cast<const float4 *>(a.Dd) +
                        (size_t)((int)blockIdx.x + j * a.nblk) * a.N * (kChunk / 4) + lane;   // the chunk's segments
    const size_t row4 = kChunk / 4;
    const int n1 = sm.uoff[j + 1];
    for (int n = sm.uoff[j] + r; n < n1; n += 8 * c) {
        float4 v[8];
        float f[8];
#pragma unroll
        for (int x = 0; x < 8; ++x) {
            const int nn = n + c * x;
            f[x] = 0.f;
            v[x] = make_float4(0.f, 0.f, 0.f, 0.f);
            if (nn < n1) {
                const int i = sm.ul[nn];
                f[x] = sm.coef[i];
                v[x] = __ldg(Dd4 + (size_t)sm.sk[i] * row4);
            }
        }
#pragma unroll
        for (int x = 0; x < 8; x += 2) {
            s1.x = fmaf(f[x], v[x].x, s1.x);
            s1.y = fmaf(f[x], v[x].y, s1.y);
            s1.z = fmaf(f[x], v[x].z, s1.z);
            s1.w = fmaf(f[x], v[x].w, s1.w);
            s2.x = fmaf(f[x + 1], v[x + 1].x, s2.x);
            s2.y = fmaf(f[x + 1], v[x + 1].y, s2.y);
            s2.z = fmaf(f[x + 1], v[x + 1].z, s2.z);
            s2.w = fmaf(f[x + 1], v[x + 1].w, s2.w);
        }
    }
}

// sums of eight values over the warp in nine exchanges: after the exchanges at 16, 8 and 4 each lane carries one
// of the eight; lane L ends with the total of value ((L >> 4) & 1) * 4 + ((L >> 3) & 1) * 2 + ((L >> 2) & 1)
__device__ __forceinline__ double warp_sum8(double (&v)[8], int lane) {
    const bool b16 = lane & 16, b8 = lane & 8, b4 = lane & 4;
#pragma unroll
    for (int x = 0; x < 4; ++x) {
        const double keep = b16 ? v[x + 4] : v[x], send = b16 ? v[x] : v[x + 4];
        v[x] = keep + __shfl_xor_sync(kFull, send, 16);
    }
#pragma unroll
    for (int x = 0; x < 2; ++x) {
        const double keep = b8 ? v[x + 2] : v[x], send = b8 ? v[x] : v[x + 2];
        v[x] = keep + __shfl_xor_sync(kFull, send, 8);
    }
    const double keep = b4 ? v[1] : v[0], send = b4 ? v[0] : v[1];
    double r = keep + __shfl_xor_sync(kFull, send, 4);
    r += __shfl_xor_sync(kFull, r, 2);
    r += __shfl_xor_sync(kFull, r, 1);
    return r;
}

// Gradient dots of the unstaged beams of group g: warp (cs, hf) takes every second entry of chunk g*kGroup + cs,
// eight beams per step; lane partials over 4 products in fp32, the warp sums in fp64 (warp_sum8), then into the
// beam's FIXED-POINT accumulator in shared memory (integer adds: order free, so the result stays reproducible
// although several warps add to one beam).  buf: the group's vector (laid out like sm.wbuf), gfx: N sums, scale scG.
__device__ __forceinline__ void grad_unstaged_listed(const MasterArgs &a, const Smem &sm, int g, const float *buf,
                                                     long long *gfx, double scG) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int cs, r, c;
    warp_share(sm, g, warp, cs, r, c);
    if (c == 0) return;
    const int j = g * kGroup + cs, n1 = sm.uoff[j + 1];
    int n = sm.uoff[j] + r;
    if (n >= n1) return;
    const float4 w4 = reinterpret_cast<const float4 *>(buf)[cs * kSeg4 + lane];
    const float4 *Dd4 = reinterpret_cast<const float4 *>(a.Dd) +
                        (size_t)((int)blockIdx.x + j * a.nblk) * a.N * (kChunk / 4) + lane;   // the chunk's segments
    const size_t row4 = kChunk / 4;
    const int mine = ((lane >> 4) & 1) * 4 + ((lane >> 3) & 1) * 2 + ((lane >> 2) & 1);   // warp_sum8's layout
    for (; n < n1; n += 8 * c) {
        float4 v[8];
        int id[8];
#pragma unroll
        for (int x = 0; x < 8; ++x) {
            const int nn = n + c * x;
            id[x] = -1;
            v[x] = make_float4(0.f, 0.f, 0.f, 0.f);
            if (nn < n1) {
                id[x] = sm.ul[nn];
                v[x] = __ldg(Dd4 + (size_t)sm.sk[id[x]] * row4);
            }
        }
        double dw[8];
#pragma unroll
        for (int x = 0; x < 8; ++x)
            dw[x] = (double)((v[x].x * w4.x + v[x].y * w4.y) + (v[x].z * w4.z + v[x].w * w4.w));
        const double rw = warp_sum8(dw, lane);
        int my_id = -1;
#pragma unroll
        for (int x = 0; x < 8; ++x)
            if (x == mine) my_id = id[x];
        if ((lane & 3) == 0 && my_id >= 0)
            atomicAdd(reinterpret_cast<unsigned long long *>(gfx) + my_id, (unsigned long long)__double2ll_rn(rw * scG));
    }
}

// value[o] = sum_i coef[i] * Dd[sk[i]][slot(o)] for the kGroup*128 slots of group g, o = tid + r*kMasterThreads.
// Staged columns: the two warps of a chunk walk its list of staged segments (every second entry each, beams
// ascending), one float4 of the segment per lane: only segments the columns really touch are visited; the
// columns that are not staged (Ku of them) follow by the same split.  The two partials of a chunk meet in
// shared memory.  The caller must __syncthreads() before sm.part2 is written again.
__device__ __forceinline__ void combine_group(const MasterArgs &a, const Smem &sm, int Ku, int g,
                                              float (&out)[kOutPerThread]) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    {
        int cs, r, c;
        warp_share(sm, g, warp, cs, r, c);
        const int n1 = c ? sm.coff[g * kGroup + cs + 1] : 0;
        int n = c ? sm.coff[g * kGroup + cs] + r : 0;
        const float4 *tile4 = reinterpret_cast<const float4 *>(sm.tile) + lane;
        float4 s1 = make_float4(0.f, 0.f, 0.f, 0.f), s2 = s1;
        for (; n + c < n1; n += 2 * c) {
            const int e1 = sm.cseg[n], e2 = sm.cseg[n + c];
            const float c1 = sm.coef[e1 >> 16], c2 = sm.coef[e2 >> 16];
            const float4 v1 = tile4[(e1 & 0xffff) * kSeg4], v2 = tile4[(e2 & 0xffff) * kSeg4];
            s1.x = fmaf(c1, v1.x, s1.x);
            s1.y = fmaf(c1, v1.y, s1.y);
            s1.z = fmaf(c1, v1.z, s1.z);
            s1.w = fmaf(c1, v1.w, s1.w);
            s2.x = fmaf(c2, v2.x, s2.x);
            s2.y = fmaf(c2, v2.y, s2.y);
            s2.z = fmaf(c2, v2.z, s2.z);
            s2.w = fmaf(c2, v2.w, s2.w);
        }
        if (n < n1) {
            const int e1 = sm.cseg[n];
            const float c1 = sm.coef[e1 >> 16];
            const float4 v1 = tile4[(e1 & 0xffff) * kSeg4];
            s1.x = fmaf(c1, v1.x, s1.x);
            s1.y = fmaf(c1, v1.y, s1.y);
            s1.z = fmaf(c1, v1.z, s1.z);
            s1.w = fmaf(c1, v1.w, s1.w);
        }
        if (c == 0) {
        } else if (Ku > 0 && a.ul_cap > 0) {
            combine_unstaged_listed(a, sm, g * kGroup + cs, r, c, lane, s1, s2);
        } else if (Ku > 0) {
            // columns that are not staged: same split, four beams per step, one float4 of the chunk per lane
            // straight from L2 / HBM; a beam that does not touch the chunk is skipped (warp-uniform test)
            const int j = g * kGroup + cs;
            const float4 *Dd4 = reinterpret_cast<const float4 *>(a.Dd) +
                                (size_t)((int)blockIdx.x + j * a.nblk) * a.N * (kChunk / 4) + lane;
            const size_t row4 = kChunk / 4;
            for (int u = r; u < Ku; u += 4 * c) {
                float4 v[4];
                float f[4];
#pragma unroll
                for (int x = 0; x < 4; ++x) {
                    const int uu = u + c * x;
                    f[x] = 0.f;
                    v[x] = make_float4(0.f, 0.f, 0.f, 0.f);
                    if (uu < Ku) {
                        const int i = sm.unc[uu];
                        if (touches(sm, a.N, i, j)) {
                            f[x] = sm.coef[i];
                            v[x] = __ldg(Dd4 + (size_t)sm.sk[i] * row4);
                        }
                    }
                }
#pragma unroll
                for (int x = 0; x < 4; x += 2) {
                    s1.x = fmaf(f[x], v[x].x, s1.x);
                    s1.y = fmaf(f[x], v[x].y, s1.y);
                    s1.z = fmaf(f[x], v[x].z, s1.z);
                    s1.w = fmaf(f[x], v[x].w, s1.w);
                    s2.x = fmaf(f[x + 1], v[x + 1].x, s2.x);
                    s2.y = fmaf(f[x + 1], v[x + 1].y, s2.y);
                    s2.z = fmaf(f[x + 1], v[x + 1].z, s2.z);
                    s2.w = fmaf(f[x + 1], v[x + 1].w, s2.w);
                }
            }
        }
        reinterpret_cast<float4 *>(sm.part2)[warp * 32 + lane] =
            make_float4(s1.x + s2.x, s1.y + s2.y, s1.z + s2.z, s1.w + s2.w);
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < kOutPerThread; ++r) {
        const int o = tid + r * kMasterThreads, ch = o >> 7, s = o & (kChunk - 1);
        const int w0 = sm.wst[g * (kGroup + 1) + ch], w1 = sm.wst[g * (kGroup + 1) + ch + 1];
        float v = 0.f;
        for (int w = w0; w < w1; ++w) v += sm.part2[w * kChunk + s];   // the chunk's warps, in order
        out[r] = v;
    }
}

// Gradient products of the staged segments of group g: two threads per segment (alternate float4s), each a plain
// dot of 64 entries with the group's vector buf (laid out like sm.wbuf) — no exchange between lanes.  Lane partials
// over 16 products in fp32, then fp64.  The partials land in gpart, two per segment; grad_total adds them per beam.
__device__ __forceinline__ void grad_staged(const Smem &sm, int g, const float *buf, double *gpart) {
    const int n0 = sm.coff[g * kGroup], n2 = 2 * (sm.coff[(g + 1) * kGroup] - n0);
    const float4 *tile4 = reinterpret_cast<const float4 *>(sm.tile);
    const float4 *wb4 = reinterpret_cast<const float4 *>(buf);
    for (int t2 = threadIdx.x; t2 < n2; t2 += kMasterThreads) {
        const int e = sm.gseg[n0 + (t2 >> 1)], hfs = t2 & 1;
        const int s = e & 0xffff, cs = e >> 16;
        const float4 *tp = tile4 + s * kSeg4 + hfs, *wp = wb4 + cs * kSeg4 + hfs;
        double dw = 0.0;
#pragma unroll
        for (int blk = 0; blk < 4; ++blk) {
            float4 aw = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
            for (int it = 0; it < 4; ++it) {
                const int x = (blk * 4 + it) * 2;
                const float4 v = tp[x], w = wp[x];
                aw.x = fmaf(v.x, w.x, aw.x);
                aw.y = fmaf(v.y, w.y, aw.y);
                aw.z = fmaf(v.z, w.z, aw.z);
                aw.w = fmaf(v.w, w.w, aw.w);
            }
            dw += (double)((aw.x + aw.y) + (aw.z + aw.w));
        }
        gpart[2 * s + hfs] = dw;
    }
}

// Columns that are not staged, when their per-chunk lists do not fit either: this warp's half of the group's chunks
// (4 chunks) and its share of those beams, two beams per step (eight masked loads), lane partials in fp32 (16
// products), the warp sums in fp64 to the row of gacc (2 x N) of this chunk half.  buf: laid out like sm.wbuf.
__device__ __forceinline__ void grad_unstaged_masked(const MasterArgs &a, const Smem &sm, int g, int Ku, const float *buf,
                                                     double *gacc2) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int kpart = warp & (kKSplit - 1), chalf = warp / kKSplit;
    float4 w4[kGroup / 2];
#pragma unroll
    for (int h = 0; h < kGroup / 2; ++h) w4[h] = reinterpret_cast<const float4 *>(buf)[(2 * h + chalf) * kSeg4 + lane];
    for (int u = kpart; u < Ku; u += 2 * kKSplit) {
        const bool has2 = u + kKSplit < Ku;
        const int i = sm.unc[u], i2 = has2 ? sm.unc[u + kKSplit] : i;
        float4 v1[kGroup / 2], v2[kGroup / 2];
        load_half(a, sm, i, g, chalf, lane, v1);
        load_half(a, sm, i2, g, chalf, lane, v2);
        float4 s1 = make_float4(0.f, 0.f, 0.f, 0.f), s2 = s1;
#pragma unroll
        for (int h = 0; h < kGroup / 2; ++h) {
            s1.x = fmaf(v1[h].x, w4[h].x, s1.x);
            s1.y = fmaf(v1[h].y, w4[h].y, s1.y);
            s1.z = fmaf(v1[h].z, w4[h].z, s1.z);
            s1.w = fmaf(v1[h].w, w4[h].w, s1.w);
            s2.x = fmaf(v2[h].x, w4[h].x, s2.x);
            s2.y = fmaf(v2[h].y, w4[h].y, s2.y);
            s2.z = fmaf(v2[h].z, w4[h].z, s2.z);
            s2.w = fmaf(v2[h].w, w4[h].w, s2.w);
        }
        double d1 = (double)((s1.x + s1.y) + (s1.z + s1.w)), d2 = (double)((s2.x + s2.y) + (s2.z + s2.w));
        // one butterfly for both rows: after the first exchange the lower half-warp carries row 1, the upper row 2
        const bool up = lane & 16;
        double r = (up ? d2 : d1) + __shfl_xor_sync(kFull, up ? d1 : d2, 16);
        r += __shfl_xor_sync(kFull, r, 8);
        r += __shfl_xor_sync(kFull, r, 4);
        r += __shfl_xor_sync(kFull, r, 2);
        r += __shfl_xor_sync(kFull, r, 1);
        double *row = gacc2 + chalf * a.N;      // entries i, i2 of this row are owned by this warp
        if (lane == 0) row[i] += r;
        if (lane == 16 && has2) row[i2] += r;
    }
}

// beam i's total over the block: staged columns add the partials of their segments in chunk order, the others
// the two chunk-half rows of sm.gacc (row0, row0 + 1)
__device__ __forceinline__ double grad_total(const Smem &sm, const double *gp, const double *gacc, int i, int N) {
    const int bs = sm.base[i];
    if (bs == kNoCache) return gacc[i] + gacc[N + i];
    double s = 0.0;
    for (int q = 0; q < sm.nseg[i]; ++q) s += gp[2 * (bs + q)] + gp[2 * (bs + q) + 1];
    return s;
}

__device__ __forceinline__ void penalty(float z, float T, float al, float be, float &w, double &F) {
    const float under = fmaxf(0.f, T - z), over = fmaxf(0.f, z - T);
    w = -2.f * al * under + 2.f * be * over;                                       // Eq. 1, derivative
    F = (double)al * (double)under * (double)under + (double)be * (double)over * (double)over;
}

// One pass over the block's chunks that evaluates the objective at a new dose:
//   FROM_Y:  z_new = sum_k y_k d_k            (coef must hold y)             -> stored to zdst, w to a.w
//   else:    z_new = zsrc + t q               (line-search trial)            -> stored to zdst
// and in the same pass F and the block's share of grad = Dc w_new, both added to the record `rec`
// in fixed point (scales scF, scG).
template <bool FROM_Y>
__device__ __forceinline__ void eval_pass(const MasterArgs &a, const Smem &sm, int K, int Ku, int ngroups, const float *zsrc,
                                          float *zdst, const float *rzsrc, float *rzdst, float tf, long long *rec,
                                          double scF, double scG, double *red) {
    const bool res = a.rslots > 0;
    const int tid = threadIdx.x;
    for (int i = tid; i < 2 * a.N; i += kMasterThreads) sm.gacc[i] = 0.0;
    if (a.ul_cap > 0)
        for (int i = tid; i < a.N; i += kMasterThreads) sm.gfx[i] = 0;
    double F = 0.0;
    __syncthreads();
    for (int g = 0; g < ngroups; ++g) {
        float zv[kOutPerThread];
        if (FROM_Y) combine_group(a, sm, Ku, g, zv);
#pragma unroll
        for (int r = 0; r < kOutPerThread; ++r) {
            const int o = tid + r * kMasterThreads, c = chunk_of(a, g, o >> 7);
            float wv = 0.f;
            if (c < a.nchunks) {
                const size_t s = (size_t)c * kChunk + (o & (kChunk - 1));
                const int ls = g * (kGroup * kChunk) + o;          // the slot's place in the resident arrays
                float z, Tv, al, be;
                if (res) {
                    z = FROM_Y ? zv[r] : fmaf(tf, sm.rq[ls], rzsrc[ls]);
                    Tv = sm.rT[ls], al = sm.ral[ls], be = sm.rbe[ls];
                    rzdst[ls] = z;
                } else {
                    z = FROM_Y ? zv[r] : fmaf(tf, a.q[s], zsrc[s]);
                    Tv = a.T[s], al = a.alpha[s], be = a.beta[s];
                }
                double f;
                penalty(z, Tv, al, be, wv, f);
                F += f;
                if (FROM_Y || !res) zdst[s] = z;   // evaluations from y publish z and w
                if (FROM_Y) a.w[s] = wv;
            }
            sm.wbuf[(o >> 7) * kSeg + (o & (kChunk - 1))] = wv;
        }
        __syncthreads();
        grad_staged(sm, g, sm.wbuf, sm.gpart);
        // columns that are not staged: through the per-chunk lists when they fit, otherwise by masked loops
        if (Ku > 0 && a.ul_cap > 0) {
            grad_unstaged_listed(a, sm, g, sm.wbuf, sm.gfx, scG);
        } else if (Ku > 0) {
            grad_unstaged_masked(a, sm, g, Ku, sm.wbuf, sm.gacc);
        }
        __syncthreads();
    }
    F = block_sum(F, red);
    if (tid == 0) fx_add(rec, F, scF);
    for (int i = tid; i < K; i += kMasterThreads) {
        if (a.ul_cap > 0 && sm.base[i] == kNoCache)   // already in fixed point
            atomicAdd(reinterpret_cast<unsigned long long *>(rec + 2 + i), (unsigned long long)sm.gfx[i]);
        else fx_add(rec + 2 + i, grad_total(sm, sm.gpart, sm.gacc, i, a.N), scG);
    }
}

// ---- control group: the first nw warps of a block (CT = 32 nw threads) share the N-vector work -----
__device__ __forceinline__ void ctl_sync(int CT) { asm volatile("bar.sync 1, %0;" ::"r"(CT) : "memory"); }

// Batched reduction over the control group: MS sums and one maximum at once, fixed order, every thread of the
// group receives the results.  One barrier per call: the scratch alternates (tog), so a call never overwrites
// what a slower warp is still reading from the call before.
template <int MS>
__device__ __forceinline__ void ctl_reduce(double (&s)[MS], double &mx, double *cred, int &tog, int nw, int CT) {
    static_assert(MS < kRedSlots, "scratch row too short");
#pragma unroll
    for (int o = 16; o; o >>= 1) {
#pragma unroll
        for (int m = 0; m < MS; ++m) s[m] += __shfl_xor_sync(kFull, s[m], o);
        mx = fmax(mx, __shfl_xor_sync(kFull, mx, o));
    }
    double *buf = cred + tog * (kMasterWarps * kRedSlots);
    tog ^= 1;
    if ((threadIdx.x & 31) == 0) {
        double *row = buf + (threadIdx.x >> 5) * kRedSlots;
#pragma unroll
        for (int m = 0; m < MS; ++m) row[m] = s[m];
        row[kRedSlots - 1] = mx;
    }
    ctl_sync(CT);
#pragma unroll
    for (int m = 0; m < MS; ++m) s[m] = 0.0;
    mx = -CUDART_INF;
    for (int w = 0; w < nw; ++w) {
#pragma unroll
        for (int m = 0; m < MS; ++m) s[m] += buf[w * kRedSlots + m];
        mx = fmax(mx, buf[w * kRedSlots + kRedSlots - 1]);
    }
}

// this thread's share of G(v) = sum_k (v_{k+1}-v_k)^2 / (theta_{k+1}-theta_k), and dG/dv_k -> sm.dG
// (Eq. 2; S2, S3)
__device__ __forceinline__ double smooth_part(const double *v, const Smem &sm, int N, int CT, bool want_dG) {
    double s = 0.0;
    for (int k = threadIdx.x; k < N; k += CT) {
        const int nx = sm.nx[k], pv = sm.pv[k];
        const double e1 = nx >= 0 ? (v[nx] - v[k]) * sm.rdt[k] : 0.0;      // (v_next - v_k) / dtheta
        if (nx >= 0) s += (v[nx] - v[k]) * e1;
        if (want_dG) {
            const double e0 = pv >= 0 ? (v[k] - v[pv]) * sm.rdt[pv] : 0.0;
            sm.dG[k] = 2.0 * (e0 - e1);
        }
    }
    return s;
}

// What both master kernels do first: carve up the block's shared memory, list the occupied beams, stage the block's
// part of Dd and build the lists over it.  NEWTON: the block also lays out what the Hessian updates of k_newton need.
struct Setup {
    int K, Ku, ngroups, segs;   // occupied beams, unstaged beams touching this block, groups of chunks, touched segments
    double l1max;               // max over occupied beams of sum |d_k|
    double *red, *cred;         // reduction scratch of the block / of its control group
};

template <bool NEWTON>
__device__ __forceinline__ Setup master_setup(const MasterArgs &a, Smem &sm, float4 *smem_raw) {
    const int N = a.N, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int F1 = NEWTON ? 1 : 0;
    sm.part2 = reinterpret_cast<float *>(smem_raw);
    sm.wbuf = sm.part2 + 2 * kGroup * kChunk;
    sm.ombuf = sm.wbuf + kGroup * kSeg;             // NEWTON: omega of the group's slots, laid out like wbuf
    sm.ubuf = sm.ombuf + F1 * kGroup * kSeg;        // NEWTON: omega d_new
    sm.fl_dw = sm.ubuf + F1 * kGroup * kSeg;        // NEWTON: change of omega at the flipped slots of each chunk
    sm.tile = sm.fl_dw + F1 * kGroup * kChunk;
    sm.rz0 = sm.tile + (size_t)a.cache_segs * kSeg;
    sm.rz1 = sm.rz0 + a.rslots;
    sm.rq = sm.rz1 + a.rslots;
    sm.rT = sm.rq + a.rslots;
    sm.ral = sm.rT + a.rslots;
    sm.rbe = sm.ral + a.rslots;
    sm.rom = sm.rbe + a.rslots;
    sm.y = reinterpret_cast<double *>(sm.rom + F1 * a.rslots);
    sm.d = sm.y + N;
    sm.grad = sm.d + N;
    sm.pg = sm.grad + N;
    sm.yn = sm.pg + N;
    sm.gn = sm.yn + N;
    sm.dG = sm.gn + N;
    sm.rdt = sm.dG + N;
    sm.gacc = sm.rdt + N;
    sm.gaccu = sm.gacc + 2 * N;  // gacc: one row per chunk half
    sm.linf = sm.gaccu + F1 * 2 * N;
    sm.gpart = sm.linf + N;
    sm.gpartu = sm.gpart + 2 * a.cache_segs;
    const int ngroups = (a.nchunks + a.nblk * kGroup - 1) / (a.nblk * kGroup);
    const int W64 = (ngroups * kGroup + 63) >> 6;   // 64-bit words of a column's local chunk mask
    sm.lmask = reinterpret_cast<unsigned long long *>(sm.gpartu + F1 * 2 * a.cache_segs);
    sm.gfx = reinterpret_cast<long long *>(sm.lmask + (size_t)W64 * N);
    sm.gfxu = sm.gfx + (a.ul_cap > 0 ? N : 0);
    double *red = reinterpret_cast<double *>(sm.gfxu + (a.ul_cap > 0 ? F1 * N : 0));
    double *cred = red + kMasterWarps;   // 2 x kMasterWarps x kRedSlots
    sm.recv = reinterpret_cast<long long *>(cred + 2 * kMasterWarps * kRedSlots);
    sm.ctl = reinterpret_cast<Ctl *>(sm.recv + 2 * N + 2);
    sm.coef = reinterpret_cast<float *>(sm.ctl + 1);
    sm.sk = reinterpret_cast<int *>(sm.coef + N);
    sm.lo = sm.sk + N;
    sm.hi = sm.lo + N;
    sm.ik = sm.hi + N;
    sm.nx = sm.ik + N;
    sm.pv = sm.nx + N;
    sm.base = sm.pv + N;
    sm.unc = sm.base + N;
    sm.cseg = sm.unc + N;
    sm.gseg = sm.cseg + a.cache_segs;
    sm.nseg = sm.gseg + a.cache_segs;
    sm.coff = sm.nseg + N;   // ngroups * kGroup + 1
    sm.wst = sm.coff + ngroups * kGroup + 1;    // ngroups * (kGroup + 1)
    sm.uoff = sm.wst + ngroups * (kGroup + 1);  // like coff, if a.ul_cap > 0
    sm.hm = sm.uoff + (a.ul_cap > 0 ? ngroups * kGroup + 1 : 0);   // NEWTON: N members of the chunk being updated
    sm.hv = sm.hm + F1 * N;                                        // NEWTON: N flags, column i is in the Hessian
    sm.fl_wc = sm.hv + F1 * N;                                     // NEWTON: kGroup x 4 flipped slots per warp of a chunk
    sm.fl_slot = reinterpret_cast<unsigned char *>(sm.fl_wc + F1 * (kGroup * 4 + 4));   // NEWTON: kGroup x kChunk
    sm.ul = reinterpret_cast<unsigned short *>(sm.fl_slot + F1 * kGroup * kChunk);   // a.ul_cap 16-bit beam numbers, last array
    __shared__ int sK, sKu, sSegs;
    __shared__ uint64_t tile_bar;

    // occupied beams in ascending order
    if (tid < 32) {
        int base = 0;
        for (int k0 = 0; k0 < N; k0 += 32) {
            const int k = k0 + tid;
            const bool f = k < N && a.occ[k];
            const unsigned m = __ballot_sync(kFull, f);
            const int i = base + __popc(m & ((1u << tid) - 1u));
            if (f) sm.sk[i] = k;
            if (k < N) sm.ik[k] = f ? i : -1;
            base += __popc(m);
        }
        if (tid == 0) {
            sK = base;
            sSegs = 0;
        }
    }
    for (int k = tid; k < N; k += kMasterThreads) {
        double yk = a.y[k];
        if (!a.occ[k]) yk = 0.0;
        else if (!(yk > a.lb)) yk = a.lb;
        else if (yk > a.ub) yk = a.ub;
        sm.y[k] = yk;
        sm.d[k] = 0.0;
        // neighbours in Eq. 2: the angles next to k (S2), or the nearest occupied beams (the other reading)
        int nxk = k + 1 < N ? k + 1 : -1, pvk = k - 1;
        if (a.occ_only) {
            if (!a.occ[k]) nxk = pvk = -1;
            else {
                while (nxk >= 0 && !a.occ[nxk]) nxk = nxk + 1 < N ? nxk + 1 : -1;
                while (pvk >= 0 && !a.occ[pvk]) --pvk;
            }
        }
        sm.nx[k] = nxk;
        sm.pv[k] = pvk;
        sm.rdt[k] = nxk >= 0 ? 1.0 / (a.theta[nxk] - a.theta[k]) : 0.0;
    }
    __syncthreads();
    const int K = sK;
    // per occupied beam: touched chunk range, max |d_k| (0 at un-occupied beams); over all: max sum |d_k|
    double l1l = 0.0;
    for (int k = tid; k < N; k += kMasterThreads) {
        const int i = sm.ik[k];
        double lf = 0.0;
        if (i >= 0) {
            const ColStat cs = a.colstat[k];
            // the block's chunks are b + jG: column k touches those with lo <= j <= hi (empty: hi < lo)
            const int b = (int)blockIdx.x, Gd_ = a.nblk;
            sm.lo[i] = cs.clo > b ? (cs.clo - b + Gd_ - 1) / Gd_ : 0;
            sm.hi[i] = cs.chi >= b ? (cs.chi - b) / Gd_ : -1;
            // which of them hold a non-zero entry of the column (the range is half empty: an aperture lights a
            // strip of every slab it crosses)
            const uint32_t *tw = a.touch + (size_t)k * a.touch_words;
            int n = 0;
            for (int w = 0; w < W64; ++w) {
                unsigned long long bits = 0ull;
                const int ja = max(sm.lo[i], w * 64), jb = min(sm.hi[i], w * 64 + 63);
                for (int j = ja; j <= jb; ++j) {
                    const int c = b + j * Gd_;
                    if ((__ldg(tw + (c >> 5)) >> (c & 31)) & 1u) bits |= 1ull << (j & 63);
                }
                sm.lmask[w * N + i] = bits;
                n += __popcll(bits);
            }
            sm.nseg[i] = n;
            if (n) atomicAdd(&sSegs, n);
            lf = (double)cs.linf * a.fx_inv * 1.000001;
            l1l = fmax(l1l, (double)cs.l1 * a.fx_inv * 1.000001);
            sm.coef[i] = (float)sm.y[k];
        }
        sm.linf[k] = lf;
    }
    const double l1max = block_max(l1l, red);

    // ---- stage the block's part of Dd in shared memory (TMA bulk copies, one per 512-byte segment) ----
    // The block's chunks are b + jG; column i touches those with j0_i <= j <= j1_i.  Segments are
    // packed column after column until the tile is full; the rest stays in L2 / HBM.
    {
        const int G = a.nblk, b = (int)blockIdx.x;
        if (tid == 0) mbar_init(&tile_bar, 1);
        __syncthreads();
        if (warp == 0) {
            int run = 0, total = 0;
            for (int i0 = 0; i0 < K; i0 += 32) {
                const int i = i0 + lane;
                int cnt = 0;
                if (i < K) cnt = sm.nseg[i];
                int incl = cnt;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const int n = __shfl_up_sync(kFull, incl, o);
                    if (lane >= o) incl += n;
                }
                const int off = run + incl - cnt;
                const bool cached = cnt > 0 && off + cnt <= a.cache_segs;
                if (i < K) sm.base[i] = cached ? off : kNoCache;
                total += cached ? cnt : 0;
                run += __shfl_sync(kFull, incl, 31);
            }
#pragma unroll
            for (int o = 16; o; o >>= 1) total += __shfl_xor_sync(kFull, total, o);
            if (lane == 0) mbar_expect_tx(&tile_bar, (unsigned)total * (kChunk * 4));
            __syncwarp();
            for (int i = lane; i < K; i += 32) {
                const int bs = sm.base[i];
                if (bs == kNoCache) continue;
                const int j0 = sm.lo[i], j1 = sm.hi[i];
                const float *src = a.Dd + (size_t)sm.sk[i] * kChunk;
                int q = 0;
                for (int j = j0; j <= j1; ++j)
                    if (touches(sm, N, i, j))
                        bulk_g2s(sm.tile + (size_t)(bs + q++) * kSeg, src + (size_t)(b + j * G) * N * kChunk, kChunk * 4, &tile_bar);
            }
        }
        __syncthreads();          // sm.base visible to all warps
    }
    // ---- lists over the staged segments, built once per solve in a fixed order (reproducible sums) ----
    const int nj = ngroups * kGroup;
    if (warp == 1) {   // beams that touch this block's chunks but are not staged, ascending
        int run = 0;
        for (int i0 = 0; i0 < K; i0 += 32) {
            const int i = i0 + lane;
            const bool f = i < K && sm.base[i] == kNoCache && sm.nseg[i] > 0;
            const unsigned m = __ballot_sync(kFull, f);
            if (f) sm.unc[run + __popc(m & ((1u << lane) - 1u))] = i;
            run += __popc(m);
        }
        if (lane == 0) sKu = run;
    }
    for (int j = warp; j < nj; j += kMasterWarps) {   // staged segments per local chunk
        int c = 0;
        for (int i0 = 0; i0 < K; i0 += 32) {
            const int i = i0 + lane;
            const bool f = i < K && sm.base[i] != kNoCache && touches(sm, N, i, j);
            c += __popc(__ballot_sync(kFull, f));
        }
        if (lane == 0) sm.coff[j + 1] = c;
        if (a.ul_cap > 0) {   // and the unstaged beams that touch it
            int cu = 0;
            for (int i0 = 0; i0 < K; i0 += 32) {
                const int i = i0 + lane;
                const bool f = i < K && sm.base[i] == kNoCache && touches(sm, N, i, j);
                cu += __popc(__ballot_sync(kFull, f));
            }
            if (lane == 0) sm.uoff[j + 1] = cu;
        }
    }
    __syncthreads();
    if (warp == 1 && a.ul_cap > 0) {   // running sums of the unstaged lists
        int run = 0;
        for (int j0 = 0; j0 < nj; j0 += 32) {
            const int j = j0 + lane;
            int incl = j < nj ? sm.uoff[j + 1] : 0;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int n = __shfl_up_sync(kFull, incl, o);
                if (lane >= o) incl += n;
            }
            if (j < nj) sm.uoff[j + 1] = run + incl;
            run += __shfl_sync(kFull, incl, 31);
        }
        if (lane == 0) sm.uoff[0] = 0;
    }
    if (warp == 0) {   // running sums: coff[j] = first entry of chunk j
        int run = 0;
        for (int j0 = 0; j0 < nj; j0 += 32) {
            const int j = j0 + lane;
            int incl = j < nj ? sm.coff[j + 1] : 0;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int n = __shfl_up_sync(kFull, incl, o);
                if (lane >= o) incl += n;
            }
            if (j < nj) sm.coff[j + 1] = run + incl;
            run += __shfl_sync(kFull, incl, 31);
        }
        if (lane == 0) sm.coff[0] = 0;
    }
    __syncthreads();
    for (int j = warp; j < nj; j += kMasterWarps) {   // chunk by chunk, beams ascending
        int pos = sm.coff[j];
        for (int i0 = 0; i0 < K; i0 += 32) {
            const int i = i0 + lane;
            const bool f = i < K && sm.base[i] != kNoCache && touches(sm, N, i, j);
            const unsigned m = __ballot_sync(kFull, f);
            if (f) sm.cseg[pos + __popc(m & ((1u << lane) - 1u))] = (sm.base[i] + seg_rank(sm, N, i, j)) | (i << 16);
            pos += __popc(m);
        }
        if (a.ul_cap > 0) {
            int pu = sm.uoff[j];
            for (int i0 = 0; i0 < K; i0 += 32) {
                const int i = i0 + lane;
                const bool f = i < K && sm.base[i] == kNoCache && touches(sm, N, i, j);
                const unsigned m = __ballot_sync(kFull, f);
                if (f) sm.ul[pu + __popc(m & ((1u << lane) - 1u))] = (unsigned short)i;
                pu += __popc(m);
            }
        }
    }
    for (int g = warp; g < ngroups; g += kMasterWarps) {   // group by group, beams ascending, then chunks
        int pos = sm.coff[g * kGroup];
        for (int i0 = 0; i0 < K; i0 += 32) {
            const int i = i0 + lane;
            unsigned bits = 0u;   // the column's touched chunks within group g
            if (i < K && sm.base[i] != kNoCache)
                bits = (unsigned)(sm.lmask[((g * kGroup) >> 6) * N + i] >> ((g * kGroup) & 63)) & 0xffu;
            const int cnt = __popc(bits);
            int incl = cnt;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int n = __shfl_up_sync(kFull, incl, o);
                if (lane >= o) incl += n;
            }
            const int at = pos + incl - cnt;
            if (cnt) {
                int sg = sm.base[i] + seg_rank(sm, N, i, g * kGroup);
                for (int q = 0, cs = 0; cs < kGroup; ++cs)
                    if ((bits >> cs) & 1u) sm.gseg[at + q++] = (sg++) | (cs << 16);
            }
            pos += __shfl_sync(kFull, incl, 31);
        }
    }
    __syncthreads();
    const int Ku = sKu;
    // the kMasterWarps warps are dealt to the chunks of every group in proportion to the work their lists hold (a
    // staged entry = 1, an unstaged one = 4; without lists every chunk walks all Ku unstaged beams), at least one
    // warp per chunk that has any: chunk lists differ several-fold in length and a pass waits for its slowest warp
    for (int g = tid; g < ngroups; g += kMasterThreads) {
        int wgt[kGroup], w[kGroup], tot = 0, sum = 0;
#pragma unroll
        for (int cs = 0; cs < kGroup; ++cs) {
            const int j = g * kGroup + cs;
            int v = sm.coff[j + 1] - sm.coff[j];
            if (a.ul_cap > 0) v += 4 * (sm.uoff[j + 1] - sm.uoff[j]);
            else if (chunk_of(a, g, cs) < a.nchunks) v += 4 * Ku;
            wgt[cs] = v;
            tot += v;
        }
#pragma unroll
        for (int cs = 0; cs < kGroup; ++cs) {
            w[cs] = wgt[cs] > 0 ? max(1, (kMasterWarps * wgt[cs]) / tot) : 0;
            sum += w[cs];
        }
        while (sum > kMasterWarps) {   // take from the chunk with the most warps
            int b = 0;
#pragma unroll
            for (int cs = 1; cs < kGroup; ++cs)
                if (w[cs] > w[b]) b = cs;
            --w[b];
            --sum;
        }
        while (tot > 0 && sum < kMasterWarps) {   // give to the chunk with the most work per warp
            int b = -1;
#pragma unroll
            for (int cs = 0; cs < kGroup; ++cs)
                if (w[cs] > 0 && (b < 0 || (long long)wgt[cs] * w[b] > (long long)wgt[b] * w[cs])) b = cs;
            ++w[b];
            ++sum;
        }
        int run = 0;
#pragma unroll
        for (int cs = 0; cs < kGroup; ++cs) {
            sm.wst[g * (kGroup + 1) + cs] = run;
            run += w[cs];
        }
        sm.wst[g * (kGroup + 1) + kGroup] = run;
    }
    __syncthreads();
    mbar_wait(&tile_bar, 0);  // the staged segments have landed (the lists were built while they were in flight)
    Setup st;
    st.K = K;
    st.Ku = Ku;
    st.ngroups = ngroups;
    st.segs = sSegs;
    st.l1max = l1max;
    st.red = red;
    st.cred = cred;
    return st;
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

// ------------------------------------------------------------------------------------------------
// Mode 1: semismooth Newton on the reduced problem (k_newton)
// ------------------------------------------------------------------------------------------------
// F is piecewise quadratic in the dose, so on the piece of the current dose the master problem is the quadratic
//     min_{lb <= y <= ub}  g.(y' - y) + 1/2 (y' - y)^T (2 H_F + 2 gamma L) (y' - y),
//     H_F[k][k'] = sum_s omega_s d_k[s] d_k'[s],  omega_s = alpha_s (z_s < T_s), beta_s (z_s > T_s), else 0,
// over the K <= N occupied beams: a problem in K unknowns that needs no pass over the columns at all once H_F is
// known.  One block of the grid (the last one) holds H_F in its shared memory and solves that quadratic by
// conjugate gradients on the faces of the box (Jacobi-preconditioned, fp64 vectors); the other blocks evaluate the
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
    double *vg = vy + N, *yc = vg + N, *vr = yc + N, *vd = vr + N, *vHd = vd + N, *vpo = vHd + N, *vyn = vpo + N;
    double *vgn = vyn + N, *vp = vgn + N, *linf = vp + N, *rdt = linf + N, *Minv = rdt + N, *dGb = Minv + N;
    double *redb = dGb + N;                                  // 2 x kMasterWarps x kSolveRed
    int *sk = reinterpret_cast<int *>(redb + 2 * kMasterWarps * kSolveRed), *ik = sk + N, *freeo = ik + N, *freen = freeo + N;
    int *nxl = freen + N, *pvl = nxl + N;   // neighbours of beam k in Eq. 2 (as in master_setup)
    float *dc = reinterpret_cast<float *>((reinterpret_cast<uintptr_t>(pvl + N) + 15) & ~(uintptr_t)15);   // compact direction
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
        // the matrix of the current piece: H32 = H_F over the occupied beams
        const long long c0 = clock64();
        {
            const int npair = K * (K + 1) / 2;
            for (int e0 = 0; e0 < npair; e0 += 8 * kMasterThreads) {
                long long v[8];
                int ri[8], ci[8];
#pragma unroll
                for (int u = 0; u < 8; ++u) {
                    const int e = e0 + u * kMasterThreads + tid;
                    ri[u] = -1;
                    v[u] = 0;
                    if (e < npair) {   // row i of the upper triangle starts at i K - i (i - 1) / 2
                        int i = (int)((2.0f * K + 1.0f - sqrtf((2.0f * K + 1.0f) * (2.0f * K + 1.0f) - 8.0f * (float)e)) * 0.5f);
                        while (i > 0 && i * K - i * (i - 1) / 2 > e) --i;
                        while ((i + 1) * K - (i + 1) * i / 2 <= e) ++i;
                        ri[u] = i;
                        ci[u] = i + e - (i * K - i * (i - 1) / 2);
                        v[u] = __ldcg(a.hess + (size_t)sk[i] * N + sk[ci[u]]);
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
        for (int e = tid; e < (Kp - K) * Kp; e += kMasterThreads) H32[(size_t)K * Kp + e] = 0.f;   // rows K..Kp-1 (read with d = 0)
        for (int k = tid; k < N; k += kMasterThreads) {
            yc[k] = vy[k];
            vr[k] = vg[k];
            vd[k] = 0.0;
            vpo[k] = 0.0;
            freeo[k] = 0;
        }
        for (int i = tid; i < Kp; i += kMasterThreads) dc[i] = 0.f;
        __syncthreads();
        for (int k = tid; k < N; k += kMasterThreads) {
            const int i = ik[k];
            double m = 0.0;
            if (i >= 0) m = 2.0 * (double)H32[i * Kp + i] + 2.0 * a.gamma * ((pvl[k] >= 0 ? rdt[pvl[k]] : 0.0) + rdt[k]);
            Minv[k] = m > 0.0 ? 1.0 / m : 1.0;
        }
        const long long c1 = clock64();
        clk_load += c1 - c0;
        // Conjugate gradients on the faces of the box for the quadratic model at (vy, vg): one beam per thread (the
        // first nv warps), all warps on the product with the matrix.  One sum over the beams per step: with the
        // residual r, the preconditioner M, the direction d and H d at hand, A = sum M r^2, B = sum M r (H d) and
        // C = sum M (H d)^2 over the face give the Polak-Ribiere numerator of the NEXT residual r + t H d without a
        // second sum, (r+ - r) M r+ = t (B + t C), and its denominator is A.  Whether the face changed, whether any
        // entry of the new projected residual is still above the tolerance and whether to give up travel as three bits
        // OR-ed into a shared word.  Step lengths, the sums and the ratios to the bounds are fp32: the iteration
        // corrects itself (the residual is updated with the step actually taken) and a beam that reaches its bound is
        // set on it explicitly.
        const double qtol = fmax(0.5 * tol, 0.05 * pgmax);
        const int k = tid;                                   // this thread's beam (k < N: checked on the host)
        const bool mine = k < N && ik[k] >= 0;
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
        int fr = mine && !at_bound(yk, rk);
        double prk = fr ? rk : 0.0, dk = -mk * prk;
        bool halt = false;
        const int maxcg = 4 * K + 20;
        int it = 0;
        int fl = any_flags(fabs(prk) > qtol ? 2 : 0);
        while ((fl & 2) && !(fl & 4) && it < maxcg) {
            if (k < N) vd[k] = dk;
            if (mine) dc[ik[k]] = (float)dk;
            __syncthreads();
            ++cg_steps;
            ++it;
            // H32 d, fp32.  The matrix is symmetric: thread (r, h) sums H[c][r] d_c over the columns c of its half h, so
            // that the lanes of a warp read consecutive words of row c (no bank conflict, 128 bytes per request) and
            // d_c is the same word for the whole warp.  Two halves: threads 0..255 and 256..511.
            {
                const int r = tid & (kMasterThreads / 2 - 1), h = tid / (kMasterThreads / 2);
                const int q0 = h * ((Kp4 + 1) / 2), q1 = min(Kp4, q0 + (Kp4 + 1) / 2);   // float4s of d of this half
                float acc0 = 0.f, acc1 = 0.f;
                if (r < K) {
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
                if (h == 1 && r < K) hpart2[r] = acc0 + acc1;
                __syncthreads();
                if (h == 0 && r < K) hpart[r] = (acc0 + acc1) + hpart2[r];
            }
            __syncthreads();
            double hdk = 0.0;
            float s5[5] = {0.f, 0.f, 0.f, 0.f, 0.f}, ntl = -CUDART_INF_F;
            if (mine) {
                const int nx = nxl[k], pv = pvl[k];
                const double e1 = nx >= 0 ? (vd[nx] - dk) * rdt[k] : 0.0;
                const double e0 = pv >= 0 ? (dk - vd[pv]) * rdt[pv] : 0.0;
                hdk = 2.0 * (double)hpart[ik[k]] + 2.0 * a.gamma * (e0 - e1);
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
            const int fn = mine && !at_bound(yk, rk);
            prk = fn ? rk : 0.0;
            fl = any_flags(warp >= nv ? 0 : (fn != fr || hit || t == 0.0 ? 1 : 0) | (fabs(prk) > qtol ? 2 : 0) | (halt ? 4 : 0));
            // (only the warps that hold beams know the sums; `halt` and the rest of the loop control travel as flags)
            beta = (fl & 1) || !(s5[2] > 0.f) ? 0.0 : (double)fmaxf(0.f, __fdividef((float)t * (s5[3] + (float)t * s5[4]), s5[2]));
            dk = fn ? -mk * prk + beta * dk : 0.0;
            fr = fn;
        }
        if (k < N) yc[k] = yk;
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

// shared memory of one master block (master_setup's carve-up); k_newton's working blocks lay out a little more
size_t seg_bytes(bool newton) { return kSeg * 4 + (newton ? 2 : 1) * 2 * 8 + 2 * 4; }   // tile, gpart (gpartu), cseg + gseg

size_t master_smem_bytes(int64_t N, int64_t rslots, int64_t cache_segs, int64_t ngroups, bool newton, int64_t ul_cap) {
    const int f1 = newton ? 1 : 0;
    return (size_t)(2 * kGroup * kChunk + (1 + 2 * f1) * kGroup * kSeg + f1 * kGroup * kChunk + (6 + f1) * rslots) * 4   // part2, wbuf (ombuf, ubuf, fl_dw), resident slots
           + (size_t)cache_segs * seg_bytes(newton)                                          // tile and the lists over it
           + (size_t)((13 + 2 * f1) * N + 2 * N + 2 + kMasterWarps + 2 * kMasterWarps * kRedSlots) * 8 + sizeof(Ctl)   // K-vectors (gaccu), recv, red, cred, ctl
           + (size_t)N * 4 * 10 + (size_t)(ngroups * kGroup + 1) * 4          // coef, sk, lo, hi, ik, nx, pv, base, unc, nseg; coff
           + (size_t)ngroups * (kGroup + 1) * 4                               // wst
           + (size_t)((ngroups * kGroup + 63) / 64) * N * 8                   // lmask
           + (size_t)f1 * ((size_t)2 * N * 4 + (kGroup * 4 + 4) * 4 + kGroup * kChunk)   // hm, hv, fl_wc, fl_slot
           + (ul_cap > 0 ? (size_t)ul_cap * 2 + 16 + (size_t)(ngroups * kGroup + 1) * 4 + (size_t)(1 + f1) * N * 8 : 0);   // ul, uoff, gfx (gfxu)
}

// shared memory of k_newton's solving block (newton_solver's carve-up)
// for N beams of which at most K are occupied
size_t solver_smem_bytes(int64_t N, int64_t K) {
    const int64_t Np = ((N + 3) / 4) | 1, Kp = 4 * (((K + 3) / 4) | 1);
    return (size_t)(14 * N + 2 * kMasterWarps * kSolveRed) * 8 + (size_t)6 * N * 4 + 16 + (size_t)4 * Np * 4 +
           (size_t)(kMasterThreads + 2 * kMasterWarps * kCgRow) * 4 + (size_t)Kp * Kp * 4;
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
    if (newton) VMAT_CUDA(p, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_newton, kMasterThreads, cfg->smem));
    else VMAT_CUDA(p, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_master, kMasterThreads, cfg->smem));
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
    cudaFuncAttributes fa0, fa1;
    VMAT_CUDA(p, cudaFuncGetAttributes(&fa0, k_master));
    VMAT_CUDA(p, cudaFuncGetAttributes(&fa1, k_newton));
    VMAT_CUDA(p, cudaFuncSetAttribute(k_master, cudaFuncAttributeMaxDynamicSharedMemorySize, optin - (int)fa0.sharedSizeBytes));
    VMAT_CUDA(p, cudaFuncSetAttribute(k_newton, cudaFuncAttributeMaxDynamicSharedMemorySize, optin - (int)fa1.sharedSizeBytes));
    int rc;
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
            while (kmax > 0 && solver_smem_bytes(p->N, kmax) > budget) --kmax;
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
        if ((rc = dev_alloc(p, (char **)&p->mail, (int64_t)sizeof(Mail) + 4 * p->N))) return rc;
        if ((rc = dev_alloc(p, &p->nsync, 4))) return rc;
        VMAT_CUDA(p, cudaMemsetAsync(p->wn_s, 0, (size_t)p->Sp * 4, p->stream));
        VMAT_CUDA(p, cudaMemsetAsync(p->mail, 0, sizeof(Mail) + 4 * (size_t)p->N, p->stream));
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
    void *args[] = {&a};
    const void *fn = newton ? (const void *)k_newton : (const void *)k_master;
    size_t smem = cfg.smem;
    if (newton && solver_smem_bytes(p->N, k_occ) > smem) smem = solver_smem_bytes(p->N, k_occ);
    VMAT_CUDA(p, cudaLaunchCooperativeKernel(fn, dim3((unsigned)cfg.grid), dim3(kMasterThreads), args, smem, p->stream));
    ++p->launches;
    return VMAT_OK;
}

int launch_master(vmat_plan *p, int trace_it, int warm, int k_occ) {
    return launch_master_impl(p, p->opt.master_max_inner, trace_it, warm, k_occ);
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
