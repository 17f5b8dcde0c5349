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
#include <cstdio>
#include <cstdlib>

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

// Dd[k][.] = fixed-point accumulator as fp32; clears the accumulator; gathers the column's
// statistics (exact integer sums / extrema, hence order free): sum and max of |d_k|, first and
// last chunk with a non-zero entry.  One block = 256 slots = 2 chunks.
__global__ void __launch_bounds__(256)
k_column_finish(unsigned long long *__restrict__ acc, long long Sp, const Sel *__restrict__ sel, int beam,
                double fx_inv, float *__restrict__ Dd, int N, ColStat *__restrict__ colstat,
                uint32_t *__restrict__ touch, int touch_words) {
    pdl_wait();      // the scatter's adds
    const int k = sel ? sel->beam : beam;
    if (k < 0) return;
    __shared__ unsigned long long s_sum[8], s_max[8];
    __shared__ int s_lo[8], s_hi[8];
    const long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    unsigned long long mag = 0ull;
    if (s < Sp) {
        const long long v = (long long)acc[s];
        Dd[((size_t)(s / kChunk) * N + k) * kChunk + (s & (kChunk - 1))] = (float)((double)v * fx_inv);   // chunk-major
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
    int stall_count;
    float Tmax, abmax;
    int max_inner;
    int rslots;                 // > 0: every block keeps z, q, T, alpha, beta of its own slots in shared memory
    int cache_segs;             // capacity of the shared-memory tile of Dd in 512-byte segments
    int ul_cap;                 // capacity of the per-chunk lists of unstaged beams (0: they do not fit, masked loops)
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
#ifdef VMAT_MASTER_PROFILE
__device__ long long g_master_prof[16];
#define PROF_DECL long long pt_ = clock64(), pacc_[16] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0}
#define PROF(i)                           \
    {                                     \
        const long long n_ = clock64();   \
        pacc_[i] += n_ - pt_;             \
        pt_ = n_;                         \
    }
#define PROFW(i, j)                       \
    {                                     \
        const long long n_ = clock64();   \
        pacc_[j] += n_ - pt_;             \
        pacc_[i] += n_ - pt_;             \
        pt_ = n_;                         \
    }
#define PROF_END                                                                  \
    if (blockIdx.x == 0 && threadIdx.x == 0)                                      \
        for (int i_ = 0; i_ < 16; ++i_) g_master_prof[i_] += pacc_[i_];
#define PROFX(j)                          \
    {                                     \
        const long long n_ = clock64();   \
        pacc_[j] += n_ - px_;             \
        px_ = n_;                         \
    }
#define PROFX_START long long px_ = clock64();
#define PROF_PARAM , long long &pt_, long long (&pacc_)[16]
#define PROF_ARG , pt_, pacc_
#else
#define PROF_PARAM
#define PROF_ARG
#define PROFX(j)
#define PROFX_START
#define PROF_DECL
#define PROF(i)
#define PROFW(i, j)
#define PROF_END
#endif

// scalars every thread of the block needs, written by warp 0 (the block's control warp)
struct Ctl {
    double scF, scG, scC, scH;   // fixed-point scales of the pass about to run
    double iF, iG, iC, iH;       // and their inverses
    float tf;               // trial step of the line search
    int state;              // what the block does next (kRunDirection, ...)
    int accepted;           // the last trial was accepted: the z buffers swap roles
    int probe;              // fused mode: the pass about to run does not move (t = 0), it only opens a new direction
};
enum { kRunDirection = 0, kRunTrial = 1, kFinish = 2, kRunFused = 3 };

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
    double *gF, *gFn, *hd, *hdn, *dnx, *gm;   // fused mode, N each: F-part of the gradient, Hessian-vector products
                                              // (accepted / pending), next direction, predicted gradient
    double *gpart, *gpartu;   // 2 per staged segment: partial dots of its two threads with w (and, fused mode, u)
    float *part2, *wbuf, *ubuf, *coef;
    float *rz0, *rz1, *rq, *rq1, *rT, *ral, *rbe;   // resident copies of the block's own slots (a.rslots each), or unused
    float *tile;       // staged 512-byte segments of the block's part of Dd, kSeg floats apart
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
    long long *gfx;    // (when a.ul_cap > 0) fixed-point gradient sums of the unstaged beams: N for w (+ N for u)
    long long *recv;   // the pass's record of grid sums, fetched by the whole block after the barrier
    Ctl *ctl;
};

// chunk handled by this block as member `ch` of its group `g`: chunks are dealt round-robin
__device__ __forceinline__ int chunk_of(int g, int ch) { return (int)blockIdx.x + (g * kGroup + ch) * (int)gridDim.x; }

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
    const int j0 = g * kGroup + chalf, G = (int)gridDim.x;
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
                        (size_t)((int)blockIdx.x + j * (int)gridDim.x) * a.N * (kChunk / 4) + lane;   // the chunk's segments
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
// although several warps add to one beam).  sm.gfx holds N entries for w and, TWO, N more for u.
template <bool TWO>
__device__ __forceinline__ void grad_unstaged_listed(const MasterArgs &a, const Smem &sm, int g, double scG, double scH) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int cs, r, c;
    warp_share(sm, g, warp, cs, r, c);
    if (c == 0) return;
    const int j = g * kGroup + cs, n1 = sm.uoff[j + 1];
    int n = sm.uoff[j] + r;
    if (n >= n1) return;
    const float4 w4 = reinterpret_cast<const float4 *>(sm.wbuf)[cs * kSeg4 + lane];
    float4 u4 = make_float4(0.f, 0.f, 0.f, 0.f);
    if (TWO) u4 = reinterpret_cast<const float4 *>(sm.ubuf)[cs * kSeg4 + lane];
    const float4 *Dd4 = reinterpret_cast<const float4 *>(a.Dd) +
                        (size_t)((int)blockIdx.x + j * (int)gridDim.x) * a.N * (kChunk / 4) + lane;   // the chunk's segments
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
        double dw[8], du[8];
#pragma unroll
        for (int x = 0; x < 8; ++x) {
            dw[x] = (double)((v[x].x * w4.x + v[x].y * w4.y) + (v[x].z * w4.z + v[x].w * w4.w));
            if (TWO) du[x] = (double)((v[x].x * u4.x + v[x].y * u4.y) + (v[x].z * u4.z + v[x].w * u4.w));
        }
        const double rw = warp_sum8(dw, lane);
        double ru = 0.0;
        if (TWO) ru = warp_sum8(du, lane);
        int my_id = -1;
#pragma unroll
        for (int x = 0; x < 8; ++x)
            if (x == mine) my_id = id[x];
        if ((lane & 3) == 0 && my_id >= 0) {
            atomicAdd(reinterpret_cast<unsigned long long *>(sm.gfx) + my_id, (unsigned long long)__double2ll_rn(rw * scG));
            if (TWO)
                atomicAdd(reinterpret_cast<unsigned long long *>(sm.gfx) + a.N + my_id,
                          (unsigned long long)__double2ll_rn(ru * scH));
        }
    }
}

// value[o] = sum_i coef[i] * Dd[sk[i]][slot(o)] for the kGroup*128 slots of group g, o = tid + r*kMasterThreads.
// Staged columns: the two warps of a chunk walk its list of staged segments (every second entry each, beams
// ascending), one float4 of the segment per lane: only segments the columns really touch are visited; the
// columns that are not staged (Ku of them) follow by the same split.  The two partials of a chunk meet in
// shared memory.  The caller must __syncthreads() before sm.part2 is written again.
__device__ __forceinline__ void combine_group(const MasterArgs &a, const Smem &sm, int Ku, int g,
                                              float (&out)[kOutPerThread] PROF_PARAM) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    PROFX_START
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
                                (size_t)((int)blockIdx.x + j * (int)gridDim.x) * a.N * (kChunk / 4) + lane;
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
    PROFX(12)
    __syncthreads();
#pragma unroll
    for (int r = 0; r < kOutPerThread; ++r) {
        const int o = tid + r * kMasterThreads, ch = o >> 7, s = o & (kChunk - 1);
        const int w0 = sm.wst[g * (kGroup + 1) + ch], w1 = sm.wst[g * (kGroup + 1) + ch + 1];
        float v = 0.f;
        for (int w = w0; w < w1; ++w) v += sm.part2[w * kChunk + s];   // the chunk's warps, in order
        out[r] = v;
    }
    PROFX(13)
}

// Gradient products of the staged segments of group g: two threads per segment (alternate float4s), each a plain
// dot of 64 entries with the group's w (TWO: and u) — no exchange between lanes.  Lane partials over 16 products
// in fp32, then fp64.  The partials land in sm.gpart (sm.gpartu), two per segment; grad_total adds them per beam.
template <bool TWO>
__device__ __forceinline__ void grad_staged(const Smem &sm, int g) {
    const int n0 = sm.coff[g * kGroup], n2 = 2 * (sm.coff[(g + 1) * kGroup] - n0);
    const float4 *tile4 = reinterpret_cast<const float4 *>(sm.tile);
    const float4 *wb4 = reinterpret_cast<const float4 *>(sm.wbuf), *ub4 = reinterpret_cast<const float4 *>(sm.ubuf);
    for (int t2 = threadIdx.x; t2 < n2; t2 += kMasterThreads) {
        const int e = sm.gseg[n0 + (t2 >> 1)], hfs = t2 & 1;
        const int s = e & 0xffff, cs = e >> 16;
        const float4 *tp = tile4 + s * kSeg4 + hfs, *wp = wb4 + cs * kSeg4 + hfs, *up = ub4 + cs * kSeg4 + hfs;
        double dw = 0.0, du = 0.0;
#pragma unroll
        for (int blk = 0; blk < 4; ++blk) {
            float4 aw = make_float4(0.f, 0.f, 0.f, 0.f), au = aw;
#pragma unroll
            for (int it = 0; it < 4; ++it) {
                const int x = (blk * 4 + it) * 2;
                const float4 v = tp[x], w = wp[x];
                aw.x = fmaf(v.x, w.x, aw.x);
                aw.y = fmaf(v.y, w.y, aw.y);
                aw.z = fmaf(v.z, w.z, aw.z);
                aw.w = fmaf(v.w, w.w, aw.w);
                if (TWO) {
                    const float4 u = up[x];
                    au.x = fmaf(v.x, u.x, au.x);
                    au.y = fmaf(v.y, u.y, au.y);
                    au.z = fmaf(v.z, u.z, au.z);
                    au.w = fmaf(v.w, u.w, au.w);
                }
            }
            dw += (double)((aw.x + aw.y) + (aw.z + aw.w));
            if (TWO) du += (double)((au.x + au.y) + (au.z + au.w));
        }
        sm.gpart[2 * s + hfs] = dw;
        if (TWO) sm.gpartu[2 * s + hfs] = du;
    }
}

// beam i's total over the block: staged columns add the partials of their segments in chunk order, the others
// the two chunk-half rows of sm.gacc (row0, row0 + 1)
__device__ __forceinline__ double grad_total(const Smem &sm, const double *gp, int i, int N, int row0) {
    const int bs = sm.base[i];
    if (bs == kNoCache) return sm.gacc[row0 * N + i] + sm.gacc[(row0 + 1) * N + i];
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
                                          double scF, double scG, double *red PROF_PARAM) {
    const bool res = a.rslots > 0;
    PROFX_START
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int kpart = warp & (kKSplit - 1), chalf = warp / kKSplit;
    for (int i = tid; i < 2 * a.N; i += kMasterThreads) sm.gacc[i] = 0.0;
    if (a.ul_cap > 0)
        for (int i = tid; i < a.N; i += kMasterThreads) sm.gfx[i] = 0;
    double F = 0.0;
    __syncthreads();
    PROFX(8)
    for (int g = 0; g < ngroups; ++g) {
        float zv[kOutPerThread];
        if (FROM_Y) combine_group(a, sm, Ku, g, zv PROF_ARG);
#pragma unroll
        for (int r = 0; r < kOutPerThread; ++r) {
            const int o = tid + r * kMasterThreads, c = chunk_of(g, o >> 7);
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
        PROFX(9)
        grad_staged<false>(sm, g);
        // columns that are not staged: through the per-chunk lists when they fit; otherwise this warp's half of the
        // group's gradient (4 chunks), and its share of those beams: two beams per step (eight masked loads), lane
        // partials in fp32 (16 products), the warp sum in fp64 to the row of sm.gacc of this chunk half
        if (Ku > 0 && a.ul_cap > 0) {
            grad_unstaged_listed<false>(a, sm, g, scG, 0.0);
        } else if (Ku > 0) {
        float4 w4[kGroup / 2];
#pragma unroll
        for (int h = 0; h < kGroup / 2; ++h) w4[h] = reinterpret_cast<const float4 *>(sm.wbuf)[(2 * h + chalf) * kSeg4 + lane];
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
            double *gacc = sm.gacc + chalf * a.N;      // entries i, i2 of this row are owned by this warp
            if (lane == 0) gacc[i] += r;
            if (lane == 16 && has2) gacc[i2] += r;
        }
        }
        PROFX(10)
        __syncthreads();
    }
    PROFX(11)
    F = block_sum(F, red);
    if (tid == 0) fx_add(rec, F, scF);
    for (int i = tid; i < K; i += kMasterThreads) {
        if (a.ul_cap > 0 && sm.base[i] == kNoCache)   // already in fixed point
            atomicAdd(reinterpret_cast<unsigned long long *>(rec + 2 + i), (unsigned long long)sm.gfx[i]);
        else fx_add(rec + 2 + i, grad_total(sm, sm.gpart, i, a.N, 0), scG);
    }
    PROFX(11)
}

// The pass of the single-barrier iteration (master_mode 1).  For the block's slots, in one sweep:
//   z_new = zsrc + t qsrc (the trial point of the direction in flight; probe: z_new = zsrc), F and w there,
//   q_new = Dc^T d_next (coef holds the next direction), the curvature sum_j omega_j q_new_j^2 of the quadratic
//   piece at z_new, and the block's share of BOTH K-vectors Dc w_new (the true gradient at the trial point) and
//   Dc (omega . q_new) (half the Hessian of F at z_new applied to d_next), so that one grid barrier per inner
//   iteration suffices.  Sums go to the record `rec` in fixed point: F, curvature, grad[0..K), Hd[K..2K).
__device__ __forceinline__ void fused_pass(const MasterArgs &a, const Smem &sm, int K, int Ku, int ngroups, const float *zsrc,
                                           float *zdst, const float *rzsrc, float *rzdst, const float *qsrc,
                                           float *qdst, const float *rqsrc, float *rqdst, float tf, bool probe,
                                           long long *rec, double scF, double scC, double scG, double scH,
                                           double *red) {
    const bool res = a.rslots > 0;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int kpart = warp & (kKSplit - 1), chalf = warp / kKSplit;
#ifdef VMAT_MASTER_PROFILE
    long long pt_ = 0, pacc_[16] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
#endif
    for (int i = tid; i < 4 * a.N; i += kMasterThreads) sm.gacc[i] = 0.0;
    if (a.ul_cap > 0)
        for (int i = tid; i < 2 * a.N; i += kMasterThreads) sm.gfx[i] = 0;
    double F = 0.0, curv = 0.0;
    __syncthreads();
    for (int g = 0; g < ngroups; ++g) {
        float om[kOutPerThread], qv[kOutPerThread];
#pragma unroll
        for (int r = 0; r < kOutPerThread; ++r) {
            const int o = tid + r * kMasterThreads, c = chunk_of(g, o >> 7);
            float wv = 0.f, omv = 0.f;
            if (c < a.nchunks) {
                const size_t s = (size_t)c * kChunk + (o & (kChunk - 1));
                const int ls = g * (kGroup * kChunk) + o;
                float z, Tv, al, be;
                if (res) {
                    z = probe ? rzsrc[ls] : fmaf(tf, rqsrc[ls], rzsrc[ls]);
                    Tv = sm.rT[ls], al = sm.ral[ls], be = sm.rbe[ls];
                    rzdst[ls] = z;
                } else {
                    z = probe ? zsrc[s] : fmaf(tf, qsrc[s], zsrc[s]);
                    Tv = a.T[s], al = a.alpha[s], be = a.beta[s];
                    zdst[s] = z;
                }
                double f;
                penalty(z, Tv, al, be, wv, f);
                F += f;
                omv = z < Tv ? al : (z > Tv ? be : 0.f);
            }
            sm.wbuf[(o >> 7) * kSeg + (o & (kChunk - 1))] = wv;
            om[r] = omv;
        }
        combine_group(a, sm, Ku, g, qv PROF_ARG);   // its barrier also publishes wbuf
#pragma unroll
        for (int r = 0; r < kOutPerThread; ++r) {
            const int o = tid + r * kMasterThreads, c = chunk_of(g, o >> 7);
            if (c < a.nchunks) {
                if (res) rqdst[g * (kGroup * kChunk) + o] = qv[r];
                else qdst[(size_t)c * kChunk + (o & (kChunk - 1))] = qv[r];
            }
            curv += (double)om[r] * (double)qv[r] * (double)qv[r];
            sm.ubuf[(o >> 7) * kSeg + (o & (kChunk - 1))] = om[r] * qv[r];
        }
        __syncthreads();
        grad_staged<true>(sm, g);
        // columns that are not staged: through the per-chunk lists when they fit; otherwise this warp's half of the
        // group (4 chunks) and its share of those beams: two beams per step, each row read once for both products;
        // lane partials in fp32, warp sums in fp64 by one butterfly for all four
        if (Ku > 0 && a.ul_cap > 0) {
            grad_unstaged_listed<true>(a, sm, g, scG, scH);
        } else if (Ku > 0) {
        float4 w4[kGroup / 2], u4[kGroup / 2];
#pragma unroll
        for (int h = 0; h < kGroup / 2; ++h) {
            w4[h] = reinterpret_cast<const float4 *>(sm.wbuf)[(2 * h + chalf) * kSeg4 + lane];
            u4[h] = reinterpret_cast<const float4 *>(sm.ubuf)[(2 * h + chalf) * kSeg4 + lane];
        }
        for (int u = kpart; u < Ku; u += 2 * kKSplit) {
            const bool has2 = u + kKSplit < Ku;
            const int i = sm.unc[u], i2 = has2 ? sm.unc[u + kKSplit] : i;
            float4 v1[kGroup / 2], v2[kGroup / 2];
            load_half(a, sm, i, g, chalf, lane, v1);
            load_half(a, sm, i2, g, chalf, lane, v2);
            float2 w1 = make_float2(0.f, 0.f), w2 = w1, u1 = w1, u2 = w1;
#pragma unroll
            for (int h = 0; h < kGroup / 2; ++h) {
                w1.x = fmaf(v1[h].x, w4[h].x, fmaf(v1[h].y, w4[h].y, w1.x));
                w1.y = fmaf(v1[h].z, w4[h].z, fmaf(v1[h].w, w4[h].w, w1.y));
                w2.x = fmaf(v2[h].x, w4[h].x, fmaf(v2[h].y, w4[h].y, w2.x));
                w2.y = fmaf(v2[h].z, w4[h].z, fmaf(v2[h].w, w4[h].w, w2.y));
                u1.x = fmaf(v1[h].x, u4[h].x, fmaf(v1[h].y, u4[h].y, u1.x));
                u1.y = fmaf(v1[h].z, u4[h].z, fmaf(v1[h].w, u4[h].w, u1.y));
                u2.x = fmaf(v2[h].x, u4[h].x, fmaf(v2[h].y, u4[h].y, u2.x));
                u2.y = fmaf(v2[h].z, u4[h].z, fmaf(v2[h].w, u4[h].w, u2.y));
            }
            const double dw1 = (double)(w1.x + w1.y), dw2 = (double)(w2.x + w2.y);
            const double du1 = (double)(u1.x + u1.y), du2 = (double)(u2.x + u2.y);
            // after the exchange at 16 the lower half-warp carries row 1, the upper row 2; after the exchange at 8
            // the quarters carry (row 1, w), (row 1, u), (row 2, w), (row 2, u)
            const bool up = lane & 16, uq = lane & 8;
            const double rw = (up ? dw2 : dw1) + __shfl_xor_sync(kFull, up ? dw1 : dw2, 16);
            const double ru = (up ? du2 : du1) + __shfl_xor_sync(kFull, up ? du1 : du2, 16);
            double r = (uq ? ru : rw) + __shfl_xor_sync(kFull, uq ? rw : ru, 8);
            r += __shfl_xor_sync(kFull, r, 4);
            r += __shfl_xor_sync(kFull, r, 2);
            r += __shfl_xor_sync(kFull, r, 1);
            double *gw = sm.gacc + chalf * a.N, *gu = sm.gacc + (2 + chalf) * a.N;   // entries owned by this warp
            if (lane == 0) gw[i] += r;
            if (lane == 8) gu[i] += r;
            if (lane == 16 && has2) gw[i2] += r;
            if (lane == 24 && has2) gu[i2] += r;
        }
        }
        __syncthreads();
    }
    F = block_sum(F, red);
    curv = block_sum(curv, red);
    if (tid == 0) {
        fx_add(rec, F, scF);
        fx_add(rec + 1, curv, scC);
    }
    for (int i = tid; i < K; i += kMasterThreads) {
        if (a.ul_cap > 0 && sm.base[i] == kNoCache) {   // already in fixed point
            atomicAdd(reinterpret_cast<unsigned long long *>(rec + 2 + i), (unsigned long long)sm.gfx[i]);
            atomicAdd(reinterpret_cast<unsigned long long *>(rec + 2 + K + i), (unsigned long long)sm.gfx[a.N + i]);
        } else {
            fx_add(rec + 2 + i, grad_total(sm, sm.gpart, i, a.N, 0), scG);
            fx_add(rec + 2 + K + i, grad_total(sm, sm.gpartu, i, a.N, 2), scH);
        }
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
        const double e1 = k + 1 < N ? (v[k + 1] - v[k]) * sm.rdt[k] : 0.0;      // (v_{k+1}-v_k)/dtheta_k
        if (k + 1 < N) s += (v[k + 1] - v[k]) * e1;
        if (want_dG) {
            const double e0 = k > 0 ? (v[k] - v[k - 1]) * sm.rdt[k - 1] : 0.0;
            sm.dG[k] = 2.0 * (e0 - e1);
        }
    }
    return s;
}

template <int MODE>   // 0: two passes and two grid barriers per inner iteration, 1: one fused pass and one barrier
__global__ void __launch_bounds__(kMasterThreads, 1) k_master(const MasterArgs a) {
    extern __shared__ float4 smem_raw[];   // 16-byte aligned: float4 tiles first, then doubles, floats, ints
    const int N = a.N, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    Smem sm;
    constexpr int F1 = MODE == 1 ? 1 : 0;   // what only the single-barrier iteration needs is not laid out in mode 0
    sm.part2 = reinterpret_cast<float *>(smem_raw);
    sm.wbuf = sm.part2 + 2 * kGroup * kChunk;
    sm.ubuf = sm.wbuf + kGroup * kSeg;
    sm.tile = sm.ubuf + F1 * kGroup * kSeg;
    sm.rz0 = sm.tile + (size_t)a.cache_segs * kSeg;
    sm.rz1 = sm.rz0 + a.rslots;
    sm.rq = sm.rz1 + a.rslots;
    sm.rq1 = sm.rq + a.rslots;
    sm.rT = sm.rq1 + F1 * a.rslots;
    sm.ral = sm.rT + a.rslots;
    sm.rbe = sm.ral + a.rslots;
    sm.y = reinterpret_cast<double *>(sm.rbe + a.rslots);
    sm.d = sm.y + N;
    sm.grad = sm.d + N;
    sm.pg = sm.grad + N;
    sm.yn = sm.pg + N;
    sm.gn = sm.yn + N;
    sm.dG = sm.gn + N;
    sm.rdt = sm.dG + N;
    sm.gacc = sm.rdt + N;
    sm.linf = sm.gacc + (2 + 2 * F1) * N;   // gacc: one row per chunk half (and per product in fused mode)
    sm.gF = sm.linf + N;
    sm.gFn = sm.gF + F1 * N;
    sm.hd = sm.gFn + F1 * N;
    sm.hdn = sm.hd + F1 * N;
    sm.dnx = sm.hdn + F1 * N;
    sm.gm = sm.dnx + F1 * N;
    sm.gpart = sm.gm + F1 * N;
    sm.gpartu = sm.gpart + 2 * a.cache_segs;
    const int ngroups = (a.nchunks + (int)gridDim.x * kGroup - 1) / ((int)gridDim.x * kGroup);
    const int W64 = (ngroups * kGroup + 63) >> 6;   // 64-bit words of a column's local chunk mask
    sm.lmask = reinterpret_cast<unsigned long long *>(sm.gpartu + F1 * 2 * a.cache_segs);
    sm.gfx = reinterpret_cast<long long *>(sm.lmask + (size_t)W64 * N);
    double *red = reinterpret_cast<double *>(sm.gfx + (a.ul_cap > 0 ? (1 + F1) * N : 0));
    double *cred = red + kMasterWarps;   // 2 x kMasterWarps x kRedSlots
    sm.recv = reinterpret_cast<long long *>(cred + 2 * kMasterWarps * kRedSlots);
    sm.ctl = reinterpret_cast<Ctl *>(sm.recv + 2 * N + 2);
    sm.coef = reinterpret_cast<float *>(sm.ctl + 1);
    sm.sk = reinterpret_cast<int *>(sm.coef + N);
    sm.lo = sm.sk + N;
    sm.hi = sm.lo + N;
    sm.ik = sm.hi + N;
    sm.base = sm.ik + N;
    sm.unc = sm.base + N;
    sm.cseg = sm.unc + N;
    sm.gseg = sm.cseg + a.cache_segs;
    sm.nseg = sm.gseg + a.cache_segs;
    sm.coff = sm.nseg + N;   // ngroups * kGroup + 1
    sm.wst = sm.coff + ngroups * kGroup + 1;    // ngroups * (kGroup + 1)
    sm.uoff = sm.wst + ngroups * (kGroup + 1);  // like coff, if a.ul_cap > 0
    sm.ul = reinterpret_cast<unsigned short *>(sm.uoff + ngroups * kGroup + 1);   // a.ul_cap 16-bit beam numbers, last array
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
        sm.rdt[k] = k + 1 < N ? 1.0 / (a.theta[k + 1] - a.theta[k]) : 0.0;
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
            const int b = (int)blockIdx.x, Gd_ = (int)gridDim.x;
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
        const int G = (int)gridDim.x, b = (int)blockIdx.x;
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
            else if (chunk_of(g, cs) < a.nchunks) v += 4 * Ku;
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
            const int c = (int)blockIdx.x + (ls >> 7) * (int)gridDim.x;
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
            if (k + 1 < N) {
                const double dv = sm.d[k + 1] - dk;
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

    // ---- single-barrier iteration (MODE 1) ---------------------------------------------------------------
    // State between passes: y (accepted point) with its true gradient grad = gF + gamma dG and projected gradient
    // pg; the direction in flight d with q = Dc^T d in the current q buffer and hd = (Hessian of F at z) d; the
    // trial step t.  make_trial_and_next sets the trial point yn = y + t d, predicts the gradient there on the
    // quadratic piece, gm = gF + t hd + gamma dG(yn) (exact while no voxel changes sides of T_j along the step),
    // and builds from it the NEXT direction dnx (Polak-Ribiere+ on the current face), whose q, curvature and
    // Hessian-vector product the coming pass computes together with the true F and gradient at yn.  Directions
    // therefore rest on a prediction, every step length, acceptance test and stop test on true values.  A probe
    // (pr = 1) is a pass with t = 0 that opens the steepest-descent direction -pg.
    int probe = 0;
    auto make_trial_and_next = [&](int pr) {
        probe = pr;
        if (pr) {
            t = 0.0;
            hit = 0;
        }
        for (int k = tid; k < N; k += CT) {
            const double yk = sm.y[k], dk = sm.d[k];
            double v = pr ? yk : yk + t * dk;
            if (!pr && sm.ik[k] >= 0) {
                if (v < lb || (hit && dk < 0.0 && (yk - lb) / (-dk) <= tmax)) v = lb;
                else if (has_ub && (v > ub || (hit && dk > 0.0 && (ub - yk) / dk <= tmax))) v = ub;
            }
            sm.yn[k] = v;
        }
        ctl_sync(CT);
        double sg[1] = {smooth_part(sm.yn, sm, N, CT, true)}, mx = 0.0;
        ctl_reduce<1>(sg, mx, cred, tog, nw, CT);   // its barrier also publishes dG
        Gn = sg[0];
        double s[3] = {0.0, 0.0, 0.0};
        mx = 0.0;
        for (int k = tid; k < N; k += CT) {
            const int i = sm.ik[k];
            const double gmk = i >= 0 ? sm.gF[k] + t * sm.hd[k] + a.gamma * sm.dG[k] : 0.0;
            const double yk = sm.yn[k], po = sm.pg[k];
            const double pn = (i < 0 || at_bound(yk, gmk)) ? 0.0 : gmk;
            sm.gm[k] = gmk;
            sm.gn[k] = pn;   // scratch until the pass returns the true gradient
            s[0] += pn * (pn - po);
            s[1] += po * po;
            s[2] += ((pn == 0.0) != (po == 0.0)) ? 1.0 : 0.0;
        }
        ctl_reduce<3>(s, mx, cred, tog, nw, CT);
        const bool changed = hit || s[2] > 0.0;
        double bpr = (pr || changed || !(s[1] > 0.0) || s[0] <= 0.0) ? 0.0 : s[0] / s[1];
        double qbn = 0.0;
        for (int pass = 0; pass < 2; ++pass) {
            double s2[2] = {0.0, 0.0};
            mx = 0.0;
            for (int k = tid; k < N; k += CT) {
                const double pn = sm.gn[k], yk = sm.yn[k];
                double dk = -pn + bpr * sm.d[k];
                if (sm.ik[k] < 0 || at_bound(yk, -dk)) dk = 0.0;   // stay feasible
                sm.dnx[k] = dk;
                s2[0] += sm.gm[k] * dk;
                s2[1] += fabs(dk) * sm.linf[k];
            }
            ctl_reduce<2>(s2, mx, cred, tog, nw, CT);
            qbn = s2[1];
            if (s2[0] < 0.0 || bpr == 0.0) break;
            bpr = 0.0;   // the conjugate direction does not descend on the prediction: steepest descent
        }
        set_eval_scales(pr ? yb : yb + t * qb);
        const FxScale sC = fx_scale_for(1.01 * Spd * ab * qbn * qbn, bad);
        const FxScale sH = fx_scale_for(1.01 * ab * qbn * l1max, bad);
        for (int i = tid; i < K; i += CT) sm.coef[i] = (float)sm.dnx[sm.sk[i]];
        if (tid == 0) {
            sm.ctl->scC = sC.scale;
            sm.ctl->iC = sC.inv;
            sm.ctl->scH = sH.scale;
            sm.ctl->iH = sH.inv;
            sm.ctl->tf = (float)t;
            sm.ctl->probe = pr;
        }
    };

    PROF_DECL;
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
    // minus the smoothing term.  The evaluation pass (and its grid barrier) is then not needed.
    const bool warm = MODE == 0 && a.warm && a.gflag[0] == 1 && a.sel->beam >= 0;
    long long *rec = nullptr;
    if (!warm) {
        rec = begin_pass();
        eval_pass<true>(a, sm, K, Ku, ngroups, nullptr, zcur, nullptr, rzcur, 0.f, rec, sm.ctl->scF, sm.ctl->scG, red PROF_ARG);
        cg::this_grid().sync();
        ++ph;
        fetch_record(rec, K + 2);
    } else if (res) {
        for (int ls = tid; ls < a.rslots; ls += kMasterThreads) {
            const int c = (int)blockIdx.x + (ls >> 7) * (int)gridDim.x;
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
            if (MODE == 1) {
                sm.gF[k] = i >= 0 ? (double)sm.recv[2 + i] * iG : 0.0;
                sm.hd[k] = 0.0;
            }
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
        } else if (MODE == 1) {
            make_trial_and_next(1);   // open the steepest-descent direction
            state = bad ? kFinish : kRunFused;
        } else if (!prepare_direction()) state = kFinish;
        if (tid == 0) {
            sm.ctl->state = state;
            sm.ctl->accepted = 0;
        }
    }
    __syncthreads();

    if constexpr (MODE == 1) {
        float *qcur = a.q, *qnext = a.q2, *rqcur = sm.rq, *rqnext = sm.rq1;
        while (sm.ctl->state != kFinish) {
            rec = begin_pass();
            fused_pass(a, sm, K, Ku, ngroups, zcur, znext, rzcur, rznext, qcur, qnext, rqcur, rqnext, sm.ctl->tf,
                       sm.ctl->probe != 0, rec, sm.ctl->scF, sm.ctl->scC, sm.ctl->scG, sm.ctl->scH, red);
            cg::this_grid().sync();
            ++ph;
            fetch_record(rec, 2 * K + 2);
            if (ctl) {
                // the true values at the trial point yn, and what the pass found along the next direction dnx
                const double iG = sm.ctl->iG, iH = sm.ctl->iH;
                const double Fn = (double)sm.recv[0] * sm.ctl->iF + a.F_out;
                const double curvF = (double)sm.recv[1] * sm.ctl->iC;
                double s[1] = {0.0}, pgm = 0.0;
                for (int k = tid; k < N; k += CT) {
                    const int i = sm.ik[k];
                    const double gf = i >= 0 ? (double)sm.recv[2 + i] * iG : 0.0;
                    const double gk = i >= 0 ? gf + a.gamma * sm.dG[k] : 0.0;
                    const double yk = sm.yn[k];
                    const double pn = (i < 0 || at_bound(yk, gk)) ? 0.0 : gk;
                    sm.gFn[k] = gf;
                    sm.gn[k] = gk;
                    sm.hdn[k] = i >= 0 ? 2.0 * (double)sm.recv[2 + K + i] * iH : 0.0;
                    s[0] += gk * sm.d[k];
                    pgm = fmax(pgm, fabs(pn));
                }
                ctl_reduce<1>(s, pgm, cred, tog, nw, CT);
                const double Phin = Fn + a.gamma * Gn;
                // sufficient decrease; below the resolution of Phi accept on the slope instead
                const bool accepted = probe || Phin <= Phi + c1a * t * phi1 ||
                                      (Phin <= Phi + noise * fabs(Phi) && fabs(s[0]) <= 0.9 * fabs(phi1));
                int state = kRunFused;
                if (accepted) {
                    const int was_probe = probe;
                    if (!was_probe) {
                        stall = (Phi - Phin <= stall_threshold(Phin) * fabs(Phi)) ? stall + 1 : 0;
                        F = Fn;
                        Gs = Gn;
                        Phi = Phin;
                        ++inner;
                    }
                    pgmax = pgm;
                    for (int k = tid; k < N; k += CT) {
                        const double yk = sm.yn[k], gk = sm.gn[k];
                        sm.y[k] = yk;
                        sm.grad[k] = gk;
                        sm.gF[k] = sm.gFn[k];
                        sm.hd[k] = sm.hdn[k];
                        sm.pg[k] = (sm.ik[k] < 0 || at_bound(yk, gk)) ? 0.0 : gk;
                        sm.d[k] = sm.dnx[k];
                    }
                    ctl_sync(CT);
                    if (!(pgmax > tol)) state = kFinish;
                    else if (stall >= a.stall_count) {
                        stop = 4;
                        state = kFinish;
                    } else if (inner >= a.max_inner) {
                        stop = 1;
                        state = kFinish;
                    } else {
                        direction_sums();   // slope, bounds, G(d) and the largest feasible step of the new direction
                        if (!(phi1 < 0.0)) {
                            if (was_probe) {
                                stop = 2;
                                state = kFinish;
                            } else make_trial_and_next(1);
                        } else {
                            const double phi2 = 2.0 * curvF + 2.0 * a.gamma * Gd;
                            t = phi2 > 0.0 ? -phi1 / phi2 : (isfinite(tmax) ? tmax : 1.0);
                            hit = 0;
                            if (t >= tmax) {
                                t = tmax;
                                hit = 1;
                            }
                            half = 0;
                            make_trial_and_next(0);
                        }
                    }
                } else {
                    t *= 0.5;
                    hit = 0;
                    ++backtracks;
                    if (++half >= 60) {
                        stop = 3;
                        state = kFinish;
                    } else make_trial_and_next(0);
                }
                if (bad) state = kFinish;
                if (tid == 0) {
                    sm.ctl->state = state;
                    sm.ctl->accepted = accepted ? 1 : 0;
                }
            }
            __syncthreads();
            if (sm.ctl->accepted) {
                float *tmp = zcur;
                zcur = znext;
                znext = tmp;
                tmp = rzcur;
                rzcur = rznext;
                rznext = tmp;
                tmp = qcur;
                qcur = qnext;
                qnext = tmp;
                tmp = rqcur;
                rqcur = rqnext;
                rqnext = tmp;
            }
        }
    }
    if constexpr (MODE == 0)
    while (sm.ctl->state != kFinish) {
        PROF(7)
        // ---- q = Dc^T d and the curvature of the quadratic piece at t = 0 ------------------------------
        rec = begin_pass();
        PROFX_START
        double curv = 0.0;
        for (int g = 0; g < ngroups; ++g) {
            float qv[kOutPerThread];
            combine_group(a, sm, Ku, g, qv PROF_ARG);
#pragma unroll
            for (int r = 0; r < kOutPerThread; ++r) {
                const int o = tid + r * kMasterThreads, c = chunk_of(g, o >> 7);
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
        PROFX(14)
        curv = block_sum(curv, red);
        if (tid == 0) fx_add(rec + 1, curv, sm.ctl->scC);
        PROFX(15)
        PROF(0)
        cg::this_grid().sync();
        PROF(1)
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
        PROF(2)
        // ---- backtracking on the true cost ----------------------------------------------------------------
        while (sm.ctl->state == kRunTrial) {
            rec = begin_pass();
            eval_pass<false>(a, sm, K, Ku, ngroups, zcur, znext, rzcur, rznext, sm.ctl->tf, rec, sm.ctl->scF,
                             sm.ctl->scG, red PROF_ARG);
            PROF(3)
            cg::this_grid().sync();
            PROF(4)
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
                    if (++half >= 60) {
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
            PROF(5)
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
    PROF_END

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
        eval_pass<true>(a, sm, K, Ku, ngroups, nullptr, a.z, nullptr, rzcur, 0.f, rec, sm.ctl->scF, sm.ctl->scG, red PROF_ARG);
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

// shared memory of one master block; mode 1 (single-barrier iteration) lays out more (k_master's carve-up)
size_t seg_bytes(int mode) { return kSeg * 4 + (mode == 1 ? 2 : 1) * 2 * 8 + 2 * 4; }   // tile, gpart (+ gpartu), cseg + gseg

size_t master_smem_bytes(int64_t N, int64_t rslots, int64_t cache_segs, int64_t ngroups, int mode, int64_t ul_cap) {
    const int f1 = mode == 1 ? 1 : 0;
    return (size_t)(2 * kGroup * kChunk + (1 + f1) * kGroup * kSeg + (6 + f1) * rslots) * 4   // part2, wbuf (ubuf), resident slots
           + (size_t)cache_segs * seg_bytes(mode)                                            // tile and the lists over it
           + (size_t)((13 + 8 * f1) * N + 2 * N + 2 + kMasterWarps + 2 * kMasterWarps * kRedSlots) * 8 + sizeof(Ctl)   // K-vectors, recv, red, cred, ctl
           + (size_t)N * 4 * 8 + (size_t)(ngroups * kGroup + 1) * 4           // coef, sk, lo, hi, ik, base, unc, nseg; coff
           + (size_t)ngroups * (kGroup + 1) * 4                               // wst
           + (size_t)((ngroups * kGroup + 63) / 64) * N * 8                   // lmask
           + (ul_cap > 0 ? (size_t)ul_cap * 2 + 16 + (size_t)(ngroups * kGroup + 1) * 4 + (size_t)(1 + f1) * N * 8 : 0);   // ul, uoff, gfx
}

}  // namespace

int master_configure(vmat_plan *p) {
    const int64_t nchunks = p->Sp / kChunk;
    int64_t grid = p->sm_count;                       // one block per SM, chunks dealt round-robin
    if (grid > nchunks) grid = nchunks;
    if (grid < 1) grid = 1;
    p->master_grid = (int)grid;
    // resident slot data (z, z trial, q, T, alpha, beta of a block's own slots) if it fits in 128 KB: on a large
    // support the tile holds a few per cent of the columns whatever its size, while slot data read from L2 / HBM
    // costs every group of every pass a round trip
    const int64_t ngroups = (nchunks + grid * kGroup - 1) / (grid * kGroup);
    int64_t rslots = ngroups * kGroup * kChunk;
    if (rslots * (p->opt.master_mode == 1 ? 7 : 6) * 4 > 128 * 1024) rslots = 0;
    p->master_rslots = (int)rslots;
    // what is left of the SM's opt-in shared memory (minus static use and room for L1) holds the tile of Dd
    int optin = 0;
    VMAT_CUDA(p, cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, p->device));
    const size_t budget = (size_t)optin > 8 * 1024 ? (size_t)optin - 8 * 1024 : 0;
    const int mode = p->opt.master_mode;
    // per-chunk lists of the unstaged beams (one entry per column and local chunk at most) if they fit in 64 KB
    int64_t ul_cap = p->N * ngroups * kGroup;
    if (ul_cap * 2 > 64 * 1024 || p->N > 65535) ul_cap = 0;
    if (getenv("VMAT_MASTER_MASKED_LOOPS")) ul_cap = 0;   // debugging aid: force the fallback path (tests)
    size_t fixed = master_smem_bytes(p->N, rslots, 0, ngroups, mode, ul_cap);
    if (fixed > budget) {
        p->master_rslots = 0;
        fixed = master_smem_bytes(p->N, 0, 0, ngroups, mode, ul_cap);
    }
    if (fixed > budget) {
        ul_cap = 0;
        fixed = master_smem_bytes(p->N, 0, 0, ngroups, mode, 0);
    }
    p->master_ul_cap = (int)ul_cap;
    if (fixed > budget) return fail(p, VMAT_EINVAL, "n_beams too large for the master kernel's shared memory");
    p->master_cache_segs = (int)((budget - fixed) / seg_bytes(mode));
    if (p->master_cache_segs > 65535 || ngroups * kGroup > 32767) p->master_cache_segs = 0;   // 16-bit fields of the lists
#ifdef VMAT_MASTER_PROFILE
    if (getenv("VMAT_NO_TILE")) p->master_cache_segs = 0;
    fprintf(stderr, "master: grid %d smem fixed %zu cache_segs %d rslots %d\n", p->master_grid, fixed, p->master_cache_segs, p->master_rslots);
#endif
    p->master_smem = master_smem_bytes(p->N, p->master_rslots, p->master_cache_segs, ngroups, mode, ul_cap);
    VMAT_CUDA(p, cudaFuncSetAttribute(k_master<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p->master_smem));
    VMAT_CUDA(p, cudaFuncSetAttribute(k_master<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p->master_smem));
    int per_sm = 0, per_sm1 = 0;
    VMAT_CUDA(p, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_master<0>, kMasterThreads, p->master_smem));
    VMAT_CUDA(p, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm1, k_master<1>, kMasterThreads, p->master_smem));
    if (per_sm1 < per_sm) per_sm = per_sm1;
    if (per_sm < 1) return fail(p, VMAT_ECUDA, "master kernel does not fit on an SM");
    int rc;
    if ((rc = dev_alloc(p, &p->accbuf, 3 * kSumGroups * (2 * p->N + 2)))) return rc;
    if ((rc = dev_alloc(p, &p->phase, 2))) return rc;
    if ((rc = dev_alloc(p, &p->mcount, 2))) return rc;
    if ((rc = dev_alloc(p, &p->gsave, p->N))) return rc;
    if ((rc = dev_alloc(p, &p->gflag, 1))) return rc;
    VMAT_CUDA(p, cudaMemsetAsync(p->gflag, 0, 4, p->stream));
    VMAT_CUDA(p, cudaMemsetAsync(p->mcount, 0, 16, p->stream));
    if ((rc = dev_alloc(p, &p->colstat, p->N))) return rc;
    p->touch_words = (int)((nchunks + 31) / 32);
    if ((rc = dev_alloc(p, &p->col_touch, p->N * p->touch_words))) return rc;
    VMAT_CUDA(p, cudaMemsetAsync(p->col_touch, 0, (size_t)p->N * p->touch_words * 4, p->stream));
    if ((rc = dev_alloc(p, &p->vbounds, 2))) return rc;
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
    return VMAT_OK;
}

int launch_column_build(vmat_plan *p, int beam) {
    const Sel *sel = beam < 0 ? p->sel : nullptr;
    const unsigned blocks = (unsigned)((p->RC + 7) / 8);
    VMAT_CUDA(p, launch_pdl(k_column_scatter, dim3(blocks), dim3(256), p->stream, p->rowq, p->val4, p->col4, sel, beam, p->left,
                            p->right, (int)p->R, (int)p->C, p->fx_scale, p->acc, p->colstat, p->col_touch, p->touch_words));
    VMAT_CUDA(p, launch_pdl(k_column_finish, dim3((unsigned)((p->Sp + 255) / 256)), dim3(256), p->stream, p->acc,
                            (long long)p->Sp, sel, beam, p->fx_inv, p->Dd, (int)p->N, p->colstat, p->col_touch,
                            p->touch_words));
    p->launches += 2;
    VMAT_CUDA(p, cudaGetLastError());
    return VMAT_OK;
}

static int launch_master_impl(vmat_plan *p, int max_inner, int trace_it, int warm) {
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
    a.lb = p->y_min;
    a.ub = p->y_max;
    a.max_inner = max_inner;
    a.rslots = p->master_rslots;
    a.cache_segs = p->master_cache_segs;
    a.ul_cap = p->master_ul_cap;
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
    void *args[] = {&a};
    const void *fn = p->opt.master_mode == 1 ? (const void *)k_master<1> : (const void *)k_master<0>;
    VMAT_CUDA(p, cudaLaunchCooperativeKernel(fn, dim3((unsigned)p->master_grid), dim3(kMasterThreads), args,
                                             p->master_smem, p->stream));
    ++p->launches;
    return VMAT_OK;
}

int launch_master(vmat_plan *p, int trace_it, int warm) {
    return launch_master_impl(p, p->opt.master_max_inner, trace_it, warm);
}

// steps (a)+(b) alone: the master kernel's evaluation pass with no iteration allowed
int launch_dose_grad(vmat_plan *p) { return launch_master_impl(p, 0, -1, 0); }

#ifdef VMAT_MASTER_PROFILE
extern "C" void vmat_debug_master_prof(long long out[16], int reset) {
    cudaMemcpyFromSymbol(out, g_master_prof, sizeof(long long) * 16);
    if (reset) {
        long long z[16] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
        cudaMemcpyToSymbol(g_master_prof, z, sizeof(z));
    }
}
#endif

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
