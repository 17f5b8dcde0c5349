// vmat_master_common.cuh — what the two master kernels share (k_master in vmat_master.cu, k_newton in vmat_newton.cu):
// the kernel arguments, the carve-up of a block's shared memory (master_setup and its host twin master_smem_bytes),
// the staged / listed / masked products with the aperture-dose columns, the penalty, the evaluation pass of mode 0,
// the fixed-point sums and the reductions of the control group.  Device code only, all of it inlined into the kernels
// (no relocatable device code); DESIGN.md sections 6 and 7.
#pragma once

#include <math_constants.h>

#include <climits>
#include <cmath>

#include "vmat_internal.cuh"

namespace vmat {

constexpr unsigned kFull = 0xffffffffu;

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

// shared memory of one master block (master_setup's carve-up); k_newton's working blocks lay out a little more
inline size_t seg_bytes(bool newton) { return kSeg * 4 + (newton ? 2 : 1) * 2 * 8 + 2 * 4; }   // tile, gpart (gpartu), cseg + gseg

inline size_t master_smem_bytes(int64_t N, int64_t rslots, int64_t cache_segs, int64_t ngroups, bool newton, int64_t ul_cap) {
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

// ---- hooks into vmat_newton.cu for the host side of the master (vmat_master.cu) --------------------------------
size_t newton_solver_smem_bytes(int64_t N, int64_t K);   // shared memory of the solving block: N beams, at most K occupied
size_t newton_mail_bytes(int64_t N);                      // the message of the solving block to the working blocks
int newton_prepare_kernel(vmat_plan *p, int optin);       // opt in to the device's maximum of dynamic shared memory
int newton_blocks_per_sm(vmat_plan *p, size_t smem, int *per_sm);
int newton_launch(vmat_plan *p, const MasterArgs &a, int grid, size_t smem);

}  // namespace vmat
