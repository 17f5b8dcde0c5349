// vmat_price.cu — step (c): beamlet prices g_i = sum_j D_ij w_j ("By checking the
// KKT optimality conditions, we can obtain the 'price' for each beamlet") for every beamlet of
// every un-occupied beam; 0 at occupied beams.
//
// D is the padded beamlet-major CSR in slot space (vmat_layout.cu): row i owns quads
// [rowq[i], rowq[i+1]) of val4/col4, 16-byte aligned, so a warp streams a row with one LDG.128 of
// values and one of indices per lane and iteration, and gathers w (|support| floats, L1/L2
// resident) four at a time.  HBM-bound: 8 bytes per stored entry, 2 flops.
#include "vmat_internal.cuh"

namespace vmat {

namespace {

__device__ __forceinline__ float4 ld_stream_f4(const float4 *ptr) {
    float4 r;
    asm volatile("ld.global.nc.L1::no_allocate.L2::128B.v4.f32 {%0,%1,%2,%3}, [%4];"
                 : "=f"(r.x), "=f"(r.y), "=f"(r.z), "=f"(r.w)
                 : "l"(ptr));
    return r;
}
__device__ __forceinline__ int4 ld_stream_i4(const int4 *ptr) {
    int4 r;
    asm volatile("ld.global.nc.L1::no_allocate.L2::128B.v4.s32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
                 : "l"(ptr));
    return r;
}

// Threads per block: 256 for long launches; 128 once a launch is short (its tail, the last blocks of the grid
// draining on a few SMs, weighs more the shorter the launch: measured 15.0 against 15.3 ms of pricing per
// configs[1] plan with 128, 334 against 332 ms on configs[4] when 128 is used throughout).
constexpr int kPriceThreadsLong = 256, kPriceThreadsShort = 128;
constexpr long long kShortLaunchRows = 600000;

// One group of LANES lanes (a warp or half a warp) per beamlet; UNROLL quads per lane are loaded
// before any gather is issued.  The grid covers only the un-occupied beams: block b works on beam
// free_list[b / blocks_per_beam] (ascending list kept current by the leaf search's commit), so a
// launch late in the plan is as short as the rows it has to stream.
template <int LANES, int UNROLL, int kPriceThreads>
__global__ void __launch_bounds__(kPriceThreads)
k_price_spmv(const uint32_t *__restrict__ rowq, const float4 *__restrict__ val4, const int4 *__restrict__ col4,
             const float *__restrict__ w, const int32_t *__restrict__ free_list, int blocks_per_beam, int RC,
             float *__restrict__ g) {
    pdl_trigger();   // the leaf search may be scheduled while this grid drains; it waits for g itself
    constexpr int kRowsPerBlock = kPriceThreads / LANES;
    const int lane = threadIdx.x & (LANES - 1);
    const int beam = free_list[blockIdx.x / blocks_per_beam];
    const int local = (blockIdx.x % blocks_per_beam) * kRowsPerBlock + threadIdx.x / LANES;
    if (local >= RC) return;
    const long long row = (long long)beam * RC + local;
    const uint32_t a = rowq[row], b = rowq[row + 1];
    float acc = 0.f;
    for (uint32_t q = a + lane; q < b; q += LANES * UNROLL) {
        float4 v[UNROLL];
        int4 c[UNROLL];
#pragma unroll
        for (int u = 0; u < UNROLL; ++u) {
            if (q + LANES * u < b) {
                v[u] = ld_stream_f4(val4 + q + LANES * u);
                c[u] = ld_stream_i4(col4 + q + LANES * u);
            } else {
                v[u] = make_float4(0.f, 0.f, 0.f, 0.f);
                c[u] = make_int4(0, 0, 0, 0);
            }
        }
#pragma unroll
        for (int u = 0; u < UNROLL; ++u) {
            acc = fmaf(v[u].x, __ldg(w + c[u].x), acc);
            acc = fmaf(v[u].y, __ldg(w + c[u].y), acc);
            acc = fmaf(v[u].z, __ldg(w + c[u].z), acc);
            acc = fmaf(v[u].w, __ldg(w + c[u].w), acc);
        }
    }
#pragma unroll
    for (int o = LANES / 2; o; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if (lane == 0) g[row] = acc;
}

__device__ __forceinline__ uint2 ld_stream_u2(const uint2 *ptr) {
    uint2 r;
    asm volatile("ld.global.nc.L1::no_allocate.v2.u32 {%0,%1}, [%2];" : "=r"(r.x), "=r"(r.y) : "l"(ptr));
    return r;
}

// d_format 1 ("compressed voxel indices to cut pricing bytes below 8 B/nnz — reported as a separate
// format"): the same product from the pair copy of D (vmat_layout.cu): a unit is an aligned pair of slots with the
// row's two values there, a group is four units = 32 bytes of values + 8 bytes of 16-bit pair ids + 1 byte of panel.
// With 8 bytes per entry the product runs at the HBM roof and, at the same time, close to the rate at which an SM
// gathers w one word at a time; the pair format lowers both: 6.35 / 5.86 bytes per entry on configs[1] / [2], and
// 0.62 / 0.57 eight-byte gathers per entry instead of one four-byte gather.  (Measured first: 16-bit ids alone, 6.1
// bytes per entry with one gather per entry, are no faster than the fp32 layout, and one entry per lane and load,
// which quarters the cache lines a warp-wide gather touches, is 2.2 times slower: the load instructions count.)
// Same row-to-lanes mapping as k_price_spmv; UNROLL groups per lane in flight before the first gather.
template <int LANES, int UNROLL, int kPriceThreads>
__global__ void __launch_bounds__(kPriceThreads)
k_price_spmv_pairs(const uint32_t *__restrict__ rowo, const float4 *__restrict__ va, const float4 *__restrict__ vb,
                   const uint2 *__restrict__ ix, const uint8_t *__restrict__ pan, const float2 *__restrict__ w2,
                   const int32_t *__restrict__ free_list, int blocks_per_beam, int RC, float *__restrict__ g) {
    pdl_trigger();
    constexpr int kRowsPerBlock = kPriceThreads / LANES;
    const int lane = threadIdx.x & (LANES - 1);
    const int beam = free_list[blockIdx.x / blocks_per_beam];
    const int local = (blockIdx.x % blocks_per_beam) * kRowsPerBlock + threadIdx.x / LANES;
    if (local >= RC) return;
    const long long row = (long long)beam * RC + local;
    const uint32_t a = rowo[row], b = rowo[row + 1];
    float acc0 = 0.f, acc1 = 0.f;
    for (uint32_t q = a + lane; q < b; q += LANES * UNROLL) {
        float4 x[UNROLL], y[UNROLL];
        uint2 c[UNROLL];
        unsigned pb[UNROLL];
#pragma unroll
        for (int u = 0; u < UNROLL; ++u) {
            if (q + LANES * u < b) {
                x[u] = ld_stream_f4(va + q + LANES * u);
                y[u] = ld_stream_f4(vb + q + LANES * u);
                c[u] = ld_stream_u2(ix + q + LANES * u);
                pb[u] = __ldg(pan + q + LANES * u);
            } else {
                x[u] = y[u] = make_float4(0.f, 0.f, 0.f, 0.f);
                c[u] = make_uint2(0u, 0u);
                pb[u] = 0u;
            }
        }
#pragma unroll
        for (int u = 0; u < UNROLL; ++u) {
            const float2 *wp = w2 + ((size_t)pb[u] << 16);
            const float2 w0 = __ldg(wp + (c[u].x & 0xffffu)), w1 = __ldg(wp + (c[u].x >> 16));
            const float2 w2v = __ldg(wp + (c[u].y & 0xffffu)), w3 = __ldg(wp + (c[u].y >> 16));
            acc0 = fmaf(x[u].x, w0.x, acc0);
            acc1 = fmaf(x[u].y, w0.y, acc1);
            acc0 = fmaf(x[u].z, w1.x, acc0);
            acc1 = fmaf(x[u].w, w1.y, acc1);
            acc0 = fmaf(y[u].x, w2v.x, acc0);
            acc1 = fmaf(y[u].y, w2v.y, acc1);
            acc0 = fmaf(y[u].z, w3.x, acc0);
            acc1 = fmaf(y[u].w, w3.y, acc1);
        }
    }
    float acc = acc0 + acc1;
#pragma unroll
    for (int o = LANES / 2; o; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if (lane == 0) g[row] = acc;
}

// ascending list of the un-occupied beams (after vmat_set_plan; the search keeps it current afterwards)
__global__ void k_free_list(const uint8_t *__restrict__ occ, int N, int32_t *__restrict__ free_list) {
    int base = 0;
    const int lane = threadIdx.x;
    for (int k0 = 0; k0 < N; k0 += 32) {
        const int k = k0 + lane;
        const bool f = k < N && !occ[k];
        const unsigned m = __ballot_sync(0xffffffffu, f);
        if (f) free_list[base + __popc(m & ((1u << lane) - 1u))] = k;
        base += __popc(m);
    }
}

template <int LANES, int UNROLL, int THREADS>
void launch_sized(vmat_plan *p, const float *w_s, float *g, int n_free) {
    const int rows_per_block = THREADS / LANES;
    const int bpb = (int)((p->RC + rows_per_block - 1) / rows_per_block);
    k_price_spmv<LANES, UNROLL, THREADS><<<(unsigned)(n_free * bpb), THREADS, 0, p->stream>>>(
        p->rowq, p->val4, p->col4, w_s, p->free_list, bpb, (int)p->RC, g);
}

template <int LANES, int UNROLL, int THREADS>
void launch_sized_pairs(vmat_plan *p, const float *w_s, float *g, int n_free) {
    const int rows_per_block = THREADS / LANES;
    const int bpb = (int)((p->RC + rows_per_block - 1) / rows_per_block);
    k_price_spmv_pairs<LANES, UNROLL, THREADS><<<(unsigned)(n_free * bpb), THREADS, 0, p->stream>>>(
        p->pr_rowo, p->pr_va, p->pr_vb, p->pr_ix, p->pr_pan, reinterpret_cast<const float2 *>(w_s), p->free_list, bpb,
        (int)p->RC, g);
}

template <int LANES, int UNROLL>
void launch_variant(vmat_plan *p, const float *w_s, float *g, int n_free) {
    if ((long long)n_free * p->RC <= kShortLaunchRows) launch_sized<LANES, UNROLL, kPriceThreadsShort>(p, w_s, g, n_free);
    else launch_sized<LANES, UNROLL, kPriceThreadsLong>(p, w_s, g, n_free);
}

}  // namespace

int launch_free_list(vmat_plan *p) {
    k_free_list<<<1, 32, 0, p->stream>>>(p->occ, (int)p->N, p->free_list);
    ++p->launches;
    VMAT_CUDA(p, cudaGetLastError());
    return VMAT_OK;
}

// g_i for the beamlets of the n_free un-occupied beams listed in p->free_list; other entries of g untouched
int launch_price_spmv(vmat_plan *p, const float *w_s, float *g, int n_free) {
    if (p->B == 0 || n_free <= 0) return VMAT_OK;
    // 16 lanes per beamlet, 4 x 16-byte loads of values and of indices in flight per lane: the best of the five
    // lanes x loads variants measured in round 1 (table of rejected variants)
    if (p->opt.d_format == 1) {
        if ((long long)n_free * p->RC <= kShortLaunchRows) launch_sized_pairs<16, 2, kPriceThreadsShort>(p, w_s, g, n_free);
        else launch_sized_pairs<16, 2, kPriceThreadsLong>(p, w_s, g, n_free);
    } else launch_variant<16, 4>(p, w_s, g, n_free);
    ++p->launches;
    VMAT_CUDA(p, cudaGetLastError());
    return VMAT_OK;
}

}  // namespace vmat
