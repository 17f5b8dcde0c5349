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
    launch_variant<16, 4>(p, w_s, g, n_free);
    ++p->launches;
    VMAT_CUDA(p, cudaGetLastError());
    return VMAT_OK;
}

}  // namespace vmat
