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

constexpr int kPriceWarps = 8;

// One warp per beamlet.  UNROLL quads per lane are loaded before any gather is issued.
template <int UNROLL>
__global__ void __launch_bounds__(kPriceWarps * 32)
k_price_spmv_warp(const uint32_t *__restrict__ rowq, const float4 *__restrict__ val4, const int4 *__restrict__ col4,
                  const float *__restrict__ w, const uint8_t *__restrict__ occ, int RC, long long B,
                  float *__restrict__ g) {
    const int lane = threadIdx.x & 31;
    const long long row = (long long)blockIdx.x * kPriceWarps + (threadIdx.x >> 5);
    if (row >= B) return;
    if (occ[row / RC]) {
        if (lane == 0) g[row] = 0.f;
        return;
    }
    const uint32_t a = rowq[row], b = rowq[row + 1];
    float acc = 0.f;
    for (uint32_t q = a + lane; q < b; q += 32 * UNROLL) {
        float4 v[UNROLL];
        int4 c[UNROLL];
#pragma unroll
        for (int u = 0; u < UNROLL; ++u) {
            if (q + 32 * u < b) {
                v[u] = ld_stream_f4(val4 + q + 32 * u);
                c[u] = ld_stream_i4(col4 + q + 32 * u);
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
    for (int o = 16; o; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if (lane == 0) g[row] = acc;
}

}  // namespace

int build_chunk_table(vmat_plan *p, const std::vector<uint32_t> &h_rowq) {
    (void)p;
    (void)h_rowq;
    return VMAT_OK;
}

int launch_price_spmv(vmat_plan *p, const float *w_s, float *g) {
    if (p->B == 0) return VMAT_OK;
    const unsigned blocks = (unsigned)((p->B + kPriceWarps - 1) / kPriceWarps);
    k_price_spmv_warp<2><<<blocks, kPriceWarps * 32, 0, p->stream>>>(p->rowq, p->val4, p->col4, w_s, p->occ, (int)p->RC,
                                                                      (long long)p->B, g);
    ++p->launches;
    VMAT_CUDA(p, cudaGetLastError());
    return VMAT_OK;
}

}  // namespace vmat
