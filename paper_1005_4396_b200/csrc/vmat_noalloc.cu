// vmat_noalloc.cu — vmat_penalty_noalloc: step (b) (Eq. 1: the one-sided quadratic penalty F(z) and its
// gradient w = dF/dz) on a caller's dose vector, for callers that may not allocate (CUDA graph capture, serving loops).
// A variant of k_dose_finish (vmat_dose.cu): the same per-voxel arithmetic and the same two-level sum of F, but the
// per-block partial sums and the ticket of the "last block adds them" hand-over live in a file-scope device array
// instead of plan memory.  Nothing here calls cudaMalloc / cudaFree or a library routine that allocates.
#include <cuda_runtime.h>

#include <mutex>
#include <string>

#include "vmat.h"
#include "vmat_internal.cuh"

namespace vmat {
namespace {

constexpr int kNaThreads = 256;
constexpr int kNaPerThread = 8;                                   // voxels per thread
constexpr int kNaPerBlock = kNaThreads * kNaPerThread;            // 2048 voxels per block
constexpr long long kNaMaxBlocks = VMAT_NOALLOC_MAX_VOXELS / kNaPerBlock;
constexpr int kNaTicketDoubles = 32;                              // 256 bytes of their own for the ticket
static_assert(VMAT_NOALLOC_MAX_VOXELS % kNaPerBlock == 0, "the maximum is a whole number of blocks");

// The scratch: kNaMaxBlocks partial sums of F, then 256 bytes whose first word is the ticket.  64 KB + 256 B, held by
// every GPU that loads the library until the process exits.  In HOST code this name is a stand-in, not a device
// address: the host gets the address from cudaGetSymbolAddress (scratch_of below), once per device.
static __device__ __align__(256) double g_na_scratch[kNaMaxBlocks + kNaTicketDoubles];

__global__ void __launch_bounds__(kNaThreads)
k_penalty_noalloc(const float *__restrict__ z, const float *__restrict__ T, const float *__restrict__ alpha,
                  const float *__restrict__ beta, long long n, float *__restrict__ w, double *__restrict__ F_out,
                  double *__restrict__ scratch) {
    __shared__ double s_sum[kNaThreads];
    __shared__ int s_last;
    double *partF = scratch;
    unsigned int *ticket = reinterpret_cast<unsigned int *>(scratch + kNaMaxBlocks);
    const long long base = (long long)blockIdx.x * kNaPerBlock + threadIdx.x;
    double F = 0.0;
#pragma unroll
    for (int r = 0; r < kNaPerThread; ++r) {      // fixed order within the thread
        const long long s = base + (long long)r * kNaThreads;
        if (s < n) {
            const float zv = z[s], t = T[s], al = alpha[s], be = beta[s];
            const float under = fmaxf(0.f, t - zv), over = fmaxf(0.f, zv - t);
            if (w) w[s] = -2.f * al * under + 2.f * be * over;                             // Eq. 1, derivative
            F += (double)al * (double)under * (double)under + (double)be * (double)over * (double)over;
        }
    }
#pragma unroll
    for (int o = 16; o; o >>= 1) F += __shfl_xor_sync(0xffffffffu, F, o);
    if ((threadIdx.x & 31) == 0) s_sum[threadIdx.x >> 5] = F;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int i = 1; i < kNaThreads / 32; ++i) F += s_sum[i];
        partF[blockIdx.x] = F;
        __threadfence();
        s_last = atomicAdd(ticket, 1u) == gridDim.x - 1u;
    }
    __syncthreads();
    if (!s_last) return;
    // the block that finishes last adds the partials in index order: the sum does not depend on the schedule
    __threadfence();
    double f = 0.0;
    for (int i = threadIdx.x; i < (int)gridDim.x; i += kNaThreads) f += __ldcg(partF + i);
    s_sum[threadIdx.x] = f;
    __syncthreads();
    for (int o = kNaThreads / 2; o; o >>= 1) {
        if (threadIdx.x < o) s_sum[threadIdx.x] += s_sum[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        if (F_out) *F_out = s_sum[0];
        *ticket = 0u;   // ready for the next call
    }
}

// device address of the scratch, looked up once per device with that device current
constexpr int kNaMaxDevices = 64;
std::mutex g_na_mutex;
double *g_na_ptr[kNaMaxDevices] = {};

int scratch_of(int device, double **out) {
    std::lock_guard<std::mutex> lock(g_na_mutex);
    if (!g_na_ptr[device]) {
        int cur = -1;
        cudaError_t e = cudaGetDevice(&cur);
        if (e != cudaSuccess) return cuda_fail(nullptr, e, "cudaGetDevice");
        if (cur != device) return fail(nullptr, VMAT_EINVAL, "vmat_penalty_noalloc: the device of the buffers is not the current device");
        double *ptr = nullptr;
        e = cudaGetSymbolAddress((void **)&ptr, g_na_scratch);
        if (e != cudaSuccess) return cuda_fail(nullptr, e, "cudaGetSymbolAddress(g_na_scratch)");
        if (!ptr) return fail(nullptr, VMAT_ECUDA, "vmat_penalty_noalloc: cudaGetSymbolAddress returned NULL");
        g_na_ptr[device] = ptr;
    }
    *out = g_na_ptr[device];
    return VMAT_OK;
}

}  // namespace
}  // namespace vmat

using namespace vmat;

extern "C" int vmat_penalty_noalloc(const float *z_dev, const float *T_dev, const float *alpha_dev, const float *beta_dev,
                                    int64_t n_voxels, float *w_dev, double *F_dev, void *cuda_stream) {
    if (n_voxels < 0) return fail(nullptr, VMAT_EINVAL, "vmat_penalty_noalloc: n_voxels must be >= 0");
    if (n_voxels > (int64_t)VMAT_NOALLOC_MAX_VOXELS)
        return fail(nullptr, VMAT_EINVAL, "vmat_penalty_noalloc: n_voxels = " + std::to_string(n_voxels) +
                                              " exceeds VMAT_NOALLOC_MAX_VOXELS = " + std::to_string((long long)VMAT_NOALLOC_MAX_VOXELS) +
                                              " (the fixed scratch holds one partial sum per 2048 voxels)");
    if (n_voxels > 0 && (!z_dev || !T_dev || !alpha_dev || !beta_dev))
        return fail(nullptr, VMAT_EINVAL, "vmat_penalty_noalloc: z_dev, T_dev, alpha_dev, beta_dev must not be NULL");
    if (!w_dev && !F_dev) return fail(nullptr, VMAT_EINVAL, "vmat_penalty_noalloc: w_dev and F_dev are both NULL");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int device = -1;
    cudaError_t e = cudaGetDevice(&device);
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "cudaGetDevice");
    if (device < 0 || device >= kNaMaxDevices) return fail(nullptr, VMAT_EINVAL, "vmat_penalty_noalloc: device ordinal out of range");
    if (n_voxels > 0) {   // the buffers must live on the current device: the scratch used is that device's copy
        cudaPointerAttributes pa;
        e = cudaPointerGetAttributes(&pa, z_dev);
        if (e != cudaSuccess) return cuda_fail(nullptr, e, "cudaPointerGetAttributes(z_dev)");
        if ((pa.type != cudaMemoryTypeDevice && pa.type != cudaMemoryTypeManaged) || (pa.type == cudaMemoryTypeDevice && pa.device != device))
            return fail(nullptr, VMAT_EINVAL, "vmat_penalty_noalloc: z_dev is not memory of the current device");
    }
    double *scratch = nullptr;
    int rc = scratch_of(device, &scratch);
    if (rc) return rc;
    if (n_voxels == 0) {   // the empty sum
        if (F_dev) {
            e = cudaMemsetAsync(F_dev, 0, sizeof(double), st);
            if (e != cudaSuccess) return cuda_fail(nullptr, e, "cudaMemsetAsync(F_dev)");
        }
        return VMAT_OK;
    }
    // The array keeps whatever the last call left.  The partial sums are all rewritten before they are read; the ticket
    // must start at zero, and a call that was torn down half-way would leave it otherwise: clear it, in stream order.
    e = cudaMemsetAsync(scratch + kNaMaxBlocks, 0, 256, st);
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "cudaMemsetAsync(ticket)");
    const unsigned blocks = (unsigned)((n_voxels + kNaPerBlock - 1) / kNaPerBlock);
    k_penalty_noalloc<<<blocks, kNaThreads, 0, st>>>(z_dev, T_dev, alpha_dev, beta_dev, (long long)n_voxels, w_dev, F_dev, scratch);
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "k_penalty_noalloc launch");
    return VMAT_OK;
}
