// vmat_engine.cu — dose-deposition matrix D on the device.
//
// "We calculate D_ij's using our in-house dose calculation engine implemented on a ... GPU" (ref 17, a
// finite-size pencil-beam engine: another paper, not available).  This is the stand-in SURVEY.md 8f #3 asks for: the
// ray / Gaussian / exponential model of BASELINE.json:configs evaluated on the GPU, so that the stress phantom's
// 1.5e9 entries are built in HBM in a fraction of a second instead of being generated on the host and uploaded.  It
// makes INPUT, none of the method's arithmetic; the model is the one DESIGN.md section 5 states:
//   parallel rays in the axial plane, gantry axis = grid z through the grid centre, beam k at theta_k = k 360/N degrees
//   travels along d = (cos, sin, 0), leaf columns run along u = (-sin, cos, 0), leaf rows stack along z; beamlet
//   (k, r, c) is the ray through a_c u + b_r zhat; a voxel centre p inside the body cylinder (radius Rb) at lateral
//   position a = p.u, along-beam position t = p.d has depth = t + sqrt(Rb^2 - a^2) and
//     D = exp(-mu depth) exp(-rho^2 / 2 sigma^2) (1 + noise U(-1,1)),  rho^2 = (a - a_c)^2 + (z - b_r)^2 <= (4.5 sigma)^2,
//   entries below cutoff x (row maximum) dropped, U a counter-based hash of (seed, beamlet, voxel).
// One warp per beamlet: the lanes take the (slice, voxel row) pairs the kernel's support meets, 32 at a time, and walk
// the few voxels of their row; a first sweep finds the row maximum, a second counts (or writes, in voxel order) what
// clears the cutoff.  Double precision throughout, values rounded to fp32 at the end, as the host generator does; exp,
// sin and cos differ from the host's by an ulp here and there, so a handful of entries at the cutoff may differ.
#include <math_constants.h>

#include "vmat_internal.cuh"

namespace vmat {

namespace {

__device__ __forceinline__ unsigned long long mix64(unsigned long long x) {   // splitmix64 finaliser
    x += 0x9E3779B97F4A7C15ull;
    x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ull;
    x = (x ^ (x >> 27)) * 0x94D049BB133111EBull;
    return x ^ (x >> 31);
}
// uniform in (-1, 1), a pure function of (seed, a, b)
__device__ __forceinline__ double hash_u11(unsigned long long seed, unsigned long long a, unsigned long long b) {
    const unsigned long long h = mix64(mix64(seed ^ mix64(a)) ^ (b * 0xD6E8FEB86659FD93ull));
    return ((double)(h >> 11) + 0.5) * (2.0 / 9007199254740992.0) - 1.0;
}

struct RowGeom {        // what the sweeps over one beamlet's support need
    double cs, sn, a_c, b_r, inv2s2, rho_max2, x0, y0, z0, vs, Rb, mu, noise;
    int iz_lo, iz_hi, iy_lo, iy_hi, nx, ny;
    unsigned long long seed;
    long long i;
};

// the voxels of row (iz, iy) the kernel may reach: [ix_lo, ix_hi], empty if ix_lo > ix_hi; dz2 = (z - b_r)^2
__device__ __forceinline__ void x_interval(const RowGeom &g, int iz, int iy, double &y, double &dz2, int &ix_lo, int &ix_hi) {
    ix_lo = 0;
    ix_hi = -1;
    const double z = g.z0 + (iz + 0.5) * g.vs, dz = z - g.b_r;
    dz2 = dz * dz;
    const double rxy2 = g.rho_max2 - dz2;
    if (rxy2 < 0.0) return;
    const double rxy = sqrt(rxy2);
    y = g.y0 + (iy + 0.5) * g.vs;
    const double bx2 = g.Rb * g.Rb - y * y;
    if (bx2 < 0.0) return;
    double xl = -sqrt(bx2), xh = -xl;                       // body chord
    if (fabs(g.sn) > 1e-12) {                               // |a - a_c| <= rxy with a = -sn x + cs y
        double e0 = (g.cs * y - g.a_c - rxy) / g.sn, e1 = (g.cs * y - g.a_c + rxy) / g.sn;
        if (e0 > e1) {
            const double t = e0;
            e0 = e1;
            e1 = t;
        }
        if (e0 > xl) xl = e0;
        if (e1 < xh) xh = e1;
    } else if (fabs(g.cs * y - g.a_c) > rxy) return;
    ix_lo = max(0, (int)floor((xl - g.x0) / g.vs - 0.5) - 1);
    ix_hi = min(g.nx - 1, (int)ceil((xh - g.x0) / g.vs - 0.5) + 1);
}

// D at voxel (ix, iy, iz), or -1 outside the body / the kernel's support
__device__ __forceinline__ double entry(const RowGeom &g, int ix, int iy, int iz, double y, double dz2) {
    const double x = g.x0 + (ix + 0.5) * g.vs;
    if (x * x + y * y > g.Rb * g.Rb) return -1.0;
    const double a = -g.sn * x + g.cs * y, t = g.cs * x + g.sn * y;
    const double da = a - g.a_c, rho2 = da * da + dz2;
    if (rho2 > g.rho_max2) return -1.0;
    const double in = g.Rb * g.Rb - a * a;
    const double depth = t + sqrt(in > 0.0 ? in : 0.0);
    const long long j = ((long long)iz * g.ny + iy) * g.nx + ix;
    return exp(-g.mu * depth - rho2 * g.inv2s2) * (1.0 + g.noise * hash_u11(g.seed, (unsigned long long)g.i, (unsigned long long)j));
}

// FILL = false: cnt[i] = entries of beamlet i; FILL = true: write them at row_ptr[i]
template <bool FILL>
__global__ void __launch_bounds__(256)
k_engine(const vmat_engine_geometry eg, long long B, long long *__restrict__ cnt, const long long *__restrict__ row_ptr,
         int32_t *__restrict__ col, float *__restrict__ val) {
    const int lane = threadIdx.x & 31;
    const long long i = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (i >= B) return;
    const int R = eg.n_rows, C = eg.n_cols;
    const int k = (int)(i / ((long long)R * C)), r = (int)((i / C) % R), c = (int)(i % C);
    RowGeom g;
    const double th = (double)k * 360.0 / (double)eg.n_beams * (CUDART_PI / 180.0);
    g.cs = cos(th);
    g.sn = sin(th);
    const double bw = eg.beamlet_mm, sigma = eg.sigma_beamlets * bw, rho_max = 4.5 * sigma;
    g.vs = eg.voxel_mm;
    g.Rb = eg.body_radius_mm;
    g.a_c = ((double)c - 0.5 * (C - 1)) * bw;
    g.b_r = ((double)r - 0.5 * (R - 1)) * bw;
    g.inv2s2 = 1.0 / (2.0 * sigma * sigma);
    g.rho_max2 = rho_max * rho_max;
    g.x0 = -0.5 * eg.nx * g.vs;
    g.y0 = -0.5 * eg.ny * g.vs;
    g.z0 = -0.5 * eg.nz * g.vs;
    g.mu = eg.mu_per_mm;
    g.noise = eg.noise;
    g.nx = eg.nx;
    g.ny = eg.ny;
    g.seed = eg.seed;
    g.i = i;
    long long n = 0;
    if (fabs(g.a_c) - rho_max < g.Rb) {                     // else the ray (with its halo) misses the body
        g.iz_lo = max(0, (int)floor((g.b_r - rho_max - g.z0) / g.vs - 0.5));
        g.iz_hi = min(eg.nz - 1, (int)ceil((g.b_r + rho_max - g.z0) / g.vs - 0.5));
        g.iy_lo = max(0, (int)floor((-g.Rb - g.y0) / g.vs - 0.5));
        g.iy_hi = min(eg.ny - 1, (int)ceil((g.Rb - g.y0) / g.vs - 0.5));
        const int nyr = g.iy_hi - g.iy_lo + 1, npairs = max(0, g.iz_hi - g.iz_lo + 1) * max(0, nyr);
        double vmax = 0.0;
        for (int p = lane; p < npairs; p += 32) {
            const int iz = g.iz_lo + p / nyr, iy = g.iy_lo + p % nyr;
            double y, dz2;
            int lo, hi;
            x_interval(g, iz, iy, y, dz2, lo, hi);
            for (int ix = lo; ix <= hi; ++ix) vmax = fmax(vmax, entry(g, ix, iy, iz, y, dz2));
        }
#pragma unroll
        for (int o = 16; o; o >>= 1) vmax = fmax(vmax, __shfl_xor_sync(0xffffffffu, vmax, o));
        if (vmax > 0.0) {
            const double keep = eg.cutoff * vmax;
            long long base = FILL ? row_ptr[i] : 0;
            for (int p0 = 0; p0 < npairs; p0 += 32) {       // 32 voxel rows at a time, in voxel order
                const int p = p0 + lane;
                int mine = 0, lo = 0, hi = -1, iz = 0, iy = 0;
                double y = 0.0, dz2 = 0.0;
                if (p < npairs) {
                    iz = g.iz_lo + p / nyr;
                    iy = g.iy_lo + p % nyr;
                    x_interval(g, iz, iy, y, dz2, lo, hi);
                    for (int ix = lo; ix <= hi; ++ix) mine += entry(g, ix, iy, iz, y, dz2) >= keep;
                }
                int incl = mine;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const int v = __shfl_up_sync(0xffffffffu, incl, o);
                    if (lane >= o) incl += v;
                }
                if (FILL && mine) {
                    long long w = base + incl - mine;
                    for (int ix = lo; ix <= hi; ++ix) {
                        const double v = entry(g, ix, iy, iz, y, dz2);
                        if (v >= keep) {
                            col[w] = (int32_t)(((long long)iz * g.ny + iy) * g.nx + ix);
                            val[w] = (float)v;
                            ++w;
                        }
                    }
                }
                const int total = __shfl_sync(0xffffffffu, incl, 31);
                base += total;
                n += total;
            }
        }
    }
    if (!FILL && lane == 0) cnt[i] = n;
}

// exclusive prefix sum of B + 1 int64 counts, in place: one block walks the array (B <= 2^31: a few milliseconds)
__global__ void __launch_bounds__(1024) k_scan_counts(long long *__restrict__ v, long long n) {
    __shared__ long long warp_tot[32];
    __shared__ long long s_carry;
    if (threadIdx.x == 0) s_carry = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (long long b0 = 0; b0 < n; b0 += 4096) {
        const long long i0 = b0 + (long long)threadIdx.x * 4;
        long long x[4], sum = 0;
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            x[u] = i0 + u < n ? v[i0 + u] : 0;
            sum += x[u];
        }
        long long incl = sum;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const long long t = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += t;
        }
        if (lane == 31) warp_tot[warp] = incl;
        __syncthreads();
        long long before = s_carry, total = 0;
        for (int w2 = 0; w2 < 32; ++w2) {
            if (w2 < warp) before += warp_tot[w2];
            total += warp_tot[w2];
        }
        long long run = before + incl - sum;
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            if (i0 + u < n) v[i0 + u] = run;
            run += x[u];
        }
        __syncthreads();
        if (threadIdx.x == 0) s_carry += total;
        __syncthreads();
    }
}

}  // namespace

}  // namespace vmat

using namespace vmat;

extern "C" {

int vmat_engine_dose_matrix(const vmat_engine_geometry *g, void *cuda_stream, int64_t **row_ptr_dev, int32_t **col_idx_dev,
                            float **val_dev, int64_t *nnz_out) {
    if (!g || !row_ptr_dev || !col_idx_dev || !val_dev || !nnz_out) return fail(nullptr, VMAT_EINVAL, "NULL argument");
    if (g->nx < 1 || g->ny < 1 || g->nz < 1 || g->n_beams < 1 || g->n_rows < 1 || g->n_cols < 1 || !(g->voxel_mm > 0.0) ||
        !(g->beamlet_mm > 0.0) || !(g->body_radius_mm > 0.0) || !(g->sigma_beamlets > 0.0) || !(g->cutoff >= 0.0) ||
        !(g->mu_per_mm >= 0.0) || !(g->noise >= 0.0 && g->noise < 1.0))
        return fail(nullptr, VMAT_EINVAL, "bad engine geometry");
    const long long B = (long long)g->n_beams * g->n_rows * g->n_cols;
    if ((long long)g->nx * g->ny * g->nz > 0x7fffffffll || B > 0x7fffffffll)
        return fail(nullptr, VMAT_EINVAL, "voxels and beamlets must fit int32");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int device = 0;
    cudaError_t e = cudaGetDevice(&device);
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "cudaGetDevice");
    long long *rp = nullptr;
    int32_t *col = nullptr;
    float *val = nullptr;
    auto bail = [&](int code) {
        pool_free(rp, device, st);
        pool_free(col, device, st);
        pool_free(val, device, st);
        return code;
    };
    if ((e = pool_alloc((void **)&rp, (size_t)(B + 1) * 8, device, st)) != cudaSuccess)
        return bail(cuda_fail(nullptr, e, "device allocation (row_ptr)"));
    if ((e = cudaMemsetAsync(rp + B, 0, 8, st)) != cudaSuccess) return bail(cuda_fail(nullptr, e, "cudaMemsetAsync"));
    const unsigned blocks = (unsigned)((B + 7) / 8);
    k_engine<false><<<blocks, 256, 0, st>>>(*g, B, rp, nullptr, nullptr, nullptr);
    k_scan_counts<<<1, 1024, 0, st>>>(rp, B + 1);
    long long nnz = 0;
    if ((e = cudaMemcpyAsync(&nnz, rp + B, 8, cudaMemcpyDeviceToHost, st)) != cudaSuccess ||
        (e = cudaStreamSynchronize(st)) != cudaSuccess)
        return bail(cuda_fail(nullptr, e, "engine count pass"));
    if ((e = pool_alloc((void **)&col, (size_t)(nnz > 0 ? nnz : 1) * 4, device, st)) != cudaSuccess ||
        (e = pool_alloc((void **)&val, (size_t)(nnz > 0 ? nnz : 1) * 4, device, st)) != cudaSuccess) {
        cudaGetLastError();
        return bail(fail(nullptr, VMAT_ENOMEM, std::string("device allocation (D) failed: ") + cudaGetErrorString(e)));
    }
    k_engine<true><<<blocks, 256, 0, st>>>(*g, B, nullptr, rp, col, val);
    if ((e = cudaGetLastError()) != cudaSuccess) return bail(cuda_fail(nullptr, e, "k_engine"));
    *row_ptr_dev = (int64_t *)rp;
    *col_idx_dev = col;
    *val_dev = val;
    *nnz_out = nnz;
    return VMAT_OK;
}

int vmat_engine_free(void *dev_ptr, void *cuda_stream) {
    if (!dev_ptr) return VMAT_OK;
    int device = 0;
    if (cudaGetDevice(&device) != cudaSuccess) return VMAT_ECUDA;
    pool_free(dev_ptr, device, (cudaStream_t)cuda_stream);
    return VMAT_OK;
}

}  // extern "C"
