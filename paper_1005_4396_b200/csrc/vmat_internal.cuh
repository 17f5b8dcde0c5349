// vmat_internal.cuh — plan state and kernel launchers shared by the translation units of
// libvmat_b200.so.  Product code: shares nothing with oracle/ (DESIGN.md section 2).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "../../include/vmat.h"

namespace vmat {

constexpr int kChunk = 128;           // slots per master chunk: one warp of float4
constexpr int kGroup = 8;             // chunks a master block works on at a time
constexpr int kMasterThreads = 512;   // 16 warps split the beam loop of one group of chunks
constexpr int kMasterWarps = kMasterThreads / 32;
constexpr int kOutPerThread = kGroup * kChunk / kMasterThreads;

struct ColStat {                      // statistics of one aperture-dose column d_k (fixed-point units)
    unsigned long long l1, linf;      // sum and max of |d_k|
    int32_t clo, chi;                 // first and last chunk with a non-zero entry (INT_MAX, -1 if none)
};

struct Sel {                          // device-side result of the beam choice (step d)
    int32_t beam;
    int32_t pad;
    double price;
};

struct MasterOut {                    // device-side mirror of vmat_master_stats
    int32_t inner, backtracks, stop_reason, pad;   // pad: passes over the columns
    double pg_entry, pg_exit, F, G, cost;
};

}  // namespace vmat

struct vmat_plan {
    // ---- sizes -------------------------------------------------------------------------
    int64_t V = 0, N = 0, R = 0, C = 0, B = 0, RC = 0;
    int64_t nnz = 0;        // entries of D as given
    int64_t nq = 0;         // quads (groups of 4 entries) of the padded layout
    int64_t S = 0;          // support: voxels with a non-empty column of D
    int64_t Sp = 0;         // S rounded up to a multiple of kChunk (>= kChunk)
    int32_t delta = 0;
    double gamma = 0.0;
    double y_min = 0.0, y_max = __builtin_huge_val();   // bounds on the dose rates of occupied beams (vmat_set_dose_rate_bounds)
    vmat_options opt{};
    cudaStream_t stream = nullptr;
    int sm_count = 0;
    int device = 0;

    // ---- D, beamlet-major padded CSR in slot space ------------------
    uint32_t *rowq = nullptr;   // B+1 row starts in quads
    float4 *val4 = nullptr;     // nq
    int4 *col4 = nullptr;       // nq, slot ids

    // ---- d_format 1: second copy of D for the pricing product, aligned slot pairs with 16-bit ids (vmat_layout.cu) ----
    uint32_t *pr_rowo = nullptr;    // B+1 row starts in groups (four units = up to eight entries)
    float4 *pr_va = nullptr, *pr_vb = nullptr;   // values of units 0-1 / 2-3 of every group
    uint2 *pr_ix = nullptr;         // four 16-bit pair ids per group, relative to its panel of 65536 pairs
    uint8_t *pr_pan = nullptr;      // panel of every group
    int64_t pr_groups = 0;

    // ---- voxel data --------------------------------------------------------------------
    float *T_V = nullptr, *alpha_V = nullptr, *beta_V = nullptr;   // V each
    int32_t *slot_of = nullptr;    // V, -1 outside the support
    int32_t *voxel_of = nullptr;   // S
    float *T_s = nullptr, *alpha_s = nullptr, *beta_s = nullptr;   // Sp each (padding: 0)
    double F_out = 0.0;            // sum over voxels outside the support of alpha_j T_j^2 (+ beta part)

    // ---- plan state on the device --------------------------------------------------------
    uint8_t *occ = nullptr;        // N
    int32_t *free_list = nullptr;  // N: un-occupied beams, ascending (first N - #occupied entries valid)
    int32_t *left = nullptr, *right = nullptr;   // N*R
    double *y = nullptr;           // N
    double *theta = nullptr;       // N

    // ---- work arrays -----------------------------------------------------------------------
    float *z_s = nullptr, *zn_s = nullptr, *q_s = nullptr, *q2_s = nullptr, *w_s = nullptr, *wtmp_s = nullptr;  // Sp each
    float *g = nullptr;            // B prices
    float *Dd = nullptr;           // N x Sp aperture-dose columns d_k (row k valid iff col_valid[k])
    unsigned long long *acc = nullptr;   // Sp fixed-point accumulator (all zero between uses)
    double fx_scale = 1.0, fx_inv = 1.0;

    int32_t *cand_left = nullptr, *cand_right = nullptr;   // N*R row optima of the last search
    double *beam_price = nullptr;  // N
    vmat::Sel *sel = nullptr;
    unsigned int *ticket = nullptr;
    unsigned long long *beam_total = nullptr;   // N, leaf search: per-beam sums of row optima (zero between launches)
    unsigned int *beam_ticket = nullptr;        // N, leaf search: per-beam block counters (zero between launches)

    long long *accbuf = nullptr;       // 3 x (2N + 2) fixed-point sums of the master kernel
    unsigned int *phase = nullptr;     // rotation counter of accbuf, barrier epoch
    unsigned long long *mcount = nullptr;   // master bookkeeping: touched segments x passes, passes
    double *gsave = nullptr;           // N: d_k . w the last master solve left (warm entry of the next one in vmat_solve)
    int *gflag = nullptr;              // device flag: gsave is valid
    bool warm_ok = false;              // host: nothing but vmat_solve's own steps touched the plan since that solve
    vmat::ColStat *colstat = nullptr;  // N
    uint32_t *col_touch = nullptr;     // N x touch_words: bit c of row k set iff chunk c of d_k holds a non-zero entry
    int touch_words = 0;
    unsigned int *vbounds = nullptr;   // bit patterns of max|T|, max(alpha, beta)
    float Tmax = 0.f, abmax = 0.f;
    // launch shape of one master kernel: mcfg[0] k_master, mcfg[1] k_newton (grid == 0: the plan cannot run it)
    struct MasterCfg {
        int grid = 0;                  // blocks launched
        int nblk = 0;                  // blocks that own chunks (k_newton: all but the solving block)
        size_t smem = 0;               // dynamic shared memory of a working block
        int cache_segs = 0;            // 512-byte segments of Dd a master block stages in shared memory
        int rslots = 0;                // slots per master block kept resident in shared memory (0: none)
        int ul_cap = 0;                // capacity of the per-chunk lists of unstaged beams (0: masked loops)
    } mcfg[2];
    // mode 1 of the master (k_newton): the Hessian of F over the occupied beams, kept on the device from solve to solve
    bool master_newton = false;        // the plan can run k_newton (master_mode 1, n_beams <= one thread per beam)
    int newton_kmax = 0;               // most occupied beams whose reduced problem fits the solving block
    bool newton_retired = false;       // a solve has outgrown it: H_F is no longer kept up (until the next reset)
    long long *hess = nullptr;         // N x N fixed point
    float *omref = nullptr;            // Sp: the omega (alpha, beta or 0 per slot) the matrix was built with
    uint8_t *hvalid = nullptr;         // N: column k is in the matrix
    int *hlive = nullptr;              // device flag: the matrix is built (a k_newton launch has run since its last reset)
    double hscale = 1.0, hinv = 1.0;
    float *wn_s = nullptr;             // Sp: second buffer of w
    void *mail = nullptr;              // message of the solving block to the working blocks
    unsigned long long *nsync = nullptr;   // arrival / epoch counters of that hand-over
    vmat::MasterOut *mout = nullptr;
    double *cost3 = nullptr;       // device {F, G, F+gamma G}
    double *rate_ratio = nullptr;  // device scalar of the dose-rate feasibility test
    double *part_dose = nullptr;   // partial F sums of the direct dose pass
    double *part_dose2 = nullptr;  // per-chunk F of the dose pass over the columns
    void *dose_scale = nullptr;    // device scalars of the direct dose pass (vmat_dose.cu)
    int32_t *dose_list = nullptr;  // B: exposed beamlets of the direct dose pass (its first dose_scale->count entries)
    int dose_blocks = 0;

    // device trace of vmat_solve
    int32_t *tr_beam = nullptr, *tr_inner = nullptr;
    double *tr_price = nullptr, *tr_F = nullptr, *tr_G = nullptr, *tr_cost = nullptr;
    int32_t tr_cap = 0;

    // ---- host mirror ------------------------------------------------------------------------
    std::vector<uint8_t> h_occ;        // occupied mask as last known to the host
    std::vector<uint8_t> col_valid;    // Dd row k matches the plan's aperture of beam k
    bool state_valid = false;          // z_s / w_s match (occ, leaves, y)
    std::string err;
    int64_t launches = 0;
    int64_t bytes = 0;
    std::vector<void *> allocs;
};

namespace vmat {

// error plumbing -------------------------------------------------------------------------------
int fail(vmat_plan *p, int code, const std::string &msg);
int cuda_fail(vmat_plan *p, cudaError_t e, const char *what);
void set_create_error(const std::string &msg);

#define VMAT_CUDA(p, call)                                                  \
    do {                                                                    \
        cudaError_t e__ = (call);                                           \
        if (e__ != cudaSuccess) return vmat::cuda_fail((p), e__, #call);    \
    } while (0)

// Device memory comes from one stream-ordered pool per device that keeps what plans free (release threshold =
// everything) until vmat_release_memory: creating and destroying plans over and over then costs no driver
// round trip (measured: cudaFree of a plan's buffers took 3 ms, with spikes of 25 - 650 ms).  Falls back to
// cudaMalloc / cudaFree where pools are not supported.
cudaError_t pool_alloc(void **ptr, size_t bytes, int device, cudaStream_t stream);
void pool_free(void *ptr, int device, cudaStream_t stream);

template <typename T>
int dev_alloc(vmat_plan *p, T **out, int64_t count) {
    void *ptr = nullptr;
    const size_t bytes = (size_t)(count > 0 ? count : 1) * sizeof(T);
    cudaError_t e = pool_alloc(&ptr, bytes, p->device, p->stream);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return fail(p, VMAT_ENOMEM, std::string("device allocation failed: ") + cudaGetErrorString(e));
    }
    p->allocs.push_back(ptr);
    p->bytes += (int64_t)bytes;
    *out = (T *)ptr;
    return VMAT_OK;
}

// Programmatic dependent launch: a kernel launched with launch_pdl may be scheduled while the previous kernel of the
// stream is still draining (provided that one has called pdl_trigger, or exited); it must call pdl_wait() before it
// touches anything earlier kernels wrote.  Used on the chain of short dependent kernels of an outer iteration
// (pricing -> leaf search -> column scatter -> column finish), where the launch gaps weigh as much as the kernels.
template <typename... KArgs, typename... Args>
cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, cudaStream_t stream, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = 0;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}
#ifdef __CUDACC__
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
#endif

// vmat_layout.cu: validation and the device layout of D ------------------------------------------
int build_layout(vmat_plan *p, const vmat_problem *pb);
int build_pairs(vmat_plan *p);

// vmat_price.cu ---------------------------------------------------------------------------------------
int launch_price_spmv(vmat_plan *p, const float *w_s, float *g, int n_free);
int launch_free_list(vmat_plan *p);

// vmat_search.cu --------------------------------------------------------------------------------------
int launch_leaf_search(vmat_plan *p, const float *g, int32_t *all_left, int32_t *all_right, double *beam_price,
                       int commit, int trace_it);

// vmat_master.cu ------------------------------------------------------------------------------------
int master_configure(vmat_plan *p);
int reset_hessian(vmat_plan *p);
int launch_column_build(vmat_plan *p, int beam /* -1: read p->sel */);
int launch_master(vmat_plan *p, int trace_it, int warm /* 1: inside vmat_solve, right after a committed search */,
                  int k_occ /* occupied beams at the launch, or an upper bound of them */);
int launch_expand(vmat_plan *p, const float *src_s, float *dst_V, int what /*0 z, 1 w*/);
int launch_compress(vmat_plan *p, const float *src_V, float *dst_s);
int launch_rate_ratio(vmat_plan *p, double rho, double *ratio_dev);

// vmat_dose.cu: steps (a)+(b) straight from D (fixed-point atomics path) ------------------------------
int dose_configure(vmat_plan *p);
int launch_direct_dose(vmat_plan *p);
int launch_columns_dose(vmat_plan *p);

}  // namespace vmat
