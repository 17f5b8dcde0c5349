// vmat_api.cu — the extern "C" boundary declared in include/vmat.h: argument checks, plan
// life-cycle, and the order in which the kernels of the other translation units are enqueued.
// No arithmetic of the method lives here.
#include <cmath>
#include <cstring>
#include <mutex>
#include <new>

#include "vmat_internal.cuh"

namespace vmat {

static thread_local std::string g_create_error;

void set_create_error(const std::string &msg) { g_create_error = msg; }

int fail(vmat_plan *p, int code, const std::string &msg) {
    if (p) p->err = msg;
    else g_create_error = msg;
    return code;
}

int cuda_fail(vmat_plan *p, cudaError_t e, const char *what) {
    cudaGetLastError();
    return fail(p, VMAT_ECUDA, std::string(what) + ": " + cudaGetErrorString(e));
}

// ---- the device memory pools (one per device, created on first use) ---------------------------------------
namespace {
constexpr int kMaxDevices = 64;
std::mutex g_pool_mutex;
cudaMemPool_t g_pool[kMaxDevices];
int g_pool_state[kMaxDevices];   // 0 not tried, 1 pool in use, -1 pools unsupported: cudaMalloc / cudaFree

cudaMemPool_t pool_of(int device) {
    if (device < 0 || device >= kMaxDevices) return nullptr;
    std::lock_guard<std::mutex> lock(g_pool_mutex);
    if (g_pool_state[device] == 0) {
        g_pool_state[device] = -1;
        int supported = 0;
        if (cudaDeviceGetAttribute(&supported, cudaDevAttrMemoryPoolsSupported, device) == cudaSuccess && supported) {
            cudaMemPoolProps props = {};
            props.allocType = cudaMemAllocationTypePinned;
            props.handleTypes = cudaMemHandleTypeNone;
            props.location.type = cudaMemLocationTypeDevice;
            props.location.id = device;
            cudaMemPool_t pool;
            if (cudaMemPoolCreate(&pool, &props) == cudaSuccess) {
                unsigned long long keep = ~0ull;
                cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
                g_pool[device] = pool;
                g_pool_state[device] = 1;
            }
        }
        cudaGetLastError();
    }
    return g_pool_state[device] == 1 ? g_pool[device] : nullptr;
}
}  // namespace

cudaError_t pool_alloc(void **ptr, size_t bytes, int device, cudaStream_t stream) {
    cudaMemPool_t pool = pool_of(device);
    if (pool) return cudaMallocFromPoolAsync(ptr, bytes, pool, stream);
    return cudaMalloc(ptr, bytes);
}

void pool_free(void *ptr, int device, cudaStream_t stream) {
    if (!ptr) return;
    if (pool_of(device)) cudaFreeAsync(ptr, stream);
    else cudaFree(ptr);
}

static void free_plan(vmat_plan *p) {
    if (!p) return;
    for (void *ptr : p->allocs) pool_free(ptr, p->device, p->stream);
    cudaStreamSynchronize(p->stream);
    delete p;
}

// Dd rows of the occupied beams that do not match the plan's apertures are rebuilt
static int ensure_columns(vmat_plan *p) {
    for (int64_t k = 0; k < p->N; ++k)
        if (p->h_occ[k] && !p->col_valid[k]) {
            int rc = launch_column_build(p, (int)k);
            if (rc) return rc;
            p->col_valid[k] = 1;
        }
    return VMAT_OK;
}

// steps (a)+(b): z, w and the cost for the current (occ, leaves, y), by the aperture-dose columns
// (path 0) or straight from D (path 1)
static int evaluate_state(vmat_plan *p, int path) {
    int rc;
    if (path == 1) {
        if ((rc = launch_direct_dose(p))) return rc;
    } else {
        if ((rc = ensure_columns(p))) return rc;
        if ((rc = launch_columns_dose(p))) return rc;
    }
    p->state_valid = true;
    return VMAT_OK;
}

static int ensure_state(vmat_plan *p) {
    if (p->state_valid) return VMAT_OK;
    return evaluate_state(p, p->opt.dose_path == 1 ? 1 : 0);
}

static int refresh_host_occ(vmat_plan *p) {
    VMAT_CUDA(p, cudaMemcpyAsync(p->h_occ.data(), p->occ, (size_t)p->N, cudaMemcpyDeviceToHost, p->stream));
    VMAT_CUDA(p, cudaStreamSynchronize(p->stream));
    return VMAT_OK;
}

static int64_t unoccupied(const vmat_plan *p) {
    int64_t n = 0;
    for (int64_t k = 0; k < p->N; ++k) n += p->h_occ[k] ? 0 : 1;
    return n;
}

}  // namespace vmat

using namespace vmat;

extern "C" {

void vmat_default_options(vmat_options *opt) {
    if (!opt) return;
    opt->validate = 1;
    opt->d_format = 0;
    opt->dose_path = 0;
    opt->master_eps = 1e-4;
    opt->master_max_inner = 500;
    opt->master_stall_rel = 1e-6;    // 100x inside the 1e-4 parity tolerance on the master cost (S11)
    opt->master_stall_count = 2;
    opt->record_phases = 0;
    opt->master_mode = 1;
    opt->stop_when_priced_out = 0;
    opt->master_unstaged_lists = 1;
    opt->occupied_only_G = 0;
    opt->master_newton_max_beams = 0;
}

int vmat_create(const vmat_problem *pb, const vmat_options *options, void *cuda_stream, vmat_plan **out) {
    if (!pb || !out) return fail(nullptr, VMAT_EINVAL, "problem and out must not be NULL");
    if (pb->n_voxels < 1 || pb->n_beams < 1 || pb->n_rows < 1 || pb->n_cols < 1)
        return fail(nullptr, VMAT_EINVAL, "n_voxels, n_beams, n_rows, n_cols must be positive");
    if (pb->n_cols > VMAT_MAX_COLS) return fail(nullptr, VMAT_EINVAL, "n_cols exceeds VMAT_MAX_COLS (255)");
    if (pb->n_voxels > 0x7fffffffll) return fail(nullptr, VMAT_EINVAL, "n_voxels must fit int32");
    if (pb->n_beams > 2048) return fail(nullptr, VMAT_EINVAL, "n_beams must be <= 2048");
    if (pb->n_rows * pb->n_cols > (1 << 20)) return fail(nullptr, VMAT_EINVAL, "n_rows*n_cols must be <= 2^20");
    if (pb->n_beams * pb->n_rows * pb->n_cols > 0x7fffffffll)
        return fail(nullptr, VMAT_EINVAL, "number of beamlets must fit int32");
    if (!pb->row_ptr || !pb->T || !pb->alpha || !pb->beta || !pb->theta_deg)
        return fail(nullptr, VMAT_EINVAL, "row_ptr, T, alpha, beta, theta_deg must not be NULL");
    if (pb->mem_space != VMAT_HOST && pb->mem_space != VMAT_DEVICE)
        return fail(nullptr, VMAT_EINVAL, "mem_space must be VMAT_HOST or VMAT_DEVICE");
    if (pb->max_leaf_travel < 0) return fail(nullptr, VMAT_EINVAL, "max_leaf_travel must be >= 0");
    if (!(pb->gamma >= 0.0) || !std::isfinite(pb->gamma)) return fail(nullptr, VMAT_EINVAL, "gamma must be finite and >= 0");
    for (int64_t k = 0; k < pb->n_beams; ++k) {
        if (!std::isfinite(pb->theta_deg[k])) return fail(nullptr, VMAT_EINVAL, "theta_deg must be finite");
        if (k > 0 && !(pb->theta_deg[k] > pb->theta_deg[k - 1]))
            return fail(nullptr, VMAT_EINVAL, "theta_deg must be strictly ascending");
    }
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        return fail(nullptr, VMAT_ECUDA, std::string("no CUDA device: ") + cudaGetErrorString(e));
    }

    vmat_plan *p = new (std::nothrow) vmat_plan();
    if (!p) return fail(nullptr, VMAT_ENOMEM, "out of host memory");
    auto bail = [&](int rc) {
        g_create_error = p->err;
        free_plan(p);
        return rc;
    };
    if (options) p->opt = *options;
    else vmat_default_options(&p->opt);
    if (!(p->opt.master_eps > 0.0)) p->opt.master_eps = 1e-4;
    if (p->opt.master_max_inner < 0) p->opt.master_max_inner = 0;
    if (!(p->opt.master_stall_rel >= 0.0)) p->opt.master_stall_rel = 1e-6;
    if (p->opt.master_stall_count < 1) p->opt.master_stall_count = 2;
    if (p->opt.master_mode != 1) p->opt.master_mode = 0;
    if (p->opt.d_format != 0 && p->opt.d_format != 1) return bail(fail(p, VMAT_EINVAL, "d_format must be 0 or 1"));
    p->V = pb->n_voxels;
    p->N = pb->n_beams;
    p->R = pb->n_rows;
    p->C = pb->n_cols;
    p->RC = p->R * p->C;
    p->B = p->N * p->RC;
    p->delta = pb->max_leaf_travel;
    p->gamma = pb->gamma;
    p->stream = (cudaStream_t)cuda_stream;
    int coop = 0;
    if ((e = cudaGetDevice(&p->device)) != cudaSuccess ||
        (e = cudaDeviceGetAttribute(&p->sm_count, cudaDevAttrMultiProcessorCount, p->device)) != cudaSuccess ||
        (e = cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, p->device)) != cudaSuccess)
        return bail(cuda_fail(p, e, "cudaDeviceGetAttribute"));
    if (!coop) return bail(fail(p, VMAT_ECUDA, "device lacks cooperative launch"));
    if (pb->row_ptr && !(pb->col_idx && pb->val)) {
        // col_idx / val may only be NULL for an empty matrix; checked against nnz in build_layout
        if (pb->mem_space == VMAT_HOST && pb->row_ptr[p->B] != 0)
            return bail(fail(p, VMAT_EINVAL, "col_idx and val must not be NULL"));
    }

    int rc = build_layout(p, pb);
    if (rc) return bail(rc);
    if (p->opt.d_format == 1 && (rc = build_pairs(p))) return bail(rc);

    const int64_t N = p->N, NR = p->N * p->R, Sp = p->Sp;
#define A(ptr, n) \
    if ((rc = dev_alloc(p, &(ptr), (n)))) return bail(rc)
    A(p->occ, N);
    A(p->free_list, N);
    A(p->left, NR);
    A(p->right, NR);
    A(p->y, N);
    A(p->theta, N);
    A(p->z_s, Sp);
    A(p->zn_s, Sp);
    A(p->q_s, Sp);
    A(p->q2_s, Sp);
    A(p->w_s, Sp);
    A(p->wtmp_s, Sp);
    A(p->g, p->B);
    A(p->Dd, N * Sp);
    A(p->acc, Sp);
    A(p->cand_left, NR);
    A(p->cand_right, NR);
    A(p->beam_price, N);
    A(p->sel, 1);
    A(p->ticket, 1);
    A(p->beam_total, N);
    A(p->beam_ticket, N);
    A(p->mout, 1);
    A(p->cost3, 3);
    A(p->rate_ratio, 1);
    p->tr_cap = (int32_t)N;
    A(p->tr_beam, N);
    A(p->tr_inner, N);
    A(p->tr_price, N);
    A(p->tr_F, N);
    A(p->tr_G, N);
    A(p->tr_cost, N);
#undef A
    cudaStream_t st = p->stream;
#define Z(ptr, bytes) \
    if ((e = cudaMemsetAsync((ptr), 0, (bytes), st)) != cudaSuccess) return bail(cuda_fail(p, e, "cudaMemsetAsync"))
    Z(p->occ, (size_t)N);
    Z(p->left, (size_t)NR * 4);
    Z(p->right, (size_t)NR * 4);
    Z(p->y, (size_t)N * 8);
    Z(p->z_s, (size_t)Sp * 4);
    Z(p->zn_s, (size_t)Sp * 4);
    Z(p->q_s, (size_t)Sp * 4);
    Z(p->q2_s, (size_t)Sp * 4);
    Z(p->w_s, (size_t)Sp * 4);
    Z(p->wtmp_s, (size_t)Sp * 4);
    Z(p->g, (size_t)p->B * 4);
    Z(p->acc, (size_t)Sp * 8);
    Z(p->cand_left, (size_t)NR * 4);
    Z(p->cand_right, (size_t)NR * 4);
    Z(p->ticket, 4);
    Z(p->beam_total, (size_t)N * 8);
    Z(p->beam_ticket, (size_t)N * 4);
    Z(p->sel, sizeof(Sel));
#undef Z
    if ((e = cudaMemcpyAsync(p->theta, pb->theta_deg, (size_t)N * 8, cudaMemcpyHostToDevice, st)) != cudaSuccess)
        return bail(cuda_fail(p, e, "cudaMemcpyAsync(theta)"));
    if ((rc = master_configure(p))) return bail(rc);
    if ((rc = dose_configure(p))) return bail(rc);
    if ((rc = launch_free_list(p))) return bail(rc);
    if ((e = cudaStreamSynchronize(st)) != cudaSuccess) return bail(cuda_fail(p, e, "cudaStreamSynchronize"));
    p->h_occ.assign((size_t)N, 0);
    p->col_valid.assign((size_t)N, 0);
    p->state_valid = false;
    p->warm_ok = false;
    *out = p;
    return VMAT_OK;
}

int vmat_release_memory(void) {
    std::lock_guard<std::mutex> lock(g_pool_mutex);
    for (int d = 0; d < kMaxDevices; ++d)
        if (g_pool_state[d] == 1 && cudaMemPoolTrimTo(g_pool[d], 0) != cudaSuccess) {
            cudaGetLastError();
            return VMAT_ECUDA;
        }
    return VMAT_OK;
}

int vmat_destroy(vmat_plan *plan) {
    if (!plan) return VMAT_OK;
    cudaStreamSynchronize(plan->stream);
    free_plan(plan);
    return VMAT_OK;
}

int vmat_get_info(const vmat_plan *p, vmat_info *out) {
    if (!p || !out) return VMAT_EINVAL;
    out->n_voxels = p->V;
    out->n_beams = p->N;
    out->n_rows = p->R;
    out->n_cols = p->C;
    out->n_beamlets = p->B;
    out->nnz = p->nnz;
    out->nnz_padded = p->nq * 4;
    out->n_support = p->S;
    out->device_bytes = p->bytes;
    out->pricing_bytes = p->opt.d_format == 1 ? p->pr_groups * 41 + (p->B + 1) * 4 : p->nq * 32 + (p->B + 1) * 4;
    return VMAT_OK;
}

int vmat_dose(vmat_plan *p, float *z_dev, float *w_dev, double cost[3]) {
    if (!p) return VMAT_EINVAL;
    int rc = ensure_state(p);
    if (rc) return rc;
    if (z_dev && (rc = launch_expand(p, p->z_s, z_dev, 0))) return rc;
    if (w_dev && (rc = launch_expand(p, p->w_s, w_dev, 1))) return rc;
    if (cost) {
        VMAT_CUDA(p, cudaMemcpyAsync(cost, p->cost3, 3 * sizeof(double), cudaMemcpyDeviceToHost, p->stream));
        VMAT_CUDA(p, cudaStreamSynchronize(p->stream));
    }
    return VMAT_OK;
}

int vmat_dose_recompute(vmat_plan *p, int dose_path) {
    if (!p) return VMAT_EINVAL;
    if (dose_path < -1 || dose_path > 1) return fail(p, VMAT_EINVAL, "dose_path must be -1, 0 or 1");
    return evaluate_state(p, dose_path < 0 ? (p->opt.dose_path == 1 ? 1 : 0) : dose_path);
}

int vmat_price_spmv(vmat_plan *p, const float *w_dev, float *g_dev) {
    if (!p || !g_dev) return fail(p, VMAT_EINVAL, "g_dev must not be NULL");
    int rc;
    const float *w_s = p->w_s;
    if (w_dev) {
        if ((rc = launch_compress(p, w_dev, p->wtmp_s))) return rc;
        w_s = p->wtmp_s;
    } else if ((rc = ensure_state(p))) return rc;
    // the kernel covers the un-occupied beams only: the caller's buffer gets its zeros here
    const int64_t n_free = unoccupied(p);
    if (n_free < p->N) VMAT_CUDA(p, cudaMemsetAsync(g_dev, 0, (size_t)p->B * 4, p->stream));
    return launch_price_spmv(p, w_s, g_dev, (int)n_free);
}

int vmat_leaf_search(vmat_plan *p, const float *g_dev, int32_t *all_left_dev, int32_t *all_right_dev,
                     double *beam_price_dev) {
    if (!p || !g_dev) return fail(p, VMAT_EINVAL, "g_dev must not be NULL");
    return launch_leaf_search(p, g_dev, all_left_dev, all_right_dev, beam_price_dev, 0, -1);
}

int vmat_price(vmat_plan *p, const float *w_override_dev, const float *g_override_dev, float *g_out_dev,
               vmat_aperture *out, int commit) {
    if (!p) return VMAT_EINVAL;
    if (!out && !commit) return fail(p, VMAT_EINVAL, "out must not be NULL unless commit = 1");
    if (out && (!out->left || !out->right)) return fail(p, VMAT_EINVAL, "out->left / out->right must not be NULL");
    if (unoccupied(p) == 0) {
        if (out) {
            out->beam = -1;
            out->price = 0.0;
        }
        return VMAT_DONE;
    }
    int rc;
    const float *g = g_override_dev;
    if (!g) {
        const float *w_s = p->w_s;
        if (w_override_dev) {
            if ((rc = launch_compress(p, w_override_dev, p->wtmp_s))) return rc;
            w_s = p->wtmp_s;
        } else if ((rc = ensure_state(p))) return rc;
        if (g_out_dev) VMAT_CUDA(p, cudaMemsetAsync(p->g, 0, (size_t)p->B * 4, p->stream));
        if ((rc = launch_price_spmv(p, w_s, p->g, (int)unoccupied(p)))) return rc;
        g = p->g;
    }
    if (g_out_dev && g_out_dev != g)
        VMAT_CUDA(p, cudaMemcpyAsync(g_out_dev, g, (size_t)p->B * 4, cudaMemcpyDeviceToDevice, p->stream));
    if ((rc = launch_leaf_search(p, g, nullptr, nullptr, nullptr, commit ? 1 : 0, -1))) return rc;
    Sel h_sel;
    VMAT_CUDA(p, cudaMemcpyAsync(&h_sel, p->sel, sizeof(Sel), cudaMemcpyDeviceToHost, p->stream));
    VMAT_CUDA(p, cudaStreamSynchronize(p->stream));
    if (h_sel.beam < 0) return fail(p, VMAT_ESTATE, "search found no beam although one is un-occupied");
    if (out) {
        out->beam = h_sel.beam;
        out->price = h_sel.price;
        VMAT_CUDA(p, cudaMemcpyAsync(out->left, p->cand_left + (size_t)h_sel.beam * p->R, (size_t)p->R * 4,
                                     cudaMemcpyDeviceToHost, p->stream));
        VMAT_CUDA(p, cudaMemcpyAsync(out->right, p->cand_right + (size_t)h_sel.beam * p->R, (size_t)p->R * 4,
                                     cudaMemcpyDeviceToHost, p->stream));
        VMAT_CUDA(p, cudaStreamSynchronize(p->stream));
    }
    if (commit) {
        p->h_occ[h_sel.beam] = 1;
        p->col_valid[h_sel.beam] = 0;
        // y_k = 0: z, w and the cost are unchanged (S2), the state stays valid
        p->warm_ok = false;   // but the saved gradient knows nothing of this beam
    }
    return VMAT_OK;
}

int vmat_master(vmat_plan *p, const vmat_master_opts *opts, vmat_master_stats *out) {
    if (!p) return VMAT_EINVAL;
    int rc = ensure_columns(p);
    if (rc) return rc;
    const vmat_options keep = p->opt;
    if (opts) {   // per-call overrides (a field <= 0 keeps the plan's value)
        if (opts->eps > 0.0) p->opt.master_eps = opts->eps;
        if (opts->max_inner > 0) p->opt.master_max_inner = opts->max_inner;
        if (opts->stall_rel > 0.0) p->opt.master_stall_rel = opts->stall_rel;
        if (opts->stall_count > 0) p->opt.master_stall_count = opts->stall_count;
    }
    rc = launch_master(p, -1, 0, (int)(p->N - unoccupied(p)));
    p->opt = keep;
    if (rc) return rc;
    p->state_valid = true;
    p->warm_ok = true;
    MasterOut h;
    VMAT_CUDA(p, cudaMemcpyAsync(&h, p->mout, sizeof(MasterOut), cudaMemcpyDeviceToHost, p->stream));
    VMAT_CUDA(p, cudaStreamSynchronize(p->stream));
    if (out) {
        out->inner = h.inner;
        out->backtracks = h.backtracks;
        out->stop_reason = h.stop_reason;
        out->passes = h.pad;
        out->pg_entry = h.pg_entry;
        out->pg_exit = h.pg_exit;
        out->F = h.F;
        out->G = h.G;
        out->cost = h.cost;
    }
    return VMAT_OK;
}

int vmat_set_dose_rate_bounds(vmat_plan *p, double y_min, double y_max) {
    if (!p) return VMAT_EINVAL;
    if (!(y_min >= 0.0) || !(y_max >= y_min) || std::isinf(y_min))
        return fail(p, VMAT_EINVAL, "dose-rate bounds need 0 <= y_min <= y_max, y_min finite");
    p->y_min = y_min;
    p->y_max = y_max;
    p->warm_ok = false;   // the next solve may clamp y: evaluate from scratch
    return VMAT_OK;
}

int vmat_enforce_dose_rate(vmat_plan *p, double rho, double factor, double tol, int32_t max_rounds,
                           vmat_rate_stats *out) {
    if (!p) return VMAT_EINVAL;
    if (!(rho > 0.0) || !std::isfinite(rho)) return fail(p, VMAT_EINVAL, "max_variation_per_deg must be finite and > 0");
    if (!(factor > 1.0) || !std::isfinite(factor)) return fail(p, VMAT_EINVAL, "gamma_factor must be finite and > 1");
    if (!(tol >= 0.0) || max_rounds < 0) return fail(p, VMAT_EINVAL, "tol and max_rounds must be >= 0");
    int rc;
    if ((rc = ensure_state(p))) return rc;
    if ((rc = ensure_columns(p))) return rc;
    auto test = [&](double &ratio) -> int {
        int r = launch_rate_ratio(p, rho, p->rate_ratio);
        if (r) return r;
        VMAT_CUDA(p, cudaMemcpyAsync(&ratio, p->rate_ratio, sizeof(double), cudaMemcpyDeviceToHost, p->stream));
        VMAT_CUDA(p, cudaStreamSynchronize(p->stream));
        return VMAT_OK;
    };
    double ratio = 0.0;
    if ((rc = test(ratio))) return rc;
    int32_t rounds = 0, inner_total = 0;
    while (ratio > 1.0 + tol && rounds < max_rounds) {
        p->gamma *= factor;                          // "gamma ... will be automatically increased"
        if (!std::isfinite(p->gamma)) return fail(p, VMAT_ESTATE, "gamma overflowed while enforcing the dose-rate limit");
        if ((rc = launch_master(p, -1, 0, (int)(p->N - unoccupied(p))))) return rc;  // "the intensity for each aperture will be re-optimized"
        MasterOut h;
        VMAT_CUDA(p, cudaMemcpyAsync(&h, p->mout, sizeof(MasterOut), cudaMemcpyDeviceToHost, p->stream));
        if ((rc = test(ratio))) return rc;           // "till the solution is feasible"
        inner_total += h.inner;
        ++rounds;
    }
    double c3[3];
    VMAT_CUDA(p, cudaMemcpyAsync(c3, p->cost3, sizeof(c3), cudaMemcpyDeviceToHost, p->stream));
    VMAT_CUDA(p, cudaStreamSynchronize(p->stream));
    if (out) {
        out->rounds = rounds;
        out->feasible = ratio <= 1.0 + tol ? 1 : 0;
        out->inner_total = inner_total;
        out->gamma = p->gamma;
        out->ratio = ratio;
        out->F = c3[0];
        out->G = c3[1];
        out->cost = c3[2];
    }
    return VMAT_OK;
}

int vmat_solve(vmat_plan *p, int32_t max_iters, vmat_solve_stats *out) {
    if (!p) return VMAT_EINVAL;
    if (max_iters < 0) return fail(p, VMAT_EINVAL, "max_iters must be >= 0");
    const int64_t n_free0 = unoccupied(p);
    int64_t todo = n_free0;
    if (todo > max_iters) todo = max_iters;
    int rc;
    cudaStream_t st = p->stream;
    const bool phases = p->opt.record_phases != 0;
    cudaEvent_t ev0 = nullptr, ev1 = nullptr;
    std::vector<cudaEvent_t> evs;
    VMAT_CUDA(p, cudaEventCreate(&ev0));
    VMAT_CUDA(p, cudaEventCreate(&ev1));
    auto cleanup = [&]() {
        cudaEventDestroy(ev0);
        cudaEventDestroy(ev1);
        for (cudaEvent_t e : evs) cudaEventDestroy(e);
    };
    if (phases) {
        evs.resize((size_t)todo * 5);
        for (auto &e : evs) {
            cudaError_t ce = cudaEventCreate(&e);
            if (ce != cudaSuccess) {
                e = nullptr;
                cleanup();
                return cuda_fail(p, ce, "cudaEventCreate");
            }
        }
    }
#define TRY(call)           \
    if ((rc = (call))) {    \
        cleanup();          \
        return rc;          \
    }
#define TRYC(call)                                   \
    {                                                \
        cudaError_t ce__ = (call);                   \
        if (ce__ != cudaSuccess) {                   \
            cleanup();                               \
            return cuda_fail(p, ce__, #call);        \
        }                                            \
    }
    TRYC(cudaMemsetAsync(p->mcount, 0, 128, st));
    TRYC(cudaEventRecord(ev0, st));
    TRY(ensure_state(p));
    TRY(ensure_columns(p));   // the master needs d_k of every occupied beam, whichever path formed z
    int64_t done = 0;
    for (int64_t it = 0; it < todo; ++it) {
        if (phases) TRYC(cudaEventRecord(evs[it * 5 + 0], st));
        TRY(launch_price_spmv(p, p->w_s, p->g, (int)(n_free0 - it)));              // (c)
        if (phases) TRYC(cudaEventRecord(evs[it * 5 + 1], st));
        if (p->opt.stop_when_priced_out) {
            // option of reading S5: look at the best price before committing (one host round trip)
            TRY(launch_leaf_search(p, p->g, nullptr, nullptr, nullptr, 0, -1));
            Sel h_sel;
            TRYC(cudaMemcpyAsync(&h_sel, p->sel, sizeof(Sel), cudaMemcpyDeviceToHost, st));
            TRYC(cudaStreamSynchronize(st));
            if (h_sel.beam < 0 || !(h_sel.price < 0.0)) break;
        }
        TRY(launch_leaf_search(p, p->g, nullptr, nullptr, nullptr, 1, (int)it));   // (d), commits
        if (phases) TRYC(cudaEventRecord(evs[it * 5 + 2], st));
        TRY(launch_column_build(p, -1));                                           // d_k of the new aperture
        if (phases) TRYC(cudaEventRecord(evs[it * 5 + 3], st));
        TRY(launch_master(p, (int)it, p->warm_ok ? 1 : 0, (int)(p->N - n_free0 + it + 1)));                      // (e), leaves z, w current
        p->warm_ok = true;
        if (phases) TRYC(cudaEventRecord(evs[it * 5 + 4], st));
        done = it + 1;
    }
    todo = done;
    TRYC(cudaEventRecord(ev1, st));
    TRYC(cudaStreamSynchronize(st));
    TRYC(cudaGetLastError());
    // bring the host mirror up to date
    std::vector<uint8_t> before = p->h_occ;
    TRY(refresh_host_occ(p));
    for (int64_t k = 0; k < p->N; ++k)
        if (p->h_occ[k] && !before[k]) p->col_valid[k] = 1;
    if (out) {
        out->iters = (int32_t)todo;
        float ms = 0.f;
        TRYC(cudaEventElapsedTime(&ms, ev0, ev1));
        out->us_total = (double)ms * 1e3;
        out->us_price = out->us_search = out->us_column = out->us_master = 0.0;
        if (phases)
            for (int64_t it = 0; it < todo; ++it) {
                float a = 0, b = 0, c = 0, d = 0;
                cudaEventElapsedTime(&a, evs[it * 5 + 0], evs[it * 5 + 1]);
                cudaEventElapsedTime(&b, evs[it * 5 + 1], evs[it * 5 + 2]);
                cudaEventElapsedTime(&c, evs[it * 5 + 2], evs[it * 5 + 3]);
                cudaEventElapsedTime(&d, evs[it * 5 + 3], evs[it * 5 + 4]);
                out->us_price += a * 1e3;
                out->us_search += b * 1e3;
                out->us_column += c * 1e3;
                out->us_master += d * 1e3;
            }
        double c3[3];
        TRYC(cudaMemcpy(c3, p->cost3, sizeof(c3), cudaMemcpyDeviceToHost));
        out->F = c3[0];
        out->G = c3[1];
        out->cost = c3[2];
        unsigned long long mc[16];
        TRYC(cudaMemcpy(mc, p->mcount, sizeof(mc), cudaMemcpyDeviceToHost));
        out->master_passes = (double)mc[1];
        out->master_bytes = (double)mc[0] * (double)(kChunk * 4);
        out->master_cg_steps = (double)mc[2];
        out->master_clk_cg = (double)mc[3];
        out->master_clk_wait = (double)mc[4];
        out->master_clk_load = (double)mc[5];
        const size_t n = (size_t)todo;
        if (n) {
            if (out->beam) TRYC(cudaMemcpy(out->beam, p->tr_beam, n * 4, cudaMemcpyDeviceToHost));
            if (out->price) TRYC(cudaMemcpy(out->price, p->tr_price, n * 8, cudaMemcpyDeviceToHost));
            if (out->trace_F) TRYC(cudaMemcpy(out->trace_F, p->tr_F, n * 8, cudaMemcpyDeviceToHost));
            if (out->trace_G) TRYC(cudaMemcpy(out->trace_G, p->tr_G, n * 8, cudaMemcpyDeviceToHost));
            if (out->trace_cost) TRYC(cudaMemcpy(out->trace_cost, p->tr_cost, n * 8, cudaMemcpyDeviceToHost));
            if (out->inner) TRYC(cudaMemcpy(out->inner, p->tr_inner, n * 4, cudaMemcpyDeviceToHost));
        }
    }
#undef TRY
#undef TRYC
    cleanup();
    return todo == 0 && unoccupied(p) == 0 ? VMAT_DONE : VMAT_OK;
}

int vmat_get_plan(vmat_plan *p, uint8_t *occupied, int32_t *left, int32_t *right, double *y) {
    if (!p) return VMAT_EINVAL;
    cudaStream_t st = p->stream;
    const size_t N = (size_t)p->N, NR = (size_t)(p->N * p->R);
    if (occupied) VMAT_CUDA(p, cudaMemcpyAsync(occupied, p->occ, N, cudaMemcpyDeviceToHost, st));
    if (left) VMAT_CUDA(p, cudaMemcpyAsync(left, p->left, NR * 4, cudaMemcpyDeviceToHost, st));
    if (right) VMAT_CUDA(p, cudaMemcpyAsync(right, p->right, NR * 4, cudaMemcpyDeviceToHost, st));
    if (y) VMAT_CUDA(p, cudaMemcpyAsync(y, p->y, N * 8, cudaMemcpyDeviceToHost, st));
    VMAT_CUDA(p, cudaStreamSynchronize(st));
    return VMAT_OK;
}

int vmat_set_plan(vmat_plan *p, const uint8_t *occupied, const int32_t *left, const int32_t *right, const double *y) {
    if (!p) return VMAT_EINVAL;
    if (!occupied || !left || !right || !y) return fail(p, VMAT_EINVAL, "occupied, left, right, y must not be NULL");
    const int64_t N = p->N, R = p->R, C = p->C;
    int64_t prev = -1;
    for (int64_t k = 0; k < N; ++k) {
        if (!std::isfinite(y[k])) return fail(p, VMAT_EINVAL, "y must be finite");
        if (!occupied[k]) continue;
        if (y[k] < 0.0) return fail(p, VMAT_EINVAL, "y must be >= 0");
        for (int64_t r = 0; r < R; ++r) {
            const int64_t l = left[k * R + r], rr = right[k * R + r];
            if (l < 0 || l > rr || rr > C) return fail(p, VMAT_EINVAL, "leaf pairs must satisfy 0 <= left <= right <= n_cols");
            if (prev >= 0) {
                const int64_t b = (int64_t)p->delta * (k - prev);
                const int64_t dl = l - left[prev * R + r], dr = rr - right[prev * R + r];
                if (dl > b || -dl > b || dr > b || -dr > b)
                    return fail(p, VMAT_EINVAL, "leaf pairs break the leaf-travel limit between successive occupied beams");
            }
        }
        prev = k;
    }
    std::vector<double> yy((size_t)N);
    std::vector<uint8_t> oo((size_t)N);
    for (int64_t k = 0; k < N; ++k) {
        oo[k] = occupied[k] ? 1 : 0;
        yy[k] = oo[k] ? y[k] : 0.0;
    }
    cudaStream_t st = p->stream;
    VMAT_CUDA(p, cudaMemcpyAsync(p->occ, oo.data(), (size_t)N, cudaMemcpyHostToDevice, st));
    VMAT_CUDA(p, cudaMemcpyAsync(p->left, left, (size_t)(N * R) * 4, cudaMemcpyHostToDevice, st));
    VMAT_CUDA(p, cudaMemcpyAsync(p->right, right, (size_t)(N * R) * 4, cudaMemcpyHostToDevice, st));
    VMAT_CUDA(p, cudaMemcpyAsync(p->y, yy.data(), (size_t)N * 8, cudaMemcpyHostToDevice, st));
    VMAT_CUDA(p, cudaStreamSynchronize(st));
    p->h_occ = oo;
    p->col_valid.assign((size_t)N, 0);
    p->state_valid = false;
    p->warm_ok = false;
    int rc = reset_hessian(p);
    if (rc) return rc;
    return launch_free_list(p);
}

int64_t vmat_launch_count(const vmat_plan *p) { return p ? p->launches : 0; }

const char *vmat_last_error(const vmat_plan *p) { return p ? p->err.c_str() : g_create_error.c_str(); }

}  // extern "C"
