/*
 * vmat.h — C ABI of the B200-native column-generation VMAT hot path.
 *
 * Method: Men, Romeijn, Jia, Jiang, "Ultra-fast treatment plan optimization for VMAT"
 * (arxiv 1005.4396).  Citations "PAPER.md:N" are lines of the paper text; "S<n>" are the
 * readings of DESIGN.md section 3 taken where the paper is silent.
 *
 * One column-generation iteration is
 *   (a) dose      z_j = sum_k y_k sum_{i in A_k} D_ij
 *   (b) gradient  w_j = dF/dz_j of the one-sided quadratic penalty (Eq. 1),
 *                 s_k = gamma dG/dy_k of the dose-rate smoothing term (Eq. 2)
 *   (c) pricing   g_i = sum_j D_ij w_j for every beamlet of every un-occupied beam
 *   (d) search    per leaf row the contiguous open interval of least total price inside the
 *                 leaf-travel box, per-beam sum, best un-occupied beam
 *   (e) master    min_{y>=0} F(z(y)) + gamma G(y) over the generated apertures by gradient
 *                 projection                                        (Eq. 3 :86-91)
 * Every step runs in hand-written sm_100a CUDA kernels on ONE GPU.  There is no CPU fallback:
 * without a CUDA device every compute entry point returns VMAT_ECUDA.
 *
 * Conventions
 *   sizes      V voxels, N beams (gantry angles), R leaf rows per beam, C beamlets per row,
 *              B = N*R*C beamlets; beamlet id i = (k*R + r)*C + c.
 *   leaves     a row's pair (left, right) = (l, r'), integers in [0, C]; column c is open iff
 *              l <= c < r'; l == r' is a closed row parked at l (S8).
 *   pointers   every pointer argument is marked HOST or DEVICE.  DEVICE pointers must belong to
 *              the CUDA device that was current when vmat_create ran.
 *   stream     all device work of a plan is ordered on the cudaStream_t given to vmat_create
 *              (NULL = legacy default stream).  Calls that return host values synchronise that
 *              stream before returning; the others are stream-ordered.
 *   ownership  the caller owns every array it passes.  vmat_create copies / re-lays-out its
 *              inputs and keeps no caller pointer.  The plan owns the device memory it
 *              allocates and frees it in vmat_destroy.  Output buffers are caller-allocated.
 *   threads    a plan is not thread-safe; different plans are independent.
 *   errors     every call returns an int: VMAT_OK, VMAT_DONE, or a negative code; no exception
 *              crosses the boundary; on error the out-parameters are unspecified but no memory
 *              is leaked.  vmat_last_error gives a message.
 */
#ifndef VMAT_H
#define VMAT_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define VMAT_OK       0
#define VMAT_DONE     1   /* nothing to do: every beam already holds an aperture               */
#define VMAT_EINVAL  (-1) /* null pointer, bad size, malformed CSR, NaN/Inf, negative weights,  */
                          /* non-ascending theta, leaf pairs outside [0,C] or breaking travel   */
#define VMAT_ENOMEM  (-2) /* host or device allocation failed                                   */
#define VMAT_ECUDA   (-3) /* CUDA runtime error (message carries the CUDA error string)         */
#define VMAT_ESTATE  (-4) /* call not valid in the plan's current state                         */

#define VMAT_HOST    0
#define VMAT_DEVICE  1

#define VMAT_MAX_COLS 255  /* C <= 255: one warp scans one leaf row                             */

typedef struct vmat_plan vmat_plan;          /* opaque; owns all device state */

/* The optimisation problem of PAPER.md:69-93. */
typedef struct {
    int64_t n_voxels, n_beams, n_rows, n_cols;   /* V, N, R, C                                   */
    /* D, the dose-deposition matrix, beamlet-major CSR.  mem_space says where
     * row_ptr/col_idx/val/T/alpha/beta live (all six in the same space).                      */
    const int64_t *row_ptr;   /* B+1, row_ptr[0] = 0, non-decreasing                            */
    const int32_t *col_idx;   /* nnz voxel ids in [0,V), strictly ascending within a row        */
    const float   *val;       /* nnz, finite                                                    */
    const float   *T;         /* V prescription / threshold dose T_j (Eq. 1)                    */
    const float   *alpha;     /* V underdose weight alpha_j >= 0                                */
    const float   *beta;      /* V overdose weight  beta_j  >= 0                                */
    const double  *theta_deg; /* HOST, N gantry angles in degrees, strictly ascending (S4)      */
    int32_t max_leaf_travel;  /* Delta >= 0: beamlets a leaf may move per angular step (S6)     */
    double  gamma;            /* weight of the smoothing term, >= 0 (Eq. 3)        */
    int32_t mem_space;        /* VMAT_HOST or VMAT_DEVICE                                       */
} vmat_problem;

/* Tunables.  Zero-initialise, then call vmat_default_options. */
typedef struct {
    int32_t validate;          /* 1: check the CSR and the voxel arrays on the device (default 1) */
    int32_t d_format;          /* device storage of D for the pricing product: 0 = fp32 value + 32-bit voxel slot per
                                  entry (8 bytes: the fp32-CSR layout of BASELINE.json north_star, default);
                                  1 = a second copy in aligned slot pairs with 16-bit pair ids (about 6 bytes per
                                  entry and 0.6 gathers of the gradient per entry, a separate
                                  format: same fp32 values, same products, the sums in another order).  Costs
                                  about 0.8 x the memory of D on top.                                    */
    int32_t dose_path;         /* how vmat_dose forms z: 0 from the aperture-dose columns d_k the
                                  master keeps (default), 1 straight from D (fixed-point atomics)  */
    double  master_eps;        /* stop when max|projected gradient| <= eps*max(1, value at entry);
                                  default 1e-4 (S11: chosen against whole plans of the oracle) */
    int32_t master_max_inner;  /* cap on inner iterations of one master solve                     */
    double  master_stall_rel;  /* a step that lowers the cost by <= this fraction of it is a stall:
                                  the decrease is below what fp32 dose arithmetic resolves.  Once a
                                  solve has lowered the cost by more than 1 % (a start far from the
                                  optimum) the fraction is applied 100x more strictly              */
    int32_t master_stall_count;/* stop after this many stalls in a row (stop_reason 4)            */
    int32_t record_phases;     /* 1: vmat_solve brackets each phase with CUDA events              */
    int32_t master_mode;       /* how step (e) reaches the minimiser (same minimiser either way, S11):
                                  0 = gradient projection with conjugate directions: two passes over the aperture-dose
                                      columns and two grid barriers per inner iteration;
                                  1 = (default) semismooth Newton on the reduced problem: F is piecewise quadratic, so
                                      the master problem restricted to the current piece is a quadratic in the K <= N
                                      dose rates with matrix 2 Dc diag(omega) Dc^T + 2 gamma L; that matrix is kept
                                      on the device from solve to solve (updated only where a voxel crossed its T_j),
                                      one thread block solves the K-dimensional box-constrained quadratic by conjugate
                                      gradients on its faces, the other blocks evaluate the true cost and gradient at
                                      the point it proposes: two or three passes per solve instead of about twenty.
                                      Needs n_beams <= 512 (one thread per beam) and, at each launch, K <= 256 occupied
                                      beams whose K x K fp32 matrix fits the block's shared memory next to 11 N
                                      doubles (K <= 212 at N = 360); a launch past that runs mode 0's kernel from
                                      the point the solve before it left, and so does every launch after it.          */
    int32_t stop_when_priced_out; /* vmat_solve stops as soon as the best aperture's price is >= 0 (the textbook
                                  column-generation stop).  Default 0: the loop goes on until every beam holds an
                                  aperture, as the paper wants (reading S5).  With 1 the
                                  call synchronises the stream once per iteration to read the price.             */
    int32_t master_unstaged_lists; /* 1 (default): aperture-dose columns that do not fit a master block's shared-memory
                                  tile are walked through per-chunk lists; 0: through masked loops over all such
                                  columns (the fallback the kernel takes by itself when the lists do not fit;
                                  exposed so that tests can reach it).  Same results.                            */
    int32_t occupied_only_G;   /* reading of Eq. 2 (S2): 0 (default) = the sum runs over all N gantry
                                  angles with y_k = 0 at un-occupied beams; 1 = over successive OCCUPIED beams only (an
                                  un-occupied beam is not part of the arc yet).  With 1 an aperture's price carries the
                                  derivative of G with its beam put into the arc, a beam that enters at y_k = 0 changes
                                  G, and the post-master cost of vmat_solve is no longer guaranteed non-increasing.
                                  vmat_enforce_dose_rate tests all N - 1 successive pairs in either reading.          */
    int32_t master_newton_max_beams; /* 0 (default): mode 1 runs while the occupied beams fit its solving block (above);
                                  > 0: and while there are at most this many of them (lets a small test reach the
                                  hand-over to mode 0's kernel; same minimiser either way).                          */
} vmat_options;

/* One deliverable aperture: a beam and one leaf pair per row. */
typedef struct {
    int32_t beam;       /* chosen beam k, -1 if none                                            */
    double  price;      /* its reduced cost: sum of row minima + gamma dG/dy_k (S10)            */
    int32_t *left;      /* HOST, R entries, caller-allocated                                    */
    int32_t *right;     /* HOST, R entries, caller-allocated                                    */
} vmat_aperture;

typedef struct {
    int32_t inner;          /* inner iterations done (mode 1: Newton steps taken)               */
    int32_t backtracks;     /* step halvings                                                    */
    int32_t stop_reason;    /* 0 converged, 1 iteration cap, 2 no descent, 3 line search failed,
                               4 decrease below fp32 resolution, 5 non-finite value,
                               6 internal hand-over timed out                                   */
    int32_t passes;         /* passes over the columns, each ended by a grid barrier            */
    double  pg_entry, pg_exit;   /* max |projected gradient| at entry / exit                    */
    double  F, G, cost;     /* at exit: F, G and F + gamma G                                    */
} vmat_master_stats;

typedef struct {
    int32_t iters;          /* outer iterations done                                            */
    double  us_total;       /* device time of the whole call (CUDA events)                      */
    double  us_price, us_search, us_column, us_master;  /* per phase, only if record_phases     */
    double  F, G, cost;     /* after the last master solve                                      */
    /* optional per-iteration trace, HOST, caller-allocated with max_iters entries, or NULL    */
    int32_t *beam;          /* chosen beam                                                      */
    double  *price;         /* its price                                                        */
    double  *trace_F, *trace_G, *trace_cost;   /* after each master solve                       */
    int32_t *inner;         /* master inner iterations                                          */
    /* bookkeeping of the master kernel over the call (algorithmic traffic of step e):                  */
    double  master_passes;  /* passes over the aperture-dose columns, each ended by a grid barrier      */
    double  master_bytes;   /* bytes of the touched 512-byte column segments those passes multiplied    */
    /* master_mode 1 only: the block that solves the reduced problems                                           */
    double  master_cg_steps;   /* conjugate-gradient steps on the K-dimensional quadratics                     */
    double  master_clk_cg, master_clk_wait, master_clk_load;   /* its SM clock cycles in those steps, waiting
                                  for the passes of the other blocks, and loading the reduced Hessian           */
} vmat_solve_stats;

typedef struct {
    int64_t n_voxels, n_beams, n_rows, n_cols, n_beamlets;
    int64_t nnz;            /* entries of D as given                                            */
    int64_t nnz_padded;     /* entries of the device layout (rows padded to multiples of 4)     */
    int64_t n_support;      /* voxels with a non-empty column of D                              */
    int64_t device_bytes;   /* device memory owned by the plan                                  */
    int64_t pricing_bytes;  /* bytes of D (values, indices, row starts) a pricing product over all rows streams */
} vmat_info;

void vmat_default_options(vmat_options *opt);

/* Build a plan from the problem statement of PAPER.md:69-93: validate, upload, re-lay-out D
 * (beamlet-major CSR, rows padded to 16-byte multiples, voxel ids compacted to the support of
 * D), allocate all state.  The plan starts empty: no beam occupied, y = 0, z = 0 (S1).
 * stream: a cudaStream_t (void*).  *out is set only on VMAT_OK.                               */
int vmat_create(const vmat_problem *problem, const vmat_options *options /* NULL = defaults */,
                void *cuda_stream, vmat_plan **out);
int vmat_destroy(vmat_plan *plan);                      /* NULL-safe */

/* Device memory of all plans comes from one stream-ordered pool per device, which keeps what vmat_destroy
 * frees so that the next vmat_create costs no driver allocation.  vmat_release_memory returns everything the
 * pools hold beyond live plans to the driver.  Thread-safe.                                              */
int vmat_release_memory(void);
int vmat_get_info(const vmat_plan *plan, vmat_info *out);

/* Steps (a)+(b) for the plan's current apertures and dose rates.
 * z_dev / w_dev: DEVICE, V floats, or NULL.  cost: HOST, {F, G, F + gamma G}, or NULL.        */
int vmat_dose(vmat_plan *plan, float *z_dev, float *w_dev, double cost[3]);

/* Steps (a)+(b) again, even if the plan's z and w are current: dose_path 0 = z = sum_k y_k d_k from
 * the aperture-dose columns, 1 = z = sum_k y_k sum_{i in A_k} D_i. straight from the CSR rows of
 * the exposed beamlets, -1 = the plan's option.  Stream-ordered, no host sync;
 * read the result with vmat_dose.  Exists so that the two layouts can be timed and compared.   */
int vmat_dose_recompute(vmat_plan *plan, int dose_path);

/* Steps (b)->(c)->(d): prices of all beamlets of un-occupied beams from the
 * current penalty gradient, the row search, the beam choice.
 *   w_override_dev  DEVICE V floats or NULL: use this gradient instead of the plan's own
 *   g_override_dev  DEVICE B floats or NULL: skip the product and search these prices
 *   g_out_dev       DEVICE B floats or NULL: receives the prices (0 at occupied beams)
 *   out             receives the chosen aperture (may be NULL when commit = 1)
 *   commit          0 report only; 1 occupy the beam with this aperture, y_k = 0
 * Returns VMAT_DONE (out->beam = -1) when no beam is un-occupied.                             */
int vmat_price(vmat_plan *plan, const float *w_override_dev, const float *g_override_dev,
               float *g_out_dev, vmat_aperture *out, int commit);

/* Step (c) alone: g = D w for the beamlets of un-occupied beams (0 elsewhere).
 * w_dev DEVICE V floats (NULL = plan's own gradient), g_dev DEVICE B floats.  Stream-ordered. */
int vmat_price_spmv(vmat_plan *plan, const float *w_dev, float *g_dev);

/* Step (d) alone on given prices: row optimum of every un-occupied beam.
 *   g_dev DEVICE B floats; all_left_dev / all_right_dev DEVICE N*R int32 (untouched at occupied
 *   beams), beam_price_dev DEVICE N doubles (+inf at occupied beams); any output may be NULL.
 * Stream-ordered; nothing is committed.                                                      */
int vmat_leaf_search(vmat_plan *plan, const float *g_dev, int32_t *all_left_dev,
                     int32_t *all_right_dev, double *beam_price_dev);

/* Per-call overrides of the master tunables of vmat_options; a field <= 0 keeps the plan's value. */
typedef struct {
    double  eps;            /* stop when max|projected gradient| <= eps*max(1, value at entry)          */
    int32_t max_inner;      /* cap on inner iterations                                                   */
    double  stall_rel;      /* see vmat_options.master_stall_rel                                         */
    int32_t stall_count;    /* see vmat_options.master_stall_count                                       */
} vmat_master_opts;

/* Step (e): solve model (3) for y >= 0 over the occupied beams, warm-started
 * from the plan's y.  Leaves z, w current.  opts may be NULL (the plan's options); out may be NULL.
 * y is kept in double precision on both sides of the boundary: the dose rates carry the plan from one
 * solve to the next, and fp32 would add 6e-8 relative noise per hand-over to a 1e-4 stop test.        */
int vmat_master(vmat_plan *plan, const vmat_master_opts *opts, vmat_master_stats *out);

/* The column-generation loop (S5): up to max_iters iterations of
 * price -> search -> occupy -> master, continuing from the plan's current state.  All iterations
 * are enqueued without a host round trip; the call synchronises once at the end.             */
int vmat_solve(vmat_plan *plan, int32_t max_iters, vmat_solve_stats *out);

/* Variant (PAPER.md:159 names "the maximum and minimum dose rate constraints" and leaves them out of "this
 * preliminary work"; reading R4): from now on step (e) solves model (3) over the box
 * y_min <= y_k <= y_max at the occupied beams (un-occupied beams deliver nothing: y_k = 0), by gradient
 * projection on that box.  Default 0, +infinity = the paper's y >= 0.  Applies to vmat_master, vmat_solve and
 * vmat_enforce_dose_rate; the plan's y is brought into the box by the next master solve.  A beam that enters
 * at y_min > 0 changes the cost on entry, so the post-master cost of vmat_solve is guaranteed non-increasing
 * only for y_min = 0.  Requires 0 <= y_min <= y_max, y_min finite.                                         */
int vmat_set_dose_rate_bounds(vmat_plan *plan, double y_min, double y_max);

/* Hard dose-rate feasibility after the last aperture ("if the final solution is not
 * feasible, the coefficient gamma in the objective function will be automatically increased and then
 * the intensity for each aperture will be re-optimized till the solution is feasible").  The constraint
 * ("the dose rate variation between neighboring angles is constrained within a certain
 * range") is read as |y_{k+1} - y_k| <= max_variation_per_deg * (theta_{k+1} - theta_k), k = 1..N-1
 * (R1-R3).  ratio = max_k |y_{k+1}-y_k| / (max_variation_per_deg (theta_{k+1}-theta_k));
 * while ratio > 1 + tol and fewer than max_rounds rounds were spent: gamma *= gamma_factor, step (e)
 * runs again (warm start).  The plan's y is tested first: a feasible plan costs zero rounds.  The
 * plan keeps the gamma at exit.  out may be NULL.  Requires max_variation_per_deg > 0,
 * gamma_factor > 1, tol >= 0, max_rounds >= 0.  Synchronises the stream once per round.       */
typedef struct {
    int32_t rounds;         /* times gamma was raised and the master re-solved                  */
    int32_t feasible;       /* 1 if ratio <= 1 + tol at exit                                    */
    int32_t inner_total;    /* master inner iterations over all rounds                          */
    double  gamma;          /* gamma at exit = gamma at entry * gamma_factor^rounds             */
    double  ratio;          /* at exit                                                          */
    double  F, G, cost;     /* at exit, cost = F + gamma G with the gamma at exit               */
} vmat_rate_stats;
int vmat_enforce_dose_rate(vmat_plan *plan, double max_variation_per_deg, double gamma_factor, double tol,
                           int32_t max_rounds, vmat_rate_stats *out);

/* Plan state: occupied mask (N bytes), leaf pairs (N*R each), dose rates (N doubles); all HOST.
 * vmat_set_plan validates 0 <= l <= r' <= C and the leaf-travel invariant between successive
 * occupied beams.  Any pointer of vmat_get_plan may be NULL.                                  */
int vmat_get_plan(vmat_plan *plan, uint8_t *occupied, int32_t *left, int32_t *right, double *y);
int vmat_set_plan(vmat_plan *plan, const uint8_t *occupied, const int32_t *left, const int32_t *right,
                  const double *y);

/* Dose-deposition matrix on the device: a stand-in for the paper's GPU dose engine ("We calculate D_ij's
 * using our in-house dose calculation engine implemented on a ... GPU", ref 17, a finite-size pencil-beam engine that is
 * another paper).  It evaluates the ray / Gaussian / exponential model of BASELINE.json:configs:
 * parallel rays in the axial plane, gantry axis = grid z through the grid centre, beam k at k 360/n_beams degrees,
 * D = exp(-mu depth) exp(-rho^2 / 2 sigma^2) (1 + noise U(-1,1)) inside a body cylinder of radius body_radius_mm,
 * sigma = sigma_beamlets x beamlet_mm, support rho <= 4.5 sigma, entries below cutoff x (row maximum) dropped, U a
 * counter-based hash of (seed, beamlet, voxel).  Voxel j = (iz ny + iy) nx + ix, beamlet i = (k n_rows + r) n_cols + c.
 * Outputs: DEVICE arrays owned by the caller afterwards (release each with vmat_engine_free), beamlet-major CSR with
 * strictly ascending voxel ids in a row, ready for vmat_create with mem_space = VMAT_DEVICE.  Synchronises the stream
 * once (the number of entries decides the allocation).  Input generation only: none of the method's arithmetic.     */
typedef struct {
    int32_t nx, ny, nz;          /* voxel grid, x fastest                                        */
    double  voxel_mm;
    int32_t n_beams, n_rows, n_cols;
    double  beamlet_mm;
    double  body_radius_mm, mu_per_mm, sigma_beamlets, noise, cutoff;
    uint64_t seed;
} vmat_engine_geometry;
int vmat_engine_dose_matrix(const vmat_engine_geometry *geometry, void *cuda_stream, int64_t **row_ptr_dev,
                            int32_t **col_idx_dev, float **val_dev, int64_t *nnz);
int vmat_engine_free(void *dev_ptr, void *cuda_stream);

/* Step (b) alone, allocation free (Eq. 1): w_j = dF/dz_j and F = sum_j alpha_j max(0, T_j - z_j)^2 +
 * beta_j max(0, z_j - T_j)^2 for a caller's dose vector, for callers that cannot call cudaMalloc (code under CUDA graph
 * capture, tight serving loops).  No plan is needed and nothing is allocated, by this call or by a library routine under
 * it: the per-block partial sums of F live in a fixed array in the library's device image (64 KB + 256 B, held by every
 * GPU that loads the library until the process exits), which bounds the size: n_voxels > VMAT_NOALLOC_MAX_VOXELS returns
 * VMAT_EINVAL and launches nothing.
 *   z_dev, T_dev, alpha_dev, beta_dev   DEVICE, n_voxels floats, memory of the CURRENT device (checked for z_dev)
 *   w_dev   DEVICE n_voxels floats or NULL;  F_dev   DEVICE one double or NULL (not both NULL)
 * Stream-ordered on cuda_stream, no host synchronisation; F is summed in a fixed order (the same bits every call).
 * Every call on a device shares that device's array, which keeps the last call's contents (the call clears what must
 * start at zero): two calls that OVERLAP on one GPU (different streams, or two graphs in flight) race on it and give a
 * wrong F - serialise them.  The first call on a device looks the array's address up (cudaGetSymbolAddress): make it
 * outside stream capture.  Errors: VMAT_EINVAL / VMAT_ECUDA, text from vmat_last_error(NULL).                       */
#define VMAT_NOALLOC_MAX_VOXELS (1 << 24)
int vmat_penalty_noalloc(const float *z_dev, const float *T_dev, const float *alpha_dev, const float *beta_dev,
                         int64_t n_voxels, float *w_dev, double *F_dev, void *cuda_stream);

/* Number of kernel launches this plan has issued since vmat_create (bench bookkeeping).     */
int64_t vmat_launch_count(const vmat_plan *plan);

const char *vmat_last_error(const vmat_plan *plan);     /* NULL plan: the last create error  */

#ifdef __cplusplus
}
#endif
#endif /* VMAT_H */
