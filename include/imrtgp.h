/*
 * imrtgp.h -- C-ABI of libimrtgp: gradient-projection IMRT fluence-map optimiser for one NVIDIA B200 (sm_100a).
 *
 * The library implements the hot path of Men et al., "GPU-based ultra fast IMRT plan optimization"
 * (arXiv 0908.4421; line numbers below are /root/reference/PAPER.md):
 *
 *   model      PAPER.md:51-66   sec. 2.1, Eq. (1)-(2)   dose z = D x, one-sided quadratic voxel penalties
 *   iteration  PAPER.md:78-90   sec. 2.2, Eq. (3)-(4)   x_{k+1} = P(x_k - lambda_k grad G(x_k)),  P(y) = max(0, y)
 *   Armijo     PAPER.md:92-95   sec. 2.2, Eq. (5)       C_k = G(x_k) - (eps/lambda) ||x_{k+1} - x_k||^2
 *   loop       PAPER.md:99-114  "Main Iterative Loop" steps 1-5, stop tolerance delta
 *
 * with the weighted, per-structure generalisation BASELINE.json's north_star asks for:
 *
 *   d_j = sum_i D_ji x_i                                   (rows of D = voxels, columns = beamlets)
 *   u_j = max(0, t_under[s] - d_j),  o_j = max(0, d_j - t_over[s]),   s = structure_id[j]
 *   G(x) = sum_j  w_under[s] u_j^2 + w_over[s] o_j^2
 *   r_j  = 2 (w_over[s] o_j - w_under[s] u_j),   g = D^T r = grad G
 *
 * Conventions
 *   - Plain C, no exceptions cross the boundary.  Every call returns an imrt_status (0 = OK).
 *   - Pointers are DEVICE pointers unless the name starts with host_.  Device arrays must be 16-byte aligned.
 *   - The library never allocates device memory: the caller asks imrt_workspace_bytes(), allocates that many
 *     bytes (e.g. a torch tensor) and passes them to imrt_plan_create().  The plan BORROWS the caller's D
 *     arrays, structure_id and the workspace: they must outlive the plan and stay unmodified.
 *   - All device work is enqueued on the stream given at creation.  Calls documented "asynchronous" return
 *     without waiting for the device; calls that fill a host_ output synchronise that stream.
 *   - The plan handle is opaque and owned by the caller between imrt_plan_create and imrt_plan_destroy.
 *   - Results of one plan are bit-reproducible from run to run (fixed-order reductions, no floating-point atomics).
 *     Two plans of the same problem may differ in the last bits of the objective: plan creation balances the dose
 *     pass over the SMs from MEASURED pass times, and the partition fixes the order in which objective partials are
 *     summed.  Set the environment variable IMRTGP_NO_TUNE to keep the modelled partition (same bits every time).
 *   - There is no CPU fallback: on a machine without an sm_100 device imrt_plan_create fails with
 *     IMRT_STATUS_UNSUPPORTED_DEVICE / IMRT_STATUS_CUDA_ERROR.
 */
#ifndef IMRTGP_H
#define IMRTGP_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum imrt_status {
    IMRT_STATUS_OK = 0,
    IMRT_STATUS_INVALID_ARG = 1,         /* null pointer, negative size, misaligned array, bad parameter value   */
    IMRT_STATUS_BAD_CSR = 2,             /* row_ptr not monotone / row_ptr[0] != 0 / row_ptr[n_v] != nnz,
                                            a column >= n_b or < 0, columns not strictly ascending in a row,
                                            a non-finite value                                                    */
    IMRT_STATUS_BAD_STRUCTURE = 3,       /* structure_id >= n_structures, negative or non-finite weight / limit  */
    IMRT_STATUS_WORKSPACE_TOO_SMALL = 4,
    IMRT_STATUS_CUDA_ERROR = 5,          /* see imrt_last_error()                                                */
    IMRT_STATUS_UNSUPPORTED_DEVICE = 6,  /* device is not compute capability 10.x                                */
    IMRT_STATUS_UNSUPPORTED = 7,         /* problem shape outside what this build handles (see imrt_last_error)  */
    IMRT_STATUS_BAD_X = 8,               /* imrt_plan_set_x: a negative or non-finite beamlet intensity          */
    IMRT_STATUS_NOT_READY = 9            /* run / get called before imrt_plan_set_x                              */
} imrt_status;

/* Why the last run stopped (PAPER.md:112-114 step 5; reading R4 for the two extra exits). */
typedef enum imrt_stop_reason {
    IMRT_STOP_MAX_ITERS = 0,             /* the requested number of accepted iterations was done                 */
    IMRT_STOP_TOLERANCE = 1,             /* |G_new - G_old| / G_new < delta (or G_new == 0)                      */
    IMRT_STOP_STATIONARY = 2,            /* G(x_k) == 0, or the first trial point equals x_k                     */
    IMRT_STOP_LINESEARCH_STALLED = 3     /* more than max_ls backtracking steps; x_k kept                        */
} imrt_stop_reason;

/* Line-search / loop parameters (PAPER.md:92 "two parameters 0 < eps < 1 and alpha > 1", :103, :114). */
typedef struct imrt_params {
    double eps;          /* Armijo parameter, 0 < eps < 1                                                        */
    double alpha;        /* backtracking divisor, > 1:  lambda <- lambda / alpha (step 4)                        */
    double lambda0;      /* step size every line search starts from (step 2), > 0                                */
    int32_t max_ls;      /* cap on backtracking steps per iteration (reading R4), >= 0                           */
    int32_t max_iters;   /* trace capacity: the total number of accepted iterations between two imrt_plan_set_x  */
    int32_t driver;      /* 0: device-resident loop (CUDA graph with nested conditional WHILE nodes, no host sync
                               per step);  1: host-driven loop (one sync per trial; same kernels; for debugging)  */
    int32_t ls_batch;    /* line-search trial points evaluated per pass over D: 1, 2 or 4 (0 = default, 4).  The
                            trials lambda, lambda/alpha, ... are the ones steps 2-4 visit one at a time; a batch
                            evaluates the next ls_batch of them in ONE dose pass (D is streamed once, each trial point
                            gets its own D x+ and objective) and step 3 is then applied to them in order, so the
                            iterates, step sizes and trial counts are bit-identical for every ls_batch.  The library
                            lowers it when the trial vectors would not fit in shared memory (imrt_plan_get_info).  */
} imrt_params;

typedef struct imrt_plan imrt_plan;

/*
 * Bytes of device workspace imrt_plan_create needs for a problem of this shape (D^T CSR, its build scratch,
 * block tables, vectors, trace).  Pure host arithmetic, no device access.
 */
imrt_status imrt_workspace_bytes(int64_t n_v, int64_t n_b, int64_t nnz, int32_t n_structures, int32_t max_iters,
                                 size_t* host_bytes);

/*
 * Create a plan from the dose-deposition matrix D in CSR (rows = voxels, cols = beamlets).
 *   row_ptr      int32 [n_v+1]    row_ptr[0] = 0, non-decreasing, row_ptr[n_v] = nnz          (device, borrowed)
 *   col_idx      int32 [nnz]      0 <= col < n_b, strictly ascending within a row              (device, borrowed)
 *   val          fp32  [nnz]      finite                                                       (device, borrowed)
 *   structure_id uint8 [n_v]      < n_structures                                               (device, borrowed)
 *   host_t_under, host_t_over, host_w_under, host_w_over   fp32 [n_structures]  (host; copied). w >= 0, finite;
 *                                 w_under = 0 means no under-dose term for that structure.
 *   host_params                   copied
 *   workspace / workspace_bytes   device memory from the caller, >= imrt_workspace_bytes(...)  (borrowed)
 *   stream                        a cudaStream_t passed as void* (NULL = the legacy default stream)
 * Validates the inputs (finite values, columns in range and strictly ascending in every row), re-packs D into the
 * block records the dose pass streams, builds the explicit transpose D^T as a second CSR (stable radix sort by
 * column) and the packed stream the transpose pass reads, balances both passes over the SMs from measured pass times
 * (a few short runs of the passes and of the loop on x = 0), and instantiates the iteration graph (driver 0).
 * Synchronises the stream.  DESIGN.md section 4 describes the layouts.
 * On failure *out is NULL unless the status is a validation error that left a handle for imrt_last_error;
 * imrt_last_error(NULL) returns the message of the last failed create on this thread.
 */
imrt_status imrt_plan_create(imrt_plan** out, int64_t n_v, int64_t n_b, int64_t nnz,
                             const int32_t* row_ptr, const int32_t* col_idx, const float* val,
                             const uint8_t* structure_id, int32_t n_structures,
                             const float* host_t_under, const float* host_t_over,
                             const float* host_w_under, const float* host_w_over,
                             const imrt_params* host_params,
                             void* workspace, size_t workspace_bytes, void* stream);

/*
 * Set the current iterate x_1 ("Select initial solution x_1 >= 0").  x0: fp32 [n_b] (device).
 * Rejects negative / non-finite entries (IMRT_STATUS_BAD_X).  Evaluates G(x_1) and r(x_1) (one dose pass), resets
 * the trace, the iteration counter and the pass counters.  Synchronises (the validity check is read back).
 */
imrt_status imrt_plan_set_x(imrt_plan* plan, const float* x0);

/*
 * Optional per-voxel limits -- the paper's own model, in which T_j is the dose of the original plan in voxel j
 * or the desired cumulative dose minus the dose already delivered:
 *   u_j = max(0, t_under_v[j] - d_j),  o_j = max(0, d_j - t_over_v[j]);   the weights stay those of the voxel's structure.
 * t_under_v, t_over_v: fp32 [n_v] (device, borrowed until the next call or imrt_plan_destroy); either may be NULL
 * (= keep the structure's limit); both NULL returns to per-structure limits.  Invalidates the current iterate:
 * call imrt_plan_set_x afterwards.  Asynchronous.
 */
imrt_status imrt_plan_set_voxel_limits(imrt_plan* plan, const float* t_under_v, const float* t_over_v);

/*
 * Run n_iters more ACCEPTED gradient-projection iterations (steps 1-4 of PAPER.md:105-111, each with its own Armijo
 * line search) unless a STATIONARY / LINESEARCH_STALLED exit happens first.  No stop test (fixed-count mode).
 * Asynchronous: with driver = 0 this is one cudaGraphLaunch.  The trace must have room (max_iters).
 */
imrt_status imrt_plan_run_iters(imrt_plan* plan, int32_t n_iters);

/*
 * Run until step 5's test |G_new - G_old| / G_new < delta holds, or max_iters more accepted
 * iterations, or a STATIONARY / STALLED exit.  Asynchronous.
 */
imrt_status imrt_plan_run_to_tol(imrt_plan* plan, double delta, int32_t max_iters);

/*
 * Per-kernel parity hook: evaluate at an arbitrary x (fp32 [n_b], device) without touching the optimiser state.
 *   d  fp32 [n_v]  dose D x            r  fp32 [n_v]  weighted residual          (device; each may be NULL)
 *   g  fp32 [n_b]  gradient D^T r      host_obj       G(x)                        (may be NULL)
 * Runs the same dose / penalty / transpose kernels the loop runs.  Synchronises.
 */
imrt_status imrt_plan_eval(imrt_plan* plan, const float* x, float* d, float* r, float* g, double* host_obj);

/*
 * g = D^T r for an arbitrary r (fp32 [n_v], device) -> g (fp32 [n_b], device): one transpose pass, the optimiser state is
 * not touched.  With imrt_plan_eval (which leaves r(x)) and imrt_trial_point this is what a host-driven loop over
 * several plans -- one per row slab of D, on one GPU each -- is made of: the partial objectives and gradients of the
 * slabs add up (paper_0908_4421_b200/sharded.py).  Asynchronous.
 */
imrt_status imrt_plan_gradient(imrt_plan* plan, const float* r, float* g);

/*
 * The trial point of PAPER.md:90 / :109-111 outside a plan: x_out = max(0, x - lambda g) (fp32 [n_b], device) and
 * *step_sq = ||x_out - x||^2 (fp64, DEVICE pointer), summed in a fixed order.  stream: a cudaStream_t as void*.
 * Asynchronous.
 */
imrt_status imrt_trial_point(const float* x, const float* g, double lambda, int64_t n_b, float* x_out, double* step_sq, void* stream);

/*
 * The two scalar decisions of the loop for a HOST-driven loop (pure host arithmetic, the formulas the device loop uses):
 *   imrt_armijo_accepts  step 3 with Eq. (5): 1 iff G_new < G_k - (eps / lambda) step_sq
 *   imrt_stop_test       step 5 (reading R5): 1 iff delta > 0 and (G_new == 0 or |G_new - G_old| / G_new < delta)
 */
int32_t imrt_armijo_accepts(double G_k, double G_new, double step_sq, double eps, double lambda);
int32_t imrt_stop_test(double G_old, double G_new, double delta);

/* Copy the current iterate to x (fp32 [n_b], device).  Asynchronous. */
imrt_status imrt_plan_get_x(imrt_plan* plan, float* x);

/* d = D x at the current iterate (fp32 [n_v], device): one dose pass.  Asynchronous. */
imrt_status imrt_plan_get_dose(imrt_plan* plan, float* d);

/*
 * Dose-volume-histogram points of the current iterate (plan evaluation): for every structure s
 * and every host_pcts[q] (percent of the structure's volume), D_p = the ceil(p n_s / 100)-th largest dose among
 * the structure's voxels (rank clamped to [1, n_s]); plus the mean dose.  host_dp is [n_structures][n_pcts]
 * doubles (NaN for a structure without voxels), host_mean [n_structures].  Computed on the device from a dose
 * pass (per-structure histogram refinement, exact).  Synchronises.
 */
imrt_status imrt_plan_dvh(imrt_plan* plan, const double* host_pcts, int32_t n_pcts, double* host_dp, double* host_mean);

/*
 * Read back the trace since the last imrt_plan_set_x.  Synchronises.
 *   host_n_iters_done   accepted iterations n
 *   host_stop_reason    imrt_stop_reason of the last run
 *   host_obj      [n+1] G(x_1) .. G(x_{n+1})          host_lambda   [n] accepted step size
 *   host_n_trials [n]   trial points evaluated          host_step_sq  [n] ||x_{k+1} - x_k||^2
 *   capacity            arrays hold at least capacity (+1 for host_obj) entries; at most that many are written.
 * Any array pointer may be NULL.
 */
imrt_status imrt_plan_get_trace(imrt_plan* plan, int32_t* host_n_iters_done, int32_t* host_stop_reason,
                                double* host_obj, double* host_lambda, int32_t* host_n_trials, double* host_step_sq,
                                int32_t capacity);

/* Dose passes (D x + penalty; one pass evaluates up to ls_batch trial points) and transpose passes (D^T r) launched
 * since the last imrt_plan_set_x, including the pass that evaluated x_1.  Synchronises. */
imrt_status imrt_plan_get_counters(imrt_plan* plan, int64_t* host_fwd_passes, int64_t* host_tr_passes);

/*
 * Introspection for tests and the benchmark.  Synchronises.
 *   host_info[0] nnz of D^T        [1] dose-pass block records   [2] dose grid (CTAs)   [3] transpose grid (CTAs)
 *   host_info[4] dynamic shared memory bytes per CTA   [5] bytes of the re-packed D the dose pass streams
 *   host_info[6] gradient partial slots   [7] non-empty rows of D   [8] SM count   [9] 16-bit column indices (1/0)
 *   host_info[10] trial points per dose pass actually used (ls_batch)   [11] dose-pass ring bytes   [12] transpose stages
 *   host_info[13] rows of D stored in quad format (4 neighbouring rows sharing one column list)
 *   host_info[14] stream the transpose pass reads: 0 plain 32-bit CSR, 1 rows with 16-bit voxel offsets, 2 row pairs
 *   host_info[15] bytes of that stream
 * d_rowT_ptr (int32 [n_b+1]), d_colT (int32 [nnz]), d_valT (fp32 [nnz]): if non-NULL receive a copy of D^T (device).
 */
imrt_status imrt_plan_get_info(imrt_plan* plan, int64_t* host_info, int32_t n_info,
                               int32_t* d_rowT_ptr, int32_t* d_colT, float* d_valT);

/*
 * Launch ONE dose pass of the line search (kind 0: ls_batch trial points -- here copies of the current iterate --,
 * D x, penalty, residual, objective partials) or ONE transpose pass (kind 1: D^T r, partial-slot reduction) on the
 * plan's stream, n_repeat times back to back, on scratch outputs, without touching the optimiser state.  For
 * per-kernel timing / profiling only.  Asynchronous.
 */
imrt_status imrt_plan_launch_pass(imrt_plan* plan, int32_t kind, int32_t n_repeat);

/*
 * Per-CTA timing of the most recent dose (kind 0) or transpose (kind 1) pass: the global-timer nanoseconds at
 * which each persistent CTA started and finished streaming its share of the matrix.  Shows how well the static
 * partition is balanced.  host_start_ns / host_end_ns hold `capacity` entries; *host_n_ctas receives the grid size.
 * Synchronises.
 */
imrt_status imrt_plan_get_pass_timing(imrt_plan* plan, int32_t kind, int64_t* host_start_ns, int64_t* host_end_ns,
                                      int32_t capacity, int32_t* host_n_ctas);

/* Message of the last error on this plan (or of the last failed imrt_plan_create when plan is NULL).
 * Owned by the library, valid until the next call on the same plan / thread. */
const char* imrt_last_error(const imrt_plan* plan);

/* Release host-side resources (graph, events).  Device memory belongs to the caller. */
imrt_status imrt_plan_destroy(imrt_plan* plan);

/* Library version string, e.g. "imrtgp 0.1 (sm_100a)". */
const char* imrt_version(void);

#ifdef __cplusplus
}
#endif
#endif /* IMRTGP_H */
