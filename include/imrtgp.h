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
 *   - Results of one plan are bit-reproducible from run to run (fixed-order reductions; the only atomics on the data
 *     path add INTEGERS, which commute).  With imrt_options.tune_level = 0 (the default) two plans of the same problem
 *     also agree bit for bit.  tune_level >= 1 balances the passes over the SMs from MEASURED pass times; the partition
 *     fixes the order in which objective partials are summed, so two tuned plans may differ in the last bits of the
 *     objective -- unless the second one is given the first one's partition (imrt_plan_get_tuning / host_tuning).
 *   - The library reads no environment variables: every switch is a field of imrt_params / imrt_options.
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
    IMRT_STOP_LINESEARCH_STALLED = 3,    /* more than max_ls backtracking steps; x_k kept                        */
    IMRT_STOP_TRACE_FULL = 4,            /* the trace (imrt_params.max_iters accepted iterations since imrt_plan_set_x)
                                            filled up before the requested number of iterations was done          */
    IMRT_STOP_PEER_TIMEOUT = 5           /* persistent driver: a wait inside the kernel -- on the other CTAs of the launch or,
                                            for a row-sharded plan, on a peer rank's partial sums -- was not answered within
                                            imrt_options.spin_timeout_ms.  The kernel left its loop instead of hanging the
                                            device; the iterate is no longer valid.  Runs are refused (they return at once
                                            with this stop reason) until the next imrt_plan_set_x; the inboxes of a sharded
                                            group must be zero-filled and imrt_plan_set_shard called again first.        */
} imrt_stop_reason;

/* Line-search / loop parameters (PAPER.md:92 "two parameters 0 < eps < 1 and alpha > 1", :103, :114). */
typedef struct imrt_params {
    double eps;          /* Armijo parameter, 0 < eps < 1                                                        */
    double alpha;        /* backtracking divisor, > 1:  lambda <- lambda / alpha (step 4)                        */
    double lambda0;      /* step size every line search starts from (step 2), > 0                                */
    int32_t max_ls;      /* cap on backtracking steps per iteration (reading R4), >= 0                           */
    int32_t max_iters;   /* trace capacity: the total number of accepted iterations between two imrt_plan_set_x  */
    int32_t driver;      /* who runs the loop (all three give bit-identical results):
                            0  CUDA graph with nested conditional WHILE nodes (one cudaGraphLaunch per run, no host
                               sync per step; one transpose pass and ceil(trials / ls_batch) dose passes per iteration)
                            1  host-driven (one launch and one sync per pass; for debugging and per-kernel profiling)
                            2  ONE cooperative persistent kernel holding the whole loop (the fast path; what the
                               Python binding and bench.py use).  Needs all n_sm CTAs co-resident: 576 threads and up
                               to 227 KB of shared memory each, i.e. an otherwise idle device.                        */
    int32_t ls_batch;    /* line-search trial points evaluated per pass over D: 1, 2 or 4 (0 = default, 4).  The
                            trials lambda, lambda/alpha, ... are the ones steps 2-4 visit one at a time; a batch
                            evaluates the next ls_batch of them in ONE dose pass (D is streamed once, each trial point
                            gets its own D x+ and objective) and step 3 is then applied to them in order, so the
                            iterates, step sizes and trial counts are bit-identical for every ls_batch.  The library
                            lowers it when the trial vectors would not fit in shared memory (imrt_plan_get_info).  */
} imrt_params;

/*
 * Layout / tuning switches of imrt_plan_create (all 0 = the defaults; pass NULL for all defaults).  None of them
 * changes what is computed, only how the matrices are laid out and the work is split.
 */
typedef struct imrt_options {
    int32_t tune_level;        /* 0: partitions from the cost model only -- plan creation is timing independent and two
                                     plans of one problem give the same bits;
                                  1: + rebalance both passes from measured per-CTA times of isolated launches;
                                  2: + a few more rounds measured inside the device-resident loop (bench.py uses this) */
    int32_t dose_format;       /* 0: quad records where smaller (4 neighbouring rows share a column list), else rows;
                                  1: row-format records only                                                          */
    int32_t col_bits;          /* 0: 16-bit column indices when n_b <= 65,536;  32: always 32-bit                     */
    int32_t transpose_format;  /* 0: smallest of {row pairs, single rows} with 16-bit voxel offsets, else plain CSR;
                                  1: single rows with 16-bit offsets (no pairs);  2: the plain 32-bit D^T CSR         */
    int32_t quad_cap;          /* union columns per quad record at most (0 = default, 384; clamped to [32, 4096])     */
    int32_t n_ctas;            /* CTAs of the persistent passes: 0 = one per SM of the device; fewer leaves SMs to other work
                                  (or to other ranks of a row-sharded problem sharing the device, imrt_plan_run_ranks)   */
    int32_t profile_create;    /* 1: synchronise after every phase of plan creation and keep the phase times for
                                  imrt_plan_get_create_times                                                           */
    int32_t spin_timeout_ms;   /* bound, in milliseconds, on every wait inside the persistent kernel (grid barrier, peer
                                  ranks' flags): 0 = default, 2000.  On expiry the run ends with IMRT_STOP_PEER_TIMEOUT          */
    const void* host_tuning;   /* a blob written by imrt_plan_get_tuning for the same problem, options and device: the
                                  plan takes its partitions from it instead of measuring (tune_level is ignored)       */
    size_t host_tuning_bytes;
} imrt_options;

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
 *   host_options                  copied; NULL = defaults
 *   workspace / workspace_bytes   device memory from the caller, >= imrt_workspace_bytes(...)  (borrowed)
 *   stream                        a cudaStream_t passed as void* (NULL = the legacy default stream)
 * Validates the inputs (finite values, columns in range and strictly ascending in every row), re-packs D into the
 * block records the dose pass streams, builds the explicit transpose D^T as a second CSR (stable radix sort by
 * column) and the packed stream the transpose pass reads, splits both passes over the SMs (cost model; with
 * imrt_options.tune_level >= 1 refined from measured pass times: a few short runs of the passes and of the loop on
 * x = 0), and instantiates the iteration graph (driver 0).  Synchronises the stream.  DESIGN.md section 4 describes
 * the layouts.
 * Limits (IMRT_STATUS_UNSUPPORTED): sizes must fit int32; a row of D may hold at most 8,192 entries; the R trial
 * vectors (4 R n_b bytes), the gradient (4 n_b) and two of the largest block records must fit in the 227 KB of shared
 * memory of one CTA -- R is lowered from 4 to 2 to 1 first, which leaves room for about 25,000 beamlets.
 * On failure *out is NULL unless the status is a validation error that left a handle for imrt_last_error;
 * imrt_last_error(NULL) returns the message of the last failed create on this thread.
 */
imrt_status imrt_plan_create(imrt_plan** out, int64_t n_v, int64_t n_b, int64_t nnz,
                             const int32_t* row_ptr, const int32_t* col_idx, const float* val,
                             const uint8_t* structure_id, int32_t n_structures,
                             const float* host_t_under, const float* host_t_over,
                             const float* host_w_under, const float* host_w_over,
                             const imrt_params* host_params, const imrt_options* host_options,
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
 * The line search's batched dose pass as a parity hook: evaluate n_points (1, 2 or 4) given points in ONE pass over D,
 * exactly as the loop evaluates a batch of trial points (the R = n_points instantiation of the kernels).
 *   x         fp32 [n_points][n_b]  the points, one after the other                           (device)
 *   r         fp32 [n_points][n_v]  weighted residual of every point, or NULL                 (device)
 *   host_obj  fp64 [n_points]       G of every point
 * The optimiser state is not touched.  Synchronises.
 */
imrt_status imrt_plan_eval_batch(imrt_plan* plan, int32_t n_points, const float* x, float* r, double* host_obj);

/*
 * g = D^T r for an arbitrary r (fp32 [n_v], device) -> g (fp32 [n_b], device): one transpose pass, the optimiser state is
 * not touched.  A parity hook (the transpose pass in isolation); with imrt_plan_eval and imrt_trial_point it is also all a
 * host-driven loop over row slabs needs (tests/host_sharded_loop.py restates the sharded protocol that way).  Asynchronous.
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
 * kind 2 / 3: the read-only STREAMING CEILING of the dose / transpose pass -- the same producers move every byte the
 * pass reads through the same shared-memory ring / stages, the consumer warps only wait and release (no arithmetic, no
 * gathers, no stores).  What the pass could reach if its consumers were free (kind 3: row-pair stream only).
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

/*
 * The partitions of the two passes as an opaque blob, for imrt_options.host_tuning of a later plan of the same problem
 * (same D, options and device): that plan skips the measurements and reproduces this plan's results bit for bit.
 * *host_bytes receives the size; the blob is written if host_buf is not NULL and capacity suffices
 * (IMRT_STATUS_INVALID_ARG otherwise).  Host only.
 */
imrt_status imrt_plan_get_tuning(imrt_plan* plan, void* host_buf, size_t capacity, size_t* host_bytes);

/*
 * Phase times of imrt_plan_create in milliseconds (only with imrt_options.profile_create = 1, else *host_n = 0):
 *   [0] validation  [1] quad union counts  [2] record layout  [3] record packing  [4] transpose (sort + gather)
 *   [5] D^T stream packing, ranges  [6] state, first schedule  [7] dose-pass tuning  [8] transpose-pass tuning  [9] graph
 */
imrt_status imrt_plan_get_create_times(imrt_plan* plan, double* host_ms, int32_t capacity, int32_t* host_n);

/*
 * Row-sharded problems (the paper is single-GPU): rank q of `world` holds a contiguous slab
 * of rows of D -- one plan per rank, created from the slab's CSR with the FULL beamlet count -- and the loop sums the
 * partial gradients (once per iteration) and the partial objectives (once per batch of trial points) over the ranks
 * INSIDE the persistent kernel: every rank pushes its partial into every rank's inbox (peer memory; NVLink stores), raises
 * a sequence flag, and adds what its own inbox holds in rank order, so all ranks compute the same bits and take the same
 * Armijo decisions with no broadcast.
 *   imrt_shard_inbox_bytes  size of one rank's inbox for n_b beamlets and `world` ranks (host arithmetic)
 *   imrt_plan_set_shard     host_inboxes [world]: device pointers to EVERY rank's inbox as this rank's device can address
 *                           them (its own included; peers' through peer access / IPC / symmetric memory), 16-byte
 *                           aligned, zero-filled before EVERY imrt_plan_set_shard (the call restarts the plan's exchange
 *                           counters at zero; all ranks of a group must be set up against the same freshly zeroed inboxes)
 *                           and never touched by the caller afterwards.  All arguments are validated before anything is
 *                           changed: a refused call leaves the plan as it was.
 *                           world = 1 returns to a stand-alone plan.  Persistent driver only.  Call imrt_plan_set_x after.
 * Every rank then calls imrt_plan_set_x (the same x0) and imrt_plan_run_iters / _run_to_tol (the same arguments); the
 * traces of all ranks are identical and hold the objective of the WHOLE problem; imrt_plan_get_dose / _eval / _dvh stay
 * per slab.
 *   imrt_plan_run_ranks     the same for ranks that are CO-RESIDENT on one device (plans created with
 *                           imrt_options.n_ctas = SMs / ranks on one stream): ONE cooperative launch runs all of them --
 *                           ranks wait on one another, so separate launches on one device could deadlock.  host_plans [n_ranks]
 *                           in rank order; they must agree in ls_batch, max_iters and n_b (checked) and must all be at the
 *                           same iteration (every rank got the same imrt_plan_set_x / run calls; not checked).  Asynchronous.
 * Failure detection: no wait inside the kernel is unbounded.  A peer that never launched, died, or runs a different number
 * of exchanges makes the waiting rank give up after imrt_options.spin_timeout_ms, mark the exchange as failed in every
 * rank's inbox (so the surviving ranks stop at once as well) and end its run with IMRT_STOP_PEER_TIMEOUT.
 */
imrt_status imrt_shard_inbox_bytes(int64_t n_b, int32_t world, size_t* host_bytes);
imrt_status imrt_plan_set_shard(imrt_plan* plan, int32_t rank, int32_t world, void* const* host_inboxes);
imrt_status imrt_plan_run_ranks(imrt_plan* const* host_plans, int32_t n_ranks, int32_t n_iters, double delta);

/*
 * Mixed-resolution row merging (section 3.1: "for unspecified tissue we increased the voxel size in each
 * dimension by a factor of 2"; reading R17).  The rows of D whose group_id is equal are replaced by ONE row,
 * their mean -- the dose of a coarse voxel is the mean dose of the fine voxels it contains.  Merged row g holds every
 * column some row of group g stores, ascending, with value (sum over the group's rows in ascending row order, fp64) /
 * (rows in the group), rounded to fp32; a group without rows gives an empty row.  The result is a CSR the caller owns and
 * can hand to imrt_plan_create; the full-resolution D stays available for plan evaluation (imrt_plan_eval / _dvh).
 *   group_id     int32 [n_v]          0 <= group_id < n_groups; the rows of a group need not be neighbours   (device)
 *   out_row_ptr  int32 [n_groups + 1]                                                                         (device)
 *   out_col      int32 [nnz_out], out_val fp32 [nnz_out]                                                      (device)
 *   workspace    >= imrt_merge_rows_workspace_bytes(n_v, n_groups); the SAME workspace, unmodified, for both calls
 * imrt_merge_rows_count checks the raw input first -- group ids in range (IMRT_STATUS_INVALID_ARG), row_ptr[0] = 0 and
 * non-decreasing, every column in [0, n_b) (IMRT_STATUS_BAD_CSR): this call runs BEFORE imrt_plan_create has seen the
 * matrix --, then sorts the rows by group, counts every merged row, fills out_row_ptr and returns nnz_out
 * (synchronises); the caller allocates out_col / out_val and calls imrt_merge_rows_fill (asynchronous).
 * Limits: n_b up to about 390,000 (the column bitmap of one group must fit 24 KB of shared memory).
 */
imrt_status imrt_merge_rows_workspace_bytes(int64_t n_v, int64_t n_groups, size_t* host_bytes);
imrt_status imrt_merge_rows_count(int64_t n_v, int64_t n_b, const int32_t* row_ptr, const int32_t* col_idx, const int32_t* group_id,
                                  int64_t n_groups, int32_t* out_row_ptr, int64_t* host_nnz_out, void* workspace, size_t workspace_bytes,
                                  void* stream);
imrt_status imrt_merge_rows_fill(int64_t n_v, int64_t n_b, const int32_t* row_ptr, const int32_t* col_idx, const float* val,
                                 int64_t n_groups, const int32_t* out_row_ptr, int32_t* out_col, float* out_val, void* workspace,
                                 size_t workspace_bytes, void* stream);

/*
 * Dose-volume-histogram points of ANY dose on the device, for callers that cannot give the library memory to work in.
 * Same definition and same kernels as imrt_plan_dvh (D_p = the ceil(p n_s / 100)-th largest dose of
 * a structure's n_s voxels, plus the mean dose), but no plan and no workspace: the histograms, counters and partial sums
 * live in an array that is part of the library image itself.  The call and everything under it makes no cudaMalloc,
 * cudaFree or other allocating CUDA call.  Who needs that: an application that has already handed all device memory to
 * its own pool (a planning server that sizes its buffers once, a process sharing the GPU under a fixed memory budget),
 * so that a further cudaMalloc would fail; and code in a latency-sensitive stretch, where the device-wide
 * synchronisation hidden in cudaMalloc / cudaFree would stall work on other streams.
 *   dose          fp32  [n_v]   any finite doses, e.g. from imrt_plan_get_dose or a full-resolution D x      (device)
 *   structure_id  uint8 [n_v]   < n_structures (checked: IMRT_STATUS_BAD_STRUCTURE)                           (device)
 *   host_pcts     fp64  [n_pcts] percent of the structure's volume;  host_dp [n_structures][n_pcts], host_mean
 *                 [n_structures] as for imrt_plan_dvh (NaN for a structure without voxels)                    (host)
 *   stream        a cudaStream_t as void* of the CURRENT device (NULL = the legacy default stream)
 * Limits (IMRT_STATUS_UNSUPPORTED, with the numbers in imrt_last_error(NULL)): n_structures <= 16, n_pcts <= 16,
 * n_structures * n_pcts <= 128, n_v <= 2^30.  The built-in array is 1,128,704 bytes (about 1.1 MB); every device on
 * which the library's code is loaded keeps that much until the process exits, whether or not this call is ever made.
 * Larger problems: imrt_plan_dvh, whose scratch is in the caller's workspace.
 * First call on a device: looks up the array's address on that device (once; the device must be current) -- make that
 * first call before starting any stream capture.
 * Sharing: all calls on a device use the one array, and it still holds what the previous call left behind; the call
 * clears what has to start from zero.  Two calls running on the GPU at the same time would corrupt each other's
 * histograms, so the call holds a library-wide lock and returns only after its stream has drained (it synchronises).
 */
imrt_status imrt_dvh_static(const float* dose, const uint8_t* structure_id, int64_t n_v, int32_t n_structures,
                            const double* host_pcts, int32_t n_pcts, double* host_dp, double* host_mean, void* stream);

/* Message of the last error on this plan (or of the last failed imrt_plan_create when plan is NULL).
 * Owned by the library, valid until the next call on the same plan / thread. */
const char* imrt_last_error(const imrt_plan* plan);

/* Release host-side resources (graph, events).  Device memory belongs to the caller. */
imrt_status imrt_plan_destroy(imrt_plan* plan);

/* Library version string, e.g. "imrtgp 0.2 (sm_100a)". */
const char* imrt_version(void);

#ifdef __cplusplus
}
#endif
#endif /* IMRTGP_H */
