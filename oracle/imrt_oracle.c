/*
 * oracle/imrt_oracle.c -- the ORACLE: a plain, serial, fp64 CPU implementation of the
 * hot path of Men et al., "GPU-based ultra fast IMRT plan optimization" (arXiv 0908.4421).
 *
 * THIS IS TEST INFRASTRUCTURE.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call it.  It shares no code,
 * header, table or helper with the CUDA library (paper_0908_4421_b200/csrc) and neither
 * includes the other.  It is deliberately slow and unblocked: every function is the paper's
 * definition written out, in the paper's order, so that it can be checked by eye.
 *
 * What it follows (line numbers are /root/reference/PAPER.md):
 *   model      : PAPER.md:51-66   section 2.1, Eq. (1)-(2)   z_j = sum_i D_ij x_i ; one-sided quadratic penalties
 *   projection : PAPER.md:90      section 2.2                P(y) = max(0, y)
 *   Armijo     : PAPER.md:92-95   section 2.2, Eq. (5)       C_k = G(x_k) - (eps/lambda) ||x_{k+1} - x_k||^2
 *   algorithm  : PAPER.md:99-112  "Main Iterative Loop" steps 1-5
 *   stop rule  : PAPER.md:112-114 step 5, delta
 *
 * Readings where the paper is silent or garbled:
 *   R1  F_j = F_j^- "U" F_j^+  is read as the SUM of the two terms.
 *   R2  Weighted, per-structure generalisation: F_j = w-_s max(0, T-_s - z_j)^2 + w+_s max(0, z_j - T+_s)^2,
 *       s = structure of voxel j.  The paper's model is w+ = 1 everywhere, w- = 1 on targets / 0 elsewhere,
 *       T- = T+ = T_j (BASELINE.json north_star asks for weights and separate limits).
 *   R3  Gradient (not printed in the paper): dG/dx_i = sum_j D_ij * 2 (w+ o_j - w- u_j); Eq. (1) has no 1/2.
 *   R4  Strict "<" in step 3 is kept; two STATIONARY exits (G_k == 0, or a first trial with zero step) and a
 *       cap max_ls on backtracking steps are added, because with "<" those cases never terminate.
 *   R5  Step 5 (operator lost in the text): |G_new - G_old| / G_new < delta with the newest pair.
 *   R6  lambda restarts at the fixed lambda0 every outer iteration.
 *   R7  "Run N iterations" = N accepted outer iterations.
 *   R16 Optional per-voxel limits T-_j / T+_j (the paper's own T_j) override the per-structure ones.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): brute-force dense D x; closed forms on hand cases; central
 * finite differences of G for the gradient; zero penalty when every voxel is at its bound; the hand-derived
 * two-trial trace on D = I; monotone decrease and Armijo invariants on the trace; KKT at convergence; agreement
 * of the converged objective with scipy.optimize.nnls when the model reduces to NNLS; scale invariance.
 * The numerical trajectory itself is "parity unpinned against the paper": the paper prints no worked example,
 * no eps / alpha / lambda0 and no iteration counts.
 *
 * Precision: fp64 throughout; D's fp32 values are promoted exactly.  (PAPER.md:179 says the authors ran in
 * single precision; BASELINE.json north_star fixes fp64 for the oracle.)
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

enum { ORACLE_STOP_MAX_ITERS = 0, ORACLE_STOP_TOLERANCE = 1, ORACLE_STOP_STATIONARY = 2, ORACLE_STOP_LS_STALLED = 3 };

/*
 * eval(x): dose, penalty, weighted residual, objective.        PAPER.md:51-66, readings R1-R3.
 *   d_j = sum_p val[p] * x[col[p]]                 (sequential, CSR order)
 *   u_j = max(0, T-_s - d_j) ; o_j = max(0, d_j - T+_s)
 *   G  += w-_s u_j^2 + w+_s o_j^2                  (plain left-to-right sum)
 *   r_j = 2 (w+_s o_j - w-_s u_j)
 * d and r may be NULL.
 *
 * Per-voxel limits (reading R16; "T_j for all j in V represents the dose distribution in the original
 * treatment plan", :195 cumulative-dose re-optimisation): when tv_under / tv_over are not NULL, voxel j uses
 * T-_j = tv_under[j] / T+_j = tv_over[j] instead of its structure's limits; the weights stay per structure.  The
 * paper's literal model is tv_under = tv_over = T_j with w- = 1 on targets, 0 elsewhere, and w+ = 1.
 */
void oracle_eval_v(int64_t n_v, const int32_t *row_ptr, const int32_t *col, const float *val, const uint8_t *sid,
                   const float *t_under, const float *t_over, const float *w_under, const float *w_over,
                   const float *tv_under, const float *tv_over,
                   const double *x, double *d, double *r, double *G_out) {
    double G = 0.0;
    for (int64_t j = 0; j < n_v; ++j) {
        double dj = 0.0;
        for (int64_t p = row_ptr[j]; p < row_ptr[j + 1]; ++p) dj += (double)val[p] * x[col[p]];
        const int s = sid[j];
        const double tu = tv_under ? (double)tv_under[j] : (double)t_under[s];
        const double to = tv_over ? (double)tv_over[j] : (double)t_over[s];
        const double u = fmax(0.0, tu - dj);
        const double o = fmax(0.0, dj - to);
        G += (double)w_under[s] * u * u + (double)w_over[s] * o * o;
        if (d) d[j] = dj;
        if (r) r[j] = 2.0 * ((double)w_over[s] * o - (double)w_under[s] * u);
    }
    *G_out = G;
}

void oracle_eval(int64_t n_v, const int32_t *row_ptr, const int32_t *col, const float *val, const uint8_t *sid,
                 const float *t_under, const float *t_over, const float *w_under, const float *w_over,
                 const double *x, double *d, double *r, double *G_out) {
    oracle_eval_v(n_v, row_ptr, col, val, sid, t_under, t_over, w_under, w_over, NULL, NULL, x, d, r, G_out);
}

/* grad(r): g = D^T r by scatter over the rows of D (the oracle never forms D^T).   Reading R3. */
void oracle_grad(int64_t n_v, int64_t n_b, const int32_t *row_ptr, const int32_t *col, const float *val,
                 const double *r, double *g) {
    for (int64_t i = 0; i < n_b; ++i) g[i] = 0.0;
    for (int64_t j = 0; j < n_v; ++j) {
        const double rj = r[j];
        for (int64_t p = row_ptr[j]; p < row_ptr[j + 1]; ++p) g[col[p]] += (double)val[p] * rj;
    }
}

/* Trial point x+ = P(x - lambda g) = max(0, x - lambda g) and Delta = ||x+ - x||^2.   PAPER.md:90, :109, Eq. (5). */
void oracle_trial_point(int64_t n_b, const double *x, const double *g, double lambda, double *x_new, double *delta_out) {
    double delta = 0.0;
    for (int64_t i = 0; i < n_b; ++i) {
        const double xn = fmax(0.0, x[i] - lambda * g[i]);
        const double dx = xn - x[i];
        delta += dx * dx;
        x_new[i] = xn;
    }
    *delta_out = delta;
}

/*
 * run: the Main Iterative Loop, with readings R4-R7.
 *
 *   delta_tol <= 0  : fixed-count mode, exactly max_iters accepted iterations unless STATIONARY / STALLED.
 *   follow_trials   : NULL = free-running.  Otherwise [max_iters] trial counts (>= 1) taken by another
 *                     implementation ("follow mode"): at iteration k the oracle accepts
 *                     the follow_trials[k]-th trial, after checking that this trial passes G+ < C and that every
 *                     earlier one fails it, each within slack tau_rel * G_k on (G+ - C).  Checks that do not hold
 *                     are counted in *n_follow_violations and the first such iteration goes to *first_violation.
 *
 * Outputs: x (in: x_1, out: last accepted iterate), obj[0..n] (G at x_1 .. x_{n+1}), lambda[k], n_trials[k],
 *          step_sq[k] (Delta of the accepted trial), margin[k] = (C - G+) / G_k of the accepted trial.
 * Returns the number of accepted iterations n.
 */
int oracle_run_v(int64_t n_v, int64_t n_b, const int32_t *row_ptr, const int32_t *col, const float *val,
               const uint8_t *sid, const float *t_under, const float *t_over, const float *w_under, const float *w_over,
               const float *tv_under, const float *tv_over,
               double eps, double alpha, double lambda0, double delta_tol, int max_ls, int max_iters,
               const int32_t *follow_trials, double tau_rel,
               double *x, double *obj, double *lambda_out, int32_t *n_trials, double *step_sq, double *margin,
               int *stop_reason, int *n_follow_violations, int *first_violation,
               int64_t *n_fwd_passes, int64_t *n_tr_passes) {
    double *g = (double *)malloc(sizeof(double) * (size_t)n_b);
    double *x_new = (double *)malloc(sizeof(double) * (size_t)n_b);
    double *r = (double *)malloc(sizeof(double) * (size_t)(n_v > 0 ? n_v : 1));
    double *r_new = (double *)malloc(sizeof(double) * (size_t)(n_v > 0 ? n_v : 1));
    int64_t fwd = 0, tr = 0;
    int viol = 0, first_viol = -1;
    int reason = ORACLE_STOP_MAX_ITERS;
    double G_k;

    oracle_eval_v(n_v, row_ptr, col, val, sid, t_under, t_over, w_under, w_over, tv_under, tv_over, x, NULL, r, &G_k);
    ++fwd;
    obj[0] = G_k;
    int k = 0; /* number of accepted iterations so far */
    while (k < max_iters) {
        /* step 1: d_k = -grad G(x_k) */
        oracle_grad(n_v, n_b, row_ptr, col, val, r, g);
        ++tr;
        if (G_k == 0.0) { reason = ORACLE_STOP_STATIONARY; break; }
        /* step 2: lambda = lambda0 */
        double lambda = lambda0, G_new = 0.0, delta = 0.0, C = 0.0;
        int m = 0, stop = 0;
        for (;;) {
            oracle_trial_point(n_b, x, g, lambda, x_new, &delta);
            if (m == 0 && delta == 0.0) { reason = ORACLE_STOP_STATIONARY; stop = 1; break; }
            oracle_eval_v(n_v, row_ptr, col, val, sid, t_under, t_over, w_under, w_over, tv_under, tv_over, x_new, NULL, r_new, &G_new);
            ++fwd;
            C = G_k - (eps / lambda) * delta; /* Eq. (5) */
            int accept;
            if (follow_trials) {
                const double slack = tau_rel * G_k;
                const int want_accept = (m + 1 == follow_trials[k]);
                const int ok = want_accept ? (G_new < C + slack) : (G_new >= C - slack);
                if (!ok) { ++viol; if (first_viol < 0) first_viol = k; }
                accept = want_accept;
            } else {
                accept = (G_new < C); /* step 3, strict as printed */
            }
            if (accept) break;
            ++m; /* step 4 */
            if (m > max_ls) { reason = ORACLE_STOP_LS_STALLED; stop = 1; break; }
            lambda = lambda / alpha;
        }
        if (stop) break;
        /* accept: x_{k+1} = x+ */
        memcpy(x, x_new, sizeof(double) * (size_t)n_b);
        { double *t = r; r = r_new; r_new = t; }
        obj[k + 1] = G_new;
        lambda_out[k] = lambda;
        n_trials[k] = m + 1;
        step_sq[k] = delta;
        margin[k] = (C - G_new) / G_k;
        const double G_old = G_k;
        G_k = G_new;
        ++k;
        /* step 5 */
        if (delta_tol > 0.0 && (G_new == 0.0 || fabs(G_new - G_old) / G_new < delta_tol)) { reason = ORACLE_STOP_TOLERANCE; break; }
    }
    *stop_reason = reason;
    if (n_follow_violations) *n_follow_violations = viol;
    if (first_violation) *first_violation = first_viol;
    if (n_fwd_passes) *n_fwd_passes = fwd;
    if (n_tr_passes) *n_tr_passes = tr;
    free(g); free(x_new); free(r); free(r_new);
    return k;
}

int oracle_run(int64_t n_v, int64_t n_b, const int32_t *row_ptr, const int32_t *col, const float *val,
               const uint8_t *sid, const float *t_under, const float *t_over, const float *w_under, const float *w_over,
               double eps, double alpha, double lambda0, double delta_tol, int max_ls, int max_iters,
               const int32_t *follow_trials, double tau_rel,
               double *x, double *obj, double *lambda_out, int32_t *n_trials, double *step_sq, double *margin,
               int *stop_reason, int *n_follow_violations, int *first_violation,
               int64_t *n_fwd_passes, int64_t *n_tr_passes) {
    return oracle_run_v(n_v, n_b, row_ptr, col, val, sid, t_under, t_over, w_under, w_over, NULL, NULL, eps, alpha, lambda0,
                        delta_tol, max_ls, max_iters, follow_trials, tau_rel, x, obj, lambda_out, n_trials, step_sq, margin,
                        stop_reason, n_follow_violations, first_violation, n_fwd_passes, n_tr_passes);
}

/*
 * Dose-volume-histogram points (plan evaluation; definition = SURVEY.md 8(c.2) #18):
 * per structure s, D_p = the ceil(p n_s / 100)-th largest dose among its voxels, and the mean dose.
 * out_dp is [n_structures][n_p]; structures without voxels give NaN.
 */
static int cmp_desc(const void *a, const void *b) {
    const double x = *(const double *)a, y = *(const double *)b;
    return (x < y) - (x > y);
}

void oracle_dvh(int64_t n_v, const uint8_t *sid, const double *d, int n_structures, const double *pcts, int n_p,
                double *out_dp, double *out_mean) {
    double *buf = (double *)malloc(sizeof(double) * (size_t)(n_v > 0 ? n_v : 1));
    for (int s = 0; s < n_structures; ++s) {
        int64_t n = 0;
        double sum = 0.0;
        for (int64_t j = 0; j < n_v; ++j)
            if (sid[j] == s) { buf[n++] = d[j]; sum += d[j]; }
        if (n == 0) {
            for (int q = 0; q < n_p; ++q) out_dp[s * n_p + q] = NAN;
            out_mean[s] = NAN;
            continue;
        }
        qsort(buf, (size_t)n, sizeof(double), cmp_desc);
        for (int q = 0; q < n_p; ++q) {
            int64_t rank = (int64_t)ceil(pcts[q] * (double)n / 100.0);
            if (rank < 1) rank = 1;
            if (rank > n) rank = n;
            out_dp[s * n_p + q] = buf[rank - 1];
        }
        out_mean[s] = sum / (double)n;
    }
    free(buf);
}

/*
 * Mixed-resolution row merging (section 3.1: "for unspecified tissue we increased the voxel size in each
 * dimension by a factor of 2"; reading R17): the rows of D that carry the same group id are replaced by ONE
 * row, their MEAN (the dose of the coarse voxel is the mean dose of the fine voxels it contains).  Written out plainly:
 * for every group, in ascending row order, add the rows into a dense fp64 accumulator over the n_b columns, divide by
 * the number of rows of the group, and emit the touched columns in ascending order, rounded to fp32.  A column counts
 * as touched if any row of the group stores it (a stored 0 is kept).
 *
 *   group[j]  in [0, n_groups) for every row j (groups need not be contiguous; a group without rows gives an empty row)
 * Two calls, as a caller that allocates the output must make them: oracle_merge_rows_count fills out_row_ptr
 * [n_groups + 1]; oracle_merge_rows_fill fills out_col / out_val [out_row_ptr[n_groups]].
 */
void oracle_merge_rows_count(int64_t n_v, int64_t n_b, const int32_t *row_ptr, const int32_t *col, const int32_t *group,
                             int64_t n_groups, int32_t *out_row_ptr) {
    unsigned char *mark = (unsigned char *)calloc((size_t)(n_b > 0 ? n_b : 1), 1);
    out_row_ptr[0] = 0;
    for (int64_t g = 0; g < n_groups; ++g) {
        int32_t cnt = 0;
        for (int64_t j = 0; j < n_v; ++j) {          /* plain and slow: every group scans every row */
            if (group[j] != g) continue;
            for (int64_t p = row_ptr[j]; p < row_ptr[j + 1]; ++p)
                if (!mark[col[p]]) { mark[col[p]] = 1; ++cnt; }
        }
        for (int64_t j = 0; j < n_v; ++j)
            if (group[j] == g)
                for (int64_t p = row_ptr[j]; p < row_ptr[j + 1]; ++p) mark[col[p]] = 0;
        out_row_ptr[g + 1] = out_row_ptr[g] + cnt;
    }
    free(mark);
}

void oracle_merge_rows_fill(int64_t n_v, int64_t n_b, const int32_t *row_ptr, const int32_t *col, const float *val,
                            const int32_t *group, int64_t n_groups, const int32_t *out_row_ptr, int32_t *out_col, float *out_val) {
    unsigned char *mark = (unsigned char *)calloc((size_t)(n_b > 0 ? n_b : 1), 1);
    double *acc = (double *)calloc((size_t)(n_b > 0 ? n_b : 1), sizeof(double));
    for (int64_t g = 0; g < n_groups; ++g) {
        int64_t size = 0;
        for (int64_t j = 0; j < n_v; ++j) {          /* ascending row order: the order of the fp64 additions */
            if (group[j] != g) continue;
            ++size;
            for (int64_t p = row_ptr[j]; p < row_ptr[j + 1]; ++p) { mark[col[p]] = 1; acc[col[p]] += (double)val[p]; }
        }
        int64_t q = out_row_ptr[g];
        for (int64_t c = 0; c < n_b; ++c) {
            if (!mark[c]) continue;
            out_col[q] = (int32_t)c;
            out_val[q] = (float)(acc[c] / (double)size);
            ++q;
            mark[c] = 0;
            acc[c] = 0.0;
        }
    }
    free(mark);
    free(acc);
}
