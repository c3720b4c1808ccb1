/*
 * dualip.h -- C ABI of the B200-native dual-gradient hot path of the ridge-regularised matching-LP
 * solver of "Large-Scale Regularized Matching on GPU Clusters" (arxiv/paper_2606_07777).
 * Citations "P:n" are line numbers of the paper text; "R<n>" are the readings listed in
 * DESIGN.md section 2.
 *
 * Problem (Eq. 1; Def. 1):   min_{x in C} c'x + (gamma/2)|x|^2   s.t.  A x <= b
 *   x_ij for eligible (user i, item j) pairs, stored as per-user CSR rows; C = product over users of a
 *   simple set C_i (unit simplex, box, box-cut); A is m families of per-item coupling rows,
 *   (A x)_{j,k} = sum_i a^k_ij x_ij.
 * Dual (Eq. 2-4):  x*(lambda) = Proj_C(-(A'lambda + c)/gamma),  grad g = A x* - b,
 *   g(lambda) = c'x* + (gamma/2)|x*|^2 + lambda'(A x* - b).
 *
 * Conventions
 *   - Every entry point returns an int: DUALIP_OK (0) or a negative DUALIP_E* code.  Nothing throws,
 *     aborts or prints.  On error, outputs are left untouched and *out handles are set to NULL.
 *   - Layouts are item-major / family-minor: a[p*m+k], b[j*m+k], lambda[j*m+k], grad[j*m+k]  (R14).
 *   - Row data is int32 / fp32; lambda, grad g, g and all scalars are fp64.
 *   - "host or device": the pointer kind is detected with cudaPointerGetAttributes.  Device pointers are
 *     used in place, asynchronously on `stream`.  Host pointers are staged through internal device
 *     buffers and the call synchronises `stream` before returning.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).
 *   - The caller keeps ownership of every buffer it passes.  The handle owns its copies.
 *   - A handle must not be used from two host threads at once.
 *   - There is no CPU fallback: without a CUDA device every call fails with DUALIP_ECUDA.
 */
#ifndef DUALIP_H
#define DUALIP_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dualip dualip_t;

enum {
    DUALIP_OK = 0,
    DUALIP_EINVAL = -1,       /* bad argument: NULL, negative size, gamma <= 0, unknown enum, m out of range */
    DUALIP_ERANGE = -2,       /* row_ptr not monotone / row_ptr[0] != 0 / item index outside [0,J) */
    DUALIP_EDUP = -3,         /* an item appears twice in one user's row (R11) */
    DUALIP_ENOMEM = -4,       /* host or device allocation failed */
    DUALIP_ECUDA = -5,        /* a CUDA runtime call failed (no device, launch failure, ...) */
    DUALIP_EUNSUPPORTED = -6, /* valid request this build cannot serve (e.g. reduction strategy needs more shared memory) */
    DUALIP_ETOOBIG = -7,      /* dualip_grad_static only: J*m exceeds DUALIP_STATIC_MAX_DUALS, the compiled-in size of its scratch */
    DUALIP_ESTALE = -8,       /* sharded handle whose c was replaced: agree on the constants again (dualip_set_shard_constants) first */
    DUALIP_EHOOK = -9         /* the caller's reduce hook returned non-zero: the evaluation was abandoned, its partial sums discarded */
};

/* Per-user simple set C_i (R5, R10, R16).  Parameters p0,p1 of dualip_opts:
 *   SIMPLEX_INEQ {x>=0, sum x <= z}: p0 = z          SIMPLEX_EQ {x>=0, sum x = z}: p0 = z
 *   BOX {lo <= x <= hi}: p0 = lo, p1 = hi             BOXCUT {0<=x<=ub, sum x<=z}: p0 = ub, p1 = z   */
enum { DUALIP_PROJ_SIMPLEX_INEQ = 0, DUALIP_PROJ_BOX = 1, DUALIP_PROJ_BOXCUT = 2, DUALIP_PROJ_SIMPLEX_EQ = 3 };

/* Item-wise reduction strategy for s_{j,k} = sum_i a^k_ij x_ij (Eq. 4; P:123 in the paper this is
 * SpMV + NCCL reduce).  All strategies accumulate in 64-bit fixed point, so results are bit-reproducible
 * run to run and independent of the launch geometry.
 *   AUTO   : SMEM when lambda and the accumulators fit in shared memory, else GLOBAL.
 *   SMEM   : per-CTA shared-memory accumulators (native 32-bit integer atomics with explicit carry),
 *            flushed once per CTA with RED.ADD.64.
 *   GLOBAL : RED.ADD.64 straight to L2 for every nonzero x; lambda still gathered from shared memory
 *            when J*m*8 bytes fit, else through the read-only path.
 *   CSC    : no atomics: x is written to HBM and each item's column is summed in fixed order (fp64, chunks of 4096
 *            entries, fixed trees) through an item-sorted permutation built at create -- for J*m beyond on-chip
 *            capacity, and the mode whose summation ORDER is fixed.  Costs nnz*(4|8) bytes for the permutation,
 *            nnz*4 for x, and three more launches per evaluation.                                       */
enum { DUALIP_RED_AUTO = 0, DUALIP_RED_SMEM = 1, DUALIP_RED_GLOBAL = 2, DUALIP_RED_CSC = 3 };

/* Preconditioning of the dual ascent ("Jacobi preconditioning ... rescaling the complex constraints using the
 * diagonal of the Hessian proxy induced by A"; Appendix B.2: D = diag(1/|A_r*|_2), A' = D A, b' = D b,
 * D_rr = 1 for rows of zero norm).  R18:
 *   NONE   : eta = gamma / L for every coordinate (R2).
 *   JACOBI : the iteration of the row-scaled system, carried out in the ORIGINAL variables lambda = D lambda': a
 *            per-coordinate step  lambda+ = max(0, y + (gamma / L') d_r^2 grad_r),  d_r^2 = 1 / sum_i (a^k_ij)^2,
 *            L' = max_j #{k : row (j,k) of A is nonzero}  (= 1 for m = 1, where A'A'^T = I exactly).  No row data is
 *            rescaled, nothing changes per iteration but one multiply per dual; lambda in and out, grad g, the
 *            residuals and the trace stay in the original units.                                             */
enum { DUALIP_PRECOND_NONE = 0, DUALIP_PRECOND_JACOBI = 1 };

/* Step rule of dualip_solve ("a fixed step size that can be derived analytically from A and gamma"; "AGD step-size
 * range [1e-5, 1e-1]"; "we scale the maximum AGD step size proportionally with the decay of gamma").  R2, R20:
 *   FIXED    : eta_t = gamma_s / L_step for every iteration of stage s.
 *   ADAPTIVE : range-clipped secant step.  hi_s = eta_max gamma_s / gamma_1, lo_s = min(eta_min, gamma_s / L_step),
 *              clip(e) = min(max(e, lo_s), hi_s): the lower end of the range never lifts a step above the analytic one (the
 *              paper's [1e-5, 1e-1] is a range for the Jacobi-scaled system, where gamma_s / L' is of that size; on an unscaled
 *              system gamma_s / L_step can be 1e-7, and a step forced up to 1e-5 would be far beyond the stability bound).
 *              The upper end is NOT adjusted: without DUALIP_PRECOND_JACOBI choose eta_max relative to gamma_1 / L yourself.
 *              First iteration of a stage (or a 0/0 secant): eta_t = clip(gamma_s / L_step);
 *              afterwards eta_t = clip(|y_t - y_{t-1}|_2 / |grad_t - grad_{t-1}|_2), the inverse of the secant estimate of the
 *              local Lipschitz constant of grad g along the last move; both norms in the system being iterated on (the
 *              row-scaled one under DUALIP_PRECOND_JACOBI).  The paper prints no formula: parity unpinned against it. */
enum { DUALIP_STEP_FIXED = 0, DUALIP_STEP_ADAPTIVE = 1 };

/* Tuning / test overrides of the launch plan; all zero = the library's choice.  stages, tile_units, lambda_plan and step_deal
 * do not change a result bit.  direct_kernel does, within the parity tolerances: k_grad forms w from the fp64 lambda and sums a
 * row's projection in another lane order than the streaming kernel (the fixed-point item sums are order-free in both). */
typedef struct {
    int32_t direct_kernel; /* 1: force the direct-load kernel k_grad instead of the streaming one (parity tests of both) */
    int32_t stages;        /* pipeline stages of the streaming kernel (2..4) */
    int32_t tile_units;    /* cap on its tile size in units (>= 256) */
    int32_t lambda_plan;   /* exact-path dual operand of the streaming kernel: 0 = chosen per launch, 1 = never stage
                              lambda's low word in shared memory, 2 = always stage it when it fits */
    int32_t step_deal;     /* how a tile's row-steps are dealt to the consumer warps: 0 = the library's choice, 1 = statically
                              (round-robin over the CTA's step sequence), 2 = dynamically (claimed from a counter) */
} dualip_tuning;

typedef struct {
    int32_t projection;   /* DUALIP_PROJ_* */
    double  p0, p1;       /* projection parameters, see above */
    int32_t reduction;    /* DUALIP_RED_* */
    int32_t borrow;       /* 1: device inputs are used in place and must outlive the handle; 0: copied */
    int32_t validate;     /* 1: check index range, monotone row_ptr, duplicates (a0); 0: trust the caller */
    int32_t momentum;     /* 1: beta_t = t/(t+3) (R1); 0: plain projected ascent (beta = 0) */
    int32_t group_lanes;  /* lanes cooperating on one row: 0 = auto from the mean row length, or 4/8/16/32 */
    int32_t grid_ctas;    /* CTAs of the gradient kernel: 0 = auto (SM count x resident CTAs per SM) */
    int32_t use_graph;    /* 1: dualip_solve replays a CUDA graph of 20 chained iteration launches per stage (stages of >= 40
                             iterations; ignored while profiling is on or with DUALIP_RED_CSC); 0: direct launches */
    dualip_tuning tuning; /* launch-plan overrides, see above */
    int32_t precondition; /* DUALIP_PRECOND_*: how dualip_solve scales its step (dualip_grad is not affected) */
    int32_t step_rule;    /* DUALIP_STEP_* */
    double  eta_min;      /* DUALIP_STEP_ADAPTIVE: the clip range [eta_min, eta_max gamma_s / gamma_1]; 0 < eta_min <= eta_max */
    double  eta_max;
} dualip_opts;

/* Fills *opts with the defaults: unit simplex (inequality), AUTO reduction, copy, validate, momentum, fixed step
 * (eta_min = 1e-5, eta_max = 1e-1 -- the paper's range, P:185 -- are filled in but unused until step_rule is ADAPTIVE). */
void dualip_opts_default(dualip_opts* opts);

/* Scalars of one evaluation (Eq. 2; "objective value and regularization term"; "slack"; R9). */
typedef struct {
    double g;      /* dual objective g(lambda) = obj + reg + lambda'grad */
    double obj;    /* c'x* */
    double reg;    /* (gamma/2)|x*|^2 */
    double r_inf;  /* max(0, max_jk grad_jk) : maximum positive constraint violation (|grad| on equality rows) */
    double r_2;    /* |max(grad, 0)|_2 (|grad| on equality rows) */
    double gap;    /* (obj + reg) - g = -lambda'grad: primal objective of x* minus dual objective -- Table 4's primal-dual gap
                      before the absolute value; tends to 0 at the optimum (complementary slackness) */
} dualip_scalars;

/* Optional per-iteration trace of dualip_solve.  All pointers are DEVICE pointers (or NULL to skip that
 * column); entry n is the n-th gradient evaluation over all stages (0 <= n < sum iters <= capacity).
 *   g[n], r_inf[n], r_2[n] : scalars at the extrapolated point y_t the gradient is taken at (R1)
 *   grad[n*R + q]          : grad g(y_t)        (R = number of duals: J*m, or J*m + 1 with the global-count row)
 *   lambda[n*R + q]        : lambda_{t+1}                                                         */
typedef struct {
    int64_t capacity;
    double* g;
    double* r_inf;
    double* r_2;
    double* grad;
    double* lambda;
    double* eta;     /* eta[n] = step of iteration n (of the iterated system; the per-coordinate factor d_q^2 not included) */
} dualip_trace;

typedef struct {
    int64_t I, nnz;
    int32_t J, m;
    double  L;               /* max_j sum_k sum_i (a^k_ij)^2 (R2) */
    int64_t max_row_len;
    int32_t group_lanes;     /* lanes per row in the gradient kernel */
    int32_t chunk_regs;      /* row chunks held in registers (rows longer than group_lanes*chunk_regs take the warp path) */
    int32_t reduction;       /* the strategy in effect (never AUTO) */
    int32_t lambda_in_smem;  /* 1 if lambda is staged in shared memory */
    int32_t grid_ctas, block_threads;
    int64_t smem_bytes;      /* dynamic shared memory per CTA of the gradient kernel */
    int64_t bytes_resident;  /* device bytes owned by the handle */
    int64_t launches;        /* kernels launched through this handle so far (all entry points) */
    double  fix_scale_s;     /* fixed-point scale of the item accumulators (a power of two) */
    int32_t streaming;       /* 1: TMA bulk-copy pipeline kernel (k_grad_tma); 0: direct-load kernel (k_grad) */
    int32_t stages;          /* pipeline stages of the streaming kernel */
    int64_t tile_units;      /* tile size TN: a tile is cut every TN units of (nonzeros + 8 per row) */
    int64_t ntiles;
    double  grad_kernel_ms;  /* profiling on: summed device time of the gradient-kernel launches since it was switched on */
    int64_t grad_kernel_count; /* ... and how many launches that sum covers */
    int32_t precondition;    /* DUALIP_PRECOND_* in effect */
    int32_t pad0;
    double  L_step;          /* the constant the step is derived from (eta = gamma / L_step): L, or L' with JACOBI
                                (+ |count row|^2 with the global-count row: nnz, or 1 with JACOBI) */
    int32_t duals;           /* length of lambda / grad vectors: J*m, or J*m + 1 with the global-count row */
    int32_t lambda_lo_smem;  /* streaming kernel: 1 if the LAST launch staged lambda's low word in shared memory */
    int32_t checked_build;   /* 1: the library was compiled with -DDUALIP_CHECKED (in-kernel bounds assertions; tests only) */
    int32_t checks_failed;   /* checked build: bit mask of the kinds of bounds violation seen so far (0 = none); else 0 */
    int64_t long_rows;       /* rows taken by the CTA-per-row kernel k_grad_long (more than long_row_threshold nonzeros) */
    int64_t long_row_threshold; /* 0: no row is treated as long */
} dualip_info;

/*
 * a0 -- build a device-resident problem from per-user CSR rows ("one column pointer, one row index
 * per nonzero, one value per nonzero"; here one block per user).
 *   I >= 0 users, J >= 1 items, 1 <= m <= 4 coupling families (Def. 1).
 *   row_ptr[I+1] int64 (host or device), row_ptr[0] = 0, non-decreasing; nnz = row_ptr[I] (may exceed 2^31).
 *   item_idx[nnz] int32 in [0,J), distinct within a row, any order;  c[nnz];  a[nnz*m];  b[J*m].
 *   opts may be NULL (defaults).
 * Work done: copy (or borrow), validation kernels, L (R2), column |a| sums and sum|c| for the fixed-point
 * scales, row-length statistics, launch plan (tile table; the list of long rows; a uint16 copy of item_idx that the
 * streaming kernel reads instead of the int32 array -- 2 bytes per nonzero of device memory, counted in
 * dualip_info.bytes_resident, also with borrow = 1); with DUALIP_RED_CSC also the item-sorted permutation.
 * Synchronises `stream`.  Errors: EINVAL, ERANGE, EDUP, ENOMEM, ECUDA, EUNSUPPORTED.
 */
int dualip_create(dualip_t** out, int64_t I, int32_t J, int32_t m, const int64_t* row_ptr,
                  const int32_t* item_idx, const float* c, const float* a, const float* b,
                  const dualip_opts* opts, void* stream);

/*
 * a1-a5 (+a8) -- one evaluation of Eq. 2-4 at `lambda` (any sign; g is defined on all of R^{mJ}) and gamma > 0.
 *   lambda[J*m] in;  grad[J*m] out (may be NULL);  scalars out (may be NULL);
 *   x[nnz] fp32 out in input nonzero order, or NULL (then x is never written to memory).
 *   Each pointer may be host or device, independently.
 */
int dualip_grad(dualip_t* h, const double* lambda, double gamma, double* grad, dualip_scalars* scalars,
                float* x, void* stream);

/*
 * a1-a8 -- gamma continuation with projected accelerated ascent (R1-R4).
 *   for each stage s < n_stages:  eta = gammas[s]/L;  y = lambda (warm start, momentum restart)
 *       repeat iters[s] times:  grad at y;  lambda+ = max(0, y + eta*grad);  y = lambda+ + beta_t (lambda+ - lambda)
 *       (with opts.precondition = DUALIP_PRECOND_JACOBI the step is per coordinate, see DUALIP_PRECOND_*)
 *   then one evaluation at the final lambda with gammas[n_stages-1] fills final_scalars / final_grad / x_out
 *   (skipped when all three are NULL, so the call is exactly sum(iters) gradient evaluations).
 *   gammas, iters: HOST arrays.  lambda_inout[J*m]: warm start in (zeros for a cold start), lambda_T out.
 *   x_out[nnz], final_scalars, final_grad[J*m] may be NULL; host or device.  trace may be NULL.
 *   n_stages = 0 is allowed (nothing happens).  No host synchronisation happens inside the loop.
 */
int dualip_solve(dualip_t* h, const double* gammas, int32_t n_stages, const int32_t* iters,
                 double* lambda_inout, float* x_out, dualip_scalars* final_scalars, double* final_grad,
                 const dualip_trace* trace, void* stream);

/* Replace c (nnz fp32, host or device) in place without rebuilding -- config 5's perturbed re-solve.
 * Recomputes the objective's fixed-point scale (not on a sharded handle: see dualip_set_shard_constants, DUALIP_ESTALE).  With borrow = 1 the handle switches to the new pointer, which must be
 * device memory and, when the streaming kernel is in use (dualip_info.streaming), 16-byte aligned like the arrays given
 * to dualip_create (its bulk copies need it): otherwise DUALIP_EINVAL and the handle keeps the old c. */
int dualip_set_c(dualip_t* h, const float* c_new, void* stream);

/* Marks coupling rows as EQUALITIES (A x)_{j,k} = b_{j,k} ("projection onto the nonnegative orthant for
 * inequality coordinates"; R19).  is_equality[J*m] (uint8, host or device; [j*m+k] != 0 = equality), or NULL to
 * make every row an inequality again (the default, Eq. 1).  An equality row's dual is free in sign: dualip_solve skips
 * the lambda >= 0 projection for it, and r_inf / r_2 (dualip_grad and dualip_solve alike) count |grad| for it instead
 * of max(grad, 0).  Nothing else changes: g and grad g are defined for any sign of lambda. */
int dualip_set_equality_rows(dualip_t* h, const uint8_t* is_equality, void* stream);

/* Global-count constraint  sum_{(i,j) in E} x_ij <= M  ("adding a global-count constraint ... only augments A and
 * lambda"; R21): one more coupling row, number J*m, with coefficient 1 on every eligible pair and its own dual mu >= 0, which
 * every nonzero gathers: w_ij = -(c_ij + sum_k a^k_ij lambda_jk + mu).  enable != 0 switches the row on with right-hand side M
 * (finite, >= 0; kept in fp64, so a budget of tens of millions of pairs is exact); enable = 0 switches it off.  While it is on, EVERY dual-sized vector at this interface -- lambda, grad,
 * lambda_inout, final_grad, the trace rows, is_equality -- has J*m + 1 entries, the last one belonging to this row
 * (dualip_info.duals).  The step constant becomes L_step + nnz (|A|_2^2 <= |A_items|_2^2 + |1|_2^2), or L' + 1 under JACOBI,
 * where the row is normalised like any other (d^2 = 1/nnz).  Switching the row on or off clears the equality mask. */
int dualip_set_global_count(dualip_t* h, int32_t enable, double M, void* stream);

/* ---- user-sharded multi-GPU (section 4.4: sources split across GPUs, lambda and b replicated, one |lambda|-sized
 * reduction per iteration; Fig. 3) ------------------------------------------------------------------------------
 * One handle per GPU holds a contiguous range of users.  The item sums are 64-bit FIXED-POINT integers, so the cross-GPU
 * reduction is an integer sum: with the same fixed-point scales on every shard (dualip_set_shard_constants) the all-reduced
 * accumulators -- and hence grad g, g, and every rank's AGD update -- are bit-identical on all ranks and to one GPU holding
 * all users.  No rank-0 update, no broadcast (the paper reduces to rank 0 and broadcasts lambda).  The library does
 * not talk to NCCL: the caller's hook does the all-reduce (the Python binding uses torch.distributed).
 *
 * Accumulator layout (int64 words, dualip_info.duals' item part first): [J*m item sums a'x][c'x][|x|^2][sum x].           */

/* Called between the gradient kernel and the epilogue of EVERY evaluation (dualip_grad, each iteration and the final evaluation
 * of dualip_solve) once set: must leave in accumulators_dev[0..n_words) the sum over all shards, enqueued on `stream` -- the
 * stream the gradient kernel was launched on and the epilogue will be; work put on any other stream races both
 * (e.g. ncclAllReduce(int64, sum) in place on `stream`).  lambda_eval_dev / gamma: the point being evaluated (identical on all
 * ranks).  Returns 0, or non-zero if the exchange could not be issued: the evaluation is then abandoned -- no epilogue, the
 * partial sums are cleared, the entry point returns DUALIP_EHOOK -- instead of finalising this shard's sums alone while the
 * other ranks wait. */
typedef int (*dualip_reduce_hook)(void* user, int64_t* accumulators_dev, int64_t n_words, const double* lambda_eval_dev,
                                  double gamma, void* stream);
/* fn = NULL removes the hook.  While a hook is set, CUDA-graph replay is off (the hook runs on the host between launches). */
int dualip_set_reduce_hook(dualip_t* h, dualip_reduce_hook fn, void* user);

/* Create-time constants (a0) of a sharded problem.  Everything a0 derives from the rows -- L (R2), the Jacobi factors
 * (R18), the fixed-point scales -- comes from per-item column sums that are themselves accumulated in fixed point, so they
 * can be made EXACTLY those of the unsharded problem with two integer all-reduces:
 *   1. dualip_get_shard_extents on every shard; all-reduce I and nnz (SUM), max_abs_a and max_abs_c (MAX) -> global extents;
 *   2. dualip_get_column_stats(h, &global, out): this shard's column sums in the fixed-point scales the GLOBAL extents imply,
 *      out[0..J*m) = sum_i (a^k_ij)^2, out[J*m..2J*m) = sum_i |a^k_ij|, out[2J*m] = sum |c|;  all-reduce (int64 SUM);
 *   3. dualip_set_shard_constants(h, &global, summed) on every shard: L, L_step, the Jacobi factors and the scales are derived
 *      from the summed integers exactly as dualip_create derives them on one GPU.
 * dualip_set_c on a handle that has been given shard constants keeps them (a shard's own sum |c| and max |c| are not the
 * problem's, and ranks with different fixed-point scales would all-reduce integers that do not add up) and marks the handle
 * stale: dualip_grad, dualip_solve and dualip_eval_partial return DUALIP_ESTALE until steps 1-3 have been repeated on every
 * shard (step 1 too: max |c| is part of the extents). */
typedef struct {
    int64_t I, nnz;                 /* users, nonzeros */
    float   max_abs_a, max_abs_c;
} dualip_shard_extents;
int dualip_get_shard_extents(dualip_t* h, dualip_shard_extents* out);
int dualip_get_column_stats(dualip_t* h, const dualip_shard_extents* global, int64_t* out /* 2*J*m + 1, host or device */, void* stream);
int dualip_set_shard_constants(dualip_t* h, const dualip_shard_extents* global, const int64_t* summed /* 2*J*m + 1, host or device */,
                               void* stream);

/* Pieces the hook-less emulation and the tests use.  dualip_eval_partial: a1-a3 + this shard's part of a4-a5 only (the
 * gradient kernel without its epilogue) at `lambda` (device), leaving the accumulators in the handle; x may be NULL.
 * dualip_export_accumulators: copies the duals' item part + 3 scalar words out (host or device) and, with clear != 0, zeroes
 * them.  dualip_import_accumulators: overwrites them (accumulate = 0) or adds to them (accumulate != 0). */
int dualip_eval_partial(dualip_t* h, const double* lambda_dev, double gamma, float* x, void* stream);
int dualip_export_accumulators(dualip_t* h, int64_t* out, int32_t clear, void* stream);
int dualip_import_accumulators(dualip_t* h, const int64_t* in, int32_t accumulate, void* stream);

/* DUALIP_RED_CSC only (else DUALIP_EUNSUPPORTED): copies out the item-sorted permutation built at create (a0).
 *   col_ptr_out[J+1] int64: column j's entries are perm[col_ptr[j] .. col_ptr[j+1]);
 *   perm_out[nnz] int64: positions into the input nonzero order, ascending inside a column -- bit-exact with a stable
 *   counting sort of item_idx.  Either pointer may be NULL; host or device.  Synchronises `stream`. */
int dualip_get_csc(dualip_t* h, int64_t* col_ptr_out, int64_t* perm_out, void* stream);

/* Profiling hook for the measurement harness: when on, every gradient-kernel launch is bracketed by CUDA
 * events recorded on the launching stream (no host synchronisation is added); dualip_get_info waits for the
 * recorded events and reports the summed device time.  Switching it on resets the counters.  At most 4096
 * launches are timed between two dualip_get_info calls; later ones run untimed. */
int dualip_set_profiling(dualip_t* h, int on);

/* Fills *info.  With profiling on, blocks until the timed launches have finished. */
int dualip_get_info(dualip_t* h, dualip_info* info);

/*
 * a1-a5 (+a8) without a handle and WITHOUT ANY ALLOCATION -- for callers that may not allocate device memory.
 *
 * Everything else in this header needs a handle, and dualip_create builds one out of cudaMalloc'd buffers.  That rules the
 * library out for code that is not allowed to allocate where it runs: a plug-in inside a host application that owns all device
 * memory and forbids cudaMalloc behind its back; a service whose memory budget was reserved in full at start-up; a
 * latency-critical path that cannot take the device-wide synchronisation cudaMalloc and cudaFree imply.  This call computes the
 * same evaluation as dualip_create + dualip_grad (Eq. 2-4: grad g = A x* - b, g, obj, reg, the residuals, optionally x)
 * for one lambda, and calls no cudaMalloc / cudaFree / allocating library routine, on the device or on the host: the scratch
 * its kernels reduce into (fixed-point item accumulators, scalar accumulators, column sums, a counter) is a fixed array
 * compiled into the library.
 *
 *   I, J, m, row_ptr[I+1], item_idx[nnz], c[nnz], a[nnz*m], b[J*m]: as for dualip_create, but ALL DEVICE pointers (a host
 *     pointer would need a staging buffer: DUALIP_EINVAL), used in place, never copied; rows are NOT validated (as with
 *     opts.validate = 0: an item index outside [0,J) is undefined behaviour); row_ptr[0] != 0 gives DUALIP_ERANGE.
 *   projection, p0, p1: DUALIP_PROJ_* and its parameters, as in dualip_opts.
 *   lambda[J*m] device in, gamma > 0;  grad[J*m], scalars, x[nnz]: DEVICE out, each may be NULL.
 *   No equality rows, no global-count row, no AGD update: one evaluation, inequality rows.
 *
 * Limit: J*m <= DUALIP_STATIC_MAX_DUALS, else DUALIP_ETOOBIG and nothing is launched.  The scratch costs
 * 8 * (8 + 2 * DUALIP_STATIC_MAX_DUALS) bytes = 448 KB of device memory on every GPU that loads the library, held until the
 * process exits, whether or not this function is ever called.
 *
 * Cost: with no handle to keep them in, the create-time constants behind the fixed-point scales (max |a|, max |c|, the largest
 * column sum of |a|, sum |c|) are recomputed on every call: two extra passes over the rows, and `stream` is synchronised three
 * times inside the call (row_ptr[I], then each pass).  The gradient kernel itself is the direct-load kernel (k_grad, lambda in
 * shared memory, RED.ADD.64 item sums), not the streaming one, and is only enqueued: the outputs are ready when `stream` is.
 * Results agree with dualip_grad on a handle of the same rows within the parity tolerances of tests/gpu_util.py (same
 * fixed-point scales; only the lane order of the projection differs).  Use a handle when you can allocate.
 *
 * Shared state -- read this:
 *   - The first call on each device looks up the device address of the scratch array and queries the device (no allocation).
 *     Make that first call, with the device current, BEFORE starting any stream capture on that device.
 *   - All calls on a device use the SAME array, which keeps the previous call's contents; every call clears the part it uses
 *     first, so calls one after another on one stream are independent.  Two calls whose GPU work can overlap -- different
 *     streams, or two host threads -- race on it and return garbage without an error.  Serialise them.
 */
#define DUALIP_STATIC_MAX_DUALS 28672
int dualip_grad_static(int64_t I, int32_t J, int32_t m, const int64_t* row_ptr, const int32_t* item_idx, const float* c,
                       const float* a, const float* b, int32_t projection, double p0, double p1, const double* lambda,
                       double gamma, double* grad, dualip_scalars* scalars, float* x, void* stream);

/* Frees everything the handle owns.  NULL is accepted. */
void dualip_destroy(dualip_t* h);

/* Static message for a return code. */
const char* dualip_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* DUALIP_H */
