/*
 * oracle/dualip_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, single-threaded fp64 CPU restatement of the dual-gradient /
 * AGD hot path of "Large-Scale Regularized Matching on GPU Clusters"
 * (arxiv/paper_2606_07777; cited below as P:<line of /root/reference/PAPER.md>).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * `--impl reference` legs may call this file.  It shares no code, header,
 * table or constant with paper_2606_07777_b200/ (the CUDA path) and neither
 * imports the other.
 *
 * What is written here, and where the paper says it:
 *   - ridge-regularised LP         min_{x in C} c'x + (gamma/2)|x|^2 s.t. Ax<=b   P:55-60  (Eq. 1)
 *   - dual function                g(l) = min_{x in C} c'x+(gamma/2)|x|^2+l'(Ax-b) P:64-67  (Eq. 2)
 *   - closed-form primal           x*(l) = Proj_C(-(A'l + c)/gamma)                P:69-71  (Eq. 3)
 *   - dual gradient (Danskin)      grad g(l) = A x*(l) - b                         P:73-75  (Eq. 4)
 *   - matching structure: per-source blocks, diagonal D_ki, m families             P:81-97  (Def. 1, Eq. 5-6)
 *   - per-source simple constraint: unit simplex sum<=1,x>=0, "or a box variant"   P:83, P:130 (Table 1)
 *   - simplex projection by Duchi et al.: sort, prefix sums, rho, theta, clamp
 *   - AGD on lambda>=0, fixed step from A and gamma, gamma continuation, warm start P:60
 *   - range-clipped adaptive step, equality rows, global-count row: oracle-defined readings
 *
 * Pins (tests/test_oracle_*.py, all `-m "not gpu"`):
 *   projections: hand-worked closed forms (tests/golden/projection_cases.txt), a second independent
 *     method (bisection on theta), brute force over supports / (lower,free,upper) partitions;
 *   g, grad g: worked example (tests/golden/worked_example_grad.txt), central finite differences,
 *     concavity, weak duality, row-scaling invariance, additivity over users;
 *   optimum: brute-force KKT active-set enumeration on <=3 users x 2 items;
 *   AGD loop: **parity unpinned against the paper** (the update rule is never printed, P:123 gives
 *     words only; reading R1/R2).  Pinned internally: I=J=1 closed-form optimum, the
 *     lambda==0 fixed point, monotone ascent of the beta==0 variant, O(1/T^2) bound on KKT instances.
 *   adaptive step (R20): **parity unpinned against the paper** (no formula printed).  Pinned internally: a clip range that
 *     is one point reproduces the fixed step bit for bit; on I=J=1 (grad g linear) the secant step IS gamma/L; every eta_t lies
 *     in the range, whose maximum scales with gamma_s/gamma_1 and whose minimum never exceeds gamma_s/L; with the paper's
 *     default range on an unscaled system (gamma/L << 1e-5) the first step of a stage is gamma/L; the KKT optimum of the tiny
 *     instances is reached.
 *   global-count row (R21): an I=1 closed form, brute-force KKT with the extra row, and J=1 instances, where the count row
 *     is literally a second coupling family with a = 1 (same gradients, same L, same trajectory) -- tests/test_oracle_extensions.py.
 *
 * Layout at this interface (same as the product's C ABI, stated independently):
 *   row_ptr[I+1] int64, item_idx[nnz] int32, c[nnz] fp32, a[nnz*m] fp32 (a[p*m+k]),
 *   b[J*m] fp32 (b[j*m+k]), lambda/grad[J*m] fp64 ([j*m+k]).  fp32 inputs are cast exactly to
 *   fp64; all arithmetic is fp64; sums over users run in index order.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

enum { ORACLE_PROJ_SIMPLEX_INEQ = 0, ORACLE_PROJ_BOX = 1, ORACLE_PROJ_BOXCUT = 2, ORACLE_PROJ_SIMPLEX_EQ = 3 };

static int cmp_desc(const void* pa, const void* pb) {
    double a = *(const double*)pa, b = *(const double*)pb;
    return (a < b) - (a > b);
}

/* Equality-form simplex {x>=0, sum x = z}: Duchi et al. 2008, Fig. 1 (the stages P:117 names:
 * sort, prefix sums, cutoff index rho, threshold theta, subtract-and-clamp). */
void dualip_oracle_project_simplex_eq(const double* v, int64_t n, double z, double* x) {
    if (n <= 0) return;
    double* u = (double*)malloc((size_t)n * sizeof(double));
    memcpy(u, v, (size_t)n * sizeof(double));
    qsort(u, (size_t)n, sizeof(double), cmp_desc);              /* u_1 >= u_2 >= ... */
    double csum = 0.0, c_rho = 0.0;
    int64_t rho = 0;
    for (int64_t k = 1; k <= n; ++k) {
        csum += u[k - 1];                                        /* c_k = sum_{l<=k} u_l */
        if (u[k - 1] - (csum - z) / (double)k > 0.0) { rho = k; c_rho = csum; }
    }
    double theta = (c_rho - z) / (double)rho;                    /* rho >= 1 whenever z > 0 */
    for (int64_t p = 0; p < n; ++p) x[p] = fmax(v[p] - theta, 0.0);
    free(u);
}

/* Inequality-form simplex {x>=0, sum x <= z} ("inequality variant").
 * Reading R5: exact early exit -- if sum max(v,0) <= z return max(v,0), no tolerance. */
void dualip_oracle_project_simplex(const double* v, int64_t n, double z, double* x) {
    double s = 0.0;
    for (int64_t p = 0; p < n; ++p) { x[p] = fmax(v[p], 0.0); s += x[p]; }
    if (s <= z) return;
    dualip_oracle_project_simplex_eq(v, n, z, x);
}

/* Box {lo <= x <= hi} element-wise ("box"). */
void dualip_oracle_project_box(const double* v, int64_t n, double lo, double hi, double* x) {
    for (int64_t p = 0; p < n; ++p) x[p] = fmin(fmax(v[p], lo), hi);
}

static double clip(double t, double lo, double hi) { return fmin(fmax(t, lo), hi); }

/* Box-cut {0 <= x <= ub, sum x <= z} (P:130 names it; reading R10).
 * p = clip(v,0,ub); if sum p <= z return p.  Otherwise phi(theta) = sum clip(v-theta,0,ub) is
 * continuous, piecewise linear and non-increasing with breakpoints {v_p, v_p-ub}; walk the
 * breakpoints in descending order, evaluating phi by its definition at each, until the segment
 * that contains phi = z is found; solve that linear piece exactly. */
void dualip_oracle_project_boxcut(const double* v, int64_t n, double ub, double z, double* x) {
    double s = 0.0;
    for (int64_t p = 0; p < n; ++p) { x[p] = clip(v[p], 0.0, ub); s += x[p]; }
    if (s <= z || n <= 0) return;
    int64_t nb = 2 * n;
    double* t = (double*)malloc((size_t)nb * sizeof(double));
    for (int64_t p = 0; p < n; ++p) { t[2 * p] = v[p]; t[2 * p + 1] = v[p] - ub; }
    qsort(t, (size_t)nb, sizeof(double), cmp_desc);
    double theta = 0.0, t_hi = t[0], phi_hi = 0.0;               /* phi(max v) = 0 */
    int found = 0;
    for (int64_t k = 1; k < nb && !found; ++k) {
        double phi_lo = 0.0;
        for (int64_t p = 0; p < n; ++p) phi_lo += clip(v[p] - t[k], 0.0, ub);
        if (phi_lo >= z) {                                       /* z in [phi_hi, phi_lo] on [t[k], t_hi] */
            theta = (phi_lo == phi_hi) ? t[k] : t[k] + (phi_lo - z) * (t_hi - t[k]) / (phi_lo - phi_hi);
            found = 1;
        } else { t_hi = t[k]; phi_hi = phi_lo; }
    }
    /* found is guaranteed: phi is non-increasing, phi(0) = s > z, and below the smallest breakpoint
     * phi is the constant n*ub = phi(t_min); so some breakpoint has phi >= z. */
    for (int64_t p = 0; p < n; ++p) x[p] = clip(v[p] - theta, 0.0, ub);
    free(t);
}

static void project(int kind, double p0, double p1, const double* v, int64_t n, double* x) {
    switch (kind) {
        case ORACLE_PROJ_SIMPLEX_INEQ: dualip_oracle_project_simplex(v, n, p0, x); break;
        case ORACLE_PROJ_BOX:          dualip_oracle_project_box(v, n, p0, p1, x); break;
        case ORACLE_PROJ_BOXCUT:       dualip_oracle_project_boxcut(v, n, p0, p1, x); break;
        default:                       dualip_oracle_project_simplex_eq(v, n, p0, x); break;
    }
}

/* One evaluation of Eq. 2-4 at lambda (any sign) and gamma > 0.
 * proj params: simplex kinds p0 = z; box p0 = lo, p1 = hi; boxcut p0 = ub, p1 = z.
 * is_eq (may be NULL = every coupling row is an inequality, Eq. 1): is_eq[q] != 0 marks row q as an EQUALITY
 *   (A x)_q = b_q, whose violation is |grad_q| instead of max(grad_q, 0) (reading R19).
 * count_coef != 0 adds the GLOBAL-COUNT row  count_coef * sum_{(i,j) in E} x_ij <= count_rhs  as coupling row number
 *   Jm ("adding a global-count constraint sum x_ij <= M only augments A and lambda"; reading R21):
 *   lambda, grad_out (and is_eq) then have Jm + 1 entries, the last one being that row's dual / gradient.  The row has
 *   the coefficient count_coef on EVERY eligible pair (1 for the plain constraint; 1/sqrt(nnz) once row-normalised).
 * scalars_out[6] = { g, obj = c'x, reg = (gamma/2)|x|^2, r_inf = max violation, r_2 = |violations|_2,
 *                    gap = (obj + reg) - g = -lambda'grad  (Table 4's primal-dual gap before the absolute value) }.
 * x_out (nnz doubles, input order) may be NULL.  Returns 0, or -1 on allocation failure. */
static int grad_f64(int64_t I, int32_t J, int32_t m, const int64_t* row_ptr, const int32_t* item_idx,
                    const float* c, const double* a, const double* b, const double* lambda, double gamma,
                    int proj_kind, double p0, double p1, const uint8_t* is_eq, double count_coef, double count_rhs,
                    double* grad_out, double* scalars_out, double* x_out) {
    int64_t max_len = 0;
    for (int64_t i = 0; i < I; ++i)
        if (row_ptr[i + 1] - row_ptr[i] > max_len) max_len = row_ptr[i + 1] - row_ptr[i];
    double* v = (double*)malloc((size_t)(max_len + 1) * sizeof(double));
    double* x = (double*)malloc((size_t)(max_len + 1) * sizeof(double));
    if (!v || !x) { free(v); free(x); return -1; }
    int64_t Jm = (int64_t)J * m;
    int64_t nrow = Jm + (count_coef != 0.0 ? 1 : 0);            /* coupling rows = duals */
    double mu = count_coef != 0.0 ? lambda[Jm] : 0.0;            /* dual of the global-count row */
    for (int64_t q = 0; q < nrow; ++q) grad_out[q] = 0.0;        /* s = A x, accumulated in user order */
    double obj = 0.0, sq = 0.0, sumx = 0.0;
    for (int64_t i = 0; i < I; ++i) {
        int64_t beg = row_ptr[i], n = row_ptr[i + 1] - beg;
        for (int64_t p = 0; p < n; ++p) {
            int64_t j = item_idx[beg + p];
            double al = 0.0;                                     /* (A' lambda)_p = sum_k a^k_p lambda_{j,k} (+ count row) */
            for (int32_t k = 0; k < m; ++k) al += a[(beg + p) * m + k] * lambda[j * m + k];
            al += count_coef * mu;
            v[p] = -((double)c[beg + p] + al) / gamma;           /* Eq. 3 argument */
        }
        project(proj_kind, p0, p1, v, n, x);
        for (int64_t p = 0; p < n; ++p) {
            int64_t j = item_idx[beg + p];
            for (int32_t k = 0; k < m; ++k) grad_out[j * m + k] += a[(beg + p) * m + k] * x[p];
            obj += (double)c[beg + p] * x[p];
            sq += x[p] * x[p];
            sumx += x[p];
            if (x_out) x_out[beg + p] = x[p];
        }
    }
    if (count_coef != 0.0) grad_out[Jm] = count_coef * sumx;
    double reg = 0.5 * gamma * sq, dot = 0.0, r_inf = 0.0, r2 = 0.0;
    for (int64_t q = 0; q < nrow; ++q) {
        grad_out[q] -= (q < Jm ? b[q] : count_rhs);              /* Eq. 4 */
        dot += lambda[q] * grad_out[q];
        double viol = (is_eq && is_eq[q]) ? fabs(grad_out[q]) : fmax(grad_out[q], 0.0);
        r2 += viol * viol;
        if (viol > r_inf) r_inf = viol;
    }
    scalars_out[0] = obj + reg + dot;                            /* Eq. 2 at its minimiser */
    scalars_out[1] = obj;
    scalars_out[2] = reg;
    scalars_out[3] = r_inf;
    scalars_out[4] = sqrt(r2);
    scalars_out[5] = -dot;
    free(v); free(x);
    return 0;
}

/* The fp32 inputs cast exactly to fp64 (a and b; c is cast where it is used). */
static double* widen(const float* v, int64_t n) {
    double* w = (double*)malloc((size_t)(n > 0 ? n : 1) * sizeof(double));
    if (w) for (int64_t q = 0; q < n; ++q) w[q] = (double)v[q];
    return w;
}

/* has_count != 0: the problem carries the global-count row sum x <= count_M (see grad_f64); lambda / grad_out / is_eq
 * then have J*m + 1 entries. */
int dualip_oracle_grad(int64_t I, int32_t J, int32_t m, const int64_t* row_ptr, const int32_t* item_idx,
                       const float* c, const float* a, const float* b, const double* lambda, double gamma,
                       int proj_kind, double p0, double p1, const uint8_t* is_eq, int32_t has_count, double count_M,
                       double* grad_out, double* scalars_out, double* x_out) {
    double* a64 = widen(a, row_ptr[I] * m);
    double* b64 = widen(b, (int64_t)J * m);
    int rc = -1;
    if (a64 && b64)
        rc = grad_f64(I, J, m, row_ptr, item_idx, c, a64, b64, lambda, gamma, proj_kind, p0, p1, is_eq,
                      has_count ? 1.0 : 0.0, count_M, grad_out, scalars_out, x_out);
    free(a64); free(b64);
    return rc;
}

/* L = max_j sum_k sum_i (a^k_ij)^2  (reading R2: |A|_2^2 exactly for m = 1 because A A' is then
 * diag(sum_i a_ij^2); a trace upper bound on the m x m Gram blocks for m > 1). */
static double lipschitz_f64(int64_t I, int32_t J, int32_t m, const int64_t* row_ptr,
                            const int32_t* item_idx, const double* a) {
    double* col = (double*)calloc((size_t)J, sizeof(double));
    if (!col) return -1.0;
    for (int64_t p = 0; p < row_ptr[I]; ++p)
        for (int32_t k = 0; k < m; ++k) col[item_idx[p]] += a[p * m + k] * a[p * m + k];
    double L = 0.0;
    for (int32_t j = 0; j < J; ++j) if (col[j] > L) L = col[j];
    free(col);
    return L;
}

/* has_count != 0: plus |count row|_2^2 = nnz (reading R21, see dualip_oracle_solve). */
double dualip_oracle_lipschitz(int64_t I, int32_t J, int32_t m, const int64_t* row_ptr,
                               const int32_t* item_idx, const float* a, int32_t has_count) {
    double* a64 = widen(a, row_ptr[I] * m);
    if (!a64) return -1.0;
    double L = lipschitz_f64(I, J, m, row_ptr, item_idx, a64);
    if (has_count) L += (double)row_ptr[I];
    free(a64);
    return L;
}

/* Jacobi preconditioning / row normalisation (Appendix B.2):
 *   D = diag(|A_r*|_2^-1) over the coupling rows r = (j,k) (rows of zero norm keep D_rr = 1),
 *   A' = D A, b' = D b.  The feasible set is unchanged and diag(A'A'^T) = I on the nonzero rows.
 * d_out[J*m] receives the diagonal of D.  |A_r*|_2^2 = sum_i (a^k_ij)^2 by Definition 1. */
void dualip_oracle_jacobi_scaling(int64_t I, int32_t J, int32_t m, const int64_t* row_ptr,
                                  const int32_t* item_idx, const float* a, double* d_out) {
    int64_t Jm = (int64_t)J * m;
    for (int64_t q = 0; q < Jm; ++q) d_out[q] = 0.0;
    for (int64_t p = 0; p < row_ptr[I]; ++p)
        for (int32_t k = 0; k < m; ++k)
            d_out[(int64_t)item_idx[p] * m + k] += (double)a[p * m + k] * (double)a[p * m + k];
    for (int64_t q = 0; q < Jm; ++q) d_out[q] = d_out[q] > 0.0 ? 1.0 / sqrt(d_out[q]) : 1.0;
}

/* gamma-continuation driver with projected Nesterov ascent (readings R1-R4 in DESIGN.md; the paper
 * gives the update in words only).
 *   for each stage s: eta = gamma_s / L;  y_0 = lambda (warm start);  t = 0
 *     repeat iters[s] times:
 *        (g_t, grad_t) = grad(y_t, gamma_s)
 *        lambda_{t+1}  = max(0, y_t + eta_t * grad_t)
 *        beta_t        = momentum ? t/(t+3) : 0
 *        y_{t+1}       = lambda_{t+1} + beta_t (lambda_{t+1} - lambda_t);   t <- t+1
 *   then one extra grad(lambda_T, gamma_S) gives final scalars / grad / x.
 * step_rule (readings R2, R20; "AGD step-size range [1e-5, 1e-1]", "we scale the maximum AGD
 *   step size proportionally with the decay of gamma"):
 *     0 FIXED     eta_t = gamma_s / L.
 *     1 ADAPTIVE  eta_fix = gamma_s / L;  hi_s = eta_max * gamma_s / gamma_1;  lo_s = min(eta_min, eta_fix);
 *                 clip(e) = min(max(e, lo_s), hi_s)  (the scaled maximum wins when it falls below lo_s).  lo_s: the lower end
 *                 of the range never lifts a step ABOVE the analytic step gamma_s / L of P:60 -- with L large (no Jacobi
 *                 scaling) gamma_s / L is far below 1e-5, and a step forced up to eta_min would be far beyond 1 / L_grad;
 *                 t = 0, or a 0/0 secant:  eta_t = clip(eta_fix);
 *                 t >= 1:  eta_t = clip(|y_t - y_{t-1}|_2 / |grad_t - grad_{t-1}|_2)   -- the inverse of the secant estimate
 *                 of the local Lipschitz constant of grad g along the last move, norms taken in the system being iterated on.
 *     The paper prints no formula for its adaptive step: PARITY UNPINNED against the paper.
 * Traces (each may be NULL) are indexed by the global iteration counter n = 0..sum(iters)-1:
 *   trace_g[n] = g(y_t), trace_rinf[n], trace_r2[n], trace_grad[n*R..] = grad(y_t), trace_lambda[n*R..] = lambda_{t+1},
 *   trace_eta[n] = eta_t (of the iterated system);  R = J*m (+1 with the global-count row).  stage_x (may be NULL) receives,
 *   per stage, x*(lambda_end) at that stage's gamma (n_stages * nnz doubles) -- used by the drift report of config 5.
 * is_eq (may be NULL = all rows are inequalities, Eq. 1): is_eq[q] != 0 marks coupling row q as an EQUALITY (A x)_q = b_q;
 *   its dual is free in sign, so the projection onto lambda >= 0 is skipped for it ("projection onto the nonnegative
 *   orthant for inequality coordinates"; reading R19) and its violation in every reported residual (traces and
 *   final scalars alike) is |grad_q| instead of max(grad_q, 0).
 * has_count != 0 (reading R21): the extra coupling row sum_{(i,j) in E} x_ij <= count_M, row number J*m,
 *   with its own dual (lambda_inout, final_grad, the traces and is_eq then have J*m + 1 entries per vector).  With that row
 *   A A^T is no longer block diagonal; the step constant becomes L = max_j sum_k sum_i (a^k_ij)^2 + |count row|_2^2
 *   (|A|_2^2 <= |A_items|_2^2 + |1|_2^2 since A^T A is the sum of the two Gram matrices).
 * jacobi != 0 (reading R18): the whole loop runs on the row-scaled system
 *   A' = D A, b' = D b with its own L' and dual lambda' (warm start lambda'_0 = D^-1 lambda_0); since
 *   A'^T lambda' = A^T (D lambda'), the dual of the ORIGINAL system is lambda = D lambda' and
 *   grad g = D^-1 grad g'.  What is returned (lambda, grad, residuals, traces) is in original units.  The global-count
 *   row is normalised like any other: D = 1/sqrt(nnz) for it. */
int dualip_oracle_solve(int64_t I, int32_t J, int32_t m, const int64_t* row_ptr, const int32_t* item_idx,
                        const float* c, const float* a, const float* b, int proj_kind, double p0, double p1,
                        const double* gammas, int32_t n_stages, const int32_t* iters, int32_t momentum, int32_t jacobi,
                        const uint8_t* is_eq, int32_t step_rule, double eta_min, double eta_max, int32_t has_count, double count_M,
                        double* lambda_inout, double* x_out, double* final_scalars, double* final_grad,
                        double* trace_g, double* trace_rinf, double* trace_r2, double* trace_grad,
                        double* trace_lambda, double* trace_eta, double* stage_x) {
    int64_t Jm = (int64_t)J * m, nnz = row_ptr[I];
    int64_t R = Jm + (has_count ? 1 : 0);                        /* coupling rows = duals */
    double* as = widen(a, nnz * m);                              /* A  (or A' = D A) */
    double* bs = widen(b, Jm);                                   /* b  (or b' = D b) */
    double* d = (double*)malloc((size_t)R * sizeof(double));
    double* y = (double*)malloc((size_t)R * sizeof(double));
    double* grad = (double*)malloc((size_t)R * sizeof(double));
    double* lam = (double*)malloc((size_t)R * sizeof(double));  /* dual of the system being iterated on */
    double* lam_new = (double*)malloc((size_t)R * sizeof(double));
    double* out = (double*)malloc((size_t)R * sizeof(double));
    double* y_prev = (double*)malloc((size_t)R * sizeof(double));
    double* g_prev = (double*)malloc((size_t)R * sizeof(double));
    if (!as || !bs || !d || !y || !grad || !lam || !lam_new || !out || !y_prev || !g_prev) {
        free(as); free(bs); free(d); free(y); free(grad); free(lam); free(lam_new); free(out); free(y_prev); free(g_prev);
        return -1;
    }
    for (int64_t q = 0; q < R; ++q) d[q] = 1.0;
    if (jacobi) {
        dualip_oracle_jacobi_scaling(I, J, m, row_ptr, item_idx, a, d);
        for (int64_t p = 0; p < nnz; ++p)
            for (int32_t k = 0; k < m; ++k) as[p * m + k] *= d[(int64_t)item_idx[p] * m + k];
        for (int64_t q = 0; q < Jm; ++q) bs[q] *= d[q];
        if (has_count) d[Jm] = nnz > 0 ? 1.0 / sqrt((double)nnz) : 1.0;   /* the count row has a 1 on each of the nnz pairs */
    }
    double count_coef = 0.0, count_rhs = 0.0;                    /* the row's coefficient (1, or 1/sqrt(nnz) row-normalised) */
    if (has_count) { count_coef = d[Jm]; count_rhs = d[Jm] * count_M; }
    for (int64_t q = 0; q < R; ++q) lam[q] = lambda_inout[q] / d[q];
    double L = lipschitz_f64(I, J, m, row_ptr, item_idx, as);
    if (has_count) L += (double)nnz * count_coef * count_coef;   /* reading R21 */
    if (!(L > 0.0)) L = 1.0;
    double sc[6];
    int64_t n = 0;
    int rc = 0;
    for (int32_t s = 0; s < n_stages && rc == 0; ++s) {
        double gamma = gammas[s], eta_fix = gamma / L;
        double hi_s = eta_max * gamma / gammas[0];               /* the maximum scales with the decay of gamma */
        memcpy(y, lam, (size_t)R * sizeof(double));              /* warm start, momentum restart */
        for (int32_t t = 0; t < iters[s] && rc == 0; ++t, ++n) {
            rc = grad_f64(I, J, m, row_ptr, item_idx, c, as, bs, y, gamma, proj_kind, p0, p1, NULL, count_coef, count_rhs,
                          grad, sc, NULL);
            if (trace_g) trace_g[n] = sc[0];
            if (trace_grad || trace_rinf || trace_r2) {          /* residuals of the original rows: grad g = D^-1 grad g' */
                double r_inf = 0.0, r2 = 0.0;
                for (int64_t q = 0; q < R; ++q) {
                    out[q] = grad[q] / d[q];
                    double viol = (is_eq && is_eq[q]) ? fabs(out[q]) : fmax(out[q], 0.0);   /* |Ax-b| on equality rows */
                    r2 += viol * viol;
                    if (viol > r_inf) r_inf = viol;
                }
                if (trace_rinf) trace_rinf[n] = r_inf;
                if (trace_r2) trace_r2[n] = sqrt(r2);
                if (trace_grad) memcpy(trace_grad + n * R, out, (size_t)R * sizeof(double));
            }
            double eta = eta_fix;
            if (step_rule == 1) {                                /* reading R20 */
                if (t >= 1) {
                    double dy2 = 0.0, dg2 = 0.0;
                    for (int64_t q = 0; q < R; ++q) {
                        dy2 += (y[q] - y_prev[q]) * (y[q] - y_prev[q]);
                        dg2 += (grad[q] - g_prev[q]) * (grad[q] - g_prev[q]);
                    }
                    if (dy2 > 0.0 && dg2 > 0.0) eta = sqrt(dy2) / sqrt(dg2);
                }
                eta = fmin(fmax(eta, fmin(eta_min, eta_fix)), hi_s);
                memcpy(y_prev, y, (size_t)R * sizeof(double));
                memcpy(g_prev, grad, (size_t)R * sizeof(double));
            }
            if (trace_eta) trace_eta[n] = eta;
            double beta = momentum ? (double)t / (double)(t + 3) : 0.0;
            for (int64_t q = 0; q < R; ++q) {
                lam_new[q] = y[q] + eta * grad[q];
                if (!(is_eq && is_eq[q])) lam_new[q] = fmax(0.0, lam_new[q]);   /* "projection onto the nonnegative
                                                                                    orthant for inequality coordinates" P:123 */
                y[q] = lam_new[q] + beta * (lam_new[q] - lam[q]);
            }
            memcpy(lam, lam_new, (size_t)R * sizeof(double));
            if (trace_lambda) for (int64_t q = 0; q < R; ++q) trace_lambda[n * R + q] = d[q] * lam[q];
        }
        if (stage_x && rc == 0)
            rc = grad_f64(I, J, m, row_ptr, item_idx, c, as, bs, lam, gamma, proj_kind, p0, p1, NULL, count_coef, count_rhs,
                          grad, sc, stage_x + (int64_t)s * nnz);
    }
    for (int64_t q = 0; q < R; ++q) lambda_inout[q] = d[q] * lam[q];
    /* final report: one evaluation of the ORIGINAL system at lambda_T = D lambda'_T (same x, same g) */
    if (rc == 0 && n_stages > 0)
        rc = dualip_oracle_grad(I, J, m, row_ptr, item_idx, c, a, b, lambda_inout, gammas[n_stages - 1],
                                proj_kind, p0, p1, is_eq, has_count, count_M, final_grad ? final_grad : grad,
                                final_scalars ? final_scalars : sc, x_out);
    free(as); free(bs); free(d); free(lam); free(out);
    free(y); free(grad); free(lam_new); free(y_prev); free(g_prev);
    return rc;
}
