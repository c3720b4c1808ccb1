// dualip_kernels.cuh -- device code of the dual-gradient hot path (sm_100a).
//
// Steps a1-a6 of SURVEY.md section 8(a); equations cited as P:n (paper line) and R<n> (DESIGN.md readings).
//   k_grad      a1 gather lambda, a2 w = -(c + sum_k a^k lambda_jk), a3 projection, a4 item reduction,
//               a5 per-lane partial scalars, a8 optional x                         (Eq. 3-4)
//   k_grad_box  the same for the element-wise box projection (no row coupling)
//   finalize_block  a4 grad = s - b, a5 g / r_inf / r_2, a6 AGD update + lambda >= 0 projection (R1),
//               run by the last CTA of every gradient launch (grid_epilogue): one launch = one iteration
//   k_validate, k_absmax, k_col_stats, k_reduce_stats      a0 create-time checks and constants (R2, R11)
//
// Numerics: lambda fp64; w by fp64 FMA from fp32 data; row maximum taken on RN_f32(w);
// u = RN_f32((w - m)/gamma) with the subtraction exact in fp64, so every quantity after the shift is O(1)
// and fp32 is accurate to ~1e-7 absolute whatever 1/gamma is.  The inequality branch (R5) is folded in as
// tau = max(theta_eq, -m/gamma):  x = max(u - tau, 0).
//
// Item reduction: 64-bit fixed point.  Shared-memory accumulators are two 32-bit words with an explicit carry,
// because ATOMS.ADD (32-bit integer) is the only native shared-memory add on sm_100a; global accumulation is
// RED.ADD.64.  Integer addition commutes, so results are bit-reproducible for any launch geometry.
#pragma once
#include <cuda_runtime.h>
#include <math_constants.h>
#include <stdint.h>

namespace dualip_dev {

constexpr int kBlockThreads = 512;
constexpr int kWarpsPerBlock = kBlockThreads / 32;
constexpr unsigned kFull = 0xffffffffu;

enum : int { PROJ_SIMPLEX_INEQ = 0, PROJ_BOX = 1, PROJ_BOXCUT = 2, PROJ_SIMPLEX_EQ = 3 };

struct GradParams {
    const long long* __restrict__ row_ptr;
    const int* __restrict__ idx;
    const float* __restrict__ c;
    const float* __restrict__ a;
    const double* __restrict__ lambda;
    unsigned long long* s_fix;   // [J*m] item accumulators, fixed point, zero on entry; nullptr = do not accumulate (CSC)
    unsigned long long* sc_fix;  // [3]   obj = c'x, |x|^2 and sum x, fixed point, zero on entry
    float* x;                    // [nnz] or nullptr
    long long I;
    long long nnz;
    int J, m;
    int proj;
    int general_boxcut;          // BOXCUT with ub < z: needs the capped threshold search
    int count_on;                // global-count row (R21): lambda[J*m] is its dual mu, gathered by EVERY nonzero
    long long long_thr;          // > 0: rows of more than this many nonzeros are k_grad_long's (dualip_long.cuh); skipped here
    float inv_gamma_f;
    float z;                     // simplex / box-cut budget
    float ub;                    // box-cut cap
    double inv_gamma;
    double box_lo, box_hi;
    double scale_s, scale_obj, scale_sq, scale_cnt;
    float scale_s_f, scale_obj_f, scale_sq_f, scale_cnt_f;   // the same powers of two as floats (streaming kernel: one FMUL + F2I)
    float max_abs_c, max_abs_a;                 // max |c|, max |a| over all nonzeros (a0): the filter's rounding bound
};

__device__ __forceinline__ long long to_fix(float v, double scale) { return __double2ll_rn((double)v * scale); }

__device__ __forceinline__ void fix_add_smem(unsigned* lo, unsigned* hi, long long v) {
    const unsigned vlo = (unsigned)(unsigned long long)v;
    const unsigned vhi = (unsigned)((unsigned long long)v >> 32);
    const unsigned old = atomicAdd(lo, vlo);
    const unsigned h = vhi + ((unsigned)(old + vlo) < vlo ? 1u : 0u);
    if (h) atomicAdd(hi, h);
}

template <int G>
__device__ __forceinline__ float group_max(float v) {
#pragma unroll
    for (int o = G / 2; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(kFull, v, o));
    return v;
}
template <int G>
__device__ __forceinline__ float group_sum(float v) {
#pragma unroll
    for (int o = G / 2; o > 0; o >>= 1) v += __shfl_xor_sync(kFull, v, o);
    return v;
}
template <int G>
__device__ __forceinline__ int group_sum_i(int v) {
#pragma unroll
    for (int o = G / 2; o > 0; o >>= 1) v += __shfl_xor_sync(kFull, v, o);
    return v;
}

// One nonzero: returns t = c + sum_k a_k * lambda[j,k] (+ mu, the dual of the global-count row, R21) in fp64 (w = -t), and
// the row data it read.
template <int M, bool LAM_SMEM>
__device__ __forceinline__ double eval_t(const GradParams& p, const double* s_lam, double mu, long long q, int mm,
                                         int& j, float& cc, float (&aa)[M > 0 ? M : 4]) {
    j = __ldg(p.idx + q);
    cc = __ldg(p.c + q);
    double t = (double)cc + mu;
    if (M > 0) {
#pragma unroll
        for (int k = 0; k < M; ++k) aa[k] = __ldg(p.a + q * M + k);
#pragma unroll
        for (int k = 0; k < M; ++k) {
            const double l = LAM_SMEM ? s_lam[j * M + k] : __ldg(p.lambda + (long long)j * M + k);
            t = fma((double)aa[k], l, t);
        }
    } else {
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            aa[k] = 0.0f;
            if (k < mm) {
                aa[k] = __ldg(p.a + q * mm + k);
                const double l = LAM_SMEM ? s_lam[j * mm + k] : __ldg(p.lambda + (long long)j * mm + k);
                t = fma((double)aa[k], l, t);
            }
        }
    }
    return t;
}

// a4 + a5 for one nonzero with x > 0.
template <int M, bool ACC_SMEM>
__device__ __forceinline__ void contribute(const GradParams& p, unsigned* s_lo, unsigned* s_hi, int mm, int j,
                                           const float (&aa)[M > 0 ? M : 4], float x) {
    const int nm = M > 0 ? M : mm;
    if (!ACC_SMEM && p.s_fix == nullptr) return;          // DUALIP_RED_CSC: the item sums are taken from x afterwards
#pragma unroll
    for (int k = 0; k < (M > 0 ? M : 4); ++k) {
        if (k < nm) {
            const long long f = to_fix(aa[k] * x, p.scale_s);
            if (ACC_SMEM) fix_add_smem(s_lo + j * nm + k, s_hi + j * nm + k, f);
            else asm volatile("red.global.add.u64 [%0], %1;" ::"l"(p.s_fix + (long long)j * nm + k), "l"((unsigned long long)f) : "memory");   // RED, not ATOM
        }
    }
}

// Iteration state kept on the device so that every launch of one stage has identical arguments (CUDA-graph replay):
// t = iteration index inside the stage (momentum restart resets it, R4), n = index over all stages (trace row).
struct IterState { int t; int pad; long long n; };

struct FinalizeParams {
    unsigned long long* s_fix;
    unsigned long long* sc_fix;
    const float* __restrict__ b;  // [JM] right-hand sides of the item rows (fp32 input data)
    double count_rhs;           // M of the global-count row (row JM) when it is on: fp64, a count above 2^24 is not an fp32 number
    const double* lam_eval;     // point the gradient was taken at
    double* grad_out;           // nullable
    double* scalars_out;        // nullable, 6 doubles {g, obj, reg, r_inf, r_2, gap}
    int JM;                     // item coupling rows J*m
    int R;                      // coupling rows = duals: JM, + 1 with the global-count row (row JM, R21)
    double inv_scale_s, inv_scale_obj, inv_scale_sq, inv_scale_cnt;
    double gamma;
    int update;                 // a6 on/off
    int momentum;               // beta_t = t/(t+3) (R1) or 0
    double eta;                 // gamma / L_step (R2)
    int step_rule;              // 0 fixed; 1 range-clipped secant step (R20)
    double eta_lo, eta_hi;      // step_rule 1: clip range of this stage, eta_hi = eta_max gamma_s / gamma_1
    double* y_prev; double* g_prev;   // step_rule 1: the previous evaluation point and gradient of this stage [R]
    const double* step_scale;   // nullable: per-coordinate factor on eta (Jacobi preconditioning, R18: d_q^2 = 1/|A_q*|^2)
    const unsigned char* row_eq; // nullable: nonzero = equality coupling row (dual free in sign, violation |grad|; R19)
    double* lam_cur;            // lambda_t -> lambda_{t+1}
    double* y;                  // y_t -> y_{t+1} (== lam_eval when update)
    IterState* state;           // read and advanced when update
    unsigned* done;             // CTAs that have flushed their partial sums (zero between launches)
    double* tr_g; double* tr_rinf; double* tr_r2; double* tr_grad; double* tr_lam; double* tr_eta;   // trace columns (nullable)
};

constexpr int kFinalizeScratchBytes = 3 * 32 * 8 + 16;   // shared memory finalize_block needs: 3 x 32 doubles + flag

// b_q: the item rows' right-hand sides are the caller's fp32 data; the global-count row's (q = JM) is the fp64 M
__device__ __forceinline__ double row_rhs(const FinalizeParams& p, int q) { return q < p.JM ? (double)__ldg(p.b + q) : p.count_rhs; }

// s_q = (A x)_q from the fixed-point accumulators: item rows from s_fix, the global-count row (q = JM) from the sum-x scalar
__device__ __forceinline__ double row_sum(const FinalizeParams& p, int q) {
    return q < p.JM ? (double)(long long)__ldcg(p.s_fix + q) * p.inv_scale_s : (double)(long long)__ldcg(p.sc_fix + 2) * p.inv_scale_cnt;
}

// a4 (grad = s - b), a5 (scalars), a6 (AGD step, R1) on the R-vector by ONE CTA of `nthreads` (<= 1024) threads;
// re-zeroes the accumulators and advances the iteration state.  `sh` = 96 doubles of shared memory.
__device__ __forceinline__ void finalize_block(const FinalizeParams& p, double* sh, int tid, int nthreads) {
    double* sh_dot = sh; double* sh_r2 = sh + 32; double* sh_inf = sh + 64;
    const int lane = tid & 31, warp = tid >> 5, nwarps = (nthreads + 31) / 32;
    int t = 0; long long n = 0;
    if (p.update) { t = p.state->t; n = p.state->n; }
    const double beta = (p.update && p.momentum) ? (double)t / (double)(t + 3) : 0.0;
    // R20: eta_t = clip(|y_t - y_{t-1}| / |grad_t - grad_{t-1}|) -- the inverse of the secant estimate of the local Lipschitz
    // constant of grad g -- with both norms taken in the system being iterated on: under Jacobi preconditioning (R18) that is
    // the row-scaled one, y' = y / d and grad' = d grad with d_q^2 = step_scale[q].  First iteration of a stage (or a 0/0
    // secant): the fixed step.  One more pass over the R-vector before the update, since every coordinate needs eta_t.
    double eta_t = p.eta;
    if (p.update && p.step_rule == 1) {
        if (t >= 1) {
            double dy2 = 0.0, dg2 = 0.0;
            for (int q = tid; q < p.R; q += nthreads) {
                const double g = row_sum(p, q) - row_rhs(p, q);
                const double d2 = p.step_scale ? __ldg(p.step_scale + q) : 1.0;
                const double dy = __ldcg(p.lam_eval + q) - __ldcg(p.y_prev + q), dg = g - __ldcg(p.g_prev + q);
                dy2 = fma(dy / d2, dy, dy2);
                dg2 = fma(dg * d2, dg, dg2);
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) { dy2 += __shfl_xor_sync(kFull, dy2, o); dg2 += __shfl_xor_sync(kFull, dg2, o); }
            if (lane == 0) { sh_dot[warp] = dy2; sh_r2[warp] = dg2; }
            __syncthreads();
            dy2 = 0.0; dg2 = 0.0;
            for (int w = 0; w < nwarps; ++w) { dy2 += sh_dot[w]; dg2 += sh_r2[w]; }
            __syncthreads();                                        // the scratch is reused below
            if (dy2 > 0.0 && dg2 > 0.0) eta_t = sqrt(dy2) / sqrt(dg2);
        }
        eta_t = fmin(fmax(eta_t, p.eta_lo), p.eta_hi);
    }
    double dot = 0.0, r2 = 0.0, rinf = 0.0;
    // four elements per thread and pass, every load issued before the first dependent store: the loop is a chain of
    // L2 round trips, and this CTA runs alone at the end of the launch
    constexpr int U = 4;
    for (int q0 = tid; q0 < p.R; q0 += U * nthreads) {
        double sv[U], bb[U], le[U], lo[U], et[U]; bool eq[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int q = q0 + u * nthreads;
            sv[u] = 0.0; bb[u] = 0.0; le[u] = 0.0; lo[u] = 0.0; et[u] = eta_t; eq[u] = false;
            if (q < p.R) {
                sv[u] = row_sum(p, q); bb[u] = row_rhs(p, q); le[u] = __ldcg(p.lam_eval + q);
                if (p.row_eq) eq[u] = __ldg(p.row_eq + q) != 0;
                if (p.update) {
                    lo[u] = __ldcg(p.lam_cur + q);
                    if (p.step_scale) et[u] = eta_t * __ldg(p.step_scale + q);
                }
            }
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int q = q0 + u * nthreads;
            if (q >= p.R) break;
            if (q < p.JM) p.s_fix[q] = 0ull;
            const double g = sv[u] - bb[u];
            dot = fma(le[u], g, dot);
            const double viol = eq[u] ? fabs(g) : fmax(g, 0.0);
            r2 = fma(viol, viol, r2); rinf = fmax(rinf, viol);
            if (p.grad_out) p.grad_out[q] = g;
            if (p.update) {
                if (p.tr_grad) p.tr_grad[n * p.R + q] = g;
                if (p.step_rule == 1) { p.y_prev[q] = le[u]; p.g_prev[q] = g; }
                const double lv = le[u] + et[u] * g;
                const double ln = eq[u] ? lv : fmax(0.0, lv);            // lambda >= 0 on inequality coordinates only
                p.lam_cur[q] = ln;
                p.y[q] = ln + beta * (ln - lo[u]);
                if (p.tr_lam) p.tr_lam[n * p.R + q] = ln;
            }
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        dot += __shfl_xor_sync(kFull, dot, o);
        r2 += __shfl_xor_sync(kFull, r2, o);
        rinf = fmax(rinf, __shfl_xor_sync(kFull, rinf, o));
    }
    if (lane == 0) { sh_dot[warp] = dot; sh_r2[warp] = r2; sh_inf[warp] = rinf; }
    __syncthreads();
    if (tid == 0) {
        dot = 0.0; r2 = 0.0; rinf = 0.0;
        for (int w = 0; w < nwarps; ++w) { dot += sh_dot[w]; r2 += sh_r2[w]; rinf = fmax(rinf, sh_inf[w]); }
        const double obj = (double)(long long)__ldcg(p.sc_fix + 0) * p.inv_scale_obj;
        const double reg = 0.5 * p.gamma * ((double)(long long)__ldcg(p.sc_fix + 1) * p.inv_scale_sq);
        p.sc_fix[0] = 0ull; p.sc_fix[1] = 0ull; p.sc_fix[2] = 0ull;
        const double g = obj + reg + dot;
        const double nr2 = sqrt(r2);
        if (p.scalars_out) {
            p.scalars_out[0] = g; p.scalars_out[1] = obj; p.scalars_out[2] = reg; p.scalars_out[3] = rinf; p.scalars_out[4] = nr2;
            p.scalars_out[5] = -dot;                                      // (obj + reg) - g: Table 4's primal-dual gap
        }
        if (p.update) {
            if (p.tr_g) p.tr_g[n] = g;
            if (p.tr_rinf) p.tr_rinf[n] = rinf;
            if (p.tr_r2) p.tr_r2[n] = nr2;
            if (p.tr_eta) p.tr_eta[n] = eta_t;
            p.state->t = t + 1; p.state->n = n + 1;
        }
    }
}

// Grid epilogue of every gradient kernel: the CTA that flushes last (threadFenceReduction pattern) runs
// finalize_block, so one launch is one whole dual-ascent iteration (a1-a6).  `sh`: kFinalizeScratchBytes of shared
// memory no longer used for anything else.  Every thread of the CTA must call it after its last accumulator flush.
__device__ __forceinline__ void grid_epilogue(const FinalizeParams& f, double* sh, int nthreads) {
    int* flag = reinterpret_cast<int*>(sh + 96);
    if (f.done == nullptr) return;                      // DUALIP_RED_CSC: a4-a6 run as launches of their own
    __threadfence();                                    // this thread's RED/atomics are visible device-wide
    __syncthreads();
    if (threadIdx.x == 0) *flag = (atomicAdd(f.done, 1u) == gridDim.x - 1) ? 1 : 0;
    __syncthreads();
    if (*flag) {
        __threadfence();
        finalize_block(f, sh, threadIdx.x, nthreads);
        if (threadIdx.x == 0) *f.done = 0u;
    }
}

// Whole-warp path for rows longer than the register budget: every pass re-reads the row (L1/L2 resident).
template <int M, bool LAM_SMEM, bool ACC_SMEM>
__device__ __noinline__ void long_row(const GradParams& p, const double* s_lam, double mu, unsigned* s_lo, unsigned* s_hi,
                                      long long beg, long long end, long long& obj_l, long long& sq_l, long long& cnt_l) {
    const int lane = threadIdx.x & 31;
    const int mm = p.m;
    int j; float cc; float aa[M > 0 ? M : 4];
    float wmax = -CUDART_INF_F;
    for (long long q = beg + lane; q < end; q += 32)
        wmax = fmaxf(wmax, (float)(-eval_t<M, LAM_SMEM>(p, s_lam, mu, q, mm, j, cc, aa)));
    const float m32 = group_max<32>(wmax);
    const bool ineq = p.proj != PROJ_SIMPLEX_EQ;
    if (ineq && !(m32 > 0.0f)) {
        if (p.x) for (long long q = beg + lane; q < end; q += 32) p.x[q] = 0.0f;
        return;
    }
    const double md = (double)m32;
    const float mv = m32 * p.inv_gamma_f, z = p.z;
    float tau;
    double ref = 0.0;                                  // box-cut: reference point (in v units) u is taken relative to
    if (!p.general_boxcut) {
        float theta = -z - (1.2e-7f * fabsf(mv) + 1e-6f);
        int n_prev = -1;
        for (;;) {
            float s = 0.0f; int n = 0;
            for (long long q = beg + lane; q < end; q += 32) {
                const float u = (float)(-eval_t<M, LAM_SMEM>(p, s_lam, mu, q, mm, j, cc, aa) - md) * p.inv_gamma_f;
                if (u > theta) { s += u; ++n; }
            }
            s = group_sum<32>(s); n = group_sum_i<32>(n);
            if (n == n_prev || n == 0) break;
            theta = fmaxf((s - z) / (float)n, theta);
            n_prev = n;
        }
        tau = ineq ? fmaxf(theta, -mv) : theta;
    } else {
        // same three steps as the register path (see there), re-reading the row on every pass
        const float ub = p.ub;
        const double ig = p.inv_gamma;
        float s0 = 0.0f;
        for (long long q = beg + lane; q < end; q += 32)
            s0 += fminf(fmaxf((float)(-eval_t<M, LAM_SMEM>(p, s_lam, mu, q, mm, j, cc, aa) * ig), 0.0f), ub);
        s0 = group_sum<32>(s0);
        if (s0 <= z) { ref = 0.0; tau = 0.0f; }
        else {
            float lo = -mv, hi = 1.2e-7f * fabsf(mv) + 1e-6f;
            for (int it = 0; it < 36; ++it) {
                const float mid = 0.5f * (lo + hi);
                float s = 0.0f;
                for (long long q = beg + lane; q < end; q += 32) {
                    const float u = (float)(-eval_t<M, LAM_SMEM>(p, s_lam, mu, q, mm, j, cc, aa) - md) * p.inv_gamma_f;
                    s += fminf(fmaxf(u - mid, 0.0f), ub);
                }
                s = group_sum<32>(s);
                if (s > z) lo = mid; else hi = mid;
            }
            const float tc = 0.5f * (lo + hi);
            const float eps = (hi - lo) + 1e-6f + 4.8e-7f * fabsf(tc);
            ref = md * ig + (double)tc;
            float dlo = -eps, dhi = eps;
            for (int it = 0; it < 26; ++it) {
                const float mid = 0.5f * (dlo + dhi);
                float s = 0.0f;
                for (long long q = beg + lane; q < end; q += 32) {
                    const float u = (float)(-eval_t<M, LAM_SMEM>(p, s_lam, mu, q, mm, j, cc, aa) * ig - ref);
                    s += fminf(fmaxf(u - mid, 0.0f), ub);
                }
                s = group_sum<32>(s);
                if (s > z) dlo = mid; else dhi = mid;
            }
            const float mid = 0.5f * (dlo + dhi);
            float sF = 0.0f; int nF = 0, nU = 0;
            for (long long q = beg + lane; q < end; q += 32) {
                const float u = (float)(-eval_t<M, LAM_SMEM>(p, s_lam, mu, q, mm, j, cc, aa) * ig - ref);
                const float d = u - mid;
                if (d >= ub) ++nU; else if (d > 0.0f) { sF += u; ++nF; }
            }
            sF = group_sum<32>(sF); nF = group_sum_i<32>(nF); nU = group_sum_i<32>(nU);
            tau = mid;
            if (nF > 0) {
                const float pol = (sF + (float)nU * ub - z) / (float)nF;
                if (pol >= dlo && pol <= dhi) tau = pol;
            }
        }
    }
    const float cap = p.general_boxcut ? p.ub : CUDART_INF_F;
    for (long long q = beg + lane; q < end; q += 32) {
        const double tq = eval_t<M, LAM_SMEM>(p, s_lam, mu, q, mm, j, cc, aa);
        const float u = p.general_boxcut ? (float)(-tq * p.inv_gamma - ref) : (float)(-tq - md) * p.inv_gamma_f;
        const float x = fminf(fmaxf(u - tau, 0.0f), cap);
        if (p.x) p.x[q] = x;
        if (x > 0.0f) {
            obj_l += to_fix(cc * x, p.scale_obj); sq_l += to_fix(x * x, p.scale_sq); cnt_l += to_fix(x, p.scale_cnt);
            contribute<M, ACC_SMEM>(p, s_lo, s_hi, mm, j, aa, x);
        }
    }
}

// The fused per-user gradient kernel.  G lanes own one row; rows of up to G*KREG nonzeros live in registers.
template <int G, int KREG, int M, bool LAM_SMEM, bool ACC_SMEM>
__global__ void __launch_bounds__(kBlockThreads, 1) k_grad(const GradParams p, const FinalizeParams f) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int MA = M > 0 ? M : 4;
    const int mm = M > 0 ? M : p.m;
    const int JM = p.J * mm;
    double* s_lam = reinterpret_cast<double*>(smem_raw);
    unsigned* s_lo = reinterpret_cast<unsigned*>(smem_raw + (LAM_SMEM ? (size_t)JM * 8 : 0));
    unsigned* s_hi = s_lo + JM;
    if (LAM_SMEM) for (int q = threadIdx.x; q < JM; q += kBlockThreads) s_lam[q] = p.lambda[q];
    if (ACC_SMEM) for (int q = threadIdx.x; q < 2 * JM; q += kBlockThreads) s_lo[q] = 0u;
    __syncthreads();

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    constexpr int RPW = 32 / G;
    const int gl = lane & (G - 1), grp = lane / G;
    const unsigned gmask = G == 32 ? kFull : (((1u << G) - 1u) << (lane & ~(G - 1)));
    const long long nsteps = (p.I + RPW - 1) / RPW;
    const bool ineq = p.proj != PROJ_SIMPLEX_EQ;
    const float z = p.z;
    // per-lane partial scalars, every product converted to fixed point on its own: the sums do not depend on which lane
    // or CTA a row lands on (bit-reproducible for any launch geometry, like the item sums)
    long long obj_l = 0, sq_l = 0, cnt_l = 0;
    const double mu = p.count_on ? __ldg(p.lambda + JM) : 0.0;      // dual of the global-count row (R21)

    for (long long step = (long long)blockIdx.x * kWarpsPerBlock + warp; step < nsteps;
         step += (long long)gridDim.x * kWarpsPerBlock) {
        const long long row = step * RPW + grp;
        long long beg = 0, end = 0;
        if (row < p.I) { beg = __ldg(p.row_ptr + row); end = __ldg(p.row_ptr + row + 1); }
        if (p.long_thr > 0 && end - beg > p.long_thr) end = beg;     // a long row: k_grad_long takes it
        const long long len = end - beg;
        const bool is_long = len > (long long)G * KREG;
        const int flen = is_long ? 0 : (int)len;
        int nch_max = (flen + G - 1) / G;
#pragma unroll
        for (int o = G; o < 32; o <<= 1) nch_max = max(nch_max, __shfl_xor_sync(kFull, nch_max, o));

        if (nch_max > 0) {
            int jj[KREG]; float cc[KREG]; float aa[KREG][MA]; double t[KREG];
            // loads first (independent, so they overlap), then the lambda gather and the fp64 FMA
#pragma unroll
            for (int k = 0; k < KREG; ++k) {
                if (k >= nch_max) break;
                const int e = k * G + gl;
                jj[k] = 0; cc[k] = 0.0f;
#pragma unroll
                for (int f = 0; f < MA; ++f) aa[k][f] = 0.0f;
                if (e < flen) {
                    const long long q = beg + e;
                    jj[k] = __ldg(p.idx + q);
                    cc[k] = __ldg(p.c + q);
                    if (M > 0) {
#pragma unroll
                        for (int f = 0; f < MA; ++f) aa[k][f] = __ldg(p.a + q * M + f);
                    } else {
#pragma unroll
                        for (int f = 0; f < MA; ++f) if (f < mm) aa[k][f] = __ldg(p.a + q * mm + f);
                    }
                }
            }
            float wmax = -CUDART_INF_F;
#pragma unroll
            for (int k = 0; k < KREG; ++k) {
                if (k >= nch_max) break;
                double tk = CUDART_INF;
                if (k * G + gl < flen) {
                    tk = (double)cc[k] + mu;
#pragma unroll
                    for (int f = 0; f < MA; ++f) {
                        if (f < mm) {
                            const double l = LAM_SMEM ? s_lam[jj[k] * mm + f] : __ldg(p.lambda + (long long)jj[k] * mm + f);
                            tk = fma((double)aa[k][f], l, tk);
                        }
                    }
                    wmax = fmaxf(wmax, (float)(-tk));
                }
                t[k] = tk;
            }
            const float gm = group_max<G>(wmax);                      // full-mask shuffles: every lane takes part
            const float m32 = flen > 0 ? gm : 0.0f;
            const bool alive = flen > 0 && (!ineq || m32 > 0.0f);
            const double md = (double)m32;
            const float mv = m32 * p.inv_gamma_f;
            const float cut = alive ? -z - (1.2e-7f * fabsf(mv) + 1e-6f) : CUDART_INF_F;

            float u[KREG];
            int cnt = 0;
#pragma unroll
            for (int k = 0; k < KREG; ++k) {
                if (k >= nch_max) break;
                u[k] = (float)(-t[k] - md) * p.inv_gamma_f;          // -inf on padding lanes
                cnt += __popc(__ballot_sync(kFull, u[k] > cut) & gmask);
            }

            float tau = CUDART_INF_F;
            bool vertex = false;
            if (!p.general_boxcut) {
                vertex = __all_sync(kFull, cnt <= 1);
                if (!vertex) {
                    // Michelot fixed point on the equality problem; theta only grows, the support only shrinks
                    float theta = cut;
                    int n_prev = cnt;
                    for (;;) {
                        float s = 0.0f;
#pragma unroll
                        for (int k = 0; k < KREG; ++k) { if (k >= nch_max) break; s += (u[k] > theta) ? u[k] : 0.0f; }
                        s = group_sum<G>(s);
                        // max(): theta is non-decreasing in exact arithmetic; enforcing it makes termination unconditional
                        const float th_new = n_prev > 0 ? fmaxf((s - z) / (float)n_prev, theta) : CUDART_INF_F;
                        int n = 0;
#pragma unroll
                        for (int k = 0; k < KREG; ++k) {
                            if (k >= nch_max) break;
                            n += __popc(__ballot_sync(kFull, u[k] > th_new) & gmask);
                        }
                        const bool changed = n != n_prev;
                        theta = th_new; n_prev = n;
                        if (!__any_sync(kFull, changed)) break;
                    }
                    tau = ineq ? fmaxf(theta, -mv) : theta;
                }
            } else if (__any_sync(kFull, alive)) {
                // box-cut with ub < z.  Free entries can sit far below the row maximum, where u (relative to the
                // maximum) has lost absolute precision in fp32; so (1) test slackness on v itself, (2) bracket
                // tau by bisection on u, (3) re-centre on the coarse tau in fp64 and solve the linear piece there.
                const float ub = p.ub;
                const double ig = p.inv_gamma;
                float s0 = 0.0f;
#pragma unroll
                for (int k = 0; k < KREG; ++k) { if (k >= nch_max) break; s0 += fminf(fmaxf((float)(-t[k] * ig), 0.0f), ub); }
                s0 = group_sum<G>(s0);
                const bool slack = !alive || s0 <= z;
                float td = 0.0f;
                if (!__all_sync(kFull, slack)) {
                    float lo = alive ? -mv : 0.0f, hi = alive ? 1.2e-7f * fabsf(mv) + 1e-6f : 0.0f;
                    for (int it = 0; it < 36; ++it) {
                        const float mid = 0.5f * (lo + hi);
                        float sm = 0.0f;
#pragma unroll
                        for (int k = 0; k < KREG; ++k) { if (k >= nch_max) break; sm += fminf(fmaxf(u[k] - mid, 0.0f), ub); }
                        sm = group_sum<G>(sm);
                        if (sm > z) lo = mid; else hi = mid;
                    }
                    const float tc = 0.5f * (lo + hi);
                    const float eps = (hi - lo) + 1e-6f + 4.8e-7f * fabsf(tc);
                    if (!slack) {
#pragma unroll
                        for (int k = 0; k < KREG; ++k) { if (k >= nch_max) break; u[k] = (float)((-t[k] - md) * ig - (double)tc); }
                    }
                    float dlo = -eps, dhi = eps;
                    for (int it = 0; it < 26; ++it) {
                        const float mid = 0.5f * (dlo + dhi);
                        float sm = 0.0f;
#pragma unroll
                        for (int k = 0; k < KREG; ++k) { if (k >= nch_max) break; sm += fminf(fmaxf(u[k] - mid, 0.0f), ub); }
                        sm = group_sum<G>(sm);
                        if (sm > z) dlo = mid; else dhi = mid;
                    }
                    const float mid = 0.5f * (dlo + dhi);
                    float sF = 0.0f; int nF = 0, nU = 0;
#pragma unroll
                    for (int k = 0; k < KREG; ++k) {
                        if (k >= nch_max) break;
                        const float d = u[k] - mid;
                        if (d >= ub) ++nU; else if (d > 0.0f) { sF += u[k]; ++nF; }
                    }
                    sF = group_sum<G>(sF); nF = group_sum_i<G>(nF); nU = group_sum_i<G>(nU);
                    td = mid;
                    if (nF > 0) {
                        const float pol = (sF + (float)nU * ub - z) / (float)nF;
                        if (pol >= dlo && pol <= dhi) td = pol;
                    }
                }
                if (slack) {
#pragma unroll
                    for (int k = 0; k < KREG; ++k) { if (k >= nch_max) break; u[k] = (float)(-t[k] * ig); }
                    td = 0.0f;
                }
                tau = alive ? td : CUDART_INF_F;
            }
            const float cap = p.general_boxcut ? p.ub : CUDART_INF_F;
#pragma unroll
            for (int k = 0; k < KREG; ++k) {
                if (k >= nch_max) break;
                float x;
                if (vertex) x = (u[k] > cut) ? (ineq ? fminf(z, u[k] + mv) : z) : 0.0f;
                else x = fminf(fmaxf(u[k] - tau, 0.0f), cap);
                const int e = k * G + gl;
                if (p.x && e < flen) p.x[beg + e] = x;
                if (x > 0.0f) {
                    obj_l += to_fix(cc[k] * x, p.scale_obj); sq_l += to_fix(x * x, p.scale_sq); cnt_l += to_fix(x, p.scale_cnt);
                    contribute<M, ACC_SMEM>(p, s_lo, s_hi, mm, jj[k], aa[k], x);
                }
            }
        }
        // rows beyond the register budget: the whole warp takes them one at a time
        unsigned long_mask = __ballot_sync(kFull, is_long && gl == 0);
        while (long_mask) {
            const int src = __ffs(long_mask) - 1;
            long_mask &= long_mask - 1;
            const long long b = __shfl_sync(kFull, beg, src), e = __shfl_sync(kFull, end, src);
            long_row<M, LAM_SMEM, ACC_SMEM>(p, s_lam, mu, s_lo, s_hi, b, e, obj_l, sq_l, cnt_l);
        }
    }

    // a5: per-lane fixed-point partials -> one atomic per warp and scalar
    {
        long long so = obj_l, ss = sq_l, sn = cnt_l;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            so += __shfl_xor_sync(kFull, so, o); ss += __shfl_xor_sync(kFull, ss, o); sn += __shfl_xor_sync(kFull, sn, o);
        }
        if (lane == 0) {
            if (so) atomicAdd(p.sc_fix + 0, (unsigned long long)so);
            if (ss) atomicAdd(p.sc_fix + 1, (unsigned long long)ss);
            if (sn) atomicAdd(p.sc_fix + 2, (unsigned long long)sn);
        }
    }
    if (ACC_SMEM) {
        __syncthreads();
        for (int q = threadIdx.x; q < JM; q += kBlockThreads) {
            const unsigned long long v = ((unsigned long long)s_hi[q] << 32) | s_lo[q];
            if (v) atomicAdd(p.s_fix + q, v);
        }
    }
    // a4-a6 by the CTA that finishes last; its scratch sits behind lambda and the accumulators
    grid_epilogue(f, reinterpret_cast<double*>(smem_raw + (LAM_SMEM ? (size_t)JM * 8 : 0) + (ACC_SMEM ? (size_t)JM * 8 : 0)), kBlockThreads);
}

// Box projection {lo <= x <= hi}: element-wise, so one thread per nonzero with fully coalesced streams.
template <int M>
__global__ void __launch_bounds__(256) k_grad_box(const GradParams p, const FinalizeParams f) {
    __shared__ double sh_fin[kFinalizeScratchBytes / 8];
    const int mm = M > 0 ? M : p.m;
    long long obj_l = 0, sq_l = 0, cnt_l = 0;
    const double mu = p.count_on ? __ldg(p.lambda + (long long)p.J * mm) : 0.0;
    for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < p.nnz; q += (long long)gridDim.x * blockDim.x) {
        int j; float cc; float aa[M > 0 ? M : 4];
        const double t = eval_t<M, false>(p, nullptr, mu, q, mm, j, cc, aa);
        const double v = -t * p.inv_gamma;
        const float x = (float)fmin(fmax(v, p.box_lo), p.box_hi);
        if (p.x) p.x[q] = x;
        if (x != 0.0f) {
            obj_l += to_fix(cc * x, p.scale_obj); sq_l += to_fix(x * x, p.scale_sq); cnt_l += to_fix(x, p.scale_cnt);
            contribute<M, false>(p, nullptr, nullptr, mm, j, aa, x);
        }
    }
    long long so = obj_l, ss = sq_l, sn = cnt_l;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        so += __shfl_xor_sync(kFull, so, o); ss += __shfl_xor_sync(kFull, ss, o); sn += __shfl_xor_sync(kFull, sn, o);
    }
    if ((threadIdx.x & 31) == 0) {
        if (so) atomicAdd(p.sc_fix + 0, (unsigned long long)so);
        if (ss) atomicAdd(p.sc_fix + 1, (unsigned long long)ss);
        if (sn) atomicAdd(p.sc_fix + 2, (unsigned long long)sn);
    }
    grid_epilogue(f, sh_fin, 256);
}

// ---- a0: create-time kernels -------------------------------------------------------------------------------

// Create-time kernels (not templates): defined in the one translation unit that launches them (dualip_api.cu).
#ifdef DUALIP_HOST_KERNELS
// flags: bit0 row_ptr not monotone, bit1 index out of range, bit2 duplicate item in a row, bit3 some row is not ascending
// (its duplicate check is k_validate_unsorted's: a strictly ascending row cannot hold a duplicate).  One thread per row.
__global__ void k_validate(const long long* __restrict__ row_ptr, const int* __restrict__ idx, long long I, int J,
                           long long nnz, int scan, int* flags, unsigned long long* max_len) {
    unsigned long long lmax = 0;
    int f = 0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < I; i += (long long)gridDim.x * blockDim.x) {
        const long long beg = row_ptr[i], end = row_ptr[i + 1];
        if (beg > end || beg < 0 || end > nnz) { f |= 1; continue; }
        if ((unsigned long long)(end - beg) > lmax) lmax = (unsigned long long)(end - beg);
        if (!scan) continue;
        int prev = -1;
        for (long long q = beg; q < end; ++q) {
            const int j = idx[q];
            if (j < 0 || j >= J) f |= 2;
            if (j <= prev) f |= 8;
            prev = j;
        }
    }
    if (f) atomicOr(flags, f);
    atomicMax(max_len, lmax);
}

// Duplicate check of the rows that are not ascending (launched only when k_validate saw one): one WARP per row, every
// element compared with the later ones lane-strided -- len^2 / 32 steps per row, rows in parallel, coalesced reads -- instead
// of one thread walking len^2 pairs.  row_ptr has been checked (bit0 clear) before this runs.
__global__ void k_validate_unsorted(const long long* __restrict__ row_ptr, const int* __restrict__ idx, long long I, int* flags) {
    const int lane = threadIdx.x & 31;
    const long long warp0 = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = ((long long)gridDim.x * blockDim.x) >> 5;
    bool dup = false;
    for (long long i = warp0; i < I; i += nwarps) {
        const long long beg = row_ptr[i], end = row_ptr[i + 1];
        bool asc = true;
        for (long long q = beg + lane; q + 1 < end; q += 32) asc = asc && idx[q] < idx[q + 1];
        if (__all_sync(kFull, asc)) continue;
        for (long long q = beg; q + 1 < end; ++q) {
            const int j = idx[q];
            for (long long r = q + 1 + lane; r < end; r += 32) dup = dup || idx[r] == j;
        }
    }
    if (dup) atomicOr(flags, 4);
}

// max |a|, max |c| as float bit patterns (order-independent)
__global__ void k_absmax(const float* __restrict__ a, long long na, const float* __restrict__ c, long long nc, unsigned* out) {
    unsigned ma = 0, mc = 0;
    for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < na; q += (long long)gridDim.x * blockDim.x)
        ma = max(ma, __float_as_uint(fabsf(a[q])));
    for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < nc; q += (long long)gridDim.x * blockDim.x)
        mc = max(mc, __float_as_uint(fabsf(c[q])));
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { ma = max(ma, __shfl_xor_sync(kFull, ma, o)); mc = max(mc, __shfl_xor_sync(kFull, mc, o)); }
    if ((threadIdx.x & 31) == 0) { atomicMax(out + 0, ma); atomicMax(out + 1, mc); }
}

// fixed-point column sums: colsq[j*m+k] += a^2 (for L, R2, and the Jacobi scaling, R18), colabs[j*m+k] += |a|, cabs += |c|
__global__ void k_col_stats(const int* __restrict__ idx, const float* __restrict__ a, const float* __restrict__ c,
                            long long nnz, int m, double scale_sq, double scale_abs, double scale_c,
                            unsigned long long* colsq, unsigned long long* colabs, unsigned long long* cabs,
                            int do_a, int do_c) {
    long long lc = 0;
    for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < nnz; q += (long long)gridDim.x * blockDim.x) {
        if (do_a) {
            const int j = idx[q];
            for (int k = 0; k < m; ++k) {
                const double v = (double)a[q * m + k];
                const long long fa = __double2ll_rn(fabs(v) * scale_abs);
                if (fa) atomicAdd(colabs + (long long)j * m + k, (unsigned long long)fa);
                const long long fq = __double2ll_rn(v * v * scale_sq);
                if (fq) atomicAdd(colsq + (long long)j * m + k, (unsigned long long)fq);
            }
        }
        if (do_c) lc += __double2ll_rn(fabs((double)c[q]) * scale_c);
    }
    if (do_c) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) lc += __shfl_xor_sync(kFull, lc, o);
        if ((threadIdx.x & 31) == 0 && lc) atomicAdd(cabs, (unsigned long long)lc);
    }
}

// out[0] = max_j sum_k colsq[j*m+k] (fixed), out[1] = max_q colabs (fixed), out[2] = max_j #{k : colsq[j*m+k] > 0}
__global__ void __launch_bounds__(1024) k_reduce_stats(const unsigned long long* colsq, int J, int m, const unsigned long long* colabs,
                                                       int JM, unsigned long long* out) {
    __shared__ unsigned long long sh[3][32];
    unsigned long long a = 0, b = 0, c = 0;
    for (int j = threadIdx.x; j < J; j += 1024) {
        unsigned long long sj = 0, nj = 0;
        for (int k = 0; k < m; ++k) { const unsigned long long v = colsq[(long long)j * m + k]; sj += v; nj += v ? 1ull : 0ull; }
        a = max(a, sj); c = max(c, nj);
    }
    for (int q = threadIdx.x; q < JM; q += 1024) b = max(b, colabs[q]);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        a = max(a, __shfl_xor_sync(kFull, a, o)); b = max(b, __shfl_xor_sync(kFull, b, o)); c = max(c, __shfl_xor_sync(kFull, c, o));
    }
    if ((threadIdx.x & 31) == 0) { sh[0][threadIdx.x >> 5] = a; sh[1][threadIdx.x >> 5] = b; sh[2][threadIdx.x >> 5] = c; }
    __syncthreads();
    if (threadIdx.x == 0) {
        a = 0; b = 0; c = 0;
        for (int w = 0; w < 32; ++w) { a = max(a, sh[0][w]); b = max(b, sh[1][w]); c = max(c, sh[2][w]); }
        out[0] = a; out[1] = b; out[2] = c;
    }
}

// Jacobi preconditioning (R18).  Row scaling A' = D A, b' = D b with D_qq = 1/|A_q*|_2 is, in the
// original variables lambda = D lambda', a per-coordinate step: lambda+ = max(0, y + eta' d_q^2 grad_q).  Only
// d_q^2 = 1/sum_i (a^k_ij)^2 is needed (1 for rows of zero norm), and no row data is rescaled.
__global__ void k_jacobi_step_scale(const unsigned long long* colsq, double inv_scale_sq, int JM, double* step_scale) {
    for (int q = blockIdx.x * blockDim.x + threadIdx.x; q < JM; q += gridDim.x * blockDim.x) {
        const double n2 = (double)(long long)colsq[q] * inv_scale_sq;
        step_scale[q] = n2 > 0.0 ? 1.0 / n2 : 1.0;
    }
}

// user-sharded multi-GPU helper: integer accumulation of another shard's sums
__global__ void k_acc_add(unsigned long long* acc, const unsigned long long* in, long long n) {
    for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < n; q += (long long)gridDim.x * blockDim.x) acc[q] += in[q];
}

#endif  // DUALIP_HOST_KERNELS

}  // namespace dualip_dev
