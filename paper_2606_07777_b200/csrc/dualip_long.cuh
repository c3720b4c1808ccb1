// dualip_long.cuh -- LONG rows at CTA granularity with shared-memory staging (BASELINE.json north_star: "long rows run at CTA
// granularity with shared-memory staging"; the paper's own fused kernel stops at 8192 nonzeros per column).
//
// A row is "long" when it does not fit the streaming kernel's stage next to a useful tile (dualip_api.cu: plan_tma's row cap;
// a few hundred to a few thousand nonzeros depending on J*m), or, on the direct-load plan, when it is beyond 4096 nonzeros.
// The other kernels skip those rows; this one takes them, ONE CTA PER ROW (persistent CTAs over the list of long rows built
// at create), before the main gradient kernel of the same evaluation, adding into the same fixed-point accumulators:
//
//   pass A   every thread streams its share of the row (coalesced idx / c / a), gathers the fp64 duals, forms t = c + a.lambda
//            (+ mu) by fp64 FMA and the block takes the maximum of RN_f32(-t): the shift of DESIGN.md "Numerics";
//   pass B   the row again (now an L2 hit), u = RN_f32((-t - max) / gamma) into SHARED memory (4 bytes per nonzero: rows of up
//            to ~56,000 nonzeros; longer ones recompute u from global memory on every pass instead);
//   Michelot's fixed point on the staged u: per iteration one strided pass over shared memory + one block reduction of
//            (sum, count); theta only grows, the support only shrinks (same arithmetic as the warp paths' slow_row);
//   last     x = max(u - tau, 0) written coalesced; the nonzero ones pushed (RED.ADD.64 per item and family, per-thread
//            fixed-point scalars reduced once per CTA).
//
// Simplex kinds only (inequality / equality form, and the box-cut with ub >= z, which IS the simplex, R10); an instance whose
// long rows would need the capped search of the genuine box-cut stays on the whole-warp path of k_grad.
#pragma once
#include "dualip_kernels.cuh"

namespace dualip_dev {

constexpr int kLongThreads = 1024;

struct LongParams {
    GradParams g;
    const long long* __restrict__ long_ids;   // rows this kernel takes
    long long n_long;
    int ucap;                                 // floats of shared memory for the staged u (0: always recompute)
};

// f(q, t, j, c, a) for every nonzero q of [beg, end) this thread owns (thread-strided: coalesced), t = c + a.lambda + mu in
// fp64.  Four nonzeros per thread and trip, all their loads issued before the first use: the dual gathers are L2 round trips
// (J*m is beyond shared memory whenever rows get this long), and one dependent chain per thread leaves the CTA latency-bound.
template <int M, class F>
__device__ __forceinline__ void for_each_t(const GradParams& p, int mm, double mu, long long beg, long long end, F&& f) {
    constexpr int U = 4, MA = M > 0 ? M : 4;                        // 1024 threads x 4 x 12 bytes = 48 KB of row data in flight per trip
    for (long long q0 = beg + threadIdx.x; q0 < end; q0 += (long long)U * kLongThreads) {
        int j[U]; float cc[U]; float aa[U][MA]; double l[U][MA];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const long long q = q0 + (long long)u * kLongThreads < end ? q0 + (long long)u * kLongThreads : q0;
            j[u] = __ldg(p.idx + q); cc[u] = __ldg(p.c + q);
#pragma unroll
            for (int k = 0; k < MA; ++k) aa[u][k] = k < mm ? __ldg(p.a + q * mm + k) : 0.0f;
        }
#pragma unroll
        for (int u = 0; u < U; ++u)
#pragma unroll
            for (int k = 0; k < MA; ++k) l[u][k] = k < mm ? __ldg(p.lambda + (long long)j[u] * mm + k) : 0.0;
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const long long q = q0 + (long long)u * kLongThreads;
            if (q < end) {
                double t = (double)cc[u] + mu;
#pragma unroll
                for (int k = 0; k < MA; ++k) if (k < mm) t = fma((double)aa[u][k], l[u][k], t);
                f(q, t, j[u], cc[u], aa[u]);
            }
        }
    }
}

// block-wide (max) / (sum, count) with every thread receiving the result; `sh` = 2 * 32 doubles of scratch
__device__ __forceinline__ float block_max(float v, float* sh) {
    v = group_max<32>(v);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    __syncthreads();
    if (lane == 0) sh[warp] = v;
    __syncthreads();
    float r = sh[0];
    for (int w = 1; w < kLongThreads / 32; ++w) r = fmaxf(r, sh[w]);
    return r;
}
__device__ __forceinline__ void block_sum(float& s, int& n, float* sh) {
    s = group_sum<32>(s); n = group_sum_i<32>(n);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    __syncthreads();
    if (lane == 0) { sh[warp] = s; reinterpret_cast<int*>(sh)[32 + warp] = n; }
    __syncthreads();
    float rs = 0.0f; int rn = 0;
    for (int w = 0; w < kLongThreads / 32; ++w) { rs += sh[w]; rn += reinterpret_cast<int*>(sh)[32 + w]; }   // fixed order
    s = rs; n = rn;
}

template <int M>
__global__ void __launch_bounds__(kLongThreads, 1) k_grad_long(const LongParams lp) {
    extern __shared__ __align__(16) unsigned char smem_long[];
    const GradParams& p = lp.g;
    float* sh = reinterpret_cast<float*>(smem_long);                 // 64 words of reduction scratch
    float* su = sh + 64;                                             // staged u
    const int mm = M > 0 ? M : p.m;
    const bool ineq = p.proj != PROJ_SIMPLEX_EQ;
    const float z = p.z;
    const double mu = p.count_on ? __ldg(p.lambda + (long long)p.J * mm) : 0.0;
    long long obj_l = 0, sq_l = 0, cnt_l = 0;
    int j; float cc; float aa[M > 0 ? M : 4];

    for (long long r = blockIdx.x; r < lp.n_long; r += gridDim.x) {
        const long long row = lp.long_ids[r];
        const long long beg = __ldg(p.row_ptr + row), end = __ldg(p.row_ptr + row + 1);
        const long long len = end - beg;
        const bool staged = len <= (long long)lp.ucap;
        // pass A: the row maximum of RN_f32(-t)
        float wmax = -CUDART_INF_F;
        for_each_t<M>(p, mm, mu, beg, end, [&](long long, double t, int, float, const float*) { wmax = fmaxf(wmax, (float)(-t)); });
        const float m32 = block_max(wmax, sh);
        if (ineq && !(m32 > 0.0f)) {                                  // nothing is positive: the whole row is zero
            if (p.x) for (long long q = beg + threadIdx.x; q < end; q += kLongThreads) p.x[q] = 0.0f;
            continue;
        }
        const double md = (double)m32;
        const float mv = m32 * p.inv_gamma_f;
        // pass B: the shifted values (exact subtraction in fp64, then fp32: every support entry is in [-z, 0])
        const float igf = p.inv_gamma_f;
        if (staged) for_each_t<M>(p, mm, mu, beg, end, [&](long long q, double t, int, float, const float*) { su[q - beg] = (float)(-t - md) * igf; });
        __syncthreads();
        float theta = -z - (1.2e-7f * fabsf(mv) + 1e-6f);
        int n_prev = -1;
        for (;;) {                                                    // Michelot: theta only grows, the support only shrinks
            float s = 0.0f; int n = 0;
            if (staged) {
                for (long long e = threadIdx.x; e < len; e += kLongThreads) { const float u = su[e]; if (u > theta) { s += u; ++n; } }
            } else {
                for_each_t<M>(p, mm, mu, beg, end, [&](long long, double t, int, float, const float*) {
                    const float u = (float)(-t - md) * igf;
                    if (u > theta) { s += u; ++n; }
                });
            }
            block_sum(s, n, sh);
            if (n == n_prev || n == 0) break;
            theta = fmaxf((s - z) / (float)n, theta);
            n_prev = n;
        }
        const float tau = ineq ? fmaxf(theta, -mv) : theta;
        if (staged) {
            for (long long e = threadIdx.x; e < len; e += kLongThreads) {
                const long long q = beg + e;
                const float x = fmaxf(su[e] - tau, 0.0f);
                if (p.x) p.x[q] = x;
                if (x > 0.0f) {
                    j = __ldg(p.idx + q); cc = __ldg(p.c + q);
#pragma unroll
                    for (int f = 0; f < (M > 0 ? M : 4); ++f) aa[f] = f < mm ? __ldg(p.a + q * mm + f) : 0.0f;
                    obj_l += to_fix(cc * x, p.scale_obj); sq_l += to_fix(x * x, p.scale_sq); cnt_l += to_fix(x, p.scale_cnt);
                    contribute<M, false>(p, nullptr, nullptr, mm, j, aa, x);
                }
            }
        } else {
            for_each_t<M>(p, mm, mu, beg, end, [&](long long q, double t, int jq, float cq, const float* aq) {
                const float x = fmaxf((float)(-t - md) * igf - tau, 0.0f);
                if (p.x) p.x[q] = x;
                if (x > 0.0f) {
                    float a2[M > 0 ? M : 4];
#pragma unroll
                    for (int f = 0; f < (M > 0 ? M : 4); ++f) a2[f] = aq[f];
                    obj_l += to_fix(cq * x, p.scale_obj); sq_l += to_fix(x * x, p.scale_sq); cnt_l += to_fix(x, p.scale_cnt);
                    contribute<M, false>(p, nullptr, nullptr, mm, jq, a2, x);
                }
            });
        }
        __syncthreads();                                              // su is reused by the next row
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
}

#ifdef DUALIP_HOST_KERNELS
// a0: the list of long rows (any order: every accumulation is an integer sum, and x is written by position)
__global__ void k_collect_long(const long long* __restrict__ row_ptr, long long I, long long thr, long long* ids, unsigned long long* count) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < I; i += (long long)gridDim.x * blockDim.x) {
        if (row_ptr[i + 1] - row_ptr[i] > thr) {
            const unsigned long long k = atomicAdd(count, 1ull);
            if (ids) ids[k] = i;
        }
    }
}
#endif

}  // namespace dualip_dev
