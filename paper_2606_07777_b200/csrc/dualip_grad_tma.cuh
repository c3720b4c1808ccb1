// dualip_grad_tma.cuh -- the streaming gradient kernel: a1-a5 with row data staged HBM -> shared memory by
// TMA bulk copies (cp.async.bulk, SASS UBLKCP) behind mbarriers, one persistent CTA per SM.
//
//   warp 0      producer: for each of this CTA's tiles, waits for a free stage, then issues one bulk copy per
//               array (16-bit item indices, c, a, row_ptr segment) that completes on the stage's "full" mbarrier.
//   warps 1..   consumers: wait for "full", take their row-steps of the tile (G lanes per row, 2*32/G rows per step,
//               steps dealt round-robin over the CTA's step sequence), read the rows straight from shared memory,
//               and release the stage.
//
// Per row the consumers run a two-level scheme:
//   fast path   fp32 filter: w' = fma(a, RN_f32(lambda_j), c) for every nonzero (one FFMA, one 4-byte gather),
//               tracking the two largest values per row.  If the top-2 gap exceeds z*gamma by more than a
//               rigorous rounding bound, x*_i is the vertex z*e_argmax capped by the inequality (min(z, v_max))
//               and only the arg-max lane redoes its nonzero in fp64.  Likewise rows whose maximum is safely
//               below zero are all-zero.  This is the common case at the small gamma the configs run at.
//   slow path   every other row: whole warp, fp64 w, exact row-maximum shift, Michelot iterations in fp32 on
//               the shifted values (or the capped search for box-cut with ub < z), re-reading the row from
//               shared memory on every pass.
//
// A tile is a run of whole rows cut where (row_ptr[r] + kRowCost*r) crosses a multiple of TN (k_build_tiles at
// create), so it holds at most TN + max_row_len nonzeros and TN/kRowCost + 1 rows whatever the row lengths
// (empty rows included).  Tiles are dealt round-robin to CTAs and row-steps round-robin to warps; every
// accumulation (items AND scalars) is 64-bit fixed point, so results do not depend on the launch geometry.
//
// Nothing here waits on DRAM latency: the only global loads in the loop are the producer's tile-table reads,
// prefetched a tile ahead.
#pragma once
#include "dualip_kernels.cuh"

namespace dualip_dev {

constexpr int kTmaConsumerWarps = 15;  // consumer warps of the streaming kernel (+ 1 producer warp)

constexpr int kRowCost = 8;            // each row costs this many "nonzero units" when cutting tiles
constexpr int kTmaStagesMax = 8;
constexpr int kTmaHeaderBytes = 256 + 256 * kTmaConsumerWarps;   // mbarriers (2 x 8) + words + per-warp candidate lists (multiple of 128)

struct TileEntry {                     // 32 bytes, one per tile (+1 sentinel)
    long long row0;                    // first row of the tile
    long long nz0;                     // row_ptr[row0]
};

struct TmaParams {
    GradParams g;
    FinalizeParams f;
    const TileEntry* __restrict__ tiles;   // [ntiles + 1]
    long long ntiles;
    int cap_nz;                        // nonzero capacity of a stage (multiple of 4)
    int cap_rows;                      // row_ptr entries per stage (even)
    int stages;
    int stage_bytes;                   // bytes of one stage (multiple of 16)
    long long nnz8;                    // nnz rounded down to a multiple of 8 (bulk copies stop there)
    const unsigned short* __restrict__ idx16;   // item_idx as 16-bit values (a0: k_encode_idx16)
    long long rows2;                   // (I+1) rounded down to a multiple of 2
    int lo_policy;                     // lambda's low word in shared memory: 0 = decided per launch (see k_grad_tma), 1 = never, 2 = always
    int smem_total;                    // dynamic shared memory of the launch (bytes)
    int* lo_flag;                      // nullable: CTA 0 records the decision here (dualip_info.lambda_lo_smem)
    int dyn_steps;                     // row-steps of a tile dealt 0 = statically (round-robin over the CTA's step sequence), 1 = dynamically
    long long row_cap;                 // > 0: a one-row tile of more than this many nonzeros is a LONG row (k_grad_long's): skipped
    unsigned* check_word;              // -DDUALIP_CHECKED builds: bit set per kind of bounds violation (dualip_info.checks_failed)
};

// ---- checked build (-DDUALIP_CHECKED): compute-sanitizer is closed on the GPU pool this was developed on, so the bounds it
// would have checked are asserted by the kernel itself: every staged-row position against the stage capacity, every item index
// against J before it is used as a shared-memory / accumulator offset, every x position against nnz, every candidate-list slot
// against the warp's list.  A violation sets a bit in a device word (dualip_info.checks_failed); the access is then skipped or
// clamped so the run can finish and report.  Compiled out of the product build.
#ifdef DUALIP_CHECKED
static __device__ unsigned* g_chk_word;
static __device__ int g_chk_cap_nz, g_chk_J, g_chk_cap_rows;
static __device__ long long g_chk_nnz;
#define DUALIP_CHECK(cond, bit) do { if (!(cond)) atomicOr(g_chk_word, 1u << (bit)); } while (0)
#define DUALIP_CHECK_POS(q) DUALIP_CHECK((unsigned)(q) < (unsigned)g_chk_cap_nz, 0)
#define DUALIP_CHECK_ITEM(j) DUALIP_CHECK((unsigned)(j) < (unsigned)g_chk_J, 1)
#define DUALIP_CHECK_X(pos) DUALIP_CHECK((unsigned long long)(pos) < (unsigned long long)g_chk_nnz, 2)
#else
#define DUALIP_CHECK(cond, bit) do { } while (0)
#define DUALIP_CHECK_POS(q) do { } while (0)
#define DUALIP_CHECK_ITEM(j) do { } while (0)
#define DUALIP_CHECK_X(pos) do { } while (0)
#endif
enum { CHK_POS = 0, CHK_ITEM = 1, CHK_X = 2, CHK_LIST = 3, CHK_ROWS = 4, CHK_ROW_EXTENT = 5, CHK_STAGE_BYTES = 6 };

// ---- PTX wrappers (mbarrier + bulk async copy) ---------------------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(void* bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(void* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(void* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(void* bar, unsigned parity) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_LOOP:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE;\n\t"
        "bra WAIT_LOOP;\n\t"
        "DONE:\n\t}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, unsigned bytes, void* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }

// One stage: [idx16 cap_nz*2][c cap_nz*4][a cap_nz*4*m][row_ptr cap_rows*8][meta: int nrows, int rpo, long long nzb, pad]
// The item indices are streamed as 16-BIT values: the streaming plan exists only while RN_f32(lambda) fits in shared memory next
// to the stages, which bounds J*m by ~48,000, so J < 65,536 always, and dualip_create keeps a uint16 copy of item_idx for this
// kernel (2 bytes per nonzero of device memory; the ABI's int32 array is untouched and still what the other kernels read).  Per
// nonzero the kernel then moves 6 + 4m bytes instead of 8 + 4m from HBM and through shared memory: a stage holds 20 % more rows.
struct StageMeta { int nrows; int rpo; long long nzb; int next_step; int pad32; long long pad; };   // next_step: dynamic dealing
struct StageView {
    const unsigned short* idx; const float* c; const float* a; const long long* rp; const StageMeta* meta;
};
__device__ __forceinline__ StageView stage_view(unsigned char* base, int cap_nz, int cap_rows, int mm) {
    StageView v;
    v.idx = reinterpret_cast<const unsigned short*>(base);
    v.c = reinterpret_cast<const float*>(base + (size_t)cap_nz * 2);
    v.a = reinterpret_cast<const float*>(base + (size_t)cap_nz * 6);
    v.rp = reinterpret_cast<const long long*>(base + (size_t)cap_nz * (6 + 4 * mm));
    v.meta = reinterpret_cast<const StageMeta*>(v.rp + cap_rows);
    return v;
}

// The x output pointer, or a compile-time nullptr in the WX = false instantiations that dualip_solve's loop launches (it
// never writes x): the x-writing code drops out of the hot kernel, which measured 2-5 % faster on every config.
template <bool WX, class P>
__device__ __forceinline__ float* xout(const P& p) { return WX ? p.x : nullptr; }

template <bool WX, class P>
__device__ __forceinline__ void store_x(const P& p, long long pos, float val) {
    DUALIP_CHECK_X(pos);
    if (WX) p.x[pos] = val;
}

// The launch constants the out-of-line row routines use, as REGISTER values.  Those routines get the kernel parameters by
// reference, i.e. as a generic pointer, and the compiler re-loads a field from memory at every use rather than keep it in
// a register (ncu on the dense regime: 40 % of the stall samples were long-scoreboard waits on exactly those loads, on the
// critical path of every fixed-point push).  pin() copies the fields once and launders them through an empty asm so they
// cannot be rematerialised from memory.  Field names are GradParams', so the routines' code reads the same.
struct GradK {
    float scale_s_f, scale_obj_f, scale_sq_f, scale_cnt_f, inv_gamma_f, z, ub;
    double inv_gamma;
    unsigned long long* s_fix;
    float* x;
    int proj, m;
};
__device__ __forceinline__ GradK pin(const GradParams& p) {
    GradK k{p.scale_s_f, p.scale_obj_f, p.scale_sq_f, p.scale_cnt_f, p.inv_gamma_f, p.z, p.ub, p.inv_gamma, p.s_fix, p.x, p.proj, p.m};
    asm volatile("" : "+f"(k.scale_s_f), "+f"(k.scale_obj_f), "+f"(k.scale_sq_f), "+f"(k.scale_cnt_f), "+f"(k.inv_gamma_f), "+f"(k.z), "+f"(k.ub));
    asm volatile("" : "+d"(k.inv_gamma), "+l"(k.s_fix), "+l"(k.x), "+r"(k.proj), "+r"(k.m));
    return k;
}

// Shared state the row routines need.
struct ConsumerCtx {
    const float* lam_hi;                          // RN_f32(lambda) in shared memory: the filter's operand
    const float* lam_lo;                          // lambda - hi in shared memory (exact to 2^-48 relative), or nullptr:
    const double* lam_g;                          //   then the exact path reads the fp64 lambda from global memory (L2)
    unsigned* acc_lo; unsigned* acc_hi;           // shared-memory item accumulators (ACC_SMEM)
    bool hi_only;                                 // RN_f32(lambda) is exact enough for this launch's gamma (see k_grad_tma)
    double mu;                                    // dual of the global-count row (R21; 0 when the row is off): every nonzero's
                                                  //   t = c + a.lambda + mu, a uniform shift of the whole row
};
__device__ __forceinline__ ConsumerCtx pin(const ConsumerCtx& c) {
    ConsumerCtx k = c;
    int hi = k.hi_only ? 1 : 0;
    asm volatile("" : "+l"(k.lam_hi), "+l"(k.lam_lo), "+l"(k.lam_g), "+l"(k.acc_lo), "+l"(k.acc_hi), "+r"(hi), "+d"(k.mu));
    k.hi_only = hi != 0;
    return k;
}
// The out-of-line routines get the stage and lambda pointers as generic pointers; telling the compiler that they point
// to shared memory turns their loads back into LDS (short scoreboard) instead of generic LD (long scoreboard + an address
// space check per access).
__device__ __forceinline__ void assume_shared(const StageView& v, const ConsumerCtx& cx) {
    __builtin_assume(__isShared(v.idx)); __builtin_assume(__isShared(v.c)); __builtin_assume(__isShared(v.a));
    __builtin_assume(__isShared(v.rp)); __builtin_assume(__isShared(v.meta));
    __builtin_assume(__isShared(cx.lam_hi)); __builtin_assume(cx.lam_lo == nullptr || __isShared(cx.lam_lo));
    __builtin_assume(__isShared(cx.acc_lo)); __builtin_assume(__isShared(cx.acc_hi));
}
struct FixPair { long long obj, sq, cnt; };       // per-lane fixed-point partial scalars c'x, |x|^2, sum x (order-independent)

// v * 2^k as a 64-bit integer.  The scales are powers of two within fp32 range (dualip_api.cu clamps the exponent), so
// the product is exact and this equals to_fix(v, (double)scale) of dualip_kernels.cuh: one FMUL + one F2I.
__device__ __forceinline__ long long to_fix32(float v, float scale) { return __float2ll_rn(v * scale); }

// RED.ADD.64 on a pointer known to be global memory (a generic atomicAdd makes ptxas emit an address-space check, a
// shared-memory CAS loop and a predicate that the caller then waits on).
__device__ __forceinline__ void red_add_u64(unsigned long long* gptr, unsigned long long v) {
    asm volatile("red.global.add.u64 [%0], %1;" ::"l"(gptr), "l"(v));
}

// (a > b) ? x : y as one SETP + SEL, whatever the surrounding control flow looks like
__device__ __forceinline__ int sel_gt(float a, float b, int x, int y) {
    int r;
    asm("{\n\t.reg .pred p;\n\tsetp.gt.f32 p, %1, %2;\n\tselp.s32 %0, %3, %4, p;\n\t}" : "=r"(r) : "f"(a), "f"(b), "r"(x), "r"(y));
    return r;
}

// a4 + a5 for one nonzero with x != 0.
template <int M, bool ACC_SMEM, class P>
__device__ __forceinline__ void push(const P& p, const ConsumerCtx& cx, FixPair& fp, int mm, int j, float cc, const float* aa, float x) {
    DUALIP_CHECK_ITEM(j);
    fp.obj += to_fix32(cc * x, p.scale_obj_f);
    fp.sq += to_fix32(x * x, p.scale_sq_f);
    fp.cnt += to_fix32(x, p.scale_cnt_f);
    if (!ACC_SMEM && p.s_fix == nullptr) return;          // DUALIP_RED_CSC
#pragma unroll
    for (int f = 0; f < (M > 0 ? M : 4); ++f) {
        if (f < mm) {
            const long long fx = to_fix32(aa[f] * x, p.scale_s_f);
            if (ACC_SMEM) fix_add_smem(cx.acc_lo + j * mm + f, cx.acc_hi + j * mm + f, fx);
            else red_add_u64(p.s_fix + (long long)j * mm + f, (unsigned long long)fx);
        }
    }
}

// The exact path's dual operand is ALWAYS the two-word value hi + lo, hi = RN_f32(lambda), lo = RN_f32(lambda - hi) (exact to
// 2^-48 relative), whether the words come from shared memory or are split on the fly from the fp64 dual read through L2: the
// per-launch choice between the two (k_grad_tma) must not change a bit of the result.
__device__ __forceinline__ double two_word(double l) {
    const float h = (float)l;
    return (double)h + (double)(float)(l - (double)h);
}

// t = c + sum_f a_f * lambda[j,f] in fp64 for the staged nonzero q (w = -t).
template <int M>
__device__ __forceinline__ double exact_t(const StageView& v, const ConsumerCtx& cx, int mm, int q, int& j, float& cc, float* aa) {
    DUALIP_CHECK_POS(q);
    j = v.idx[q];
    DUALIP_CHECK_ITEM(j);
    cc = v.c[q];
    double t = (double)cc + cx.mu;
#pragma unroll
    for (int f = 0; f < (M > 0 ? M : 4); ++f) {
        aa[f] = 0.0f;
        if (f < mm) {
            aa[f] = v.a[q * mm + f];
            const double l = cx.hi_only ? (double)cx.lam_hi[j * mm + f]
                                        : (cx.lam_lo ? (double)cx.lam_hi[j * mm + f] + (double)cx.lam_lo[j * mm + f] : two_word(__ldg(cx.lam_g + j * mm + f)));
            t = fma((double)aa[f], l, t);
        }
    }
    return t;
}

// exact_t for K staged nonzeros at once: all index loads first, then all lambda gathers (an L2 round trip each when lambda's
// low word is not in shared memory), then the arithmetic -- K independent chains in flight instead of K serial ones.  Every
// position must be inside the stage (callers clamp the slots they do not own to a valid one and discard the result).  Same
// operations in the same order as exact_t, so the values are bit-identical to it.
template <int K, int M>
__device__ __forceinline__ void exact_t_batch(const StageView& v, const ConsumerCtx& cx, int mm, const int (&q)[K], double (&t)[K]) {
    constexpr int MA = M > 0 ? M : 4;
    int j[K];
    double l[K][MA];
#pragma unroll
    for (int k = 0; k < K; ++k) { DUALIP_CHECK_POS(q[k]); j[k] = v.idx[q[k]]; DUALIP_CHECK_ITEM(j[k]); }
    if (cx.hi_only) {
#pragma unroll
        for (int k = 0; k < K; ++k)
#pragma unroll
            for (int f = 0; f < MA; ++f) l[k][f] = f < mm ? (double)cx.lam_hi[j[k] * mm + f] : 0.0;
    } else if (cx.lam_lo) {
#pragma unroll
        for (int k = 0; k < K; ++k)
#pragma unroll
            for (int f = 0; f < MA; ++f) l[k][f] = f < mm ? (double)cx.lam_hi[j[k] * mm + f] + (double)cx.lam_lo[j[k] * mm + f] : 0.0;
    } else {
#pragma unroll
        for (int k = 0; k < K; ++k)
#pragma unroll
            for (int f = 0; f < MA; ++f) l[k][f] = f < mm ? two_word(__ldg(cx.lam_g + j[k] * mm + f)) : 0.0;
    }
#pragma unroll
    for (int k = 0; k < K; ++k) {
        double tt = (double)v.c[q[k]] + cx.mu;
#pragma unroll
        for (int f = 0; f < MA; ++f)
            if (f < mm) tt = fma((double)v.a[q[k] * mm + f], l[k][f], tt);
        t[k] = tt;
    }
}

// The filter's view of 4 nonzeros of one row: this lane's slots at q (M != 2: q..q+3; M = 2: the pairs (q, q+1) and
// (q+2G, q+2G+1), so that the 64-bit idx / c loads and the 128-bit a loads of a group are each one contiguous,
// conflict-free run -- four consecutive nonzeros per lane would put the a loads 32 bytes apart, a two-way bank conflict).
// w[e] = -(c + a . RN_f32(lambda)) in fp32 (one FFMA per family), -inf for slots outside [beg, beg+len); pe[e] = the
// slot's position in the stage.
template <int G, int M>
__device__ __forceinline__ void filter_load(const StageView& v, const float* __restrict__ s_hi32, int mm, int q, int beg, int len,
                                            float (&w)[4], int (&pe)[4]) {
    DUALIP_CHECK_POS(q); DUALIP_CHECK_POS(M == 2 ? q + 2 * G + 1 : q + 3);
    if (M == 2) {
        const int q2 = q + 2 * G;
        const unsigned wA = *reinterpret_cast<const unsigned*>(v.idx + q), wB = *reinterpret_cast<const unsigned*>(v.idx + q2);
        const int2 jA = make_int2((int)(wA & 0xffffu), (int)(wA >> 16)), jB = make_int2((int)(wB & 0xffffu), (int)(wB >> 16));
        const float2 cA = *reinterpret_cast<const float2*>(v.c + q), cB = *reinterpret_cast<const float2*>(v.c + q2);
        const float4 aA = *reinterpret_cast<const float4*>(v.a + 2 * q), aB = *reinterpret_cast<const float4*>(v.a + 2 * q2);
        const int jj[4] = {jA.x, jA.y, jB.x, jB.y};
        DUALIP_CHECK_ITEM(jj[0]); DUALIP_CHECK_ITEM(jj[1]); DUALIP_CHECK_ITEM(jj[2]); DUALIP_CHECK_ITEM(jj[3]);
        const float cv[4] = {cA.x, cA.y, cB.x, cB.y};
        const float ax[4] = {aA.x, aA.z, aB.x, aB.z}, ay[4] = {aA.y, aA.w, aB.y, aB.w};
        pe[0] = q; pe[1] = q + 1; pe[2] = q2; pe[3] = q2 + 1;
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const float2 l2 = *reinterpret_cast<const float2*>(s_hi32 + 2 * jj[e]);
            w[e] = -fmaf(ay[e], l2.y, fmaf(ax[e], l2.x, cv[e]));
        }
    } else {
        const uint2 w4 = *reinterpret_cast<const uint2*>(v.idx + q);
        const int4 j4 = make_int4((int)(w4.x & 0xffffu), (int)(w4.x >> 16), (int)(w4.y & 0xffffu), (int)(w4.y >> 16));
        const float4 c4 = *reinterpret_cast<const float4*>(v.c + q);
        const int jj[4] = {j4.x, j4.y, j4.z, j4.w};
        DUALIP_CHECK_ITEM(jj[0]); DUALIP_CHECK_ITEM(jj[1]); DUALIP_CHECK_ITEM(jj[2]); DUALIP_CHECK_ITEM(jj[3]);
        const float cv[4] = {c4.x, c4.y, c4.z, c4.w};
        if (M == 1) {
            const float4 a4 = *reinterpret_cast<const float4*>(v.a + q);
            const float aa4[4] = {a4.x, a4.y, a4.z, a4.w};
#pragma unroll
            for (int e = 0; e < 4; ++e) w[e] = -fmaf(aa4[e], s_hi32[jj[e]], cv[e]);
        } else {
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                float t = cv[e];
                for (int f = 0; f < mm; ++f) t = fmaf(v.a[(q + e) * mm + f], s_hi32[jj[e] * mm + f], t);
                w[e] = -t;
            }
        }
#pragma unroll
        for (int e = 0; e < 4; ++e) pe[e] = q + e;
    }
#pragma unroll
    for (int e = 0; e < 4; ++e) w[e] = (unsigned)(pe[e] - beg) < (unsigned)len ? w[e] : -CUDART_INF_F;
}

// One pass of the fp32 filter for one row: updates the running two largest w' (m1 >= m2) and the position of the largest.
// The four values are first reduced among themselves (depth 2), then merged into the running pair, so the dependent
// chain per pass is ~4 min/max deep instead of 8.  Equal maxima give m2 = m1 (no vertex).
template <int G, int M>
__device__ __forceinline__ void filter_pass(const StageView& v, const float* __restrict__ s_hi32, int mm, int q, int beg, int len,
                                            float& m1, float& m2, int& pb) {
    float w[4]; int pe[4];
    filter_load<G, M>(v, s_hi32, mm, q, beg, len, w, pe);
    const float hi01 = fmaxf(w[0], w[1]), lo01 = fminf(w[0], w[1]), hi23 = fmaxf(w[2], w[3]), lo23 = fminf(w[2], w[3]);
    const int p01 = sel_gt(w[1], w[0], pe[1], pe[0]), p23 = sel_gt(w[3], w[2], pe[3], pe[2]);
    const float top = fmaxf(hi01, hi23);
    const float sec = fmaxf(fminf(hi01, hi23), fmaxf(lo01, lo23));
    const int p4 = sel_gt(hi23, hi01, p23, p01);
    m2 = fmaxf(fmaxf(m2, sec), fminf(m1, top));
    pb = sel_gt(top, m1, p4, pb);
    m1 = fmaxf(m1, top);
}

// Slow path: one row, whole warp, any length; every pass re-reads the staged row.  Same arithmetic as long_row()
// in dualip_kernels.cuh (which documents the three box-cut steps).
template <int M, bool ACC_SMEM, bool GBOX, bool WX>
__device__ __noinline__ FixPair slow_row(const GradParams& p_in, const StageView v, const ConsumerCtx cx_in, int beg, int len, long long nzb) {
    const GradK p = pin(p_in);
    const ConsumerCtx cx = pin(cx_in);
    assume_shared(v, cx);
    FixPair fp{0ll, 0ll, 0ll};                              // returned in registers: the caller's accumulators never live in local memory
    const int lane = threadIdx.x & 31;
    const int mm = M > 0 ? M : p.m;
    const int end = beg + len;
    int j; float cc; float aa[M > 0 ? M : 4];
    const bool ineq = p.proj != PROJ_SIMPLEX_EQ;
    constexpr int KS = 4;                              // register-resident rows: up to 32*KS nonzeros
    if (!GBOX && len <= 32 * KS) {
        // Rows of up to 128 nonzeros (all but the tail of every config): the fp64 t = c + a.lambda is formed ONCE per
        // nonzero and kept in registers, and the Michelot iterations run on the shifted fp32 values there.  Same values,
        // same per-lane summation order (k ascending) and same reductions as the re-reading loops below, so the result is
        // bit-identical to them; it only drops the 5-8 re-evaluations per nonzero that dominate the fractional regime
        // (large gamma, binding constraints).
        double tk[KS];
        float wmax = -CUDART_INF_F;
        {
            int qk[KS];
#pragma unroll
            for (int k = 0; k < KS; ++k) qk[k] = min(beg + lane + 32 * k, end - 1);      // len >= 1 here
            exact_t_batch<KS, M>(v, cx, mm, qk, tk);
#pragma unroll
            for (int k = 0; k < KS; ++k) {
                if (beg + lane + 32 * k < end) wmax = fmaxf(wmax, (float)(-tk[k]));
                else tk[k] = CUDART_INF;
            }
        }
        const float m32 = group_max<32>(wmax);
        if (ineq && !(m32 > 0.0f)) {
            if (xout<WX>(p)) for (int q = beg + lane; q < end; q += 32) store_x<WX>(p, nzb + q, 0.0f);
            return fp;
        }
        const double md = (double)m32;
        const float mv = m32 * p.inv_gamma_f, z = p.z;
        float u[KS];
#pragma unroll
        for (int k = 0; k < KS; ++k) u[k] = (beg + lane + 32 * k < end) ? (float)(-tk[k] - md) * p.inv_gamma_f : -CUDART_INF_F;
        float theta = -z - (1.2e-7f * fabsf(mv) + 1e-6f);
        int n_prev = -1;
        for (;;) {
            float sm = 0.0f; int n = 0;
#pragma unroll
            for (int k = 0; k < KS; ++k) {
                const bool in = u[k] > theta;
                if (in) sm += u[k];
                if (32 * k < len) n += __popc(__ballot_sync(kFull, in));     // the count needs no shuffle tree
            }
            sm = group_sum<32>(sm);
            if (n == n_prev || n == 0) break;
            theta = fmaxf((sm - z) / (float)n, theta);
            n_prev = n;
        }
        const float tau = ineq ? fmaxf(theta, -mv) : theta;
#pragma unroll
        for (int k = 0; k < KS; ++k) {
            const int q = beg + lane + 32 * k;
            if (q < end) {
                const float x = fmaxf(u[k] - tau, 0.0f);
                if (xout<WX>(p)) store_x<WX>(p, nzb + q, x);
                if (x > 0.0f) {
                    j = v.idx[q]; cc = v.c[q];
#pragma unroll
                    for (int f = 0; f < (M > 0 ? M : 4); ++f) aa[f] = f < mm ? v.a[q * mm + f] : 0.0f;
                    push<M, ACC_SMEM>(p, cx, fp, mm, j, cc, aa, x);
                }
            }
        }
        return fp;
    }
    float wmax = -CUDART_INF_F;
    for (int q = beg + lane; q < end; q += 32) wmax = fmaxf(wmax, (float)(-exact_t<M>(v, cx, mm, q, j, cc, aa)));
    const float m32 = group_max<32>(wmax);
    if (ineq && !(m32 > 0.0f)) {
        if (xout<WX>(p)) for (int q = beg + lane; q < end; q += 32) store_x<WX>(p, nzb + q, 0.0f);
        return fp;
    }
    const double md = (double)m32;
    const float mv = m32 * p.inv_gamma_f, z = p.z;
    float tau;
    double ref = 0.0;
    if (!GBOX) {
        float theta = -z - (1.2e-7f * fabsf(mv) + 1e-6f);
        int n_prev = -1;
        for (;;) {
            float s = 0.0f; int n = 0;
            for (int q = beg + lane; q < end; q += 32) {
                const float u = (float)(-exact_t<M>(v, cx, mm, q, j, cc, aa) - md) * p.inv_gamma_f;
                if (u > theta) { s += u; ++n; }
            }
            s = group_sum<32>(s); n = group_sum_i<32>(n);
            if (n == n_prev || n == 0) break;
            theta = fmaxf((s - z) / (float)n, theta);
            n_prev = n;
        }
        tau = ineq ? fmaxf(theta, -mv) : theta;
    } else {
        const float ub = p.ub;
        const double ig = p.inv_gamma;
        float s0 = 0.0f;
        for (int q = beg + lane; q < end; q += 32) s0 += fminf(fmaxf((float)(-exact_t<M>(v, cx, mm, q, j, cc, aa) * ig), 0.0f), ub);
        s0 = group_sum<32>(s0);
        if (s0 <= z) { ref = 0.0; tau = 0.0f; }
        else {
            float lo = -mv, hi = 1.2e-7f * fabsf(mv) + 1e-6f;
            for (int it = 0; it < 36; ++it) {
                const float mid = 0.5f * (lo + hi);
                float s = 0.0f;
                for (int q = beg + lane; q < end; q += 32) {
                    const float u = (float)(-exact_t<M>(v, cx, mm, q, j, cc, aa) - md) * p.inv_gamma_f;
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
                for (int q = beg + lane; q < end; q += 32) {
                    const float u = (float)(-exact_t<M>(v, cx, mm, q, j, cc, aa) * ig - ref);
                    s += fminf(fmaxf(u - mid, 0.0f), ub);
                }
                s = group_sum<32>(s);
                if (s > z) dlo = mid; else dhi = mid;
            }
            const float mid = 0.5f * (dlo + dhi);
            float sF = 0.0f; int nF = 0, nU = 0;
            for (int q = beg + lane; q < end; q += 32) {
                const float u = (float)(-exact_t<M>(v, cx, mm, q, j, cc, aa) * ig - ref);
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
    const float cap = GBOX ? p.ub : CUDART_INF_F;
    for (int q = beg + lane; q < end; q += 32) {
        const double tq = exact_t<M>(v, cx, mm, q, j, cc, aa);
        const float u = GBOX ? (float)(-tq * p.inv_gamma - ref) : (float)(-tq - md) * p.inv_gamma_f;
        const float x = fminf(fmaxf(u - tau, 0.0f), cap);
        if (xout<WX>(p)) store_x<WX>(p, nzb + q, x);
        if (x > 0.0f) push<M, ACC_SMEM>(p, cx, fp, mm, j, cc, aa, x);
    }
    return fp;
}

// Two slow rows at once, one per half-warp, K nonzeros per lane (rows of at most 16*K nonzeros, simplex kinds): lanes 0-15
// take (b0, l0), lanes 16-31 take (b1, l1); l1 = 0 means "no partner".  The arithmetic is slow_row's (fp64 t once per
// nonzero, exact maximum, Michelot on the shifted fp32 values) with 16-lane reductions.
template <int K, int M, bool ACC_SMEM, bool WX>
__device__ __forceinline__ void half_warp_rows(const GradK& p, const StageView& v, const ConsumerCtx& cx, FixPair& fp, int b0, int l0, int b1,
                                               int l1, long long nzb) {
    const int lane = threadIdx.x & 31, h = lane & 15;
    const int mm = M > 0 ? M : p.m;
    const bool ineq = p.proj != PROJ_SIMPLEX_EQ;
    const float z = p.z;
    const unsigned hmask = lane < 16 ? 0x0000ffffu : 0xffff0000u;
    const int beg = lane < 16 ? b0 : b1, len = lane < 16 ? l0 : l1;
    int j; float cc; float aa[M > 0 ? M : 4];
    double tk[K];
    float wmax = -CUDART_INF_F;
    {
        int qk[K];
#pragma unroll
        for (int k = 0; k < K; ++k) qk[k] = beg + min(h + 16 * k, max(len - 1, 0));       // slots past the row: a valid position, discarded
        exact_t_batch<K, M>(v, cx, mm, qk, tk);
#pragma unroll
        for (int k = 0; k < K; ++k) {
            if (h + 16 * k < len) wmax = fmaxf(wmax, (float)(-tk[k]));
            else tk[k] = CUDART_INF;
        }
    }
    const float m16 = group_max<16>(wmax);
    const bool alive = len > 0 && (!ineq || m16 > 0.0f);
    const double md = (double)m16;
    const float mv = m16 * p.inv_gamma_f;
    float u[K];
#pragma unroll
    for (int k = 0; k < K; ++k) u[k] = (alive && h + 16 * k < len) ? (float)(-tk[k] - md) * p.inv_gamma_f : -CUDART_INF_F;
    float theta = -z - (1.2e-7f * fabsf(mv) + 1e-6f);
    int n_prev = -1;
    bool stop = !alive;
    // (The sums as 32-bit fixed-point integers added across the half-warp by redux.sync -- two instructions instead of a shuffle
    // tree and a ballot per register -- were built and measured: cfg3-tight steady 6.8 -> 9.4 ms; REDUX under a sub-warp mask is
    // far slower than four shuffles on sm_100a.)
    for (;;) {
        float sm = 0.0f; int n = 0;
#pragma unroll
        for (int k = 0; k < K; ++k) {
            const bool in = u[k] > theta;
            if (in) sm += u[k];
            n += __popc(__ballot_sync(kFull, in) & hmask);
        }
        sm = group_sum<16>(sm);
        if (!stop) {
            if (n == n_prev || n == 0) stop = true;
            else { theta = fmaxf((sm - z) / (float)n, theta); n_prev = n; }
        }
        if (__all_sync(kFull, stop)) break;
    }
    const float tau = ineq ? fmaxf(theta, -mv) : theta;
#pragma unroll
    for (int k = 0; k < K; ++k) {
        if (h + 16 * k < len) {
            const int q = beg + h + 16 * k;
            const float x = fmaxf(u[k] - tau, 0.0f);
            if (xout<WX>(p)) store_x<WX>(p, nzb + q, x);
            if (x > 0.0f) {
                j = v.idx[q]; cc = v.c[q];
#pragma unroll
                for (int f = 0; f < (M > 0 ? M : 4); ++f) aa[f] = f < mm ? v.a[q * mm + f] : 0.0f;
                push<M, ACC_SMEM>(p, cx, fp, mm, j, cc, aa, x);
            }
        }
    }
}

// All slow rows of one row-step.  `mask`: lanes whose (fbeg, flen) describe a slow row.  Rows of at most 32 / at most 64
// nonzeros (simplex kinds) run two at a time on half-warps with 2 / 4 nonzeros per lane -- always in the layout of their
// own length class, partner or not, so a row's arithmetic does not depend on what else is in its step; everything else
// goes to slow_row one row at a time.
template <int M, bool ACC_SMEM, bool GBOX, bool WX>
__device__ __noinline__ FixPair slow_rows_all(const GradParams& p_in, const StageView v, const ConsumerCtx cx_in, int fbeg, int flen, unsigned mask,
                                              long long nzb) {
    const GradK p = pin(p_in);
    const ConsumerCtx cx = pin(cx_in);
    assume_shared(v, cx);
    FixPair fp{0ll, 0ll, 0ll};
    while (mask) {
        const int s0 = __ffs(mask) - 1;
        mask &= mask - 1;
        const int b0 = __shfl_sync(kFull, fbeg, s0), l0 = __shfl_sync(kFull, flen, s0);
        if (GBOX || l0 > 64) {
            const FixPair sp = slow_row<M, ACC_SMEM, GBOX, WX>(p_in, v, cx_in, b0, l0, nzb);
            fp.obj += sp.obj; fp.sq += sp.sq; fp.cnt += sp.cnt;
            continue;
        }
        const bool small = l0 <= 32;
        int b1 = 0, l1 = 0;                                  // partner: the next slow row of the same length class
        for (unsigned m2 = mask; m2; m2 &= m2 - 1) {
            const int s1 = __ffs(m2) - 1;
            const int lc = __shfl_sync(kFull, flen, s1);
            if (lc <= 64 && (lc <= 32) == small) { b1 = __shfl_sync(kFull, fbeg, s1); l1 = lc; mask &= ~(1u << s1); break; }
        }
        if (small) half_warp_rows<2, M, ACC_SMEM, WX>(p, v, cx, fp, b0, l0, b1, l1, nzb);
        else half_warp_rows<4, M, ACC_SMEM, WX>(p, v, cx, fp, b0, l0, b1, l1, nzb);
    }
    return fp;
}

template <int G, int M, bool ACC_SMEM, bool GBOX, bool WX, int NWC>
__global__ void __launch_bounds__(32 * (NWC + 1), 1) k_grad_tma(const __grid_constant__ TmaParams tp) {
    extern __shared__ __align__(128) unsigned char smem_tma[];
    const GradParams& p = tp.g;
    constexpr int MA = M > 0 ? M : 4;
    constexpr int NT = 32 * (NWC + 1);
    const int mm = M > 0 ? M : p.m;
    const int JM = p.J * mm;
    // layout: [full[8], empty[8] mbarriers: 128 B][words: 128 B][candidate lists: 256 B per consumer warp][lam_hi JM*4]
    //         [acc 2*JM*4 (ACC_SMEM)][lam_lo JM*4 (decided per launch, below)][stages]
    unsigned long long* bars = reinterpret_cast<unsigned long long*>(smem_tma);
    unsigned* s_words = reinterpret_cast<unsigned*>(smem_tma + 128);      // [0] = max |lambda_hi| as float bits
    int* cand_list = reinterpret_cast<int*>(smem_tma + 256);              // 64 positions per consumer warp (candidate path B)
    float* s_hi32 = reinterpret_cast<float*>(smem_tma + kTmaHeaderBytes);
    unsigned* a_lo = reinterpret_cast<unsigned*>(s_hi32 + JM);
    unsigned* a_hi = a_lo + JM;
    float* s_lo32 = s_hi32 + (ACC_SMEM ? 3 : 1) * JM;

#ifdef DUALIP_CHECKED
    if (threadIdx.x == 0) {
        g_chk_word = tp.check_word; g_chk_cap_nz = tp.cap_nz; g_chk_J = p.J; g_chk_cap_rows = tp.cap_rows; g_chk_nnz = p.nnz;
        if ((size_t)tp.stage_bytes < (size_t)tp.cap_nz * (6 + 4 * mm) + (size_t)tp.cap_rows * 8 + sizeof(StageMeta)) atomicOr(tp.check_word, 1u << CHK_STAGE_BYTES);
    }
    __syncthreads();
#endif
    if (threadIdx.x == 0) s_words[0] = 0u;
    __syncthreads();
    {
        float lmax = 0.0f;
        for (int q = threadIdx.x; q < JM; q += NT) {
            const float h = (float)p.lambda[q];
            s_hi32[q] = h;
            lmax = fmaxf(lmax, fabsf(h));
        }
        // max |lambda|: the filter's rounding bound (M > 1) and the hi_only test below need it
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) lmax = fmaxf(lmax, __shfl_xor_sync(kFull, lmax, o));
        if ((threadIdx.x & 31) == 0) atomicMax(&s_words[0], __float_as_uint(lmax));
    }
    if (ACC_SMEM) for (int q = threadIdx.x; q < 2 * JM; q += NT) a_lo[q] = 0u;
    __syncthreads();

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    // The exact path needs lambda beyond fp32 only when 1/gamma amplifies its rounding into x: dropping the low word moves
    // w by at most m max|a| max|lambda| 2^-25, v = w/gamma by that over gamma, and any x by at most twice that.  When the
    // bound is below 1e-7 (two orders inside the 1e-5 bar, the size of the fp32 steps that follow anyway) the exact path
    // reads RN_f32(lambda) from shared memory instead of the fp64 dual -- which is what makes rows in the
    // fractional regime (large gamma, or lambda = 0) cost one shared-memory latency instead of one L2 round trip each.
    const bool hi_only = (float)mm * p.max_abs_a * __uint_as_float(s_words[0]) * p.inv_gamma_f * 5.9604645e-8f <= 1e-7f;
    // When the test fails, the exact path needs lambda's low word as well.  THIS launch stages it in shared memory, next to
    // the high word, if that still leaves two pipeline stages (the tiles were sized at create without it: a launch that needs
    // the low word is in the fractional regime, far from the HBM roof, where a shallower pipeline costs nothing; a launch
    // that does not need it keeps every stage).  Otherwise the exact path reads the fp64 dual through L2.  The decision
    // depends on lambda and gamma only, so every CTA takes the same one.  lo_policy: 0 = as described, 1 = never, 2 = always.
    int nstages = tp.stages;
    size_t off = kTmaHeaderBytes + (size_t)JM * 4 * (ACC_SMEM ? 3 : 1);
    bool lo_smem = false;
    if (tp.lo_policy == 2 || (tp.lo_policy == 0 && !hi_only)) {
        const size_t off_lo = (off + (size_t)JM * 4 + 127) & ~(size_t)127;
        const long long fit = ((long long)tp.smem_total - (long long)off_lo) / tp.stage_bytes;
        if (fit >= 2) { lo_smem = true; off = off_lo; nstages = fit < nstages ? (int)fit : nstages; }
    }
    off = (off + 127) & ~(size_t)127;
    unsigned char* stage0 = smem_tma + off;
    if (lo_smem) {
        for (int q = threadIdx.x; q < JM; q += NT) {
            const double l = p.lambda[q];
            s_lo32[q] = (float)(l - (double)(float)l);
        }
    }
    {   // consumers read whole 16-byte vectors around a row, beyond the part of the stage the tile's copies wrote: every word of
        // the INDEX array of a stage must always hold a valid item index (c and a may hold anything: those slots are masked)
        for (int s = 0; s < nstages; ++s) {
            uint4* sp = reinterpret_cast<uint4*>(stage0 + (size_t)s * tp.stage_bytes);
            for (int q = threadIdx.x; q < tp.cap_nz / 8; q += NT) sp[q] = make_uint4(0u, 0u, 0u, 0u);
        }
        fence_proxy_async();                                             // generic-proxy zeros before the first bulk copy
    }
    if (threadIdx.x == 0) {
        for (int s = 0; s < nstages; ++s) { mbar_init(&bars[s], 1); mbar_init(&bars[kTmaStagesMax + s], NWC); }
        fence_mbar_init();
        fence_proxy_async();
        if (blockIdx.x == 0 && tp.lo_flag) *tp.lo_flag = lo_smem ? 1 : 0;
    }
    __syncthreads();

    const bool dyn = tp.dyn_steps != 0;
    const double mu = p.count_on ? p.lambda[JM] : 0.0;
    const ConsumerCtx cx{s_hi32, lo_smem ? s_lo32 : nullptr, p.lambda, a_lo, a_hi, hi_only, mu};
    FixPair fp{0ll, 0ll, 0ll};

    if (warp == 0) {
        // ================= producer =================
        if (lane == 0) {
            long long t = blockIdx.x;
            TileEntry cur{0, 0}, nxt{0, 0};
            if (t < tp.ntiles) { cur = tp.tiles[t]; nxt = tp.tiles[t + 1]; }
            int s = 0;
            unsigned ph = 0;
            for (; t < tp.ntiles; t += gridDim.x) {
                const long long tn = t + gridDim.x;                                  // prefetch the next table entries
                TileEntry ncur{0, 0}, nnxt{0, 0};
                if (tn < tp.ntiles) { ncur = tp.tiles[tn]; nnxt = tp.tiles[tn + 1]; }
                mbar_wait(&bars[kTmaStagesMax + s], ph ^ 1u);                        // stage free?
                unsigned char* sb = stage0 + (size_t)s * tp.stage_bytes;
                unsigned short* d_idx = reinterpret_cast<unsigned short*>(sb);
                float* d_c = reinterpret_cast<float*>(sb + (size_t)tp.cap_nz * 2);
                float* d_a = reinterpret_cast<float*>(sb + (size_t)tp.cap_nz * 6);
                long long* d_rp = reinterpret_cast<long long*>(sb + (size_t)tp.cap_nz * (6 + 4 * mm));
                StageMeta* d_meta = reinterpret_cast<StageMeta*>(d_rp + tp.cap_rows);
                const long long r0 = cur.row0, p0 = cur.nz0;
                long long r1 = nxt.row0, p1 = nxt.nz0;
                if (tp.row_cap > 0 && r1 - r0 == 1 && p1 - p0 > tp.row_cap) { r1 = r0; p1 = p0; }   // a long row's own tile: nothing to stage
                const long long p0a = p0 & ~7ll;                                      // 8 nonzeros = 16 bytes of 16-bit indices
                long long p1a = (p1 + 7) & ~7ll;
                if (p1a > tp.nnz8) p1a = tp.nnz8 > p0a ? tp.nnz8 : p0a;              // never read past the arrays
                const long long r0a = r0 & ~1ll;
                long long r1a = (r1 + 2) & ~1ll;                                       // rows r0a .. r1 inclusive, even count
                if (r1a > tp.rows2) r1a = tp.rows2 > r0a ? tp.rows2 : r0a;
                d_meta->nrows = (int)(r1 - r0); d_meta->rpo = (int)(r0 - r0a); d_meta->nzb = p0a; d_meta->next_step = 0;
                // tails that are not a whole 16-byte chunk (only at the very end of the arrays): plain copies
                for (long long q = p1a > p0a ? p1a : p0a; q < p1; ++q) {
                    d_idx[q - p0a] = tp.idx16[q]; d_c[q - p0a] = p.c[q];
                    for (int f = 0; f < mm; ++f) d_a[(q - p0a) * mm + f] = p.a[q * mm + f];
                }
                for (long long r = r1a > r0a ? r1a : r0a; r <= r1; ++r) d_rp[r - r0a] = p.row_ptr[r];
                const unsigned nz = (unsigned)(p1a > p0a ? p1a - p0a : 0), nr = (unsigned)(r1a > r0a ? r1a - r0a : 0);
                mbar_expect_tx(&bars[s], nz * (6u + 4u * (unsigned)mm) + nr * 8u);     // release: meta/claim/tail stores
                if (nz) {
                    bulk_g2s(d_idx, tp.idx16 + p0a, nz * 2u, &bars[s]);
                    bulk_g2s(d_c, p.c + p0a, nz * 4u, &bars[s]);
                    bulk_g2s(d_a, p.a + p0a * mm, nz * 4u * (unsigned)mm, &bars[s]);
                }
                if (nr) bulk_g2s(d_rp, p.row_ptr + r0a, nr * 8u, &bars[s]);
                cur = ncur; nxt = nnxt;
                if (++s == nstages) { s = 0; ph ^= 1u; }
            }
        }
    } else {
        // ================= consumers =================
        constexpr int GPW = 32 / G;                  // row groups per warp
        constexpr int RPG = G >= 2 ? 2 : 1;          // rows a group takes per step (finalised together)
        constexpr int RPW = GPW * RPG;               // rows per warp step
        constexpr int HG = G >= 2 ? G / 2 : 1;
        const int gl = lane & (G - 1), grp = lane / G;
        const bool ineq = p.proj != PROJ_SIMPLEX_EQ;
        const float z = p.z;
        const float gz = (float)((double)p.z / p.inv_gamma);            // z * gamma: the vertex gap in w units
        const bool upper = RPG == 2 && (gl & HG) != 0;                   // this lane ends up holding the group's row 1
        const bool fin = RPG == 2 ? (gl & (HG - 1)) == 0 : true;        // lanes 0 and G/2 of a group finalise rows 0 and 1
        // rounding bound of the filter (see below): the part that does not depend on the row
        const float bnd0 = M == 1 ? p.max_abs_c : p.max_abs_c + (float)mm * p.max_abs_a * __uint_as_float(s_words[0]);
        const float gz_sat = gz * (1.0f + 4.8e-7f);                      // w_max above this (plus tol): v_max >= z for sure
        // The global-count dual mu shifts every w of every row by the same amount, so the filter leaves it out (the top two,
        // their gap and the candidate set do not see it); only the two tests against absolute levels (row dead: w_max < 0,
        // row saturated: w_max >= z gamma) take it, with its fp32 rounding added to their tolerance.
        const float mu_f = (float)mu, mu_tol = 2.4e-7f * fabsf(mu_f);
        int s = 0;
        unsigned ph = 0;
        int step_off = 0;                                                // (steps of all earlier tiles) mod NWC
        for (long long t = blockIdx.x; t < tp.ntiles; t += gridDim.x) {
            mbar_wait(&bars[s], ph);
            const StageView v = stage_view(stage0 + s * tp.stage_bytes, tp.cap_nz, tp.cap_rows, mm);
            const int nrows = v.meta->nrows;
            const int nsteps = (nrows + RPW - 1) / RPW;
            // Row-steps are dealt round-robin over the CTA's whole step sequence (not per tile): step st of this tile is
            // number step_off + st of the sequence and belongs to warp (step_off + st) mod NWC.  Every warp sees every
            // tile's nsteps, so each keeps the running offset itself: no shared counter, no atomics.
            // That is the STATIC deal: right when every step costs the same (the vertex regime).  When most rows take the
            // candidate / slow paths a step's cost varies several-fold, a warp that draws a heavy step holds its stage, and with
            // only ~1 step per warp resident the others idle at the next "full" barrier (ncu: 16 % of the stall samples on cfg5
            // at gamma = 0.1).  The DYNAMIC deal -- a warp claims the tile's next step from a counter in the stage's meta words
            // (one shared-memory atomic by lane 0 + a broadcast per claim) -- lets whoever is free take it.  dyn is per launch.
            int st0 = (warp - 1) - step_off;
            if (st0 < 0) st0 += NWC;
            step_off = (step_off + nsteps) % NWC;
            int* const next_step = const_cast<int*>(&v.meta->next_step);
            auto claim = [&]() { int c = 0; if (lane == 0) c = atomicAdd(next_step, 1); return __shfl_sync(kFull, c, 0); };
            for (int st = dyn ? claim() : st0; st < nsteps; st = dyn ? claim() : st + NWC) {
                const int rpo = v.meta->rpo;
                const int nzb32 = (int)v.meta->nzb;                       // low word is enough for local offsets
                int rbeg[RPG], rlen[RPG];
                float rm1[RPG], rm2[RPG];
                int rpos[RPG];
#pragma unroll
                for (int r = 0; r < RPG; ++r) {
                    const int lr = st * RPW + r * GPW + grp;
                    int beg = 0, len = 0;
                    if (lr < nrows) {
                        const int b = (int)v.rp[rpo + lr], e = (int)v.rp[rpo + lr + 1];   // differences fit in 32 bits
                        beg = b - nzb32; len = e - b;
                        DUALIP_CHECK(rpo + lr + 1 < tp.cap_rows, CHK_ROWS);
                        DUALIP_CHECK(beg >= 0 && len >= 0 && (beg & ~3) + ((len + (beg & 3) + 4 * G - 1) / (4 * G)) * (4 * G) <= tp.cap_nz, CHK_ROW_EXTENT);
                    }
                    rbeg[r] = beg; rlen[r] = len;
                    rm1[r] = -CUDART_INF_F; rm2[r] = -CUDART_INF_F; rpos[r] = 0;
                }
                if (!GBOX) {
                    // ---- fp32 filter: the two largest w' = -(c + a.lambda_hi) of each row and where the largest sits.
                    // A lane takes 4 nonzeros of a row per pass (filter_pass) starting from the 16-byte aligned position at
                    // or below the row start; the G lanes of a group cover 4G consecutive nonzeros.  Slots outside
                    // [beg, beg+len) hold other rows' data (or zeros): their lambda index is in range, their value is
                    // masked to -inf.
                    constexpr int LS = M == 2 ? 2 : 4;                        // first-slot spacing of the lanes
                    int q[RPG], qe[RPG];
#pragma unroll
                    for (int r = 0; r < RPG; ++r) { q[r] = (rbeg[r] & ~3) + LS * gl; qe[r] = rbeg[r] + rlen[r]; }
#pragma unroll
                    for (int r = 0; r < RPG; ++r)
                        for (; q[r] < qe[r]; q[r] += 4 * G)
                            filter_pass<G, M>(v, s_hi32, mm, q[r], rbeg[r], rlen[r], rm1[r], rm2[r], rpos[r]);
                }
                unsigned slow_mask;
                int fbeg = rbeg[0], flen = rlen[0];
                if (RPG == 2 && upper) { fbeg = rbeg[RPG - 1]; flen = rlen[RPG - 1]; }
                const bool active = fin && flen > 0;
                if (GBOX) {
                    slow_mask = __ballot_sync(kFull, active);
                } else {
                    // group reduction of (m1, m2, argmax position, bound).  With two rows per group the first exchange
                    // is a transposition: the lower half of the group keeps row 0 and hands over its part of row 1,
                    // the upper half the reverse; the remaining levels then run on both rows at once.  Equal maxima in
                    // two lanes give m2 = m1 (no vertex).
                    float m1 = rm1[0], m2 = rm2[0];
                    int fpos = rpos[0];
                    if (RPG == 2) {
                        float g1 = rm1[RPG - 1], g2 = rm2[RPG - 1];
                        int gp = rpos[RPG - 1];
                        if (upper) {
                            float tf; int ti;
                            tf = m1; m1 = g1; g1 = tf; tf = m2; m2 = g2; g2 = tf; ti = fpos; fpos = gp; gp = ti;
                        }
                        const float o1 = __shfl_xor_sync(kFull, g1, HG), o2 = __shfl_xor_sync(kFull, g2, HG);
                        const int op = __shfl_xor_sync(kFull, gp, HG);
                        const bool gt = o1 > m1;
                        m2 = fmaxf(fminf(m1, o1), fmaxf(m2, o2));
                        fpos = gt ? op : fpos;
                        m1 = fmaxf(m1, o1);
                    }
#pragma unroll
                    for (int o = HG / 2; o > 0; o >>= 1) {
                        const float o1 = __shfl_xor_sync(kFull, m1, o), o2 = __shfl_xor_sync(kFull, m2, o);
                        const int op = __shfl_xor_sync(kFull, fpos, o);
                        const bool gt = o1 > m1;
                        m2 = fmaxf(fminf(m1, o1), fmaxf(m2, o2));
                        fpos = gt ? op : fpos;
                        m1 = fmaxf(m1, o1);
                    }
                    // rounding bound of the filter.  Every FFMA rounds once, relative to its own result, and lambda is
                    // truncated to fp32 (2^-24 relative to |a lam|).  M = 1: error <= 2^-24 (|w'| + |a lam|) and
                    // |a lam| <= |w'| + |c|, so B = 2|w'| + max|c| covers the top two; a value far below them has a larger
                    // error but is further away by more than that.  M > 1: every partial sum is at most
                    // B = max|c| + m max|a| max|lam|, and there are m roundings plus the truncations.  2.4e-7 = 2^-22 gives
                    // slack.  The maxima are global (a0 / this launch's lambda): a looser bound only sends more rows to
                    // the exact path.
                    const float mag = fmaxf(fabsf(m1), m2 > -CUDART_INF_F ? fabsf(m2) : 0.0f);
                    const float B = M == 1 ? 2.0f * mag + bnd0 : bnd0;
                    const float tol = 2.4e-7f * (float)(mm + 1) * B + 1e-30f;
                    const bool vertex = (m1 - m2) > gz + 2.0f * tol;
                    const float m1s = m1 - mu_f, tol_s = tol + mu_tol;
                    const bool dead = ineq && m1s < -tol_s;
                    const bool fast = vertex || dead;
                    float xo = 0.0f;
                    if (active && vertex && !dead) {
                        // x = clamp(v_max, 0, z) on the arg-max nonzero (z for the equality simplex).  When v_max >= z is
                        // certain in fp32 the answer is z itself; otherwise that one nonzero is redone in fp64.
                        int j; float cc; float aa[MA];
                        if (!ineq || m1s - tol_s > gz_sat) {
                            j = v.idx[fpos]; cc = v.c[fpos];
#pragma unroll
                            for (int f = 0; f < MA; ++f) aa[f] = f < mm ? v.a[fpos * mm + f] : 0.0f;
                            xo = z;
                        } else {
                            const double tq = exact_t<M>(v, cx, mm, fpos, j, cc, aa);
                            xo = fmaxf((float)fmin((double)z, -tq * p.inv_gamma), 0.0f);
                        }
                        if (xo > 0.0f) push<M, ACC_SMEM>(p, cx, fp, mm, j, cc, aa, xo);
                    }
                    if (xout<WX>(p)) {
                        const long long nzb = v.meta->nzb;
#pragma unroll
                        for (int r = 0; r < RPG; ++r) {
                            const int src = (lane & ~(G - 1)) + r * HG;
                            const bool fr = __shfl_sync(kFull, (int)(active && fast), src) != 0;
                            const float xr = __shfl_sync(kFull, xo, src);
                            const int pr = __shfl_sync(kFull, fpos, src);
                            if (fr) for (int e = gl; e < rlen[r]; e += G) store_x<WX>(p, nzb + rbeg[r] + e, (rbeg[r] + e == pr) ? xr : 0.0f);
                        }
                    }
                    // ---- candidate path: rows that are neither a vertex nor dead.  Only nonzeros with w > w_max - z gamma
                    // can be in the support (theta >= v_max - z for both simplex forms): the CANDIDATES, typically 2-4 of
                    // a row.  They are brought to one per lane (two per lane when a row has more candidates than its group
                    // has lanes), redone in fp64 and projected in registers by the group; the rest of the row is zero.
                    //   (A) the filter already knows each lane's two largest w': if no lane's SECOND value passes the
                    //       candidate threshold, every lane holds at most one candidate, at a known position;
                    //   (B) otherwise the group scans the staged row once more and compacts the candidates' positions
                    //       through a per-warp list in shared memory (ballot + prefix popc), up to 2G of them;
                    //   rows with more than 2G candidates (gamma of the order of the spread of w) go to slow_rows_all.
                    bool handled = false;
                    const bool want = active && !fast;
                    if (__any_sync(kFull, want)) {
                        const unsigned gmask = G == 32 ? kFull : (((1u << G) - 1u) << (lane & ~(G - 1)));
                        const unsigned lt_mask = (1u << lane) - 1u;
                        const float thr_own = m1 - gz_sat - 2.0f * tol;
                        int* const clist = cand_list + (warp - 1) * 64 + grp * (2 * G);
#pragma unroll
                        for (int r = 0; r < RPG; ++r) {
                            const int src = (lane & ~(G - 1)) + r * HG;
                            const bool rw = __shfl_sync(kFull, (int)want, src) != 0;
                            const float thr = __shfl_sync(kFull, thr_own, src);
                            const unsigned okb = __ballot_sync(kFull, !(rm2[r] > thr));
                            const bool rowA = rw && (okb & gmask) == gmask;
                            // (B) holds up to 2G candidates.  The filter already knows a lower bound on their number (lanes whose
                            // largest / second largest value is one); when that alone reaches 2G on a row longer than 2G -- a
                            // dense row: gamma of the order of the spread of w -- the re-scan would only find out that the row
                            // does not fit, so it goes to the slow path directly.  The test reads the row's own data only.
                            const unsigned c1b = __ballot_sync(kFull, rm1[r] > thr);
                            const bool dense = __popc(~okb & gmask) + __popc(c1b & gmask) >= 2 * G && rlen[r] > 2 * G;
                            const bool needB = rw && !rowA && !dense;
                            bool row_ok = rowA;
                            int cp0 = (rowA && rm1[r] > thr) ? rpos[r] : -1, cp1 = -1;
                            if (__any_sync(kFull, needB)) {
                                constexpr int LS = M == 2 ? 2 : 4;
                                int qq = (rbeg[r] & ~3) + LS * gl;
                                const int qe = rbeg[r] + rlen[r];
                                int ncand = 0;                                   // candidates of this group's row so far
                                while (__any_sync(kFull, needB && qq < qe)) {
                                    float w[4]; int pe[4];
                                    if (needB && qq < qe) filter_load<G, M>(v, s_hi32, mm, qq, rbeg[r], rlen[r], w, pe);
                                    else {
#pragma unroll
                                        for (int e = 0; e < 4; ++e) { w[e] = -CUDART_INF_F; pe[e] = 0; }
                                    }
                                    // one ballot + prefix popc per slot.  (A per-lane count + an inclusive prefix sum over the
                                    // group's lanes -- a third of the instructions -- was measured SLOWER: cfg5 at gamma = 0.1
                                    // 4.36 -> 4.69 ms; the shuffle chain is serial, the four ballots are independent.)
#pragma unroll
                                    for (int e = 0; e < 4; ++e) {
                                        const bool isc = w[e] > thr;
                                        const unsigned bal = __ballot_sync(kFull, isc) & gmask;
                                        const int k = ncand + __popc(bal & lt_mask);
                                        DUALIP_CHECK(!(isc && k < 2 * G) || (clist + k) - cand_list < 64 * NWC, CHK_LIST);
                                        if (isc && k < 2 * G) clist[k] = pe[e];
                                        ncand += __popc(bal);
                                    }
                                    qq += 4 * G;
                                }
                                __syncwarp();
                                const bool rowB = needB && ncand <= 2 * G;
                                if (rowB) { cp0 = gl < ncand ? clist[gl] : -1; cp1 = gl + G < ncand ? clist[gl + G] : -1; }
                                row_ok = rowA || rowB;
                                __syncwarp();                                    // the list is reused by the group's next row
                            }
                            if (!__any_sync(kFull, row_ok)) continue;
                            const bool two = __any_sync(kFull, cp1 >= 0);        // warp-uniform: a second candidate per lane is rare
                            int j = 0; float cc = 0.0f; float aa[MA];
                            double wq0 = -CUDART_INF, wq1 = -CUDART_INF;
                            if (cp0 >= 0) wq0 = -exact_t<M>(v, cx, mm, cp0, j, cc, aa);
                            if (two && cp1 >= 0) wq1 = -exact_t<M>(v, cx, mm, cp1, j, cc, aa);
                            const float m32 = group_max<G>(fmaxf((float)wq0, (float)wq1));   // the row maximum is always a candidate
                            const bool alive = row_ok && (!ineq || m32 > 0.0f);
                            const float mv = m32 * p.inv_gamma_f;
                            const float u0 = cp0 >= 0 ? (float)(wq0 - (double)m32) * p.inv_gamma_f : -CUDART_INF_F;
                            const float u1 = (two && cp1 >= 0) ? (float)(wq1 - (double)m32) * p.inv_gamma_f : -CUDART_INF_F;
                            float theta = -z - (1.2e-7f * fabsf(mv) + 1e-6f);
                            // Michelot's fixed point on the candidates.  (A closed form -- every lane ranking its value among the
                            // group's with G - 1 exchanges, Duchi's criterion evaluated per lane -- was built and measured: equal at
                            // G = 4, slower from G = 8 up, where 3-4 iterations of a log G reduction cost less than G - 1 exchanges.)
                            int n_prev = -1;
                            for (;;) {
                                const bool in0 = alive && u0 > theta, in1 = alive && u1 > theta;
                                const float sg = group_sum<G>((in0 ? u0 : 0.0f) + (in1 ? u1 : 0.0f));
                                int n = __popc(__ballot_sync(kFull, in0) & gmask);
                                if (two) n += __popc(__ballot_sync(kFull, in1) & gmask);
                                const bool stop = n == n_prev || n == 0;
                                if (!stop) { theta = fmaxf((sg - z) / (float)n, theta); n_prev = n; }
                                if (__all_sync(kFull, stop)) break;
                            }
                            const float tau = ineq ? fmaxf(theta, -mv) : theta;
                            const float xq0 = alive ? fmaxf(u0 - tau, 0.0f) : 0.0f;
                            const float xq1 = alive ? fmaxf(u1 - tau, 0.0f) : 0.0f;
                            if (xq0 > 0.0f) {
                                j = v.idx[cp0]; cc = v.c[cp0];
#pragma unroll
                                for (int f = 0; f < MA; ++f) aa[f] = f < mm ? v.a[cp0 * mm + f] : 0.0f;
                                push<M, ACC_SMEM>(p, cx, fp, mm, j, cc, aa, xq0);
                            }
                            if (two && xq1 > 0.0f) {
                                j = v.idx[cp1]; cc = v.c[cp1];
#pragma unroll
                                for (int f = 0; f < MA; ++f) aa[f] = f < mm ? v.a[cp1 * mm + f] : 0.0f;
                                push<M, ACC_SMEM>(p, cx, fp, mm, j, cc, aa, xq1);
                            }
                            if (xout<WX>(p)) {
                                const long long nzb = v.meta->nzb;
                                if (row_ok) for (int e = gl; e < rlen[r]; e += G) store_x<WX>(p, nzb + rbeg[r] + e, 0.0f);
                                __syncwarp();
                                if (cp0 >= 0) store_x<WX>(p, nzb + cp0, xq0);
                                if (cp1 >= 0) store_x<WX>(p, nzb + cp1, xq1);
                            }
                            if (lane == src && row_ok) handled = true;
                        }
                    }
                    slow_mask = __ballot_sync(kFull, want && !handled);
                }
                if (slow_mask) {
                    const FixPair sp = slow_rows_all<M, ACC_SMEM, GBOX, WX>(p, v, cx, fbeg, flen, slow_mask, v.meta->nzb);
                    fp.obj += sp.obj; fp.sq += sp.sq; fp.cnt += sp.cnt;
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&bars[kTmaStagesMax + s]);           // this warp is done with the stage
            if (++s == nstages) { s = 0; ph ^= 1u; }
        }
    }

    {
        long long so = fp.obj, ss = fp.sq, sn = fp.cnt;
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
        for (int q = threadIdx.x; q < JM; q += NT) {
            const unsigned long long val = ((unsigned long long)a_hi[q] << 32) | a_lo[q];
            if (val) atomicAdd(p.s_fix + q, val);
        }
    }
    // a4-a6 by the CTA that finishes last.  Its scratch is the first stage buffer: grid_epilogue's barrier comes after
    // every consumer has seen the last "full" phase, so no bulk copy is in flight any more.
    grid_epilogue(tp.f, reinterpret_cast<double*>(stage0), NT);
}

#ifdef DUALIP_HOST_KERNELS
// a0: the 16-bit copy of the item indices the streaming kernel reads (J < 65,536 on that plan)
__global__ void k_encode_idx16(const int* __restrict__ idx, long long nnz, unsigned short* out) {
    for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < nnz; q += (long long)gridDim.x * blockDim.x) out[q] = (unsigned short)idx[q];
}

// a0: tile table from an explicit list of cut rows (the streaming plan with long rows isolated: dualip_api.cu)
__global__ void k_fill_tiles(const long long* __restrict__ row_ptr, const long long* __restrict__ cuts, long long ntiles, TileEntry* tiles) {
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t <= ntiles; t += (long long)gridDim.x * blockDim.x) {
        tiles[t].row0 = cuts[t];
        tiles[t].nz0 = row_ptr[cuts[t]];
    }
}

// a0: tile table.  Tile t starts at the first row r with row_ptr[r] + kRowCost*r >= t*TN (parallel binary search).
__global__ void k_build_tiles(const long long* __restrict__ row_ptr, long long I, long long TN, long long ntiles, TileEntry* tiles) {
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t <= ntiles; t += (long long)gridDim.x * blockDim.x) {
        long long r;
        if (t == ntiles) r = I;
        else {
            const long long target = t * TN;
            long long lo = 0, hi = I;                       // first r in [0,I] with key(r) >= target; key(I) >= target holds
            while (lo < hi) {
                const long long mid = (lo + hi) >> 1;
                if (row_ptr[mid] + kRowCost * mid >= target) hi = mid; else lo = mid + 1;
            }
            r = lo;
        }
        tiles[t].row0 = r;
        tiles[t].nz0 = row_ptr[r];
    }
}

#endif  // DUALIP_HOST_KERNELS

// Kernel table of one translation unit: dualip_tma_wx0.cu / dualip_tma_wx1.cu each instantiate every (G, M, ACC_SMEM,
// GBOX) variant for their WX and export this lookup, so the two halves compile in parallel.
template <bool WX>
struct TmaKernelTable {
    template <int G, int M>
    static const void* acc(bool a, bool gbox) {
        if (a) return gbox ? (const void*)k_grad_tma<G, M, true, true, WX, kTmaConsumerWarps>
                           : (const void*)k_grad_tma<G, M, true, false, WX, kTmaConsumerWarps>;
        return gbox ? (const void*)k_grad_tma<G, M, false, true, WX, kTmaConsumerWarps>
                    : (const void*)k_grad_tma<G, M, false, false, WX, kTmaConsumerWarps>;
    }
    template <int G>
    static const void* fam(int M, bool a, bool gbox) {
        if (M == 1) return acc<G, 1>(a, gbox);
        if (M == 2) return acc<G, 2>(a, gbox);
        return nullptr;
    }
    static const void* get(int G, int M, bool a, bool gbox) {
        if (M == 0) return acc<8, 0>(a, gbox);
        switch (G) {
            case 1: return fam<1>(M, a, gbox);
            case 2: return fam<2>(M, a, gbox);
            case 4: return fam<4>(M, a, gbox);
            case 8: return fam<8>(M, a, gbox);
            case 16: return fam<16>(M, a, gbox);
            default: return fam<32>(M, a, gbox);
        }
    }
};

}  // namespace dualip_dev
