// dualip_api.cu -- the C ABI of include/dualip.h: argument checking, device residency, launch plan and the
// gamma-continuation driver (a0, a7).  Every arithmetic step of the path runs in the kernels of
// dualip_kernels.cuh; the host only sizes buffers, picks fixed-point exponents and launches.
#include "../../include/dualip.h"
#define DUALIP_HOST_KERNELS 1
#include "dualip_kernels.cuh"
#include "dualip_grad_tma.cuh"
#include "dualip_csc.cuh"
#include "dualip_long.cuh"

#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

using namespace dualip_dev;

// kernel tables of the two streaming-kernel translation units (dualip_tma_wx0.cu: never writes x; dualip_tma_wx1.cu: writes x)
const void* dualip_tma_kernel_wx0(int G, int M, bool acc_smem, bool gbox);
const void* dualip_tma_kernel_wx1(int G, int M, bool acc_smem, bool gbox);

namespace {

constexpr size_t kSmemBudget = 227 * 1024;  // bytes of dynamic shared memory one CTA may opt in to on sm_100a

constexpr size_t kLoSmemBytes = 64 * 1024;  // lambda as an fp32 pair is always staged in shared memory while the pair stays under this

struct Plan {
    int G = 32, KREG = 5, M = 1;
    bool lam_smem = true, acc_smem = true;
    int grid = 0;
    size_t smem = 0;
    const void* fn = nullptr;
    const void* fn_x = nullptr;     // streaming path: the x-writing instantiation (fn never writes x)
    // streaming (TMA) path
    bool tma = false;
    int lo_policy = 0;              // lambda's low word in shared memory: 0 per launch (kernel decides), 1 never, 2 always (sized in)
    long long TN = 0, ntiles = 0;
    int cap_nz = 0, cap_rows = 0, stages = 0, stage_bytes = 0;
};

}  // namespace

struct dualip {
    long long I = 0, nnz = 0;
    int J = 0, m = 0;
    dualip_opts opts{};
    // row data (owned unless borrowed)
    const long long* row_ptr = nullptr; const int* idx = nullptr; const float* c = nullptr; const float* a = nullptr;
    bool own_rows = false, own_c = false;
    float* b = nullptr;
    // scratch
    unsigned long long* s_fix = nullptr;   // JM item accumulators, then the 3 scalars obj, sq, cnt (sc_fix)
    unsigned long long* sc_fix = nullptr;
    double* lam_cur = nullptr; double* y = nullptr; double* lam_stage = nullptr; double* grad_stage = nullptr;
    double* y_prev = nullptr; double* g_prev = nullptr;   // DUALIP_STEP_ADAPTIVE: previous evaluation point / gradient (R20)
    bool count_on = false;                                 // global-count row (R21): duals = J*m + 1
    double count_M = 0.0;                                  // ... and its right-hand side, in fp64 (budgets above 2^24 are not fp32 numbers)
    // user-sharded multi-GPU: the caller's all-reduce between the gradient kernel and the epilogue
    dualip_reduce_hook hook = nullptr; void* hook_user = nullptr;
    long long nnz_total = 0;                               // nonzeros over all shards (= nnz unless dualip_set_shard_constants said otherwise)
    bool sharded = false;                                  // dualip_set_shard_constants has been called: the constants are GLOBAL ones
    bool shard_stale = false;                              // ... and dualip_set_c has changed c since: they must be agreed on again
    double* scalars_dev = nullptr;
    float* x_stage = nullptr;
    dualip_dev::TileEntry* tiles = nullptr;
    unsigned short* idx16 = nullptr;       // streaming plan: item_idx as 16-bit values (owned, 2 bytes per nonzero)
    unsigned char* ctl = nullptr;          // [IterState (16 B)][done counter (4 B)] -- see grid_epilogue
    // DUALIP_RED_CSC: item-sorted permutation (a0) and the per-iteration scratch of the atomics-free reduction
    bool csc = false, perm64 = false;
    void* csc_perm = nullptr;              // unsigned[nnz] (nnz < 2^32) or long long[nnz]
    long long* col_ptr = nullptr;          // [J+1]
    long long* chunk_ptr = nullptr;        // [J+1]
    int* chunk_item = nullptr;             // [nchunks]
    long long nchunks = 0;
    double* csc_partial = nullptr;         // [nchunks*m]
    float* x_csc = nullptr;                // [nnz] x of the current evaluation when the caller does not ask for it
    // CUDA graph of kGraphUnroll chained iteration launches (use_graph), re-parameterised per stage
    cudaGraph_t graph = nullptr; cudaGraphExec_t graph_exec = nullptr;
    std::vector<cudaGraphNode_t> graph_nodes;
    long long graph_launches = 0;
    // constants from a0
    double L = 0.0, max_colabs = 0.0, sum_abs_c = 0.0;
    double L_step = 0.0;                   // the constant the step is derived from: L, or L' of the row-scaled system (Jacobi)
    double* step_scale = nullptr;          // [JM] d_q^2 (Jacobi) or nullptr
    unsigned char* row_eq = nullptr;       // [JM] equality-row mask (dualip_set_equality_rows) or nullptr
    float max_abs_a = 0.0f, max_abs_c = 0.0f;
    long long max_row_len = 0;
    // long rows (dualip_long.cuh): rows of more than long_thr nonzeros are skipped by the main gradient kernel and taken by
    // k_grad_long, one CTA per row, in a launch of its own before it.  long_thr = 0: no such rows.
    long long long_thr = 0, n_long = 0;
    long long* long_ids = nullptr;
    double scale_s = 1.0, scale_obj = 1.0, scale_sq = 1.0, scale_cnt = 1.0;
    double xmax = 1.0;
    Plan plan;
    int num_sms = 0;
    long long launches = 0;
    long long bytes_resident = 0;
    // profiling hook: event pairs around gradient-kernel launches
    bool profile = false;
    std::vector<cudaEvent_t> events;
    size_t ev_used = 0;
    double prof_ms = 0.0;
    long long prof_count = 0;
};

namespace {

#define CK(call) do { if ((call) != cudaSuccess) { cudaGetLastError(); return DUALIP_ECUDA; } } while (0)

bool is_device_ptr(const void* p) {
    if (!p) return false;
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged;
}

template <typename T>
int dev_alloc(dualip* h, T** out, size_t n) {
    void* p = nullptr;
    if (cudaMalloc(&p, n ? n * sizeof(T) : sizeof(T)) != cudaSuccess) { cudaGetLastError(); return DUALIP_ENOMEM; }
    h->bytes_resident += (long long)(n * sizeof(T));
    *out = static_cast<T*>(p);
    return DUALIP_OK;
}

// 2^e with |bound| * 2^e < 2^61
double fix_scale(double bound) {
    if (!(bound > 0.0) || !std::isfinite(bound)) return 1.0;
    int e = 0;
    std::frexp(bound, &e);
    int s = 61 - e;
    if (s > 96) s = 96;       // keeps the scale (and value * scale for fp32 values below 2^31) inside fp32 range
    if (s < -96) s = -96;
    return std::ldexp(1.0, s);
}

template <int G, int KREG, int M>
const void* pick_mode(bool lam, bool acc) {
    if (lam && acc) return (const void*)k_grad<G, KREG, M, true, true>;
    if (lam) return (const void*)k_grad<G, KREG, M, true, false>;
    return (const void*)k_grad<G, KREG, M, false, false>;
}
template <int G, int KREG>
const void* pick_m(int M, bool lam, bool acc) {
    if (M == 1) return pick_mode<G, KREG, 1>(lam, acc);
    if (M == 2) return pick_mode<G, KREG, 2>(lam, acc);
    return nullptr;
}
template <int G>
const void* pick_k(int KREG, int M, bool lam, bool acc) {
    if (KREG == 2) return pick_m<G, 2>(M, lam, acc);
    if (KREG == 3) return pick_m<G, 3>(M, lam, acc);
    return pick_m<G, 5>(M, lam, acc);
}
const void* pick_kernel(const Plan& pl) {
    if (pl.M == 0) return pick_mode<32, 5, 0>(pl.lam_smem, pl.acc_smem);
    if (pl.G == 8) return pick_k<8>(pl.KREG, pl.M, pl.lam_smem, pl.acc_smem);
    if (pl.G == 16) return pick_k<16>(pl.KREG, pl.M, pl.lam_smem, pl.acc_smem);
    return pick_k<32>(pl.KREG, pl.M, pl.lam_smem, pl.acc_smem);
}

// Streaming plan: lambda (and for small J*m the accumulators) in shared memory, the rest of the 227 KB split into
// `stages` tile buffers.  Returns false if this problem cannot use it.
bool plan_tma(dualip* h, Plan& pl, long long max_len) {
    const size_t JM = (size_t)h->J * h->m;
    const int red = h->opts.reduction;
    if (h->opts.projection == DUALIP_PROJ_BOX || h->nnz == 0) return false;
    if (max_len > 8192 || h->J > 65535) return false;       // (J is far below that whenever lambda fits in shared memory)
    if (((uintptr_t)h->row_ptr | (uintptr_t)h->idx | (uintptr_t)h->c | (uintptr_t)h->a) & 15) return false;
    // Shared memory: RN_f32(lambda) always (the filter's operand, 4 B per dual).  Its low word joins it while the
    // pair stays under 64 KB (otherwise the exact path reads the fp64 lambda through L2: it runs once per row at
    // most).  The fixed-point item accumulators (8 B per dual) are privatised per CTA only for small J*m, where the
    // same few addresses would otherwise serialise in L2; beyond that RED.ADD.64 goes straight to L2.
    const size_t fixed = kTmaHeaderBytes + 128;
    if (fixed + 4 * JM + 32 * 1024 > kSmemBudget) return false;
    // small J*m: the low word is always staged (the plan is sized with it); larger: the kernel decides per launch whether
    // to trade a pipeline stage for it (k_grad_tma); tuning.lambda_plan overrides
    const int lp = h->opts.tuning.lambda_plan;
    const bool lo = lp != 1 && 8 * JM <= kLoSmemBytes;
    const size_t lam_bytes = (lo ? 8 : 4) * JM;
    bool acc = (red == DUALIP_RED_AUTO && 16 * JM <= 64 * 1024) ||
               (red == DUALIP_RED_SMEM && fixed + lam_bytes + 8 * JM + 32 * 1024 <= kSmemBudget);
    if (red == DUALIP_RED_SMEM && !acc) return false;
    const size_t avail = kSmemBudget - fixed - lam_bytes - (acc ? 8 : 0) * JM;
    pl.lo_policy = lo ? 2 : (lp == 1 ? 1 : (lp == 2 ? 2 : 0));
    const int m = h->m;
    const long long units = h->nnz + (long long)kRowCost * h->I;
    long long TN = 0; int stages = 0; size_t stage_bytes = 0;
    const int s_hi = h->opts.tuning.stages ? h->opts.tuning.stages : 3, s_lo = h->opts.tuning.stages ? h->opts.tuning.stages : 2;
    for (int S = s_hi; S >= s_lo && TN < 256; --S) {
        stage_bytes = (avail / S) & ~(size_t)127;
        const long long over = 80 + (max_len + 16 + 72) * (6 + 4 * m);
        long long tn = ((long long)stage_bytes - over) / (7 + 4 * m);
        tn = tn > 0 ? (tn & ~63ll) : 0;
        if (tn >= (S >= 3 ? 512 : 256)) { TN = tn; stages = S; }
    }
    if (TN < 256) return false;
    // small problems: keep at least ~8 tiles per CTA so the static deal stays balanced
    const long long want = units / ((long long)h->num_sms * 8);
    if (TN > 8192) TN = 8192;
    if (TN > want) TN = want > 256 ? (want & ~63ll) : 256;
    if (h->opts.tuning.tile_units >= 256 && h->opts.tuning.tile_units < TN) TN = h->opts.tuning.tile_units & ~63ll;
    pl.tma = true; pl.acc_smem = acc; pl.lam_smem = true;
    pl.TN = TN; pl.stages = stages;
    pl.cap_nz = (int)((TN + max_len + 16 + 72 + 7) & ~7ll);  // +72: lanes may read up to 2*32+2 slots past a row end (m = 2)
    pl.cap_rows = (int)((TN / kRowCost + 6 + 1) & ~1ll);
    size_t sb = (size_t)pl.cap_nz * (6 + 4 * m) + (size_t)pl.cap_rows * 8 + 32;
    pl.stage_bytes = (int)((sb + 127) & ~(size_t)127);
    pl.ntiles = (units + TN - 1) / TN;
    size_t off = kTmaHeaderBytes + lam_bytes + (acc ? 8 : 0) * JM;
    off = (off + 127) & ~(size_t)127;
    pl.smem = off + (size_t)pl.stage_bytes * stages;
    if (pl.smem > kSmemBudget) return false;
    // room for lambda's low word where the budget has it (small plans): a launch that stages it then keeps all its stages
    if (!lo) pl.smem = std::min(kSmemBudget, pl.smem + 4 * JM + 128);
    return true;
}

int make_plan(dualip* h) {
    Plan pl;
    const size_t JM = (size_t)h->J * h->m;
    const int red = h->opts.reduction;
    const size_t kScratch = (kFinalizeScratchBytes + 15) & ~(size_t)15;
    const bool fits_both = 16 * JM + kScratch <= kSmemBudget, fits_lam = 8 * JM + kScratch <= kSmemBudget;
    if (red == DUALIP_RED_SMEM && !fits_both) return DUALIP_EUNSUPPORTED;
    pl.acc_smem = (red == DUALIP_RED_AUTO || red == DUALIP_RED_SMEM) && fits_both;
    pl.lam_smem = pl.acc_smem || fits_lam;
    pl.M = (h->m <= 2) ? h->m : 0;
    const double mean = h->I > 0 ? (double)h->nnz / (double)h->I : 0.0;
    int G = h->opts.group_lanes;
    if (G == 0) G = mean > 20.0 ? 32 : (mean > 10.0 ? 16 : 8);
    if (G != 1 && G != 2 && G != 4 && G != 8 && G != 16 && G != 32) return DUALIP_EINVAL;
    if (pl.M == 0) G = 32;
    // Rows the streaming kernel cannot stage next to a useful tile are LONG rows: k_grad_long takes them, CTA per row, and the
    // streaming kernel's tile table isolates each of them in a tile of its own that the producer skips.  The cap is the
    // largest row length (tried downwards from 8192 in steps of a quarter) that still gives a 3-stage plan; simplex kinds only.
    const bool simplex_kind = h->opts.projection == DUALIP_PROJ_SIMPLEX_INEQ || h->opts.projection == DUALIP_PROJ_SIMPLEX_EQ ||
                              (h->opts.projection == DUALIP_PROJ_BOXCUT && h->opts.p0 >= h->opts.p1);
    bool streaming = false;
    h->long_thr = 0;
    if (h->opts.tuning.direct_kernel != 1) {                        // tuning.direct_kernel forces the non-streaming kernel (tests)
        streaming = plan_tma(h, pl, h->max_row_len);
        if (!streaming && simplex_kind && h->max_row_len > 256) {
            for (long long cap = std::min<long long>(8192, h->max_row_len - 1) & ~63ll; cap >= 256 && !streaming; cap = (cap * 3 / 4) & ~63ll) {
                Plan trial = pl;
                if (plan_tma(h, trial, cap) && trial.stages >= 3) { pl = trial; streaming = true; h->long_thr = cap; }
            }
        }
    }
    if (streaming) {
        // narrow lane groups: several rows share one pass of the chunk loop, which amortises the per-row work
        int Gs = h->opts.group_lanes;
        if (Gs == 0) {
            Gs = mean <= 6.0 ? 1 : (mean <= 12.0 ? 2 : (mean <= 32.0 ? 4 : (mean <= 256.0 ? 8 : (mean <= 1024.0 ? 16 : 32))));
            // a tile is released only when its slowest row-step is done, so it should split into about as many steps
            // (2 * 32/G rows each) as there are consumer warps: long rows (few per tile) get wider groups
            const double rows_per_tile = (double)pl.TN / (mean + kRowCost);
            int Gt = 1;
            while (Gt < 32 && (double)Gt * rows_per_tile < 360.0) Gt <<= 1;     // measured: cfg5 (92 rows per tile) is faster at 4, cfg3 (82) at 8
            if (Gt > Gs) Gs = Gt;
        }
        if (pl.M == 0) Gs = 8;
        pl.G = Gs;
        pl.KREG = 0;
        const bool gbox = h->opts.projection == DUALIP_PROJ_BOXCUT && h->opts.p0 < h->opts.p1;
        pl.fn = dualip_tma_kernel_wx0(pl.G, pl.M, pl.acc_smem, gbox);
        pl.fn_x = dualip_tma_kernel_wx1(pl.G, pl.M, pl.acc_smem, gbox);
        if (!pl.fn || !pl.fn_x) return DUALIP_EUNSUPPORTED;
        // the attribute is per function and process-wide: always the full budget, so that handles with different plans
        // (several may share one instantiation) never shrink it under each other
        CK(cudaFuncSetAttribute(pl.fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBudget));
        CK(cudaFuncSetAttribute(pl.fn_x, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBudget));
        pl.grid = h->opts.grid_ctas > 0 ? h->opts.grid_ctas : (int)(pl.ntiles < h->num_sms ? pl.ntiles : h->num_sms);
        if (pl.grid < 1) pl.grid = 1;
        h->plan = pl;
        return DUALIP_OK;
    }
    pl.tma = false;
    if (simplex_kind && h->max_row_len > 4096) h->long_thr = 4096;   // direct-load plan: beyond this a row gets a CTA, not a warp
    if (G < 8) G = 8;
    pl.acc_smem = (red == DUALIP_RED_AUTO || red == DUALIP_RED_SMEM) && fits_both;
    pl.lam_smem = pl.acc_smem || fits_lam;
    pl.G = G;
    pl.KREG = 5;
    if (pl.M != 0) {
        if ((long long)G * 2 >= h->max_row_len) pl.KREG = 2;
        else if ((long long)G * 3 >= h->max_row_len) pl.KREG = 3;
    }
    pl.smem = (pl.lam_smem ? 8 * JM : 0) + (pl.acc_smem ? 8 * JM : 0) + kScratch;
    pl.fn = pick_kernel(pl);
    if (!pl.fn) return DUALIP_EUNSUPPORTED;
    CK(cudaFuncSetAttribute(pl.fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBudget));
    int nb = 0;
    CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, pl.fn, kBlockThreads, pl.smem));
    if (nb < 1) return DUALIP_EUNSUPPORTED;
    pl.grid = h->opts.grid_ctas > 0 ? h->opts.grid_ctas : h->num_sms * nb;
    h->plan = pl;
    return DUALIP_OK;
}

void set_xmax(dualip* h) {
    const dualip_opts& o = h->opts;
    switch (o.projection) {
        case DUALIP_PROJ_BOX: h->xmax = std::fmax(std::fabs(o.p0), std::fabs(o.p1)); break;
        case DUALIP_PROJ_BOXCUT: h->xmax = std::fmin(o.p0, o.p1); break;
        default: h->xmax = o.p0; break;
    }
}

void set_scales(dualip* h) {
    h->scale_s = fix_scale(h->xmax * h->max_colabs * 1.000001);
    h->scale_obj = fix_scale(h->xmax * h->sum_abs_c * 1.000001);
    h->scale_sq = fix_scale(h->xmax * h->xmax * (double)(h->nnz_total > 0 ? h->nnz_total : 1) * 1.000001);
    h->scale_cnt = fix_scale(h->xmax * (double)(h->nnz_total > 0 ? h->nnz_total : 1) * 1.000001);
}

// duals = coupling rows: J*m, + 1 with the global-count row (R21)
size_t n_duals(const dualip* h) { return (size_t)h->J * h->m + (h->count_on ? 1 : 0); }

int grid_for(long long n, int threads, int num_sms) {
    long long g = (n + threads - 1) / threads;
    const long long cap = (long long)num_sms * 16;
    if (g > cap) g = cap;
    if (g < 1) g = 1;
    return (int)g;
}

// Fixed-point scales of the a0 column statistics, from the problem's extents (the GLOBAL extents of a sharded problem, so
// that every shard accumulates in the same scales and the integer sums add up exactly to the unsharded ones).
struct StatScales { double sq, abs, c; };
StatScales stat_scales(long long I, long long nnz, int m, float maxa, float maxc) {
    const double rows = (double)(I > 0 ? I : 1);
    StatScales sc;
    sc.sq = fix_scale((double)maxa * maxa * m * rows * 1.000001);
    sc.abs = fix_scale((double)maxa * rows * 1.000001);
    sc.c = fix_scale((double)maxc * (double)(nnz > 0 ? nnz : 1) * 1.000001);
    return sc;
}

// max |a|, max |c| of this handle's rows
int absmax_rows(dualip* h, cudaStream_t st, float& maxa, float& maxc) {
    unsigned* d_mx = nullptr;
    if (cudaMalloc(&d_mx, 2 * sizeof(unsigned)) != cudaSuccess) { cudaGetLastError(); return DUALIP_ENOMEM; }
    unsigned mx[2] = {0u, 0u};
    const bool ok = cudaMemsetAsync(d_mx, 0, 2 * sizeof(unsigned), st) == cudaSuccess;
    if (ok) { k_absmax<<<grid_for(h->nnz * h->m, 256, h->num_sms), 256, 0, st>>>(h->a, h->nnz * h->m, h->c, h->nnz, d_mx); h->launches++; }
    const bool ok2 = ok && cudaMemcpyAsync(mx, d_mx, sizeof(mx), cudaMemcpyDeviceToHost, st) == cudaSuccess &&
                     cudaStreamSynchronize(st) == cudaSuccess && cudaGetLastError() == cudaSuccess;
    cudaFree(d_mx);
    if (!ok2) { cudaGetLastError(); return DUALIP_ECUDA; }
    std::memcpy(&maxa, &mx[0], 4); std::memcpy(&maxc, &mx[1], 4);
    return DUALIP_OK;
}

// d_fix = [colsq JM][colabs JM][cabs 1][out 3] (zeroed by the caller where it accumulates): this handle's column sums
void launch_col_stats(dualip* h, cudaStream_t st, const StatScales& sc, unsigned long long* d_fix, bool do_a, bool do_c) {
    const int JM = h->J * h->m;
    k_col_stats<<<grid_for(h->nnz, 256, h->num_sms), 256, 0, st>>>(h->idx, h->a, h->c, h->nnz, h->m, sc.sq, sc.abs, sc.c,
                                                                   d_fix, d_fix + JM, d_fix + 2 * JM, do_a ? 1 : 0, do_c ? 1 : 0);
    h->launches++;
}

// L (R2), max column |a| sum, sum |c|, the Jacobi factors (R18): derived from the fixed-point column sums in d_fix
int derive_constants(dualip* h, cudaStream_t st, const StatScales& sc, unsigned long long* d_fix, bool do_a, bool do_c) {
    const int J = h->J, m = h->m, JM = J * m;
    unsigned long long* colsq = d_fix; unsigned long long* colabs = d_fix + JM; unsigned long long* cabs = colabs + JM;
    unsigned long long* out = cabs + 1;
    k_reduce_stats<<<1, 1024, 0, st>>>(colsq, J, m, colabs, JM, out); h->launches++;
    if (do_a && h->step_scale) {
        k_jacobi_step_scale<<<grid_for(JM, 256, h->num_sms), 256, 0, st>>>(colsq, 1.0 / sc.sq, JM, h->step_scale); h->launches++;
        const double d2_count = h->nnz_total > 0 ? 1.0 / (double)h->nnz_total : 1.0;   // the count row has a 1 on each of the nnz pairs
        if (cudaMemcpyAsync(h->step_scale + JM, &d2_count, 8, cudaMemcpyHostToDevice, st) != cudaSuccess) { cudaGetLastError(); return DUALIP_ECUDA; }
    }
    unsigned long long res[4];
    if (cudaMemcpyAsync(res, cabs, sizeof(res), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
        cudaStreamSynchronize(st) != cudaSuccess || cudaGetLastError() != cudaSuccess) { cudaGetLastError(); return DUALIP_ECUDA; }
    if (do_c) h->sum_abs_c = (double)(long long)res[0] / sc.c;
    if (do_a) {
        h->L = (double)(long long)res[1] / sc.sq; h->max_colabs = (double)(long long)res[2] / sc.abs;
        // Jacobi: every nonzero row of A' has unit norm, so L' = max_j sum_k |A'_(j,k)*|^2 = max_j #{k : row (j,k) != 0}
        h->L_step = h->step_scale ? (double)(res[3] > 0 ? res[3] : 1) : h->L;
    }
    return DUALIP_OK;
}

// a0 constants of an unsharded problem; all through order-independent fixed point.
int compute_stats(dualip* h, cudaStream_t st, bool do_a, bool do_c) {
    const int JM = h->J * h->m;
    float maxa = 0.0f, maxc = 0.0f;
    int rc = absmax_rows(h, st, maxa, maxc);
    if (rc != 0) return rc;
    h->max_abs_a = maxa; h->max_abs_c = maxc;
    unsigned long long* d_fix = nullptr;  // colsq[JM], colabs[JM], cabs[1], out[3]
    const size_t nfix = (size_t)2 * JM + 4;
    if (cudaMalloc(&d_fix, nfix * sizeof(unsigned long long)) != cudaSuccess) { cudaGetLastError(); return DUALIP_ENOMEM; }
    if (cudaMemsetAsync(d_fix, 0, nfix * sizeof(unsigned long long), st) != cudaSuccess) { cudaGetLastError(); cudaFree(d_fix); return DUALIP_ECUDA; }
    const StatScales sc = stat_scales(h->I, h->nnz, h->m, maxa, maxc);
    launch_col_stats(h, st, sc, d_fix, do_a, do_c);
    rc = derive_constants(h, st, sc, d_fix, do_a, do_c);
    cudaFree(d_fix);
    return rc;
}

void fill_grad_params(const dualip* h, GradParams& p, const double* lam_dev, double gamma, float* x_dev) {
    const dualip_opts& o = h->opts;
    p.row_ptr = h->row_ptr; p.idx = h->idx; p.c = h->c; p.a = h->a;
    p.lambda = lam_dev; p.s_fix = h->s_fix; p.sc_fix = h->sc_fix; p.x = x_dev;
    p.I = h->I; p.nnz = h->nnz; p.J = h->J; p.m = h->m; p.proj = o.projection;
    p.inv_gamma = 1.0 / gamma; p.inv_gamma_f = (float)(1.0 / gamma);
    p.general_boxcut = 0; p.z = 1.0f; p.ub = 0.0f; p.box_lo = 0.0; p.box_hi = 0.0;
    switch (o.projection) {
        case DUALIP_PROJ_BOX: p.box_lo = o.p0; p.box_hi = o.p1; break;
        case DUALIP_PROJ_BOXCUT:
            p.ub = (float)o.p0; p.z = (float)o.p1;
            p.general_boxcut = (o.p0 < o.p1) ? 1 : 0;       // ub >= z is the simplex itself (R10)
            if (!p.general_boxcut) p.proj = PROJ_SIMPLEX_INEQ;
            break;
        default: p.z = (float)o.p0; break;
    }
    p.count_on = h->count_on ? 1 : 0;
    p.long_thr = h->long_thr;
    p.scale_s = h->scale_s; p.scale_obj = h->scale_obj; p.scale_sq = h->scale_sq; p.scale_cnt = h->scale_cnt;
    p.scale_s_f = (float)h->scale_s; p.scale_obj_f = (float)h->scale_obj; p.scale_sq_f = (float)h->scale_sq;
    p.scale_cnt_f = (float)h->scale_cnt;
    p.max_abs_c = h->max_abs_c; p.max_abs_a = h->max_abs_a;
}

constexpr size_t kMaxTimedLaunches = 4096;

bool prof_begin(dualip* h, cudaStream_t st) {
    if (!h->profile || h->ev_used + 2 > 2 * kMaxTimedLaunches) return false;
    while (h->events.size() < h->ev_used + 2) {
        cudaEvent_t e;
        if (cudaEventCreate(&e) != cudaSuccess) { cudaGetLastError(); return false; }
        h->events.push_back(e);
    }
    return cudaEventRecord(h->events[h->ev_used], st) == cudaSuccess;
}
void prof_end(dualip* h, cudaStream_t st) {
    cudaEventRecord(h->events[h->ev_used + 1], st);
    h->ev_used += 2;
}
void prof_collect(dualip* h) {
    for (size_t e = 0; e + 1 < h->ev_used; e += 2) {
        float ms = 0.0f;
        if (cudaEventSynchronize(h->events[e + 1]) == cudaSuccess &&
            cudaEventElapsedTime(&ms, h->events[e], h->events[e + 1]) == cudaSuccess) { h->prof_ms += ms; h->prof_count++; }
        else cudaGetLastError();
    }
    h->ev_used = 0;
}

// Common fields of the per-launch epilogue (a4-a6).  The caller sets lam_eval/gamma/update/... before launch_iter.
void fill_finalize_common(const dualip* h, FinalizeParams& f) {
    f.s_fix = h->s_fix; f.sc_fix = h->sc_fix; f.b = h->b; f.count_rhs = h->count_M; f.JM = h->J * h->m; f.R = (int)n_duals(h);
    f.inv_scale_s = 1.0 / h->scale_s; f.inv_scale_obj = 1.0 / h->scale_obj; f.inv_scale_sq = 1.0 / h->scale_sq;
    f.inv_scale_cnt = 1.0 / h->scale_cnt;
    f.row_eq = h->row_eq;
    f.state = reinterpret_cast<IterState*>(h->ctl);
    f.done = reinterpret_cast<unsigned*>(h->ctl + sizeof(IterState));
}

// Everything one launch needs: function, geometry and the argument block (kept alive by the caller).
struct IterLaunch {
    const void* fn; dim3 grid, block; size_t smem;
    GradParams p; FinalizeParams f, f_after; TmaParams tp;
    void* args[2];
};

void prepare_iter(const dualip* h, IterLaunch& L, const double* lam_dev, double gamma, float* x_dev, const FinalizeParams& f_in) {
    fill_grad_params(h, L.p, lam_dev, gamma, x_dev);
    L.f = f_in;
    fill_finalize_common(h, L.f);
    L.f_after = L.f;
    if (h->csc) {                       // the kernel only writes x and the scalars; a4-a6 follow as launches of their own
        L.p.s_fix = nullptr;
        if (!L.p.x) L.p.x = h->x_csc;
        L.f.done = nullptr;
    }
    if (h->hook) L.f.done = nullptr;    // sharded: the cross-GPU sum of the accumulators comes between the kernel and a4-a6
    if (h->opts.projection == DUALIP_PROJ_BOX) {
        L.fn = h->m == 1 ? (const void*)k_grad_box<1> : (h->m == 2 ? (const void*)k_grad_box<2> : (const void*)k_grad_box<0>);
        L.grid = dim3(grid_for(h->nnz, 256, h->num_sms)); L.block = dim3(256); L.smem = 0;
        L.args[0] = &L.p; L.args[1] = &L.f;
    } else if (h->plan.tma) {
        TmaParams& tp = L.tp;
        tp.g = L.p; tp.f = L.f; tp.tiles = h->tiles; tp.ntiles = h->plan.ntiles; tp.cap_nz = h->plan.cap_nz; tp.cap_rows = h->plan.cap_rows;
        tp.stages = h->plan.stages; tp.stage_bytes = h->plan.stage_bytes;
        tp.nnz8 = h->nnz & ~7ll; tp.idx16 = h->idx16; tp.rows2 = (h->I + 1) & ~1ll; tp.lo_policy = h->plan.lo_policy;
        tp.smem_total = (int)h->plan.smem; tp.lo_flag = reinterpret_cast<int*>(h->ctl + 32);
        tp.check_word = reinterpret_cast<unsigned*>(h->ctl + 36);
        tp.dyn_steps = h->opts.tuning.step_deal == 2 ? 1 : 0;
        tp.row_cap = h->long_thr;
        L.fn = L.p.x ? h->plan.fn_x : h->plan.fn; L.grid = dim3(h->plan.grid); L.block = dim3(32 * (kTmaConsumerWarps + 1)); L.smem = h->plan.smem;
        L.args[0] = &L.tp; L.args[1] = nullptr;
    } else {
        L.fn = h->plan.fn; L.grid = dim3(h->plan.grid); L.block = dim3(kBlockThreads); L.smem = h->plan.smem;
        L.args[0] = &L.p; L.args[1] = &L.f;
    }
}

int launch_long(dualip* h, const GradParams& p, cudaStream_t st);

// One launch = one evaluation a1-a5 (+ the AGD update a6 when f.update): gradient kernel with the grid epilogue.
int launch_iter(dualip* h, IterLaunch& L, cudaStream_t st) {
    const bool timed = prof_begin(h, st);
    struct End { dualip* h; cudaStream_t st; bool on; ~End() { if (on) prof_end(h, st); } } end_guard{h, st, timed};
    { int rc = launch_long(h, L.p, st); if (rc != 0) return rc; }     // long rows first (none on the BASELINE configs)
    CK(cudaLaunchKernel(L.fn, L.grid, L.block, L.args, L.smem, st));
    h->launches++;
    CK(cudaGetLastError());
    if (h->csc) {
        const int rg = (int)std::min<long long>((h->nchunks + 7) / 8, (long long)h->num_sms * 8);
        if (h->nchunks > 0) {
            if (h->perm64) k_csc_reduce<long long><<<rg, 256, 0, st>>>((const long long*)h->csc_perm, h->col_ptr, h->chunk_ptr, h->chunk_item,
                                                                      h->nchunks, h->a, L.p.x, h->m, h->csc_partial);
            else k_csc_reduce<unsigned><<<rg, 256, 0, st>>>((const unsigned*)h->csc_perm, h->col_ptr, h->chunk_ptr, h->chunk_item,
                                                          h->nchunks, h->a, L.p.x, h->m, h->csc_partial);
            h->launches++;
        }
        const long long JM = (long long)h->J * h->m;
        k_csc_combine<<<(unsigned)((JM + 7) / 8), 256, 0, st>>>(h->chunk_ptr, h->J, h->m, h->csc_partial, h->scale_s, h->s_fix);
        h->launches++;
        CK(cudaGetLastError());
    }
    if (h->csc || h->hook) {
        if (h->hook && h->hook(h->hook_user, reinterpret_cast<int64_t*>(h->s_fix), (int64_t)h->J * h->m + 3, L.f_after.lam_eval, L.f_after.gamma, st) != 0) {
            // the exchange failed: finalising local sums would silently diverge from the other ranks.  Drop them (the epilogue,
            // which normally re-zeroes the accumulators, does not run) and report.
            CK(cudaMemsetAsync(h->s_fix, 0, ((size_t)h->J * h->m + 3) * 8, st));
            return DUALIP_EHOOK;
        }
        k_finalize_only<<<1, kBlockThreads, 0, st>>>(L.f_after);
        h->launches++;
        CK(cudaGetLastError());
    }
    return DUALIP_OK;
}

// a0 for DUALIP_RED_CSC: stable counting sort of the nonzero positions by item (dualip_csc.cuh)
int build_csc(dualip* h, cudaStream_t st) {
    const long long nnz = h->nnz;
    const int J = h->J;
    h->perm64 = nnz >= (1ll << 32);
    int rc;
    if ((rc = dev_alloc(h, &h->col_ptr, (size_t)J + 1)) != 0) return rc;
    if ((rc = dev_alloc(h, &h->chunk_ptr, (size_t)J + 1)) != 0) return rc;
    if ((rc = dev_alloc(h, &h->x_csc, (size_t)nnz)) != 0) return rc;
    {
        void* pp = nullptr;
        const size_t bytes = (size_t)(nnz > 0 ? nnz : 1) * (h->perm64 ? 8 : 4);
        if (cudaMalloc(&pp, bytes) != cudaSuccess) { cudaGetLastError(); return DUALIP_ENOMEM; }
        h->csc_perm = pp; h->bytes_resident += (long long)bytes;
    }
    // blocks of positions, one warp each; the (block, item) table is capped at 2^26 entries
    long long nblocks = (1ll << 26) / J;
    if (nblocks > 8192) nblocks = 8192;
    if (nblocks > (nnz + 1023) / 1024) nblocks = (nnz + 1023) / 1024;
    if (nblocks < 1) nblocks = 1;
    long long blk_len = (nnz + nblocks - 1) / nblocks;
    blk_len = (blk_len + 31) & ~31ll;
    if (blk_len < 32) blk_len = 32;
    if (blk_len >= (1ll << 32)) return DUALIP_EUNSUPPORTED;                  // a block's per-item count must fit 32 bits
    unsigned* table = nullptr; long long* total = nullptr; long long* nch = nullptr;
    if (cudaMalloc(&table, (size_t)nblocks * J * 4) != cudaSuccess) { cudaGetLastError(); return DUALIP_ENOMEM; }
    if (cudaMalloc(&total, (size_t)J * 16) != cudaSuccess) { cudaGetLastError(); cudaFree(table); return DUALIP_ENOMEM; }
    nch = total + J;
    rc = DUALIP_OK;
    do {
        if (cudaMemsetAsync(table, 0, (size_t)nblocks * J * 4, st) != cudaSuccess) { rc = DUALIP_ECUDA; break; }
        const unsigned wg = (unsigned)((nblocks + 7) / 8);
        k_csc_count<<<wg, 256, 0, st>>>(h->idx, nnz, J, nblocks, blk_len, table);
        k_csc_block_offsets<<<(J + 255) / 256, 256, 0, st>>>(table, J, nblocks, total, nch);
        k_scan_exclusive<<<1, 1024, 0, st>>>(total, J, h->col_ptr);
        k_scan_exclusive<<<1, 1024, 0, st>>>(nch, J, h->chunk_ptr);
        if (h->perm64) k_csc_scatter<long long><<<wg, 256, 0, st>>>(h->idx, nnz, J, nblocks, blk_len, table, h->col_ptr, (long long*)h->csc_perm);
        else k_csc_scatter<unsigned><<<wg, 256, 0, st>>>(h->idx, nnz, J, nblocks, blk_len, table, h->col_ptr, (unsigned*)h->csc_perm);
        h->launches += 5;
        long long nc = 0;
        if (cudaMemcpyAsync(&nc, h->chunk_ptr + J, 8, cudaMemcpyDeviceToHost, st) != cudaSuccess ||
            cudaStreamSynchronize(st) != cudaSuccess || cudaGetLastError() != cudaSuccess) { rc = DUALIP_ECUDA; break; }
        h->nchunks = nc;
    } while (0);
    cudaFree(table); cudaFree(total);
    if (rc != 0) return rc;
    if ((rc = dev_alloc(h, &h->chunk_item, (size_t)h->nchunks)) != 0) return rc;
    if ((rc = dev_alloc(h, &h->csc_partial, (size_t)h->nchunks * h->m)) != 0) return rc;
    k_csc_chunk_items<<<(J + 255) / 256, 256, 0, st>>>(h->chunk_ptr, J, h->chunk_item);
    h->launches++;
    CK(cudaGetLastError());
    return DUALIP_OK;
}

// a0: the rows k_grad_long takes (more than long_thr nonzeros)
int build_long_list(dualip* h, cudaStream_t st) {
    unsigned long long* d_cnt = nullptr;
    if (cudaMalloc(&d_cnt, 8) != cudaSuccess) { cudaGetLastError(); return DUALIP_ENOMEM; }
    unsigned long long n = 0;
    int rc = DUALIP_OK;
    do {
        const int g = grid_for(h->I, 256, h->num_sms);
        if (cudaMemsetAsync(d_cnt, 0, 8, st) != cudaSuccess) { rc = DUALIP_ECUDA; break; }
        k_collect_long<<<g, 256, 0, st>>>(h->row_ptr, h->I, h->long_thr, nullptr, d_cnt); h->launches++;
        if (cudaMemcpyAsync(&n, d_cnt, 8, cudaMemcpyDeviceToHost, st) != cudaSuccess || cudaStreamSynchronize(st) != cudaSuccess) { rc = DUALIP_ECUDA; break; }
        h->n_long = (long long)n;
        if (n == 0) { h->long_thr = 0; break; }
        if ((rc = dev_alloc(h, &h->long_ids, (size_t)n)) != 0) break;
        if (cudaMemsetAsync(d_cnt, 0, 8, st) != cudaSuccess) { rc = DUALIP_ECUDA; break; }
        k_collect_long<<<g, 256, 0, st>>>(h->row_ptr, h->I, h->long_thr, h->long_ids, d_cnt); h->launches++;
        if (cudaStreamSynchronize(st) != cudaSuccess || cudaGetLastError() != cudaSuccess) { rc = DUALIP_ECUDA; break; }
        const void* fn = h->m == 1 ? (const void*)k_grad_long<1> : (h->m == 2 ? (const void*)k_grad_long<2> : (const void*)k_grad_long<0>);
        if (cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBudget) != cudaSuccess) { rc = DUALIP_ECUDA; break; }
    } while (0);
    cudaFree(d_cnt);
    if (rc == DUALIP_ECUDA) cudaGetLastError();
    return rc;
}

// Streaming plan with long rows: every long row becomes a tile of its own (which the producer skips), i.e. the tile table gets
// a cut before and after each of them.  The table is a sorted list of row numbers, so this is a merge, done on the host at
// create; the rest of a split tile keeps its bounds (a piece of a tile is smaller than the tile).
int isolate_long_rows(dualip* h, cudaStream_t st) {
    const long long nt = h->plan.ntiles;
    std::vector<TileEntry> tiles((size_t)nt + 1);
    std::vector<long long> ids((size_t)h->n_long);
    CK(cudaMemcpyAsync(tiles.data(), h->tiles, ((size_t)nt + 1) * sizeof(TileEntry), cudaMemcpyDeviceToHost, st));
    CK(cudaMemcpyAsync(ids.data(), h->long_ids, (size_t)h->n_long * 8, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    std::vector<long long> cuts;
    cuts.reserve((size_t)nt + 1 + 2 * ids.size());
    for (const TileEntry& t : tiles) cuts.push_back(t.row0);
    for (long long r : ids) { cuts.push_back(r); cuts.push_back(r + 1); }
    std::sort(cuts.begin(), cuts.end());
    cuts.erase(std::unique(cuts.begin(), cuts.end()), cuts.end());           // first cut is row 0, last is row I
    const long long nt2 = (long long)cuts.size() - 1;
    long long* d_cuts = nullptr;
    if (cudaMalloc(&d_cuts, cuts.size() * 8) != cudaSuccess) { cudaGetLastError(); return DUALIP_ENOMEM; }
    cudaFree(h->tiles); h->tiles = nullptr; h->bytes_resident -= (long long)(((size_t)nt + 1) * sizeof(TileEntry));
    int rc = dev_alloc(h, &h->tiles, (size_t)nt2 + 1);
    if (rc == 0) {
        if (cudaMemcpyAsync(d_cuts, cuts.data(), cuts.size() * 8, cudaMemcpyHostToDevice, st) != cudaSuccess) rc = DUALIP_ECUDA;
        else {
            k_fill_tiles<<<grid_for(nt2 + 1, 128, h->num_sms), 128, 0, st>>>(h->row_ptr, d_cuts, nt2, h->tiles); h->launches++;
            if (cudaStreamSynchronize(st) != cudaSuccess || cudaGetLastError() != cudaSuccess) rc = DUALIP_ECUDA;
        }
    }
    cudaFree(d_cuts);
    if (rc != 0) { cudaGetLastError(); return rc; }
    h->plan.ntiles = nt2;
    if (h->opts.grid_ctas <= 0) h->plan.grid = (int)(nt2 < h->num_sms ? (nt2 > 0 ? nt2 : 1) : h->num_sms);
    return DUALIP_OK;
}

// the long rows of one evaluation: launched before the main gradient kernel, same accumulators, no epilogue
int launch_long(dualip* h, const GradParams& p, cudaStream_t st) {
    if (h->n_long <= 0) return DUALIP_OK;
    LongParams lp;
    lp.g = p; lp.long_ids = h->long_ids; lp.n_long = h->n_long;
    const size_t scratch = 64 * 4;
    lp.ucap = (int)((kSmemBudget - scratch) / 4);
    const int grid = (int)std::min<long long>(h->n_long, (long long)h->num_sms);
    if (h->m == 1) k_grad_long<1><<<grid, kLongThreads, kSmemBudget, st>>>(lp);
    else if (h->m == 2) k_grad_long<2><<<grid, kLongThreads, kSmemBudget, st>>>(lp);
    else k_grad_long<0><<<grid, kLongThreads, kSmemBudget, st>>>(lp);
    h->launches++;
    CK(cudaGetLastError());
    return DUALIP_OK;
}

constexpr int kGraphUnroll = 20;   // iterations per graph replay

void drop_graph(dualip* h) {
    if (h->graph_exec) cudaGraphExecDestroy(h->graph_exec);
    if (h->graph) cudaGraphDestroy(h->graph);
    h->graph_exec = nullptr; h->graph = nullptr; h->graph_nodes.clear();
}

// (Re)parameterise the graph of kGraphUnroll chained launches of L.  Built node by node (no stream capture, so it
// also works when the caller's stream is the legacy default stream).
int set_graph(dualip* h, IterLaunch& L) {
    cudaKernelNodeParams kp{};
    kp.func = const_cast<void*>(L.fn); kp.gridDim = L.grid; kp.blockDim = L.block;
    kp.sharedMemBytes = (unsigned)L.smem; kp.kernelParams = L.args; kp.extra = nullptr;
    if (h->graph_exec) {
        bool ok = true;
        for (cudaGraphNode_t nd : h->graph_nodes)
            if (cudaGraphExecKernelNodeSetParams(h->graph_exec, nd, &kp) != cudaSuccess) { cudaGetLastError(); ok = false; break; }
        if (ok) return DUALIP_OK;
        drop_graph(h);
    }
    CK(cudaGraphCreate(&h->graph, 0));
    h->graph_nodes.resize(kGraphUnroll);
    for (int k = 0; k < kGraphUnroll; ++k) {
        const cudaGraphNode_t* dep = k ? &h->graph_nodes[k - 1] : nullptr;
        if (cudaGraphAddKernelNode(&h->graph_nodes[k], h->graph, dep, k ? 1 : 0, &kp) != cudaSuccess) { cudaGetLastError(); drop_graph(h); return DUALIP_ECUDA; }
    }
    if (cudaGraphInstantiate(&h->graph_exec, h->graph, 0) != cudaSuccess) { cudaGetLastError(); drop_graph(h); return DUALIP_ECUDA; }
    return DUALIP_OK;
}

int ensure_x_stage(dualip* h) {
    if (!h->x_stage) return dev_alloc(h, &h->x_stage, (size_t)h->nnz);
    return DUALIP_OK;
}

}  // namespace

extern "C" {

void dualip_opts_default(dualip_opts* o) {
    if (!o) return;
    std::memset(o, 0, sizeof(*o));
    o->projection = DUALIP_PROJ_SIMPLEX_INEQ; o->p0 = 1.0; o->p1 = 0.0;
    o->reduction = DUALIP_RED_AUTO; o->borrow = 0; o->validate = 1; o->momentum = 1;
    o->step_rule = DUALIP_STEP_FIXED; o->eta_min = 1e-5; o->eta_max = 1e-1;
}

const char* dualip_strerror(int code) {
    switch (code) {
        case DUALIP_OK: return "ok";
        case DUALIP_EINVAL: return "invalid argument";
        case DUALIP_ERANGE: return "row_ptr not monotone or item index out of range";
        case DUALIP_EDUP: return "duplicate item within a user's row";
        case DUALIP_ENOMEM: return "out of memory";
        case DUALIP_ECUDA: return "CUDA runtime error";
        case DUALIP_EUNSUPPORTED: return "unsupported configuration";
        case DUALIP_ETOOBIG: return "J*m exceeds DUALIP_STATIC_MAX_DUALS, the fixed scratch size of dualip_grad_static";
        case DUALIP_ESTALE: return "sharded handle: c changed, call dualip_set_shard_constants again before evaluating";
        case DUALIP_EHOOK: return "the reduce hook failed; evaluation abandoned";
        default: return "unknown error code";
    }
}

void dualip_destroy(dualip_t* h) {
    if (!h) return;
    if (h->own_rows) { cudaFree((void*)h->row_ptr); cudaFree((void*)h->idx); cudaFree((void*)h->a); }
    if (h->own_c) cudaFree((void*)h->c);
    cudaFree(h->b); cudaFree(h->s_fix); cudaFree(h->lam_cur); cudaFree(h->y); cudaFree(h->lam_stage);
    cudaFree(h->grad_stage); cudaFree(h->y_prev); cudaFree(h->g_prev); cudaFree(h->scalars_dev); cudaFree(h->step_scale); cudaFree(h->row_eq); cudaFree(h->x_stage); cudaFree(h->tiles); cudaFree(h->idx16);
    drop_graph(h);
    cudaFree(h->ctl);
    cudaFree(h->csc_perm); cudaFree(h->col_ptr); cudaFree(h->chunk_ptr); cudaFree(h->chunk_item); cudaFree(h->csc_partial);
    cudaFree(h->x_csc); cudaFree(h->long_ids);
    for (cudaEvent_t e : h->events) cudaEventDestroy(e);
    cudaGetLastError();
    delete h;
}

int dualip_set_profiling(dualip_t* h, int on) {
    if (!h) return DUALIP_EINVAL;
    prof_collect(h);
    h->profile = on != 0;
    h->prof_ms = 0.0; h->prof_count = 0;
    return DUALIP_OK;
}

int dualip_create(dualip_t** out, int64_t I, int32_t J, int32_t m, const int64_t* row_ptr, const int32_t* item_idx,
                  const float* c, const float* a, const float* b, const dualip_opts* opts_in, void* stream) {
    if (!out) return DUALIP_EINVAL;
    *out = nullptr;
    if (I < 0 || J < 1 || m < 1 || m > 4 || !row_ptr || !b) return DUALIP_EINVAL;
    if ((long long)J * m > (1ll << 30)) return DUALIP_EINVAL;
    dualip_opts o;
    if (opts_in) o = *opts_in; else dualip_opts_default(&o);
    if (o.tuning.direct_kernel != 0 && o.tuning.direct_kernel != 1) return DUALIP_EINVAL;
    if (o.tuning.stages != 0 && (o.tuning.stages < 2 || o.tuning.stages > kTmaStagesMax)) return DUALIP_EINVAL;
    if (o.tuning.tile_units < 0 || o.tuning.lambda_plan < 0 || o.tuning.lambda_plan > 2) return DUALIP_EINVAL;
    if (o.tuning.step_deal < 0 || o.tuning.step_deal > 2) return DUALIP_EINVAL;
    if (o.step_rule != DUALIP_STEP_FIXED && o.step_rule != DUALIP_STEP_ADAPTIVE) return DUALIP_EINVAL;
    if (o.step_rule == DUALIP_STEP_ADAPTIVE && !(o.eta_min > 0.0 && o.eta_min <= o.eta_max && std::isfinite(o.eta_max))) return DUALIP_EINVAL;
    if (o.precondition != DUALIP_PRECOND_NONE && o.precondition != DUALIP_PRECOND_JACOBI) return DUALIP_EINVAL;
    switch (o.projection) {
        case DUALIP_PROJ_SIMPLEX_INEQ: case DUALIP_PROJ_SIMPLEX_EQ: if (!(o.p0 > 0.0)) return DUALIP_EINVAL; break;
        case DUALIP_PROJ_BOX: if (!(o.p0 <= o.p1)) return DUALIP_EINVAL; break;
        case DUALIP_PROJ_BOXCUT: if (!(o.p0 > 0.0) || !(o.p1 > 0.0)) return DUALIP_EINVAL; break;
        default: return DUALIP_EINVAL;
    }
    if (o.reduction < DUALIP_RED_AUTO || o.reduction > DUALIP_RED_CSC) return DUALIP_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { cudaGetLastError(); return DUALIP_ECUDA; }
    cudaStream_t st = static_cast<cudaStream_t>(stream);

    // nnz = row_ptr[I]; row_ptr[0] must be 0
    long long ends[2] = {0, 0};
    const bool rp_dev = is_device_ptr(row_ptr);
    if (rp_dev) {
        CK(cudaMemcpyAsync(&ends[0], row_ptr, 8, cudaMemcpyDeviceToHost, st));
        CK(cudaMemcpyAsync(&ends[1], row_ptr + I, 8, cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
    } else { ends[0] = row_ptr[0]; ends[1] = row_ptr[I]; }
    if (ends[0] != 0 || ends[1] < 0) return DUALIP_ERANGE;
    const long long nnz = ends[1];
    if (nnz > 0 && (!item_idx || !c || !a)) return DUALIP_EINVAL;

    dualip* h = new (std::nothrow) dualip();
    if (!h) return DUALIP_ENOMEM;
    h->I = I; h->nnz = nnz; h->nnz_total = nnz; h->J = J; h->m = m; h->opts = o;
    int dev = 0;
    int rc = DUALIP_OK;
#define FAIL(code) do { rc = (code); goto fail; } while (0)
#define CKF(call) do { if ((call) != cudaSuccess) { cudaGetLastError(); FAIL(DUALIP_ECUDA); } } while (0)
    {
        CKF(cudaGetDevice(&dev));
        CKF(cudaDeviceGetAttribute(&h->num_sms, cudaDevAttrMultiProcessorCount, dev));
        const bool all_dev = rp_dev && (nnz == 0 || (is_device_ptr(item_idx) && is_device_ptr(c) && is_device_ptr(a)));
        if (o.borrow && all_dev) {
            h->row_ptr = reinterpret_cast<const long long*>(row_ptr); h->idx = item_idx; h->c = c; h->a = a;
        } else {
            long long* d_rp = nullptr; int* d_idx = nullptr; float* d_c = nullptr; float* d_a = nullptr;
            h->own_rows = true; h->own_c = true;
            if ((rc = dev_alloc(h, &d_rp, (size_t)I + 1)) != 0) goto fail;
            h->row_ptr = d_rp;
            if ((rc = dev_alloc(h, &d_idx, (size_t)nnz)) != 0) goto fail;
            h->idx = d_idx;
            if ((rc = dev_alloc(h, &d_c, (size_t)nnz)) != 0) goto fail;
            h->c = d_c;
            if ((rc = dev_alloc(h, &d_a, (size_t)nnz * m)) != 0) goto fail;
            h->a = d_a;
            CKF(cudaMemcpyAsync(d_rp, row_ptr, ((size_t)I + 1) * 8, cudaMemcpyDefault, st));
            if (nnz > 0) {
                CKF(cudaMemcpyAsync(d_idx, item_idx, (size_t)nnz * 4, cudaMemcpyDefault, st));
                CKF(cudaMemcpyAsync(d_c, c, (size_t)nnz * 4, cudaMemcpyDefault, st));
                CKF(cudaMemcpyAsync(d_a, a, (size_t)nnz * m * 4, cudaMemcpyDefault, st));
            }
        }
        const size_t JM = (size_t)J * m;
        // every dual-sized buffer has room for the global-count row's entry (index JM; dualip_set_global_count)
        if ((rc = dev_alloc(h, &h->b, JM + 1)) != 0) goto fail;
        CKF(cudaMemsetAsync(h->b, 0, (JM + 1) * 4, st));
        CKF(cudaMemcpyAsync(h->b, b, JM * 4, cudaMemcpyDefault, st));
        if ((rc = dev_alloc(h, &h->s_fix, JM + 3)) != 0) goto fail;
        h->sc_fix = h->s_fix + JM;
        CKF(cudaMemsetAsync(h->s_fix, 0, (JM + 3) * 8, st));
        if ((rc = dev_alloc(h, &h->lam_cur, JM + 1)) != 0) goto fail;
        if ((rc = dev_alloc(h, &h->y, JM + 1)) != 0) goto fail;
        if ((rc = dev_alloc(h, &h->lam_stage, JM + 1)) != 0) goto fail;
        if ((rc = dev_alloc(h, &h->grad_stage, JM + 1)) != 0) goto fail;
        if ((rc = dev_alloc(h, &h->scalars_dev, 6)) != 0) goto fail;
        if (o.step_rule == DUALIP_STEP_ADAPTIVE) {
            if ((rc = dev_alloc(h, &h->y_prev, JM + 1)) != 0) goto fail;
            if ((rc = dev_alloc(h, &h->g_prev, JM + 1)) != 0) goto fail;
        }
        if ((rc = dev_alloc(h, &h->ctl, 64)) != 0) goto fail;
        CKF(cudaMemsetAsync(h->ctl, 0, 64, st));

        // validation (R11) and row-length statistics.  Monotone row_ptr and the maximum row length are always
        // computed (the kernels index with them); `validate` switches the index-range / duplicate scan.
        {
            int* d_flags = nullptr; unsigned long long* d_maxlen = nullptr;
            if (cudaMalloc(&d_flags, sizeof(int)) != cudaSuccess) { cudaGetLastError(); FAIL(DUALIP_ENOMEM); }
            if (cudaMalloc(&d_maxlen, 8) != cudaSuccess) { cudaGetLastError(); cudaFree(d_flags); FAIL(DUALIP_ENOMEM); }
            cudaMemsetAsync(d_flags, 0, sizeof(int), st); cudaMemsetAsync(d_maxlen, 0, 8, st);
            k_validate<<<grid_for(I, 128, h->num_sms), 128, 0, st>>>(h->row_ptr, h->idx, I, J, nnz, o.validate ? 1 : 0, d_flags, d_maxlen);
            h->launches++;
            int flags = 0; unsigned long long maxlen = 0;
            cudaError_t e1 = cudaMemcpyAsync(&flags, d_flags, sizeof(int), cudaMemcpyDeviceToHost, st);
            cudaError_t e2 = cudaMemcpyAsync(&maxlen, d_maxlen, 8, cudaMemcpyDeviceToHost, st);
            cudaError_t e3 = cudaStreamSynchronize(st);
            if (e1 == cudaSuccess && e2 == cudaSuccess && e3 == cudaSuccess && (flags & 8) && !(flags & 3)) {
                // some row is not ascending: its duplicate check is warp-cooperative (k_validate_unsorted)
                k_validate_unsorted<<<grid_for(I * 32, 256, h->num_sms), 256, 0, st>>>(h->row_ptr, h->idx, I, d_flags);
                h->launches++;
                e1 = cudaMemcpyAsync(&flags, d_flags, sizeof(int), cudaMemcpyDeviceToHost, st);
                e3 = cudaStreamSynchronize(st);
            }
            cudaFree(d_flags); cudaFree(d_maxlen);
            if (e1 != cudaSuccess || e2 != cudaSuccess || e3 != cudaSuccess || cudaGetLastError() != cudaSuccess) FAIL(DUALIP_ECUDA);
            if (flags & 3) FAIL(DUALIP_ERANGE);
            if (flags & 4) FAIL(DUALIP_EDUP);
            h->max_row_len = (long long)maxlen;
        }
        if (o.precondition == DUALIP_PRECOND_JACOBI && (rc = dev_alloc(h, &h->step_scale, JM + 1)) != 0) goto fail;
        if ((rc = compute_stats(h, st, true, true)) != 0) goto fail;
        set_xmax(h);
        set_scales(h);
        if ((rc = make_plan(h)) != 0) goto fail;
        if (o.reduction == DUALIP_RED_CSC) {
            h->csc = true;
            if ((rc = build_csc(h, st)) != 0) goto fail;
        }
        if (h->long_thr > 0 && (rc = build_long_list(h, st)) != 0) goto fail;
        if (h->plan.tma) {
            if ((rc = dev_alloc(h, &h->idx16, (size_t)nnz + 16)) != 0) goto fail;
            k_encode_idx16<<<grid_for(nnz, 256, h->num_sms), 256, 0, st>>>(h->idx, nnz, h->idx16); h->launches++;
            if ((rc = dev_alloc(h, &h->tiles, (size_t)h->plan.ntiles + 1)) != 0) goto fail;
            k_build_tiles<<<grid_for(h->plan.ntiles + 1, 128, h->num_sms), 128, 0, st>>>(h->row_ptr, I, h->plan.TN, h->plan.ntiles, h->tiles);
            h->launches++;
            CKF(cudaGetLastError());
            if (h->n_long > 0 && (rc = isolate_long_rows(h, st)) != 0) goto fail;
        }
        CKF(cudaStreamSynchronize(st));
    }
    *out = h;
    return DUALIP_OK;
fail:
    dualip_destroy(h);
    return rc;
#undef FAIL
#undef CKF
}

int dualip_get_info(dualip_t* h, dualip_info* info) {
    if (!h || !info) return DUALIP_EINVAL;
    prof_collect(h);
    std::memset(info, 0, sizeof(*info));
    info->I = h->I; info->nnz = h->nnz; info->J = h->J; info->m = h->m; info->L = h->L;
    info->max_row_len = h->max_row_len; info->long_rows = h->n_long; info->long_row_threshold = h->long_thr;
    info->group_lanes = h->plan.G; info->chunk_regs = h->plan.KREG;
    info->reduction = h->csc ? DUALIP_RED_CSC : (h->plan.acc_smem ? DUALIP_RED_SMEM : DUALIP_RED_GLOBAL);
    info->lambda_in_smem = h->plan.lam_smem ? 1 : 0;
    info->grid_ctas = h->plan.grid; info->block_threads = h->plan.tma ? 32 * (kTmaConsumerWarps + 1) : kBlockThreads;
    info->streaming = h->plan.tma ? 1 : 0; info->stages = h->plan.stages; info->tile_units = h->plan.TN; info->ntiles = h->plan.ntiles;
    info->smem_bytes = (int64_t)h->plan.smem;
    info->bytes_resident = h->bytes_resident; info->launches = h->launches;
    info->fix_scale_s = h->scale_s;
    info->grad_kernel_ms = h->prof_ms; info->grad_kernel_count = h->prof_count;
    info->precondition = h->step_scale ? DUALIP_PRECOND_JACOBI : DUALIP_PRECOND_NONE;
    info->L_step = h->L_step + (h->count_on ? (h->step_scale ? 1.0 : (double)h->nnz_total) : 0.0);
    info->duals = (int32_t)n_duals(h);
#ifdef DUALIP_CHECKED
    info->checked_build = 1;
#endif
    if (h->plan.tma) {                                       // what the last streaming launch decided (it has finished: default-stream copy)
        int flag = 0;
        int flag2[2] = {0, 0};
        if (cudaMemcpy(flag2, h->ctl + 32, sizeof(flag2), cudaMemcpyDeviceToHost) == cudaSuccess) { flag = flag2[0]; info->lambda_lo_smem = flag; info->checks_failed = flag2[1]; }
        else cudaGetLastError();
    }
    return DUALIP_OK;
}

int dualip_set_reduce_hook(dualip_t* h, dualip_reduce_hook fn, void* user) {
    if (!h) return DUALIP_EINVAL;
    h->hook = fn; h->hook_user = fn ? user : nullptr;
    return DUALIP_OK;
}

int dualip_get_shard_extents(dualip_t* h, dualip_shard_extents* out) {
    if (!h || !out) return DUALIP_EINVAL;
    out->I = h->I; out->nnz = h->nnz;
    // the handle's current maxima are the shard's own until dualip_set_shard_constants replaced them: recompute
    float maxa = 0.0f, maxc = 0.0f;
    int rc = absmax_rows(h, nullptr, maxa, maxc);
    if (rc != 0) return rc;
    out->max_abs_a = maxa; out->max_abs_c = maxc;
    return DUALIP_OK;
}

int dualip_get_column_stats(dualip_t* h, const dualip_shard_extents* g, int64_t* out, void* stream) {
    if (!h || !g || !out || g->I < h->I || g->nnz < h->nnz) return DUALIP_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const int JM = h->J * h->m;
    const size_t n = (size_t)2 * JM + 1;
    unsigned long long* d_fix = nullptr;
    if (cudaMalloc(&d_fix, n * 8) != cudaSuccess) { cudaGetLastError(); return DUALIP_ENOMEM; }
    int rc = DUALIP_OK;
    if (cudaMemsetAsync(d_fix, 0, n * 8, st) != cudaSuccess) rc = DUALIP_ECUDA;
    if (rc == 0) {
        launch_col_stats(h, st, stat_scales(g->I, g->nnz, h->m, g->max_abs_a, g->max_abs_c), d_fix, true, true);
        if (cudaGetLastError() != cudaSuccess || cudaMemcpyAsync(out, d_fix, n * 8, cudaMemcpyDefault, st) != cudaSuccess ||
            cudaStreamSynchronize(st) != cudaSuccess) rc = DUALIP_ECUDA;
    }
    cudaFree(d_fix);
    if (rc != 0) cudaGetLastError();
    return rc;
}

int dualip_set_shard_constants(dualip_t* h, const dualip_shard_extents* g, const int64_t* summed, void* stream) {
    if (!h || !g || !summed || g->I < h->I || g->nnz < h->nnz) return DUALIP_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const int JM = h->J * h->m;
    const size_t n = (size_t)2 * JM + 1;
    unsigned long long* d_fix = nullptr;                     // + out[3] of k_reduce_stats
    if (cudaMalloc(&d_fix, (n + 3) * 8) != cudaSuccess) { cudaGetLastError(); return DUALIP_ENOMEM; }
    int rc = DUALIP_OK;
    if (cudaMemcpyAsync(d_fix, summed, n * 8, cudaMemcpyDefault, st) != cudaSuccess) rc = DUALIP_ECUDA;
    if (rc == 0) {
        h->nnz_total = g->nnz; h->max_abs_a = g->max_abs_a; h->max_abs_c = g->max_abs_c;
        rc = derive_constants(h, st, stat_scales(g->I, g->nnz, h->m, g->max_abs_a, g->max_abs_c), d_fix, true, true);
    }
    cudaFree(d_fix);
    if (rc != 0) { cudaGetLastError(); return rc; }
    set_scales(h);
    h->sharded = true; h->shard_stale = false;
    return DUALIP_OK;
}

int dualip_eval_partial(dualip_t* h, const double* lambda_dev, double gamma, float* x, void* stream) {
    if (!h || !lambda_dev || !(gamma > 0.0) || !std::isfinite(gamma)) return DUALIP_EINVAL;
    if (!is_device_ptr(lambda_dev) || (x && !is_device_ptr(x)) || h->csc) return DUALIP_EINVAL;
    if (h->shard_stale) return DUALIP_ESTALE;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    FinalizeParams f{};
    f.lam_eval = lambda_dev; f.gamma = gamma; f.update = 0;
    IterLaunch L;
    prepare_iter(h, L, lambda_dev, gamma, x, f);
    L.f.done = nullptr;                                      // no epilogue: the accumulators stay in the handle
    if (h->plan.tma) L.tp.f = L.f;
    const bool timed = prof_begin(h, st);
    { int rc = launch_long(h, L.p, st); if (rc != 0) { if (timed) prof_end(h, st); return rc; } }
    CK(cudaLaunchKernel(L.fn, L.grid, L.block, L.args, L.smem, st));
    if (timed) prof_end(h, st);
    h->launches++;
    CK(cudaGetLastError());
    return DUALIP_OK;
}

int dualip_export_accumulators(dualip_t* h, int64_t* out, int32_t clear, void* stream) {
    if (!h || !out) return DUALIP_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const size_t n = (size_t)h->J * h->m + 3;
    CK(cudaMemcpyAsync(out, h->s_fix, n * 8, cudaMemcpyDefault, st));
    if (clear) CK(cudaMemsetAsync(h->s_fix, 0, n * 8, st));
    if (!is_device_ptr(out)) CK(cudaStreamSynchronize(st));
    return DUALIP_OK;
}

int dualip_import_accumulators(dualip_t* h, const int64_t* in, int32_t accumulate, void* stream) {
    if (!h || !in) return DUALIP_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const size_t n = (size_t)h->J * h->m + 3;
    if (!accumulate) {
        CK(cudaMemcpyAsync(h->s_fix, in, n * 8, cudaMemcpyDefault, st));
        if (!is_device_ptr(in)) CK(cudaStreamSynchronize(st));
        return DUALIP_OK;
    }
    const unsigned long long* src = reinterpret_cast<const unsigned long long*>(in);
    unsigned long long* tmp = nullptr;
    if (!is_device_ptr(in)) {
        if (cudaMalloc(&tmp, n * 8) != cudaSuccess) { cudaGetLastError(); return DUALIP_ENOMEM; }
        if (cudaMemcpyAsync(tmp, in, n * 8, cudaMemcpyHostToDevice, st) != cudaSuccess) { cudaGetLastError(); cudaFree(tmp); return DUALIP_ECUDA; }
        src = tmp;
    }
    k_acc_add<<<grid_for((long long)n, 256, h->num_sms), 256, 0, st>>>(h->s_fix, src, (long long)n);
    h->launches++;
    const cudaError_t e = cudaGetLastError();
    if (tmp) { cudaStreamSynchronize(st); cudaFree(tmp); }
    return e == cudaSuccess ? DUALIP_OK : DUALIP_ECUDA;
}

int dualip_get_csc(dualip_t* h, int64_t* col_ptr_out, int64_t* perm_out, void* stream) {
    if (!h) return DUALIP_EINVAL;
    if (!h->csc) return DUALIP_EUNSUPPORTED;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (col_ptr_out) CK(cudaMemcpyAsync(col_ptr_out, h->col_ptr, ((size_t)h->J + 1) * 8, cudaMemcpyDefault, st));
    if (perm_out && h->nnz > 0) {
        if (h->perm64) CK(cudaMemcpyAsync(perm_out, h->csc_perm, (size_t)h->nnz * 8, cudaMemcpyDefault, st));
        else {
            long long* tmp = nullptr;
            if (cudaMalloc(&tmp, (size_t)h->nnz * 8) != cudaSuccess) { cudaGetLastError(); return DUALIP_ENOMEM; }
            k_perm_widen<<<grid_for(h->nnz, 256, h->num_sms), 256, 0, st>>>((const unsigned*)h->csc_perm, h->nnz, tmp);
            h->launches++;
            const cudaError_t e1 = cudaMemcpyAsync(perm_out, tmp, (size_t)h->nnz * 8, cudaMemcpyDefault, st);
            const cudaError_t e2 = cudaStreamSynchronize(st);
            cudaFree(tmp);
            if (e1 != cudaSuccess || e2 != cudaSuccess) { cudaGetLastError(); return DUALIP_ECUDA; }
        }
    }
    CK(cudaStreamSynchronize(st));
    return DUALIP_OK;
}

int dualip_set_c(dualip_t* h, const float* c_new, void* stream) {
    if (!h || (!c_new && h->nnz > 0)) return DUALIP_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (h->nnz == 0) return DUALIP_OK;
    if (h->own_c) {
        CK(cudaMemcpyAsync((void*)h->c, c_new, (size_t)h->nnz * 4, cudaMemcpyDefault, st));
    } else {
        if (!is_device_ptr(c_new)) return DUALIP_EINVAL;     // borrowed rows: the new c must be device memory too
        if (h->plan.tma && ((uintptr_t)c_new & 15)) return DUALIP_EINVAL;   // the streaming kernel's bulk copies need 16-byte alignment
        h->c = c_new;
    }
    // A shard's sum |c| and max |c| are not the problem's: recomputing them here would give every rank its own fixed-point
    // scale for c'x, and the all-reduce would then add integers of different scales.  Keep the agreed constants and refuse to
    // evaluate until the shards have agreed again (dualip_get_shard_extents .. dualip_set_shard_constants).
    if (h->sharded) { h->shard_stale = true; return DUALIP_OK; }
    int rc = compute_stats(h, st, false, true);
    if (rc != 0) return rc;
    set_scales(h);
    return DUALIP_OK;
}

int dualip_set_equality_rows(dualip_t* h, const uint8_t* is_equality, void* stream) {
    if (!h) return DUALIP_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const size_t JM = (size_t)h->J * h->m, R = n_duals(h);
    if (!is_equality) {                                      // back to all-inequality rows
        if (h->row_eq) { CK(cudaStreamSynchronize(st)); cudaFree(h->row_eq); h->row_eq = nullptr; h->bytes_resident -= (long long)(JM + 1); }
        return DUALIP_OK;
    }
    if (!h->row_eq) { int rc = dev_alloc(h, &h->row_eq, JM + 1); if (rc != 0) return rc; }
    CK(cudaMemcpyAsync(h->row_eq, is_equality, R, cudaMemcpyDefault, st));
    if (!is_device_ptr(is_equality)) CK(cudaStreamSynchronize(st));
    return DUALIP_OK;
}

int dualip_set_global_count(dualip_t* h, int32_t enable, double M, void* stream) {
    if (!h) return DUALIP_EINVAL;
    if (enable && !(M >= 0.0 && std::isfinite(M))) return DUALIP_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    CK(cudaStreamSynchronize(st));                           // earlier launches still read the old layout
    if (h->row_eq) { cudaFree(h->row_eq); h->row_eq = nullptr; h->bytes_resident -= (long long)((size_t)h->J * h->m + 1); }
    h->count_on = enable != 0;
    h->count_M = enable ? M : 0.0;                           // read by the epilogue as row J*m's right-hand side (FinalizeParams.count_rhs)
    return DUALIP_OK;
}

int dualip_grad(dualip_t* h, const double* lambda, double gamma, double* grad, dualip_scalars* scalars, float* x,
                void* stream) {
    if (!h || !lambda || !(gamma > 0.0) || !std::isfinite(gamma)) return DUALIP_EINVAL;
    if (h->shard_stale) return DUALIP_ESTALE;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const size_t JM = n_duals(h);
    const bool lam_dev = is_device_ptr(lambda), grad_dev = is_device_ptr(grad), sc_dev = is_device_ptr(scalars),
               x_dev = is_device_ptr(x);
    const double* lam_d = lambda;
    if (!lam_dev) { CK(cudaMemcpyAsync(h->lam_stage, lambda, JM * 8, cudaMemcpyHostToDevice, st)); lam_d = h->lam_stage; }
    float* x_d = x;
    if (x && !x_dev) { int rc = ensure_x_stage(h); if (rc != 0) return rc; x_d = h->x_stage; }
    FinalizeParams f{};
    f.lam_eval = lam_d; f.gamma = gamma; f.update = 0;
    f.grad_out = grad ? (grad_dev ? grad : h->grad_stage) : nullptr;
    f.scalars_out = scalars ? (sc_dev ? reinterpret_cast<double*>(scalars) : h->scalars_dev) : nullptr;
    IterLaunch L;
    prepare_iter(h, L, lam_d, gamma, x_d, f);
    int rc = launch_iter(h, L, st);
    if (rc != 0) return rc;
    bool sync = !lam_dev;
    if (grad && !grad_dev) { CK(cudaMemcpyAsync(grad, h->grad_stage, JM * 8, cudaMemcpyDeviceToHost, st)); sync = true; }
    if (scalars && !sc_dev) { CK(cudaMemcpyAsync(scalars, h->scalars_dev, sizeof(dualip_scalars), cudaMemcpyDeviceToHost, st)); sync = true; }
    if (x && !x_dev && h->nnz > 0) { CK(cudaMemcpyAsync(x, h->x_stage, (size_t)h->nnz * 4, cudaMemcpyDeviceToHost, st)); sync = true; }
    if (sync) CK(cudaStreamSynchronize(st));
    return DUALIP_OK;
}

int dualip_solve(dualip_t* h, const double* gammas, int32_t n_stages, const int32_t* iters, double* lambda_inout,
                 float* x_out, dualip_scalars* final_scalars, double* final_grad, const dualip_trace* trace, void* stream) {
    if (!h || n_stages < 0 || !lambda_inout) return DUALIP_EINVAL;
    if (n_stages > 0 && (!gammas || !iters)) return DUALIP_EINVAL;
    long long total = 0;
    for (int s = 0; s < n_stages; ++s) {
        if (!(gammas[s] > 0.0) || !std::isfinite(gammas[s]) || iters[s] < 0) return DUALIP_EINVAL;
        total += iters[s];
    }
    if (trace && trace->capacity < total) return DUALIP_EINVAL;
    if (n_stages == 0) return DUALIP_OK;
    if (h->shard_stale) return DUALIP_ESTALE;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const size_t JM = n_duals(h);
    const bool lam_dev = is_device_ptr(lambda_inout), grad_dev = is_device_ptr(final_grad),
               sc_dev = is_device_ptr(final_scalars), x_dev = is_device_ptr(x_out);
    CK(cudaMemcpyAsync(h->lam_cur, lambda_inout, JM * 8, cudaMemcpyDefault, st));
    // R21: with the global-count row A A^T is no longer block diagonal; |A|_2^2 <= |A_items|_2^2 + |count row|_2^2, and the
    // row's squared norm is nnz (1 once row-normalised)
    double L = h->L_step + (h->count_on ? (h->step_scale ? 1.0 : (double)h->nnz_total) : 0.0);
    if (!(L > 0.0)) L = 1.0;
    const bool adaptive = h->opts.step_rule == DUALIP_STEP_ADAPTIVE;
    CK(cudaMemsetAsync(h->ctl, 0, sizeof(IterState), st));                                 // t = 0, n = 0
    for (int s = 0; s < n_stages; ++s) {
        const double gamma = gammas[s], eta = gamma / L;
        CK(cudaMemcpyAsync(h->y, h->lam_cur, JM * 8, cudaMemcpyDeviceToDevice, st));   // warm start, momentum restart (R4)
        CK(cudaMemsetAsync(h->ctl, 0, sizeof(int), st));                                   // t = 0; n runs on
        FinalizeParams f{};
        f.lam_eval = h->y; f.gamma = gamma; f.update = 1; f.eta = eta; f.momentum = h->opts.momentum ? 1 : 0;
        f.lam_cur = h->lam_cur; f.y = h->y; f.step_scale = h->step_scale;
        if (adaptive) {                                      // R20: clip range of this stage; the maximum scales with gamma
            // the lower end never lifts a step above the analytic one, gamma_s / L_step: without Jacobi scaling that is far
            // below the paper's 1e-5, and a step forced up to eta_min would be far beyond the stability bound
            f.step_rule = 1; f.eta_lo = std::min(h->opts.eta_min, eta); f.eta_hi = h->opts.eta_max * gamma / gammas[0];
            f.y_prev = h->y_prev; f.g_prev = h->g_prev;
        }
        if (trace) {
            f.tr_g = trace->g; f.tr_rinf = trace->r_inf; f.tr_r2 = trace->r_2; f.tr_grad = trace->grad; f.tr_lam = trace->lambda;
            f.tr_eta = trace->eta;
        }
        IterLaunch it;
        prepare_iter(h, it, h->y, gamma, nullptr, f);
        int t = 0;
        // beta_t and the trace row come from the device-side iteration state, so every launch of a stage has the
        // same arguments: replay a graph of kGraphUnroll chained launches, then finish with direct launches
        if (h->opts.use_graph && !h->profile && !h->csc && !h->hook && h->n_long == 0 && iters[s] >= 2 * kGraphUnroll) {
            int rc = set_graph(h, it);
            if (rc != 0) return rc;
            for (; t + kGraphUnroll <= iters[s]; t += kGraphUnroll) {
                CK(cudaGraphLaunch(h->graph_exec, st));
                h->launches += kGraphUnroll; h->graph_launches++;
            }
        }
        for (; t < iters[s]; ++t) {
            int rc = launch_iter(h, it, st);
            if (rc != 0) return rc;
        }
    }
    // final evaluation at lambda_T (R3); skipped when nobody asked for its outputs
    if (x_out || final_scalars || final_grad) {
        float* x_d = x_out;
        if (x_out && !x_dev) { int rc = ensure_x_stage(h); if (rc != 0) return rc; x_d = h->x_stage; }
        FinalizeParams f{};
        f.lam_eval = h->lam_cur; f.gamma = gammas[n_stages - 1]; f.update = 0;
        f.grad_out = final_grad ? (grad_dev ? final_grad : h->grad_stage) : nullptr;
        f.scalars_out = final_scalars ? (sc_dev ? reinterpret_cast<double*>(final_scalars) : h->scalars_dev) : nullptr;
        IterLaunch it;
        prepare_iter(h, it, h->lam_cur, gammas[n_stages - 1], x_d, f);
        int rc = launch_iter(h, it, st);
        if (rc != 0) return rc;
    }
    bool sync = false;
    CK(cudaMemcpyAsync(lambda_inout, h->lam_cur, JM * 8, cudaMemcpyDefault, st));
    if (!lam_dev) sync = true;
    if (final_grad && !grad_dev) { CK(cudaMemcpyAsync(final_grad, h->grad_stage, JM * 8, cudaMemcpyDeviceToHost, st)); sync = true; }
    if (final_scalars && !sc_dev) { CK(cudaMemcpyAsync(final_scalars, h->scalars_dev, sizeof(dualip_scalars), cudaMemcpyDeviceToHost, st)); sync = true; }
    if (x_out && !x_dev && h->nnz > 0) { CK(cudaMemcpyAsync(x_out, h->x_stage, (size_t)h->nnz * 4, cudaMemcpyDeviceToHost, st)); sync = true; }
    if (sync) CK(cudaStreamSynchronize(st));
    return DUALIP_OK;
}

}  // extern "C"
