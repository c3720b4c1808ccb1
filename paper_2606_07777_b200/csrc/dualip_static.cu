// dualip_static.cu -- dualip_grad_static (include/dualip.h): one evaluation of Eq. 2-4 that allocates nothing.
//
// Who needs it.  Every other entry point works on a handle, and dualip_create fills that handle with cudaMalloc'd
// buffers -- among them the scratch the gradient kernel reduces into (the 64-bit fixed-point item accumulators, three
// scalar accumulators and the arrival counter of its grid epilogue).  Some programs may not allocate device memory at
// the point where they want a gradient: a plug-in inside a host application that hands out all device memory itself and
// forbids cudaMalloc behind its back, a service whose memory budget was fixed and fully reserved at start-up, code on a
// latency-critical path where cudaMalloc's implicit device-wide synchronisation is not acceptable.  For them the same
// kernel (k_grad / k_grad_box of dualip_kernels.cuh, unchanged) is launched here with its scratch in a file-scope
// `static __device__` array of this translation unit instead.  Inputs and outputs are still the caller's device buffers.
//
// Cost of having no handle: the fixed-point scales that dualip_create derives once (max |a|, max |c|, the largest column
// sum of |a|, sum |c|) are recomputed by every call -- two extra passes over the rows and two stream synchronisations.
//
// Rules of the static scratch (also in the header):
//   * it is g_static_scratch below: (8 + 2 * DUALIP_STATIC_MAX_DUALS) 8-byte words = 448 KB + 64 B of device memory on
//     EVERY GPU whose context loads this library, from load until the process exits;
//   * in host code the name g_static_scratch is only a host-side shadow symbol, not a device address -- the device address
//     comes from cudaGetSymbolAddress, once per device with that device current (device_setup), and that pointer is what
//     the kernels receive.  The three small kernels of this file name the array directly, which device code may do;
//   * every call shares it and it keeps whatever the previous call left, so each call first clears the part it uses;
//   * two calls that overlap on the GPU (different streams, or two host threads) race on it.
#include "../../include/dualip.h"
#include "dualip_kernels.cuh"

#include <cmath>
#include <cstring>
#include <mutex>

using namespace dualip_dev;

namespace {

constexpr int kMaxDuals = DUALIP_STATIC_MAX_DUALS;
constexpr size_t kSmemBudget = 227 * 1024;   // dynamic shared memory one CTA may opt in to on sm_100a
constexpr size_t kEpilogueSmem = ((size_t)kFinalizeScratchBytes + 15) & ~(size_t)15;
static_assert(8 * (size_t)kMaxDuals + kEpilogueSmem <= kSmemBudget, "lambda for DUALIP_STATIC_MAX_DUALS duals must fit in shared memory");

// Word layout (8-byte words).  D = J*m of the current call; the two D-sized blocks are packed behind the header, so one
// memset of (8 + 2 D) words clears everything a call uses.
enum : int {
    W_ABSMAX = 0,   // two 32-bit words: bit patterns of max |a| and max |c|
    W_SUM_C = 1,    // sum |c|, fixed point
    W_MAX_COL = 2,  // max over coupling rows of the column sum of |a|, fixed point
    W_DONE = 3,     // low 32 bits: arrival counter of the gradient kernel's grid epilogue
    W_SCALARS = 4,  // c'x, |x|^2, sum x, fixed point (sc_fix of GradParams); word 7 unused
    W_BLOCKS = 8    // [W_BLOCKS, W_BLOCKS + D): column sums of |a|;  [W_BLOCKS + D, W_BLOCKS + 2 D): item accumulators (s_fix)
};
constexpr size_t kScratchWords = W_BLOCKS + 2 * (size_t)kMaxDuals;

static __device__ __align__(256) unsigned long long g_static_scratch[kScratchWords];

// ---- the create-time constants, recomputed per call; same arithmetic as k_absmax / k_col_stats / k_reduce_stats so that
// the fixed-point scales come out exactly as dualip_create's.  Device code: the array is named directly.

__global__ void k_static_absmax(const float* __restrict__ a, long long na, const float* __restrict__ c, long long nc) {
    unsigned ma = 0, mc = 0;
    for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < na; q += (long long)gridDim.x * blockDim.x)
        ma = max(ma, __float_as_uint(fabsf(a[q])));
    for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < nc; q += (long long)gridDim.x * blockDim.x)
        mc = max(mc, __float_as_uint(fabsf(c[q])));
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { ma = max(ma, __shfl_xor_sync(kFull, ma, o)); mc = max(mc, __shfl_xor_sync(kFull, mc, o)); }
    unsigned* out = reinterpret_cast<unsigned*>(g_static_scratch + W_ABSMAX);
    if ((threadIdx.x & 31) == 0) { atomicMax(out + 0, ma); atomicMax(out + 1, mc); }
}

__global__ void k_static_col_abs(const int* __restrict__ idx, const float* __restrict__ a, const float* __restrict__ c,
                                 long long nnz, int m, double scale_abs, double scale_c) {
    unsigned long long* colabs = g_static_scratch + W_BLOCKS;
    long long lc = 0;
    for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < nnz; q += (long long)gridDim.x * blockDim.x) {
        const int j = idx[q];
        for (int k = 0; k < m; ++k) {
            const long long fa = __double2ll_rn(fabs((double)a[q * m + k]) * scale_abs);
            if (fa) atomicAdd(colabs + (long long)j * m + k, (unsigned long long)fa);
        }
        lc += __double2ll_rn(fabs((double)c[q]) * scale_c);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) lc += __shfl_xor_sync(kFull, lc, o);
    if ((threadIdx.x & 31) == 0 && lc) atomicAdd(g_static_scratch + W_SUM_C, (unsigned long long)lc);
}

__global__ void __launch_bounds__(1024) k_static_max_col(int JM) {
    __shared__ unsigned long long sh[32];
    const unsigned long long* colabs = g_static_scratch + W_BLOCKS;
    unsigned long long b = 0;
    for (int q = threadIdx.x; q < JM; q += 1024) b = max(b, colabs[q]);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) b = max(b, __shfl_xor_sync(kFull, b, o));
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = b;
    __syncthreads();
    if (threadIdx.x == 0) {
        b = 0;
        for (int w = 0; w < 32; ++w) b = max(b, sh[w]);
        g_static_scratch[W_MAX_COL] = b;
    }
}

// ---- host side ------------------------------------------------------------------------------------------------------

#define CKS(call) do { if ((call) != cudaSuccess) { cudaGetLastError(); return DUALIP_ECUDA; } } while (0)

// 2^e with |bound| * 2^e < 2^61 -- the rule dualip_create uses for every fixed-point scale (dualip_api.cu fix_scale)
double fix_scale(double bound) {
    if (!(bound > 0.0) || !std::isfinite(bound)) return 1.0;
    int e = 0;
    std::frexp(bound, &e);
    int s = 61 - e;
    if (s > 96) s = 96;
    if (s < -96) s = -96;
    return std::ldexp(1.0, s);
}

bool on_device(const void* p) {
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged;
}

int grid_for(long long n, int threads, int num_sms) {
    long long g = (n + threads - 1) / threads;
    const long long cap = (long long)num_sms * 16;
    if (g > cap) g = cap;
    if (g < 1) g = 1;
    return (int)g;
}

// Per-device set-up, done by the first call on each device with that device current: the DEVICE address of the scratch
// array (g_static_scratch itself means nothing to a kernel when written in host code) and the SM count.
constexpr int kMaxDevices = 64;
struct DeviceSetup { bool ready = false; unsigned long long* scratch = nullptr; int num_sms = 0; };
DeviceSetup g_setup[kMaxDevices];
std::mutex g_setup_mutex;

int device_setup(const DeviceSetup** out) {
    int dev = -1;
    CKS(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices) return DUALIP_EUNSUPPORTED;
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    DeviceSetup& s = g_setup[dev];
    if (!s.ready) {
        void* p = nullptr;
        CKS(cudaGetSymbolAddress(&p, g_static_scratch));
        if (!p) return DUALIP_ECUDA;
        CKS(cudaDeviceGetAttribute(&s.num_sms, cudaDevAttrMultiProcessorCount, dev));
        s.scratch = static_cast<unsigned long long*>(p);
        s.ready = true;
    }
    *out = &s;
    return DUALIP_OK;
}

// the direct-load kernel with lambda in shared memory and the item sums reduced straight into the scratch (RED.ADD.64)
template <int G>
const void* pick_grad(int M) {
    if (M == 1) return (const void*)k_grad<G, 5, 1, true, false>;
    if (M == 2) return (const void*)k_grad<G, 5, 2, true, false>;
    return nullptr;
}

}  // namespace

extern "C" int dualip_grad_static(int64_t I, int32_t J, int32_t m, const int64_t* row_ptr, const int32_t* item_idx, const float* c,
                                  const float* a, const float* b, int32_t projection, double p0, double p1, const double* lambda,
                                  double gamma, double* grad, dualip_scalars* scalars, float* x, void* stream) {
    if (I < 0 || J < 1 || m < 1 || m > 4 || !row_ptr || !b || !lambda) return DUALIP_EINVAL;
    if (!(gamma > 0.0) || !std::isfinite(gamma)) return DUALIP_EINVAL;
    switch (projection) {
        case DUALIP_PROJ_SIMPLEX_INEQ: case DUALIP_PROJ_SIMPLEX_EQ: if (!(p0 > 0.0)) return DUALIP_EINVAL; break;
        case DUALIP_PROJ_BOX: if (!(p0 <= p1)) return DUALIP_EINVAL; break;
        case DUALIP_PROJ_BOXCUT: if (!(p0 > 0.0) || !(p1 > 0.0)) return DUALIP_EINVAL; break;
        default: return DUALIP_EINVAL;
    }
    if ((long long)J * m > (long long)kMaxDuals) return DUALIP_ETOOBIG;        // the scratch is sized at compile time
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { cudaGetLastError(); return DUALIP_ECUDA; }
    // nothing can be staged without allocating: every buffer has to be device memory already
    if (!on_device(row_ptr) || !on_device(b) || !on_device(lambda)) return DUALIP_EINVAL;
    if ((grad && !on_device(grad)) || (scalars && !on_device(scalars)) || (x && !on_device(x))) return DUALIP_EINVAL;

    const DeviceSetup* dv = nullptr;
    { int rc = device_setup(&dv); if (rc != 0) return rc; }
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    unsigned long long* const W = dv->scratch;
    const int JM = J * m;

    long long ends[2] = {0, 0};
    CKS(cudaMemcpyAsync(&ends[0], row_ptr, 8, cudaMemcpyDeviceToHost, st));
    CKS(cudaMemcpyAsync(&ends[1], row_ptr + I, 8, cudaMemcpyDeviceToHost, st));
    CKS(cudaStreamSynchronize(st));
    if (ends[0] != 0 || ends[1] < 0) return DUALIP_ERANGE;
    const long long nnz = ends[1];
    if (nnz > 0 && (!item_idx || !c || !a)) return DUALIP_EINVAL;
    if (nnz > 0 && (!on_device(item_idx) || !on_device(c) || !on_device(a))) return DUALIP_EINVAL;

    // the array holds the previous call's leftovers (or those of a call that failed half-way): clear what this call uses
    CKS(cudaMemsetAsync(W, 0, ((size_t)W_BLOCKS + 2 * (size_t)JM) * 8, st));

    // create-time constants (a0; R2 and the fixed-point scales), in the arithmetic of dualip_create
    float max_abs_a = 0.0f, max_abs_c = 0.0f;
    double max_colabs = 0.0, sum_abs_c = 0.0;
    if (nnz > 0) {
        k_static_absmax<<<grid_for(nnz * m, 256, dv->num_sms), 256, 0, st>>>(a, nnz * m, c, nnz);
        unsigned mx[2] = {0u, 0u};
        CKS(cudaMemcpyAsync(mx, W + W_ABSMAX, sizeof(mx), cudaMemcpyDeviceToHost, st));
        CKS(cudaStreamSynchronize(st));
        CKS(cudaGetLastError());
        std::memcpy(&max_abs_a, &mx[0], 4); std::memcpy(&max_abs_c, &mx[1], 4);
        const double rows = (double)(I > 0 ? I : 1);
        const double scale_abs = fix_scale((double)max_abs_a * rows * 1.000001);
        const double scale_c = fix_scale((double)max_abs_c * (double)nnz * 1.000001);
        k_static_col_abs<<<grid_for(nnz, 256, dv->num_sms), 256, 0, st>>>(item_idx, a, c, nnz, m, scale_abs, scale_c);
        k_static_max_col<<<1, 1024, 0, st>>>(JM);
        unsigned long long res[2] = {0ull, 0ull};
        CKS(cudaMemcpyAsync(res, W + W_SUM_C, sizeof(res), cudaMemcpyDeviceToHost, st));      // W_SUM_C, W_MAX_COL are adjacent
        CKS(cudaStreamSynchronize(st));
        CKS(cudaGetLastError());
        sum_abs_c = (double)(long long)res[0] / scale_c;
        max_colabs = (double)(long long)res[1] / scale_abs;
    }
    double xmax = p0;
    if (projection == DUALIP_PROJ_BOX) xmax = std::fmax(std::fabs(p0), std::fabs(p1));
    else if (projection == DUALIP_PROJ_BOXCUT) xmax = std::fmin(p0, p1);
    const double nz = (double)(nnz > 0 ? nnz : 1);
    const double scale_s = fix_scale(xmax * max_colabs * 1.000001), scale_obj = fix_scale(xmax * sum_abs_c * 1.000001);
    const double scale_sq = fix_scale(xmax * xmax * nz * 1.000001), scale_cnt = fix_scale(xmax * nz * 1.000001);

    GradParams p{};
    p.row_ptr = reinterpret_cast<const long long*>(row_ptr); p.idx = item_idx; p.c = c; p.a = a; p.lambda = lambda;
    p.s_fix = W + W_BLOCKS + JM; p.sc_fix = W + W_SCALARS; p.x = x;
    p.I = I; p.nnz = nnz; p.J = J; p.m = m; p.proj = projection;
    p.inv_gamma = 1.0 / gamma; p.inv_gamma_f = (float)(1.0 / gamma);
    p.general_boxcut = 0; p.z = 1.0f; p.ub = 0.0f; p.box_lo = 0.0; p.box_hi = 0.0;
    switch (projection) {
        case DUALIP_PROJ_BOX: p.box_lo = p0; p.box_hi = p1; break;
        case DUALIP_PROJ_BOXCUT:
            p.ub = (float)p0; p.z = (float)p1;
            p.general_boxcut = (p0 < p1) ? 1 : 0;                      // ub >= z is the simplex itself (R10)
            if (!p.general_boxcut) p.proj = PROJ_SIMPLEX_INEQ;
            break;
        default: p.z = (float)p0; break;
    }
    p.count_on = 0; p.long_thr = 0;
    p.scale_s = scale_s; p.scale_obj = scale_obj; p.scale_sq = scale_sq; p.scale_cnt = scale_cnt;
    p.scale_s_f = (float)scale_s; p.scale_obj_f = (float)scale_obj; p.scale_sq_f = (float)scale_sq; p.scale_cnt_f = (float)scale_cnt;
    p.max_abs_c = max_abs_c; p.max_abs_a = max_abs_a;

    FinalizeParams f{};
    f.s_fix = p.s_fix; f.sc_fix = p.sc_fix; f.b = b; f.lam_eval = lambda;
    f.grad_out = grad; f.scalars_out = reinterpret_cast<double*>(scalars);
    f.JM = JM; f.R = JM;
    f.inv_scale_s = 1.0 / scale_s; f.inv_scale_obj = 1.0 / scale_obj; f.inv_scale_sq = 1.0 / scale_sq; f.inv_scale_cnt = 1.0 / scale_cnt;
    f.gamma = gamma; f.update = 0;
    f.done = reinterpret_cast<unsigned*>(W + W_DONE);

    void* args[2] = {&p, &f};
    if (projection == DUALIP_PROJ_BOX) {
        const void* fn = m == 1 ? (const void*)k_grad_box<1> : (m == 2 ? (const void*)k_grad_box<2> : (const void*)k_grad_box<0>);
        CKS(cudaLaunchKernel(fn, dim3(grid_for(nnz, 256, dv->num_sms)), dim3(256), args, 0, st));
    } else {
        const double mean = I > 0 ? (double)nnz / (double)I : 0.0;
        const int G = mean > 20.0 ? 32 : (mean > 10.0 ? 16 : 8);
        const void* fn = m > 2 ? (const void*)k_grad<32, 5, 0, true, false>
                               : (G == 32 ? pick_grad<32>(m) : (G == 16 ? pick_grad<16>(m) : pick_grad<8>(m)));
        const size_t smem = 8 * (size_t)JM + kEpilogueSmem;
        CKS(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBudget));
        int per_sm = 0;
        CKS(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, kBlockThreads, smem));
        if (per_sm < 1) return DUALIP_EUNSUPPORTED;
        CKS(cudaLaunchKernel(fn, dim3(dv->num_sms * per_sm), dim3(kBlockThreads), args, smem, st));
    }
    CKS(cudaGetLastError());
    return DUALIP_OK;
}
