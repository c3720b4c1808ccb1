// dualip_csc.cuh -- the atomics-free item reduction (DUALIP_RED_CSC): a4 through a precomputed item-sorted
// permutation, for J*m beyond what per-CTA accumulators or L2 atomics serve well, and as the mode whose summation
// ORDER is fixed (not only its result).
//
//   a0 (create)   stable counting sort of the nonzero positions by item: col_ptr[J+1], perm[nnz] with
//                 perm[col_ptr[j] .. col_ptr[j+1]) = positions of item j's nonzeros in ascending order -- bit-exact
//                 with a CPU stable counting sort.  The position range is cut into `nblocks` contiguous blocks, one
//                 warp each; table[b][j] first counts item j inside block b, then becomes the block's cursor.
//   per iteration k_csc_reduce: one warp per column chunk (kCscChunk entries) sums a^k * x over its entries in a fixed
//                 lane-strided order + a fixed shuffle tree (fp64);  k_csc_combine: one warp per (item, family) adds the
//                 chunk partials in order and stores the 64-bit fixed-point sum the epilogue expects;  k_finalize_only:
//                 a4-a6 (finalize_block).  The gradient kernel runs before them with x written to memory and its own
//                 item accumulation and epilogue switched off.
#pragma once
#include "dualip_kernels.cuh"

namespace dualip_dev {

constexpr int kCscChunk = 4096;          // column entries per reduction chunk

// ---- a0: stable counting sort --------------------------------------------------------------------------------------

// table[b*J + j] = number of nonzeros of item j among positions [b*blk_len, (b+1)*blk_len)
__global__ void k_csc_count(const int* __restrict__ idx, long long nnz, int J, long long nblocks, long long blk_len,
                            unsigned* table) {
    const long long b = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    if (b >= nblocks) return;
    const int lane = threadIdx.x & 31;
    const long long beg = b * blk_len, end = min(nnz, beg + blk_len);
    unsigned* row = table + b * J;
    for (long long q = beg + lane; q < end; q += 32) atomicAdd(row + idx[q], 1u);
}

// per item: table[b][j] <- number of item-j nonzeros in blocks before b (exclusive running count); total[j] = column length
__global__ void k_csc_block_offsets(unsigned* table, int J, long long nblocks, long long* total, long long* nchunks) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= J) return;
    unsigned long long run = 0;
    for (long long b = 0; b < nblocks; ++b) {
        const unsigned t = table[b * J + j];
        table[b * J + j] = (unsigned)run;
        run += t;
    }
    total[j] = (long long)run;
    nchunks[j] = (long long)((run + kCscChunk - 1) / kCscChunk);
}

// out[0..n] = exclusive prefix sums of in[0..n) (out[n] = total); one CTA of 1024 threads
__global__ void __launch_bounds__(1024) k_scan_exclusive(const long long* in, int n, long long* out) {
    __shared__ long long sh[32];
    __shared__ long long carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int base = 0; base < n; base += 1024) {
        const int q = base + threadIdx.x;
        const long long v = q < n ? in[q] : 0;
        long long s = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const long long t = __shfl_up_sync(kFull, s, o); if (lane >= o) s += t; }
        if (lane == 31) sh[warp] = s;
        __syncthreads();
        if (warp == 0) {
            long long w = sh[lane];
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { const long long t = __shfl_up_sync(kFull, w, o); if (lane >= o) w += t; }
            sh[lane] = w;
        }
        __syncthreads();
        const long long before = carry + (warp ? sh[warp - 1] : 0) + s - v;
        if (q < n) out[q] = before;
        __syncthreads();
        if (threadIdx.x == 1023) carry = before + v;
        __syncthreads();
    }
    if (threadIdx.x == 0) out[n] = carry;
}

// stable scatter: warp b walks its block in order, 32 positions at a time; equal items inside the 32 keep lane order
template <typename PT>
__global__ void k_csc_scatter(const int* __restrict__ idx, long long nnz, int J, long long nblocks, long long blk_len,
                              unsigned* table, const long long* __restrict__ col_ptr, PT* perm) {
    const long long b = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    if (b >= nblocks) return;
    const int lane = threadIdx.x & 31;
    const long long beg = b * blk_len, end = min(nnz, beg + blk_len);
    unsigned* row = table + b * J;
    for (long long q0 = beg; q0 < end; q0 += 32) {
        const long long q = q0 + lane;
        const bool valid = q < end;
        const int j = valid ? idx[q] : J + lane;                    // padding lanes get distinct keys outside [0,J)
        const unsigned peers = __match_any_sync(kFull, j);
        const unsigned base = valid ? row[j] : 0u;
        __syncwarp();                                                // every peer has read the cursor before it moves
        if (valid) {
            const unsigned rank = __popc(peers & ((1u << lane) - 1u));
            perm[col_ptr[j] + base + rank] = (PT)q;
            if ((peers >> lane) == 1u) row[j] = base + __popc(peers);   // the highest peer lane advances the cursor
        }
        __syncwarp();
    }
}

// chunk_item[c] = item of reduction chunk c (chunk_ptr = exclusive scan of the per-item chunk counts)
__global__ void k_csc_chunk_items(const long long* __restrict__ chunk_ptr, int J, int* chunk_item) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= J) return;
    for (long long c = chunk_ptr[j]; c < chunk_ptr[j + 1]; ++c) chunk_item[c] = j;
}

// ---- per iteration ---------------------------------------------------------------------------------------------------

template <typename PT>
__global__ void __launch_bounds__(256) k_csc_reduce(const PT* __restrict__ perm, const long long* __restrict__ col_ptr,
                                                    const long long* __restrict__ chunk_ptr, const int* __restrict__ chunk_item,
                                                    long long nchunks, const float* __restrict__ a, const float* __restrict__ x,
                                                    int m, double* partial) {
    const int lane = threadIdx.x & 31;
    const long long warp0 = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const long long nwarps = ((long long)gridDim.x * blockDim.x) >> 5;
    for (long long c = warp0; c < nchunks; c += nwarps) {
        const int j = chunk_item[c];
        const long long beg = col_ptr[j] + (c - chunk_ptr[j]) * kCscChunk;
        const long long end = min(col_ptr[j + 1], beg + kCscChunk);
        double acc[4] = {0.0, 0.0, 0.0, 0.0};
        for (long long p = beg + lane; p < end; p += 32) {
            const long long pos = (long long)perm[p];
            const float xv = x[pos];
            if (xv != 0.0f) {
#pragma unroll
                for (int k = 0; k < 4; ++k) if (k < m) acc[k] = fma((double)a[pos * m + k], (double)xv, acc[k]);
            }
        }
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            if (k < m) {
                double v = acc[k];
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(kFull, v, o);
                if (lane == 0) partial[c * m + k] = v;
            }
        }
    }
}

// one warp per (item, family): chunk partials added in chunk order (lane-strided, then a fixed tree) -> fixed point
__global__ void __launch_bounds__(256) k_csc_combine(const long long* __restrict__ chunk_ptr, int J, int m,
                                                     const double* __restrict__ partial, double scale_s, unsigned long long* s_fix) {
    const int lane = threadIdx.x & 31;
    const long long q = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    if (q >= (long long)J * m) return;
    const int j = (int)(q / m), k = (int)(q % m);
    double v = 0.0;
    for (long long c = chunk_ptr[j] + lane; c < chunk_ptr[j + 1]; c += 32) v += partial[c * m + k];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(kFull, v, o);
    if (lane == 0) s_fix[q] = (unsigned long long)__double2ll_rn(v * scale_s);
}

__global__ void k_perm_widen(const unsigned* __restrict__ in, long long n, long long* out) {
    for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < n; q += (long long)gridDim.x * blockDim.x) out[q] = (long long)in[q];
}

// a4-a6 as a launch of its own (the CSC path; every other path runs finalize_block in the gradient kernel's epilogue)
// Launched with kBlockThreads threads: the same count as the gradient kernels' epilogue CTA, so the scalar reductions run in the
// same order and a sharded / two-phase evaluation gives the same bits as the fused one.
__global__ void __launch_bounds__(1024) k_finalize_only(const FinalizeParams f) {
    __shared__ double sh[kFinalizeScratchBytes / 8];
    finalize_block(f, sh, threadIdx.x, blockDim.x);
}

}  // namespace dualip_dev
