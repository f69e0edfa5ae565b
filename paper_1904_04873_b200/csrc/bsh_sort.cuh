// bsh_sort.cuh -- stable LSD radix sort of candidate records by (key descending, index ascending) (R-11) for the LARGE
// toplists of SURVEY NEXT-1 (a fraction N_C = 5-10 % of all templates goes to stage 2: millions of candidates).
// The bitonic network of bsh_kernels.cuh needs log^2(n) / 2 passes over the buffer (276 for 2^23 records: 72 ms); this needs
// one pass per byte of the composite key that actually varies (5-8 passes: ~3 ms).
//
// One pass = radix_hist_kernel (per-tile digit histograms) -> radix_scan_kernel (exclusive scan, digit-major) ->
// radix_scatter_kernel (stable scatter: tiles are walked in order, 256 records at a time; the rank of a record among the
// equal digits of its group comes from __match_any_sync inside the warp and a per-digit prefix over the warps).
// Digit d of pass q: byte q of the index (ascending) for q < 8, byte q - 8 of the key, inverted, for q >= 8 (descending).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "bsh_core.cuh"

namespace bsh {

constexpr int kRadixThreads = 256;
constexpr int kRadixPerThread = 64;
constexpr int kRadixTile = kRadixThreads * kRadixPerThread;      // records per block

__device__ __forceinline__ uint32_t radix_digit(const RawCand &rc, int pass)
{
    return pass < 8 ? (uint32_t)(rc.index >> (8 * pass)) & 255u : 255u - ((rc.key >> (8 * (pass - 8))) & 255u);
}

// bits in which the records differ: out[0..1] = OR of (index ^ index_0), out[2] = OR of (key ^ key_0)
__global__ void __launch_bounds__(256) radix_diff_kernel(const RawCand *__restrict__ in, unsigned int n, unsigned int *out)
{
    const RawCand first = in[0];
    uint64_t di = 0;
    uint32_t dk = 0;
    for (unsigned int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const RawCand rc = in[i];
        di |= rc.index ^ first.index;
        dk |= rc.key ^ first.key;
    }
    const uint32_t lo = __reduce_or_sync(0xFFFFFFFFu, (uint32_t)di), hi = __reduce_or_sync(0xFFFFFFFFu, (uint32_t)(di >> 32));
    dk = __reduce_or_sync(0xFFFFFFFFu, dk);
    if ((threadIdx.x & 31) == 0) {
        if (lo) atomicOr(out + 0, lo);
        if (hi) atomicOr(out + 1, hi);
        if (dk) atomicOr(out + 2, dk);
    }
}

__global__ void __launch_bounds__(kRadixThreads) radix_hist_kernel(const RawCand *__restrict__ in, unsigned int n, int pass,
                                                                   unsigned int n_tiles, unsigned int *__restrict__ hist)
{
    __shared__ unsigned int h[256];
    h[threadIdx.x] = 0u;
    __syncthreads();
    const unsigned int base = blockIdx.x * kRadixTile;
    for (int q = 0; q < kRadixPerThread; ++q) {
        const unsigned int i = base + q * kRadixThreads + threadIdx.x;
        if (i < n) atomicAdd(&h[radix_digit(in[i], pass)], 1u);
    }
    __syncthreads();
    hist[threadIdx.x * n_tiles + blockIdx.x] = h[threadIdx.x];      // digit-major
}

// exclusive scan of m = 256 n_tiles counters, one block
__global__ void __launch_bounds__(1024) radix_scan_kernel(unsigned int *hist, unsigned int m)
{
    __shared__ unsigned int s_warp[32], s_base;
    if (threadIdx.x == 0) s_base = 0u;
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (unsigned int i0 = 0; i0 < m; i0 += 4096) {
        const unsigned int i = i0 + 4 * threadIdx.x;
        unsigned int v[4], t = 0u;
#pragma unroll
        for (int c = 0; c < 4; ++c) { v[c] = i + c < m ? hist[i + c] : 0u; t += v[c]; }
        unsigned int x = t;
        for (int d = 1; d < 32; d <<= 1) {
            const unsigned int y = __shfl_up_sync(0xFFFFFFFFu, x, d);
            if (lane >= d) x += y;
        }
        if (lane == 31) s_warp[warp] = x;
        __syncthreads();
        unsigned int o = s_base + x - t;
        for (int w = 0; w < warp; ++w) o += s_warp[w];
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            if (i + c < m) hist[i + c] = o;
            o += v[c];
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            unsigned int s = 0u;
            for (int w = 0; w < 32; ++w) s += s_warp[w];
            s_base += s;
        }
        __syncthreads();
    }
}

__global__ void __launch_bounds__(kRadixThreads) radix_scatter_kernel(const RawCand *__restrict__ in, unsigned int n, int pass,
                                                                      unsigned int n_tiles, const unsigned int *__restrict__ offs,
                                                                      RawCand *__restrict__ out)
{
    __shared__ unsigned int run[256];                     // next output slot of each digit for this tile
    __shared__ unsigned int wcnt[kRadixThreads / 32][256];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    run[threadIdx.x] = offs[threadIdx.x * n_tiles + blockIdx.x];
    const unsigned int base = blockIdx.x * kRadixTile;
    for (int q = 0; q < kRadixPerThread; ++q) {
        const unsigned int i = base + q * kRadixThreads + threadIdx.x;
        if (base + q * kRadixThreads >= n) break;         // uniform
#pragma unroll
        for (int w = 0; w < kRadixThreads / 32; ++w) wcnt[w][threadIdx.x] = 0u;
        __syncthreads();
        const bool live = i < n;
        RawCand rc;
        uint32_t d = 256u + lane;                         // dead lanes: a digit nobody shares
        if (live) { rc = in[i]; d = radix_digit(rc, pass); }
        const uint32_t peers = __match_any_sync(0xFFFFFFFFu, d);
        const uint32_t rank_in_warp = __popc(peers & ((1u << lane) - 1u));
        if (live && rank_in_warp == 0) wcnt[warp][d] = __popc(peers);
        __syncthreads();
        if (live) {
            unsigned int pos = run[d] + rank_in_warp;
            for (int w = 0; w < warp; ++w) pos += wcnt[w][d];
            out[pos] = rc;
        }
        __syncthreads();
        {
            unsigned int t = 0u;
#pragma unroll
            for (int w = 0; w < kRadixThreads / 32; ++w) t += wcnt[w][threadIdx.x];
            run[threadIdx.x] += t;
        }
        __syncthreads();
    }
}

}  // namespace bsh
