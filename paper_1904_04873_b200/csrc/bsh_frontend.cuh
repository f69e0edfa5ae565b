// bsh_frontend.cuh -- front end of the search: complex SFT bins -> normalised powers -> peakgram, fused.
//
//   PAPER.md L167-L174, Eq. (20)-(21): rho_Jk = |x_Jk|^2 / <n_Jk>^2, "<n_Jk>^2 is usually estimated with a running median
//   over a number of frequency bins (usually 101 bins are used)";  L176: bit = rho > rho_th.
//
// Reading R-22: n_raw = K + window - 1 raw bins per SFT, slab column k = raw bin k + h, h = (window - 1) / 2
// (the caller supplies h wing bins on each side, so there is no edge rule);
//   p_q = fl32(fl32(re re) + fl32(im im));  med_k = (h + 1)-th smallest of p_k .. p_{k + window - 1} (NaN ranks last);
//   n2_k = fl32(med_k / bias);  rho_k = fl32(p_{k + h} / n2_k)        -- IEEE FP32 operations, no FMA, no fast division.
//
// One block of 256 threads per SFT row; everything after the load stays in shared memory:
//   1. every warp sorts runs of 32 powers in registers (bitonic network over __shfl_xor_sync on 64-bit (power bits, position)
//      keys: unique, so the order is total);
//   2. the rank of an element = sum over the runs of the number of smaller keys in that run (a 5-step binary search per run);
//      spos[rank] = position;
//   3. for every rank threshold 32 (b + 1) and every block of 32 positions: the ballot of "rank below the threshold" and its
//      running count -- so that "how many elements of window k rank below 32 b" is two table reads and a popcount;
//   4. thread = output column: binary search over b for the chunk of 32 ranks that holds the median, then at most 32 steps
//      through that chunk's positions.  A selection, so exact.
// (The first version sorted the row with a block-wide bitonic network, 45 barriers, and scanned half the sorted row per
// column: 1800 instead of ~500 instructions per thread, 0.25 ms at config-3 size.)
// HBM traffic: 8 n_raw bytes in, 4 K + K / 8 bytes out per row.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace bsh {

constexpr int kFrontThreads = 256;
constexpr int kFrontMaxRaw = 2048;                    // raw bins per row the shared-memory sort is sized for

// shared-memory bytes of a row of n_raw bins (n_runs = ceil(n_raw / 32) runs of 32)
__host__ __device__ constexpr size_t front_smem_bytes(int n_raw)
{
    const size_t nr = (size_t)((n_raw + 31) / 32);
    return nr * 32 * 8 * 2 + nr * 32 * 4 * 3 + nr * nr * 8;
}

__global__ void __launch_bounds__(kFrontThreads) normalise_peakgram_kernel(const float2 *__restrict__ sft, int n_raw,
                                                                            int64_t sft_stride, int window, float bias,
                                                                            float rho_th, float *__restrict__ rho,
                                                                            int64_t rho_stride, uint32_t *__restrict__ peak,
                                                                            int words_per_row)
{
    extern __shared__ __align__(16) unsigned char fsm[];
    const int nr = (n_raw + 31) >> 5, n32 = nr * 32;
    uint64_t *keys = reinterpret_cast<uint64_t *>(fsm);                       // [n32] (ordered power bits, position), by position
    uint64_t *sk = keys + n32;                                                // [n32] the same keys, each run of 32 sorted
    float *pw = reinterpret_cast<float *>(sk + n32);                          // [n32] powers by position
    uint32_t *spos = reinterpret_cast<uint32_t *>(pw + n32);                  // [n32] position of the element of rank r
    uint32_t *rnk = spos + n32;                                               // [n32] rank of the element at position p
    uint32_t *bm = rnk + n32;                                                 // [nr][nr] ballots: rank < 32 (b + 1), positions 32 pb ..
    uint32_t *bc = bm + nr * nr;                                              // [nr][nr] running count of those ballots before pb
    const int row = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const float2 *x = sft + (int64_t)row * sft_stride;

    // 1. load, |x|^2, keys; every warp sorts its runs in registers
    for (int run = warp; run < nr; run += kFrontThreads / 32) {
        const int q = run * 32 + lane;
        uint64_t key = ~0ull - (uint64_t)(n32 - q);                           // padding ranks last (still unique)
        float p = 0.0f;
        if (q < n_raw) {
            const float2 v = x[q];
            p = __fadd_rn(__fmul_rn(v.x, v.x), __fmul_rn(v.y, v.y));          // |x|^2, Eq. (20) numerator
            const uint32_t b = (p != p) ? 0xFFFFFFFEu : __float_as_uint(p);   // p >= 0: the bit pattern is monotone; NaN last
            key = ((uint64_t)b << 32) | (uint32_t)q;
        }
        pw[q] = p;
        keys[q] = key;
#pragma unroll
        for (int k = 2; k <= 32; k <<= 1)
#pragma unroll
            for (int j = k >> 1; j > 0; j >>= 1) {
                const uint64_t other = __shfl_xor_sync(0xFFFFFFFFu, key, j);
                const bool up = (lane & k) == 0, lower = (lane & j) == 0;
                const uint64_t mn = key < other ? key : other, mx = key < other ? other : key;
                key = (lower == up) ? mn : mx;
            }
        sk[q] = key;
    }
    __syncthreads();
    // 2. rank = number of smaller keys, run by run
    for (int q = tid; q < n32; q += kFrontThreads) {
        const uint64_t kq = keys[q];
        uint32_t r = 0;
        for (int run = 0; run < nr; ++run) {
            const uint64_t *s = sk + run * 32;
            int pos = 0;
#pragma unroll
            for (int st = 16; st > 0; st >>= 1)
                if (s[pos + st - 1] < kq) pos += st;
            if (s[pos] < kq) pos += 1;
            r += (uint32_t)pos;
        }
        rnk[q] = r;
        spos[r] = (uint32_t)q;
    }
    __syncthreads();
    // 3. ballots and their running counts
    for (int pb = warp; pb < nr; pb += kFrontThreads / 32) {
        const uint32_t r = rnk[pb * 32 + lane];
        for (int b = 0; b < nr; ++b) {
            const uint32_t m = __ballot_sync(0xFFFFFFFFu, r < 32u * (uint32_t)(b + 1));
            if (lane == 0) bm[b * nr + pb] = m;
        }
    }
    __syncthreads();
    for (int b = tid; b < nr; b += kFrontThreads) {
        uint32_t c = 0;
        for (int pb = 0; pb < nr; ++pb) {
            bc[b * nr + pb] = c;
            c += __popc(bm[b * nr + pb]);
        }
    }
    __syncthreads();

    // 4. the median of every window
    const int h = (window - 1) >> 1;
    const int K = n_raw - window + 1;
    const int k_words = (K + 31) >> 5;
    auto below = [&](int b, int p) -> int {                                   // elements at positions < p with rank < 32 (b + 1)
        const int pb = p >> 5;                                                // (p <= n_raw <= n32; p = n32 only when n_raw = n32)
        if (pb >= nr) return (int)(bc[b * nr + nr - 1] + __popc(bm[b * nr + nr - 1]));
        return (int)(bc[b * nr + pb] + __popc(bm[b * nr + pb] & ((1u << (p & 31)) - 1u)));
    };
    for (int k0 = tid - lane; k0 < k_words * 32; k0 += kFrontThreads) {       // a warp takes 32 consecutive columns
        const int k = k0 + lane;
        const bool live = k < K;
        bool bit = false;
        if (live) {
            int lo = -1, hi = nr - 1;                                         // count(lo) < h + 1 <= count(hi); count(-1) = 0
            while (hi - lo > 1) {
                const int mid = (lo + hi) >> 1;
                if (below(mid, k + window) - below(mid, k) >= h + 1) hi = mid; else lo = mid;
            }
            int cnt = lo >= 0 ? below(lo, k + window) - below(lo, k) : 0;
            uint32_t mpos = 0;
            for (int r = 32 * hi; r < 32 * hi + 32; ++r) {                    // the median is among the ranks of chunk hi
                const uint32_t pos = spos[r];
                if ((uint32_t)(pos - (uint32_t)k) < (uint32_t)window && ++cnt == h + 1) { mpos = pos; break; }
            }
            const float med = pw[mpos];
            const float n2v = __fdiv_rn(med, bias);                           // <n>^2, Eq. (21)
            const float rv = __fdiv_rn(pw[k + h], n2v);                       // Eq. (20)
            if (rho) rho[(int64_t)row * rho_stride + k] = rv;
            bit = rv > rho_th;                                                // L176, strict, NaN -> 0
        }
        const uint32_t word = __ballot_sync(0xFFFFFFFFu, bit);
        if (peak && lane == 0) peak[(int64_t)row * words_per_row + (k0 >> 5)] = word;
    }
    if (peak)
        for (int wd = k_words + tid; wd < words_per_row; wd += kFrontThreads) peak[(int64_t)row * words_per_row + wd] = 0u;
}

}  // namespace bsh
