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
// One block per SFT row.  The row's powers are sorted once in shared memory (bitonic network on (key, position) pairs);
// the median of a window is then the (h + 1)-th entry, in ascending order, whose position lies inside the window:
// thread = output column, scanning the sorted positions (one broadcast shared-memory read per step) and stopping at the
// median -- on average half the row.  Selection only, so the median is exact whatever the order of equal keys.
// HBM traffic: 8 n_raw bytes in, 4 K + K / 8 bytes out per row; everything else stays on chip.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace bsh {

constexpr int kFrontThreads = 256;
constexpr int kFrontMaxRaw = 2048;                    // raw bins per row the shared-memory sort is sized for

__global__ void __launch_bounds__(kFrontThreads) normalise_peakgram_kernel(const float2 *__restrict__ sft, int n_raw,
                                                                            int64_t sft_stride, int window, float bias,
                                                                            float rho_th, float *__restrict__ rho,
                                                                            int64_t rho_stride, uint32_t *__restrict__ peak,
                                                                            int words_per_row, int n2)
{
    extern __shared__ __align__(16) unsigned char fsm[];
    uint64_t *keys = reinterpret_cast<uint64_t *>(fsm);                       // [n2]  (ordered power bits, position)
    float *pw = reinterpret_cast<float *>(fsm + (size_t)n2 * 8);              // [n_raw] powers by position
    uint32_t *spos = reinterpret_cast<uint32_t *>(fsm + (size_t)n2 * 8 + (size_t)n_raw * 4);   // [n_raw] positions, ascending power
    const int row = blockIdx.x, tid = threadIdx.x;
    const float2 *x = sft + (int64_t)row * sft_stride;

    for (int q = tid; q < n2; q += kFrontThreads) {
        uint64_t key = ~0ull;                                                 // padding sorts last
        if (q < n_raw) {
            const float2 v = x[q];
            const float p = __fadd_rn(__fmul_rn(v.x, v.x), __fmul_rn(v.y, v.y));   // |x|^2, Eq. (20) numerator
            pw[q] = p;
            const uint32_t b = (p != p) ? 0xFFFFFFFEu : __float_as_uint(p);   // p >= 0: the bit pattern is monotone; NaN last
            key = ((uint64_t)b << 32) | (uint32_t)q;
        }
        keys[q] = key;
    }
    __syncthreads();
    for (int k = 2; k <= n2; k <<= 1)
        for (int j = k >> 1; j > 0; j >>= 1) {
            for (int t = tid; t < (n2 >> 1); t += kFrontThreads) {
                const int lo = ((t & ~(j - 1)) << 1) | (t & (j - 1)), hi = lo | j;
                const uint64_t a = keys[lo], b = keys[hi];
                const bool up = (lo & k) == 0;
                if ((a > b) == up) { keys[lo] = b; keys[hi] = a; }
            }
            __syncthreads();
        }
    for (int q = tid; q < n_raw; q += kFrontThreads) spos[q] = (uint32_t)keys[q];
    __syncthreads();

    const int h = (window - 1) >> 1;
    const int K = n_raw - window + 1;
    const int k_words = (K + 31) >> 5;
    const int lane = tid & 31;
    for (int k0 = tid - lane; k0 < k_words * 32; k0 += kFrontThreads) {       // a warp takes 32 consecutive columns
        const int k = k0 + lane;
        const bool live = k < K;
        int cnt = 0, r = 0;
        uint32_t med_rank = 0;
        bool found = !live;
        while (!__all_sync(0xFFFFFFFFu, found)) {
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                const int rr = r + u;
                const uint32_t pos = rr < n_raw ? spos[rr] : 0xFFFFFFFFu;
                const bool in = (uint32_t)(pos - (uint32_t)k) < (uint32_t)window;
                cnt += in ? 1 : 0;
                if (in && !found && cnt == h + 1) { med_rank = (uint32_t)rr; found = true; }
            }
            r += 8;
            if (r >= n_raw) found = true;
        }
        bool bit = false;
        if (live) {
            const uint32_t mb = (uint32_t)(keys[med_rank] >> 32);
            const float med = mb == 0xFFFFFFFEu ? __uint_as_float(0x7FC00000u) : __uint_as_float(mb);
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
