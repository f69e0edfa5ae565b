// bsh_kernels.cuh -- device kernels of the BinarySkyHough hot path for sm_100a (included by bsh_api.cu only).
//
//   peakgram_kernel            L176:   rho > rho_th -> bit-packed rows (coalesced / 128-bit loads + warp OR-reduce)
//   prep_table_kernel          builds the window table the accumulation kernels stage with TMA bulk copies, and the
//                              per-row peak fractions the threshold estimate uses
//   threshold_kernel           in-kernel emission threshold from the Poisson-binomial moments of the data
//   dtable_kernel              D[pix][i] = v_i.n_pix / c in canonical operation order (R-5)
//   stage1_unweighted_kernel   Eq. (15) track + bit-sliced carry-save count of up to 96 f0 bins per thread  (L223)
//   stage1_weighted_kernel     same track, FP32 weighted count                                            (L223, Eq. 22)
//   stage1_naive_kernel        diagnostic: one thread per template, one track evaluation per accumulation
//   bitonic_* / finalize_*     candidate sort by (statistic desc, index asc) and toplist records          (L217, L225)
//   rescore_kernel             count / weighted count of the toplist entries (warp per candidate)
//   stage2_kernel              Eq. (26) power statistic, warp per candidate                               (L227)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <utility>

#include "bsh_core.cuh"

namespace bsh {

constexpr int kChunk = 64;            // SFTs per shared-memory stage (2 unrolled blocks of 32)
constexpr int kStages = 2;
constexpr int kSmemHeader = 128;      // mbarriers live here
constexpr int kSortTile = 2048;       // RawCand per CTA in the shared-memory sort (32 KB)

// ---------------------------------------------------------------------------------------------------------------------
// small PTX wrappers: mbarrier + 1-D TMA bulk copy (global -> shared), SASS: UBLKCP + SYNCS
// ---------------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
#ifndef BSH_SPIN_DELAY
#define BSH_SPIN_DELAY 0
#endif
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
#if BSH_SPIN_DELAY == 0
    asm volatile(
        "{\n\t"
        ".reg .pred P1;\n\t"
        "WAIT_LOOP:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n\t"   // plain polling: a suspend-time hint or a
                                                                          // nanosleep back-off measured 5-10 % slower
        "@P1 bra WAIT_DONE;\n\t"
        "bra WAIT_LOOP;\n\t"
        "WAIT_DONE:\n\t"
        "}" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
#else
    // a failed poll is followed by a chain of dependent MUFU operations (a pipe the accumulation kernels leave idle): the
    // waiting warp then issues ~1 instruction per 20 cycles instead of spinning on the issue port the other warps need
    uint32_t ok;
    float x = 1.5f;
    for (;;) {
        asm volatile("{\n\t.reg .pred P1;\n\tmbarrier.try_wait.parity.shared::cta.b64 P1, [%1], %2;\n\tselp.u32 %0, 1, 0, P1;\n\t}"
                     : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
        if (ok) break;
#pragma unroll
        for (int d = 0; d < BSH_SPIN_DELAY; ++d) asm volatile("rsqrt.approx.ftz.f32 %0, %0;" : "+f"(x));
        if (x == 123.456f) break;                         // never true: keeps the chain live
    }
#endif
}
__device__ __forceinline__ void tma_bulk_g2s(void *smem_dst, const void *gmem_src, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(smem_dst)),
                 "l"(gmem_src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

// ---------------------------------------------------------------------------------------------------------------------
// Peakgram, L176.  One warp per 128 slab columns of one row when rows are 16-byte aligned (float4 loads, 4 compare bits
// per lane, OR-reduce inside groups of 8 lanes); otherwise one warp per 32 columns with a ballot.
// ---------------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) peakgram_vec4_kernel(const float *__restrict__ rho, int n_sft, int n_bins,
                                                            int64_t stride, float rho_th, uint32_t *__restrict__ peak,
                                                            int words_per_row)
{
    const int lane = threadIdx.x & 31;
    const int segs = (words_per_row + 3) >> 2;                               // 128-column segments per row
    const int64_t gw = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (gw >= (int64_t)n_sft * segs) return;
    const int i = (int)(gw / segs), seg = (int)(gw % segs);
    const int k0 = seg * 128 + lane * 4;
    uint32_t nib = 0u;
    if (k0 + 3 < n_bins) {
        const float4 v = *reinterpret_cast<const float4 *>(rho + (int64_t)i * stride + k0);
        nib = (v.x > rho_th ? 1u : 0u) | (v.y > rho_th ? 2u : 0u) | (v.z > rho_th ? 4u : 0u) | (v.w > rho_th ? 8u : 0u);
    } else {
        for (int c = 0; c < 4; ++c)
            if (k0 + c < n_bins && rho[(int64_t)i * stride + k0 + c] > rho_th) nib |= 1u << c;
    }
    uint32_t word = nib << (4 * (lane & 7));
    word |= __shfl_xor_sync(0xFFFFFFFFu, word, 1);
    word |= __shfl_xor_sync(0xFFFFFFFFu, word, 2);
    word |= __shfl_xor_sync(0xFFFFFFFFu, word, 4);
    const int wd = seg * 4 + (lane >> 3);
    if ((lane & 7) == 0 && wd < words_per_row) peak[(int64_t)i * words_per_row + wd] = word;
}

__global__ void __launch_bounds__(256) peakgram_scalar_kernel(const float *__restrict__ rho, int n_sft, int n_bins,
                                                              int64_t stride, float rho_th, uint32_t *__restrict__ peak,
                                                              int words_per_row)
{
    const int lane = threadIdx.x & 31;
    const int64_t gw = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (gw >= (int64_t)n_sft * words_per_row) return;
    const int i = (int)(gw / words_per_row), wd = (int)(gw % words_per_row);
    const int k = wd * 32 + lane;
    const bool on = k < n_bins && rho[(int64_t)i * stride + k] > rho_th;
    const uint32_t word = __ballot_sync(0xFFFFFFFFu, on);
    if (lane == 0) peak[(int64_t)i * words_per_row + wd] = word;
}

// ---------------------------------------------------------------------------------------------------------------------
// Window table + row statistics.  wtab[i][e] = row words [e - off_words, e - off_words + 4) of SFT i (zero outside the
// row, zero rows for the padding SFTs i >= n_sft).  stats[0] += w_i p_i, stats[1] += w_i^2 p_i (1 - p_i), with
// p_i the fraction of ones in row i: the Poisson-binomial mean and variance of a count whose track visits row i once.
// ---------------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) prep_table_kernel(const uint32_t *__restrict__ peak, int words_per_row, int n_sft,
                                                         int n_pad, int n_bins, int n_entries, int off_words,
                                                         const float *__restrict__ w, uint4 *__restrict__ wtab,
                                                         float *__restrict__ w_pad, double *__restrict__ stats)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    double s_mean = 0.0, s_var = 0.0;
    if (i < n_pad) {
        const int row_words = (n_bins + 31) >> 5;
        const uint32_t *row = peak + (int64_t)i * words_per_row;
        int ones = 0;
        for (int e = 0; e < n_entries; ++e) {
            uint32_t v[4];
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                const int wd = e + c - off_words;
                v[c] = (i < n_sft && wd >= 0 && wd < row_words) ? row[wd] : 0u;
            }
            wtab[(int64_t)i * n_entries + e] = make_uint4(v[0], v[1], v[2], v[3]);
        }
        if (i < n_sft)
            for (int wd = 0; wd < row_words; ++wd) ones += __popc(row[wd]);
        const float wi = (i < n_sft) ? (w ? w[i] : 1.0f) : 0.0f;
        if (w_pad) w_pad[i] = wi;
        const double p = (double)ones / (double)n_bins;
        s_mean = (double)wi * p;
        s_var = (double)wi * (double)wi * p * (1.0 - p);
    }
    // block reduce, one atomic pair per block
    __shared__ double sh[2][8];
    for (int o = 16; o > 0; o >>= 1) {
        s_mean += __shfl_xor_sync(0xFFFFFFFFu, s_mean, o);
        s_var += __shfl_xor_sync(0xFFFFFFFFu, s_var, o);
    }
    if ((threadIdx.x & 31) == 0) { sh[0][threadIdx.x >> 5] = s_mean; sh[1][threadIdx.x >> 5] = s_var; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double a = 0.0, b = 0.0;
        for (int k = 0; k < (int)(blockDim.x >> 5); ++k) { a += sh[0][k]; b += sh[1][k]; }
        atomicAdd(&stats[0], a);
        atomicAdd(&stats[1], b);
    }
}

struct Threshold {
    int32_t tau_i;      // unweighted: emit when count >= tau_i
    float tau_f;        // weighted:   emit when n_w   >= tau_f
    float mean, sigma;  // of the noise model                                   (the host reads back these first 16 bytes)
    // Massive ties at the cut (more templates AT the k-th value than the candidate buffer holds: a cleaned / notched band,
    // constant rows, very few SFTs): of the templates whose statistic has exactly the bit pattern tie_key only those with
    // template index < tie_limit are candidates -- the order is (value desc, index asc), so the lowest indices are the
    // ones a toplist can need.  A normal pass has tie_limit = 2^64 - 1: nothing is held back.
    uint32_t tie_key;
    uint32_t pad;
    uint64_t tie_limit;
};
constexpr size_t kThresholdHostBytes = 16;

// First pass: tau = mean + z sigma with z from the normal tail for the wanted survivor fraction, minus a safety margin.
// When too few or too many templates pass, the host (bsh_stage1_collect) searches for the threshold and re-runs with
// fixed != 0: tau_i / tau_f / tie_key / tie_limit as given (stats -> n_passes).
__global__ void threshold_kernel(const double *__restrict__ stats, double frac, int emit_all, int fixed, int32_t fixed_tau_i,
                                 float fixed_tau_f, uint32_t tie_key, uint64_t tie_limit, Threshold *__restrict__ out)
{
    const double mean = stats[0], sigma = sqrt(stats[1] > 0.0 ? stats[1] : 0.0);
    double z = -1.0e30;
    if (!emit_all && frac < 0.5) z = -normcdfinv(frac) - 0.4;
    const double tau = emit_all ? -1.0e30 : mean + z * sigma;
    out->mean = (float)mean;
    out->sigma = (float)sigma;
    out->tau_f = tau < -1.0e29 ? -3.0e38f : (float)tau;
    out->tau_i = tau < -1.0e29 ? -(1 << 30) : (int32_t)floor(tau);
    if (fixed && !emit_all) {
        out->tau_f = fixed_tau_f;
        out->tau_i = fixed_tau_i;
    }
    out->tie_key = tie_key;
    out->pad = 0u;
    out->tie_limit = tie_limit;
}

// A template that passed the threshold goes into the candidate buffer (key = the count, or the bits of the FP32 weighted
// count) -- unless it is one of the ties held back by tie_limit.  cand_count counts every survivor, also those beyond the
// buffer's capacity: the host sees the overflow there.
__device__ __forceinline__ void emit_survivor(const Threshold *__restrict__ thr, RawCand *__restrict__ cand,
                                              unsigned int *__restrict__ cand_count, unsigned int cand_cap, uint64_t index,
                                              uint32_t key)
{
    if (key == thr->tie_key && index >= thr->tie_limit) return;
    const unsigned int pos = atomicAdd(cand_count, 1u);
    if (pos < cand_cap) {
        RawCand rc;
        rc.index = index;
        rc.key = key;
        rc.pad = 0u;
        cand[pos] = rc;
    }
}

// ---------------------------------------------------------------------------------------------------------------------
// D table (R-5): D = fl(fl(fl(vx nx) + fl(vy ny)) + fl(vz nz)).  Layout [n_groups][n_pad][R]; padding SFTs get 0 and
// padding pixels repeat the last real pixel (their results are never written out).
// ---------------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) dtable_kernel(const double *__restrict__ v_over_c, const double *__restrict__ nvec,
                                                     int n_sft, int n_pad, int n_pix, int n_groups, int R,
                                                     double *__restrict__ dtab)
{
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t total = (int64_t)n_groups * n_pad * R;
    if (t >= total) return;
    const int r = (int)(t % R);
    const int i = (int)((t / R) % n_pad);
    const int g = (int)(t / ((int64_t)R * n_pad));
    int pix = g * R + r;
    if (pix >= n_pix) pix = n_pix - 1;
    double D = 0.0;
    if (i < n_sft) {
        const double a = __dmul_rn(v_over_c[3 * i + 0], nvec[3 * pix + 0]);
        const double b = __dmul_rn(v_over_c[3 * i + 1], nvec[3 * pix + 1]);
        const double c = __dmul_rn(v_over_c[3 * i + 2], nvec[3 * pix + 2]);
        D = __dadd_rn(__dadd_rn(a, b), c);
    }
    dtab[t] = D;
}

// ---------------------------------------------------------------------------------------------------------------------
// Stage-1 accumulation kernels
// ---------------------------------------------------------------------------------------------------------------------
struct Stage1Params {
    const uint4 *wtab;          // [n_pad][n_entries]
    const double2 *cs;          // [n_P][n_pad]  (cos, sin)(Omega_p t_i)
    const double *dtab;         // [n_groups][n_pad][R]
    const float *w_pad;         // [n_pad]
    const double *A;            // [n_ap][n_P]   fl(a_p Omega_p)
    const double2 *casa;        // [n_P][n_tasc] (cos, sin)(Omega_p t_asc)
    const double2 *ke;          // [n_tasc] (e cos omega, e sin omega) of the combined (t_asc, eccentricity) axis, or NULL
    int n_pad, n_entries, n_chunks;
    int n_pix, n_ap, n_P, n_tasc, n_f0;
    int j0, n_fj;               // f0 tile
    int n_groups, n_aq, n_aq_tiles;
    double u0;                  // k_band0 + j0
    int off, s_max, s_zero;     // table coordinates (see TrackConst)
    int list_cap;               // deferred-break list entries per (thread, pixel)
    const Threshold *thr;
    RawCand *cand;
    unsigned int *cand_count;
    unsigned int cand_cap;
    void *counts_full;          // int32 (unweighted) / float (weighted) [n_templates] or NULL
};

struct BlockCoord {
    int grp, ip, ia, it;
    bool active;
};

__device__ __forceinline__ BlockCoord block_coord(const Stage1Params &p)
{
    BlockCoord c;
    int b = blockIdx.x;
    const int tile = b % p.n_aq_tiles;
    b /= p.n_aq_tiles;
    c.ip = b % p.n_P;
    c.grp = b / p.n_P;
    int aq = tile * blockDim.x + threadIdx.x;
    c.active = aq < p.n_aq;
    if (!c.active) aq = p.n_aq - 1;
    c.ia = aq / p.n_tasc;
    c.it = aq - c.ia * p.n_tasc;
    return c;
}

__device__ __forceinline__ TrackConst make_track_const(const Stage1Params &p, const BlockCoord &c)
{
    TrackConst tc;
    tc.u0 = p.u0;
    tc.uL = p.u0 + (double)(p.n_fj - 1);
    tc.A = p.A[c.ia * p.n_P + c.ip];
    const double2 q = p.casa[c.ip * p.n_tasc + c.it];
    tc.CA = q.x;
    tc.SA = q.y;
    const double2 ke = p.ke ? p.ke[c.it] : make_double2(0.0, 0.0);
    tc.kap = ke.x;
    tc.eta = ke.y;
    tc.off = p.off;
    tc.magic = kMagic + (double)p.off;
    tc.s_max = p.s_max;
    tc.s_zero = p.s_zero;
    tc.n_fj = p.n_fj;
    return tc;
}

// The same, compiled out of line, for the weighted pixel-lane kernel (bsh_wpix.cuh): its epilogue tests 90 accumulators one
// after the other, and 90 inlined copies of the emission cost the kernel 10 registers and 296 bytes of spills in the hot
// loop (168 -> 158 registers, none spilled; config 3: 730 -> 644 ms per launch, profiles/r03_stage1_wpix_full.md).  The
// unweighted kernels keep the inline form: they lose nothing to it, and a toplist of a fraction N_C of the bank (L225)
// emits millions of survivors, where a call per survivor costs (27.8 -> 36.0 ms on the N_C = 5 % pass of config 2).
__device__ __noinline__ void emit_survivor_out_of_line(const Threshold *__restrict__ thr, RawCand *__restrict__ cand,
                                                       unsigned int *__restrict__ cand_count, unsigned int cand_cap,
                                                       uint64_t index, uint32_t key)
{
    emit_survivor(thr, cand, cand_count, cand_cap, index, key);
}

__device__ __forceinline__ void emit_candidate(const Stage1Params &p, uint64_t index, uint32_t key)
{
    emit_survivor(p.thr, p.cand, p.cand_count, p.cand_cap, index, key);
}

// Shared-memory staging of one chunk of kChunk SFTs: window-table rows, (cos, sin) rows of this period, D rows of this
// pixel group and (weighted only) the weights -- four 1-D TMA bulk copies completing on one mbarrier.
template <int R, bool WEIGHTED>
struct StageLayout {
    int wt_bytes, cs_bytes, d_bytes, w_bytes, stride;
    __device__ __host__ StageLayout(int n_entries)
    {
        wt_bytes = kChunk * n_entries * 16;
        cs_bytes = kChunk * 16;
        d_bytes = kChunk * R * 8;
        w_bytes = WEIGHTED ? kChunk * 4 : 0;
        stride = wt_bytes + cs_bytes + d_bytes + w_bytes;
    }
    __device__ __host__ int total() const { return kSmemHeader + kStages * stride; }
};

template <int R, bool WEIGHTED>
__device__ __forceinline__ void issue_chunk(const Stage1Params &p, const StageLayout<R, WEIGHTED> &L, unsigned char *stage,
                                            uint64_t *bar, int chunk, int ip, int grp)
{
    const int64_t i0 = (int64_t)chunk * kChunk;
    mbar_expect_tx(bar, (uint32_t)L.stride);
    tma_bulk_g2s(stage, p.wtab + i0 * p.n_entries, (uint32_t)L.wt_bytes, bar);
    tma_bulk_g2s(stage + L.wt_bytes, p.cs + (int64_t)ip * p.n_pad + i0, (uint32_t)L.cs_bytes, bar);
    tma_bulk_g2s(stage + L.wt_bytes + L.cs_bytes, p.dtab + ((int64_t)grp * p.n_pad + i0) * R, (uint32_t)L.d_bytes, bar);
    if (WEIGHTED) tma_bulk_g2s(stage + L.wt_bytes + L.cs_bytes + L.d_bytes, p.w_pad + i0, (uint32_t)L.w_bytes, bar);
}

// One SFT of the unrolled block: binary term once, then per pixel the window (or the zero window + a bit in brk[r] when
// the shift breaks inside the f0 tile) pushed into the carry-save tree at compile-time position K.
template <int K, int NW, int HP, int R, bool CLAMP>
__device__ __forceinline__ void sft_step_unweighted(const TrackConst &tc, const uint4 *wt, int n_entries,
                                                    const double2 *cs, const double *d, Counter<NW, HP> (&cnt)[R],
                                                    uint32_t (&brk)[R])
{
    const double2 c = cs[K];
    const double B = binary_term(tc, c.x, c.y);
    double Dv[R];
    if constexpr (R == 2) {
        const double2 dd = reinterpret_cast<const double2 *>(d)[K];
        Dv[0] = dd.x;
        Dv[1] = dd.y;
    } else {
#pragma unroll
        for (int r = 0; r < R; ++r) Dv[r] = d[K * R + r];
    }
#pragma unroll
    for (int r = 0; r < R; ++r) {
        bool b;
        const Win<NW> x = track_window_deferred<NW, CLAMP>(tc, wt + K * n_entries, Dv[r], B, b);
        brk[r] |= b ? (1u << K) : 0u;
        push<K, NW, HP>(cnt[r], x);
    }
}

template <int NW, int HP, int R, bool CLAMP, int... Ks>
__device__ __forceinline__ void block_unweighted(const TrackConst &tc, const uint4 *wt, int n_entries, const double2 *cs,
                                                 const double *d, Counter<NW, HP> (&cnt)[R], uint32_t (&brk)[R],
                                                 std::integer_sequence<int, Ks...>)
{
    (sft_step_unweighted<Ks, NW, HP, R, CLAMP>(tc, wt, n_entries, cs, d, cnt, brk), ...);
}

// Exact window of one deferred (pixel r, SFT i) read from the global tables, added by ripple carry.
template <int NW, int HP, int R, bool CLAMP>
__device__ __forceinline__ void fixup_from_global(const Stage1Params &p, const TrackConst &tc, const BlockCoord &bc, int r,
                                                  int i, Counter<NW, HP> &cnt)
{
    const double2 c = p.cs[(int64_t)bc.ip * p.n_pad + i];
    const double B = binary_term(tc, c.x, c.y);
    const double D = p.dtab[((int64_t)bc.grp * p.n_pad + i) * R + r];
    const Win<NW> x = track_window<NW, CLAMP>(tc, p.wtab + (int64_t)i * p.n_entries, D, B);
    add_window(cnt, x);
}

// Stage-1 unweighted accumulation (L223, L241-L247).  Block = (pixel group, period, tile of (a_p, t_asc) pairs);
// thread = one (a_p, t_asc) pair x R pixels x up to 32 NW f0 bins.  SFTs stream through shared memory in chunks of
// kChunk (TMA bulk copies, two stages).  Breaks are parked in a per-thread list in shared memory (uint16 SFT indices,
// cap entries per pixel) and resolved in bulk when some list in the block runs full, and at the end.
template <int NW, int HP, int R, bool CLAMP>
__global__ void __launch_bounds__(256, 2) stage1_unweighted_kernel(const Stage1Params p)
{
    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t *bars = reinterpret_cast<uint64_t *>(smem);
    const StageLayout<R, false> L(p.n_entries);
    const BlockCoord bc = block_coord(p);
    const TrackConst tc = make_track_const(p, bc);
    uint16_t *list = reinterpret_cast<uint16_t *>(smem + kSmemHeader + kStages * L.stride);
    const int cap = p.list_cap, tpb = blockDim.x, tid = threadIdx.x;

    if (tid == 0) {
        mbar_init(&bars[0], 1);
        mbar_init(&bars[1], 1);
        mbar_fence_init();
    }
    __syncthreads();
    if (tid == 0) issue_chunk<R, false>(p, L, smem + kSmemHeader, &bars[0], 0, bc.ip, bc.grp);

    Counter<NW, HP> cnt[R];
    int npend[R];
#pragma unroll
    for (int r = 0; r < R; ++r) { cnt[r].clear(); npend[r] = 0; }

    for (int c = 0; c < p.n_chunks; ++c) {
        const int s = c & 1;
        if (tid == 0 && c + 1 < p.n_chunks)
            issue_chunk<R, false>(p, L, smem + kSmemHeader + (s ^ 1) * L.stride, &bars[s ^ 1], c + 1, bc.ip, bc.grp);
        mbar_wait(&bars[s], (uint32_t)((c >> 1) & 1));
        const unsigned char *st = smem + kSmemHeader + s * L.stride;
        const uint4 *wt = reinterpret_cast<const uint4 *>(st);
        const double2 *cs = reinterpret_cast<const double2 *>(st + L.wt_bytes);
        const double *d = reinterpret_cast<const double *>(st + L.wt_bytes + L.cs_bytes);
        bool want_flush = false;
#pragma unroll 1
        for (int blk = 0; blk < kChunk / kBlock; ++blk) {
            uint32_t brk[R];
#pragma unroll
            for (int r = 0; r < R; ++r) brk[r] = 0u;
            block_unweighted<NW, HP, R, CLAMP>(tc, wt + blk * kBlock * p.n_entries, p.n_entries, cs + blk * kBlock,
                                               d + blk * kBlock * R, cnt, brk, std::make_integer_sequence<int, kBlock>{});
#pragma unroll
            for (int r = 0; r < R; ++r) {
                uint32_t m = brk[r];
                while (m) {
                    const int k = __ffs(m) - 1;
                    m &= m - 1;
                    const int i = c * kChunk + blk * kBlock + k;
                    if (npend[r] < cap) {
                        list[(r * cap + npend[r]) * tpb + tid] = (uint16_t)i;
                        npend[r] += 1;
                    } else {
                        fixup_from_global<NW, HP, R, CLAMP>(p, tc, bc, r, i, cnt[r]);   // list full: resolve now
                    }
                }
                want_flush |= npend[r] > (cap >> 1) + (cap >> 2);
            }
        }
        const bool flush = __syncthreads_or(want_flush) != 0 || c + 1 == p.n_chunks;
        if (flush) {
#pragma unroll
            for (int r = 0; r < R; ++r) {
                for (int n = 0; n < npend[r]; ++n)
                    fixup_from_global<NW, HP, R, CLAMP>(p, tc, bc, r, (int)list[(r * cap + n) * tpb + tid], cnt[r]);
                npend[r] = 0;
            }
        }
    }

    // epilogue: threshold in bit-sliced form, emit the (rare) survivors
    const int32_t tau = p.thr->tau_i;
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int pix = bc.grp * R + r;
        if (!bc.active || pix >= p.n_pix) continue;
        const uint64_t base =
            ((((uint64_t)pix * p.n_ap + bc.ia) * p.n_P + bc.ip) * p.n_tasc + bc.it) * (uint64_t)p.n_f0 + p.j0;
        const Win<NW> ge = count_ge(cnt[r], tau);
        int32_t *out = p.counts_full ? reinterpret_cast<int32_t *>(p.counts_full) + base : nullptr;
#pragma unroll
        for (int w = 0; w < NW; ++w) {
            if (out) {
                for (int b = 0; b < 32; ++b)
                    if (32 * w + b < p.n_fj) out[32 * w + b] = count_at(cnt[r], w, b);
            }
            uint32_t m = ge.x[w] & valid_mask(p.n_fj, w);
            while (m) {
                const int b = __ffs(m) - 1;
                m &= m - 1;
                emit_candidate(p, base + 32 * w + b, (uint32_t)count_at(cnt[r], w, b));
            }
        }
    }
}

template <int NW, bool CLAMP>
__global__ void __launch_bounds__(256, 1) stage1_weighted_kernel(const Stage1Params p)
{
    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t *bars = reinterpret_cast<uint64_t *>(smem);
    const StageLayout<1, true> L(p.n_entries);
    const BlockCoord bc = block_coord(p);
    const TrackConst tc = make_track_const(p, bc);

    if (threadIdx.x == 0) {
        mbar_init(&bars[0], 1);
        mbar_init(&bars[1], 1);
        mbar_fence_init();
    }
    __syncthreads();
    if (threadIdx.x == 0) issue_chunk<1, true>(p, L, smem + kSmemHeader, &bars[0], 0, bc.ip, bc.grp);

    float acc[32 * NW];
#pragma unroll
    for (int j = 0; j < 32 * NW; ++j) acc[j] = 0.0f;

    for (int c = 0; c < p.n_chunks; ++c) {
        const int s = c & 1;
        if (threadIdx.x == 0 && c + 1 < p.n_chunks)
            issue_chunk<1, true>(p, L, smem + kSmemHeader + (s ^ 1) * L.stride, &bars[s ^ 1], c + 1, bc.ip, bc.grp);
        mbar_wait(&bars[s], (uint32_t)((c >> 1) & 1));
        const unsigned char *st = smem + kSmemHeader + s * L.stride;
        const uint4 *wt = reinterpret_cast<const uint4 *>(st);
        const double2 *cs = reinterpret_cast<const double2 *>(st + L.wt_bytes);
        const double *d = reinterpret_cast<const double *>(st + L.wt_bytes + L.cs_bytes);
        const float *wv = reinterpret_cast<const float *>(st + L.wt_bytes + L.cs_bytes + L.d_bytes);
#pragma unroll 2
        for (int k = 0; k < kChunk; ++k) {
            const double2 csk = cs[k];
            const double B = binary_term(tc, csk.x, csk.y);
            const Win<NW> x = track_window<NW, CLAMP>(tc, wt + k * p.n_entries, d[k], B);
            accumulate_weighted<NW>(acc, x, wv[k]);
        }
        __syncthreads();
    }

    const float tau = p.thr->tau_f;
    const int pix = bc.grp;
    if (bc.active && pix < p.n_pix) {
        const uint64_t base =
            ((((uint64_t)pix * p.n_ap + bc.ia) * p.n_P + bc.ip) * p.n_tasc + bc.it) * (uint64_t)p.n_f0 + p.j0;
        float *out = p.counts_full ? reinterpret_cast<float *>(p.counts_full) + base : nullptr;
#pragma unroll
        for (int j = 0; j < 32 * NW; ++j) {
            if (j < p.n_fj) {
                if (out) out[j] = acc[j];
                if (acc[j] >= tau) emit_candidate(p, base + j, __float_as_uint(acc[j]));
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------------
// Canonical single-accumulation track (used by the naive, rescoring and stage-2 kernels): slab column or -1.
// ---------------------------------------------------------------------------------------------------------------------
struct TemplateCoord {
    int pix, ia, ip, it, j;
};

struct TrackTables {
    const double2 *cs;     // [n_P][n_pad]
    const double *dtab;    // [n_groups][n_pad][R]
    const double *A;       // [n_ap][n_P]
    const double2 *casa;   // [n_P][n_tasc]
    const double2 *ke;     // [n_tasc] (e cos omega, e sin omega), or NULL (circular orbits)
    const double2 *cs_t;   // [n_pad][n_P] transposed copy of cs for the one-thread-per-candidate kernels, or NULL
    int n_pad, R;
    int n_pix, n_ap, n_P, n_tasc, n_f0;
    int64_t k_band0;
    int m;                 // k_band0 - k_slab0
    int n_bins;
    int n_sft;
};

__device__ __forceinline__ TemplateCoord decode_template(const TrackTables &t, uint64_t idx)
{
    TemplateCoord c;
    c.j = (int)(idx % (uint64_t)t.n_f0);    idx /= (uint64_t)t.n_f0;
    c.it = (int)(idx % (uint64_t)t.n_tasc); idx /= (uint64_t)t.n_tasc;
    c.ip = (int)(idx % (uint64_t)t.n_P);    idx /= (uint64_t)t.n_P;
    c.ia = (int)(idx % (uint64_t)t.n_ap);   idx /= (uint64_t)t.n_ap;
    c.pix = (int)idx;
    return c;
}

struct TemplateConst {
    double A, CA, SA, u, kap, eta;
    const double2 *cs;
    const double *d;
    int d_stride, cs_stride, mj;
};

__device__ __forceinline__ TemplateConst template_const(const TrackTables &t, const TemplateCoord &c)
{
    TemplateConst k;
    k.A = t.A[c.ia * t.n_P + c.ip];
    const double2 q = t.casa[c.ip * t.n_tasc + c.it];
    k.CA = q.x;
    k.SA = q.y;
    const double2 ke = t.ke ? t.ke[c.it] : make_double2(0.0, 0.0);
    k.kap = ke.x;
    k.eta = ke.y;
    k.u = (double)(t.k_band0 + c.j);
    k.cs = t.cs_t ? t.cs_t + c.ip : t.cs + (int64_t)c.ip * t.n_pad;
    k.cs_stride = t.cs_t ? t.n_P : 1;
    k.d = t.dtab + ((int64_t)(c.pix / t.R) * t.n_pad) * t.R + (c.pix % t.R);
    k.d_stride = t.R;
    k.mj = t.m + c.j;
    return k;
}

// ECC = false: the grid is circular (Eq. 15), the eccentric terms are not even compiled in (as a run-time test of kap, eta the
// compiler evaluated both brackets and selected: 19 instead of 9 FP64 operations per evaluation in the large-list kernels)
template <bool ECC = true>
__device__ __forceinline__ int track_column(const TemplateConst &k, int i, int n_bins)
{
    const double2 cs = k.cs[(int64_t)i * k.cs_stride];
    const double B = dmul(k.A, ECC ? orbit_bracket(cs.x, cs.y, k.CA, k.SA, k.kap, k.eta)
                                   : dadd(dmul(cs.x, k.CA), dmul(cs.y, k.SA)));
    const double g = dsub(k.d[(int64_t)i * k.d_stride], B);
    const int col = shift_of(k.u, g, k.mj);
    return (col >= 0 && col < n_bins) ? col : -1;
}

// diagnostic kernel: one thread per template
__global__ void __launch_bounds__(256) stage1_naive_kernel(const TrackTables t, const uint32_t *__restrict__ peak,
                                                           int words_per_row, const float *__restrict__ w,
                                                           int weighted, uint64_t n_templates, const Threshold *thr,
                                                           RawCand *cand, unsigned int *cand_count,
                                                           unsigned int cand_cap, void *counts_full)
{
    const uint64_t idx = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= n_templates) return;
    const TemplateCoord c = decode_template(t, idx);
    const TemplateConst k = template_const(t, c);
    int n = 0;
    float nw = 0.0f;
    for (int i = 0; i < t.n_sft; ++i) {
        const int col = track_column(k, i, t.n_bins);
        if (col >= 0 && ((peak[(int64_t)i * words_per_row + (col >> 5)] >> (col & 31)) & 1u)) {
            n += 1;
            if (weighted) nw += w[i];
        }
    }
    bool pass;
    uint32_t key;
    if (weighted) {
        if (counts_full) reinterpret_cast<float *>(counts_full)[idx] = nw;
        pass = nw >= thr->tau_f;
        key = __float_as_uint(nw);
    } else {
        if (counts_full) reinterpret_cast<int32_t *>(counts_full)[idx] = n;
        pass = n >= thr->tau_i;
        key = (uint32_t)n;
    }
    if (pass) emit_survivor(thr, cand, cand_count, cand_cap, idx, key);
}

// ---------------------------------------------------------------------------------------------------------------------
// Candidate ordering: (key descending, index ascending).  Bitonic network over a power-of-two padded buffer; strides
// below kSortTile run in shared memory.
// ---------------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ bool cand_before(const RawCand &a, const RawCand &b)
{
    return a.key > b.key || (a.key == b.key && a.index < b.index);
}

// Pre-selection for the toplist (L217, L225): the k-th largest key of the n candidates is found by an MSB-first radix
// select (4 passes of 8 bits, 256-bin shared-memory histogram), then every candidate with key >= that value is copied
// to `out` (all ties AT the cut are kept, so the (key desc, index asc) order of R-11 is decided by the sort that
// follows).  One block; n <= 2^20.  out_count[0] = number of candidates kept (>= k).
__global__ void __launch_bounds__(1024) select_cut_kernel(const RawCand *__restrict__ cand, unsigned int n, unsigned int k,
                                                          RawCand *__restrict__ out, unsigned int *__restrict__ out_count)
{
    __shared__ unsigned int hist[256];
    __shared__ unsigned int s_prefix, s_k, s_n_out;
    __shared__ unsigned int s_min[32], s_max[32];
    // common leading bits of all keys need no pass (number counts of a patch differ in their low bits only, and a pass
    // over identical digits would serialise every shared-memory atomic on one address)
    unsigned int kmin = 0xFFFFFFFFu, kmax = 0u;
    for (unsigned int i = threadIdx.x; i < n; i += blockDim.x) {
        const unsigned int key = cand[i].key;
        kmin = key < kmin ? key : kmin;
        kmax = key > kmax ? key : kmax;
    }
    kmin = __reduce_min_sync(0xFFFFFFFFu, kmin);
    kmax = __reduce_max_sync(0xFFFFFFFFu, kmax);
    if ((threadIdx.x & 31) == 0) { s_min[threadIdx.x >> 5] = kmin; s_max[threadIdx.x >> 5] = kmax; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (unsigned int w = 1; w < (blockDim.x >> 5); ++w) {
            kmin = s_min[w] < kmin ? s_min[w] : kmin;
            kmax = s_max[w] > kmax ? s_max[w] : kmax;
        }
        const unsigned int diff = kmin ^ kmax;
        const int top = diff ? 31 - __clz(diff) : -1;    // highest bit in which two keys differ
        const int first_shift = top < 0 ? -8 : (top / 8) * 8;
        s_prefix = first_shift + 8 >= 32 ? 0u : (kmax & (0xFFFFFFFFu << (first_shift + 8)));
        s_k = k;
        s_n_out = 0u;
        s_min[0] = (unsigned int)(first_shift + 8);      // passes start below this bit
    }
    __syncthreads();
    for (int shift = (int)s_min[0] - 8; shift >= 0; shift -= 8) {
        for (unsigned int t = threadIdx.x; t < 256; t += blockDim.x) hist[t] = 0u;
        __syncthreads();
        const unsigned int prefix = s_prefix;
        const unsigned int hi_mask = shift == 24 ? 0u : (0xFFFFFFFFu << (shift + 8));
        for (unsigned int i = threadIdx.x; i < n; i += blockDim.x) {
            const unsigned int key = cand[i].key;
            if ((key & hi_mask) == prefix) atomicAdd(&hist[(key >> shift) & 255u], 1u);
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            unsigned int need = s_k, d = 255u;
            for (;; --d) {                               // digits above d hold fewer than `need` candidates
                if (hist[d] >= need || d == 0u) break;
                need -= hist[d];
            }
            s_k = need;
            s_prefix = prefix | (d << shift);
        }
        __syncthreads();
    }
    const unsigned int cut = s_prefix;
    for (unsigned int i = threadIdx.x; i < n; i += blockDim.x) {
        const RawCand rc = cand[i];
        if (rc.key >= cut) out[atomicAdd(&s_n_out, 1u)] = rc;
    }
    __syncthreads();
    if (threadIdx.x == 0) out_count[0] = s_n_out;
}

__global__ void pad_candidates_kernel(RawCand *buf, unsigned int n, unsigned int n_pow2)
{
    const unsigned int i = blockIdx.x * blockDim.x + threadIdx.x + n;
    if (i < n_pow2) {
        RawCand rc;
        rc.index = ~0ull;
        rc.key = 0u;
        rc.pad = 1u;                     // padding marker
        buf[i] = rc;
    }
}

__device__ __forceinline__ void bitonic_cmpx(RawCand &a, RawCand &b, bool up)
{
    // up: a must come before b
    if (cand_before(b, a) == up) {
        const RawCand t = a;
        a = b;
        b = t;
    }
}

// all (k, j) with k <= min(n, kSortTile) when k_lo == 2; or for one k > kSortTile the strides j < kSortTile
__global__ void __launch_bounds__(1024) bitonic_tile_kernel(RawCand *buf, unsigned int n, unsigned int k_lo,
                                                            unsigned int k_hi)
{
    __shared__ RawCand sh[kSortTile];
    const unsigned int base = blockIdx.x * kSortTile;
    for (unsigned int t = threadIdx.x; t < kSortTile; t += blockDim.x)
        if (base + t < n) sh[t] = buf[base + t];
    __syncthreads();
    for (unsigned int k = k_lo; k <= k_hi; k <<= 1) {
        unsigned int j = (k >> 1) < (unsigned)kSortTile ? (k >> 1) : (unsigned)kSortTile >> 1;
        for (; j > 0; j >>= 1) {
            for (unsigned int t = threadIdx.x; t < kSortTile / 2; t += blockDim.x) {
                const unsigned int lo = ((t & ~(j - 1)) << 1) | (t & (j - 1));
                const unsigned int hi = lo | j;
                if (base + hi < n) bitonic_cmpx(sh[lo], sh[hi], ((base + lo) & k) == 0);
            }
            __syncthreads();
        }
    }
    for (unsigned int t = threadIdx.x; t < kSortTile; t += blockDim.x)
        if (base + t < n) buf[base + t] = sh[t];
}

__global__ void __launch_bounds__(256) bitonic_global_kernel(RawCand *buf, unsigned int n, unsigned int k, unsigned int j)
{
    const unsigned int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n / 2) return;
    const unsigned int lo = ((t & ~(j - 1)) << 1) | (t & (j - 1));
    const unsigned int hi = lo | j;
    RawCand a = buf[lo], b = buf[hi];
    const bool up = (lo & k) == 0;
    if (cand_before(b, a) == up) {
        buf[lo] = b;
        buf[hi] = a;
    }
}

// toplist records from the sorted candidates
__global__ void finalize_top_kernel(const RawCand *__restrict__ sorted, int n_keep, int topk, int weighted,
                                    bsh_cand *__restrict__ top)
{
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= topk) return;
    bsh_cand o;
    o.index = 0;
    o.count = 0;
    o.wcount = 0.0f;
    o.power = 0.0f;
    o.flags = 0u;
    if (c < n_keep) {
        const RawCand rc = sorted[c];
        o.index = rc.index;
        if (weighted) o.wcount = __uint_as_float(rc.key);
        else o.count = (int32_t)rc.key;
        o.flags = 1u;
    }
    top[c] = o;
}

// ---------------------------------------------------------------------------------------------------------------------
// Warp per candidate: lanes take SFTs i = lane, lane + 32, ...; FP32 partial sums per lane in that order, then a fixed
// xor-shuffle tree (R-20).  rescore fills count / wcount from the peakgram, stage 2 fills power from rho (Eq. 26).
// ---------------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ float warp_sum(float v)
{
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, o);
    return v;
}
__device__ __forceinline__ int warp_sum_int(int v)
{
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, o);
    return v;
}

// One block of kCandThreads threads per candidate: thread t takes SFTs t, t + kCandThreads, ... in order, then a fixed
// xor-shuffle tree inside each warp and the warp partials in warp order (R-20: deterministic run to run).
constexpr int kCandThreads = 128;

__global__ void __launch_bounds__(kCandThreads) rescore_kernel(const TrackTables t, const uint32_t *__restrict__ peak,
                                                               int words_per_row, const float *__restrict__ w,
                                                               int weighted_rank, bsh_cand *__restrict__ cands, int n_cands)
{
    __shared__ int sh_n[kCandThreads / 32];
    __shared__ float sh_w[kCandThreads / 32];
    const int c = blockIdx.x;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (c >= n_cands) return;
    const TemplateCoord tc = decode_template(t, cands[c].index);
    const TemplateConst k = template_const(t, tc);
    int n = 0;
    float nw = 0.0f;
    for (int i = threadIdx.x; i < t.n_sft; i += kCandThreads) {
        const int col = track_column(k, i, t.n_bins);
        if (col >= 0 && ((peak[(int64_t)i * words_per_row + (col >> 5)] >> (col & 31)) & 1u)) {
            n += 1;
            nw += w ? w[i] : 1.0f;
        }
    }
    n = warp_sum_int(n);
    nw = warp_sum(nw);
    if (lane == 0) { sh_n[warp] = n; sh_w[warp] = nw; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int q = 1; q < kCandThreads / 32; ++q) { n += sh_n[q]; nw += sh_w[q]; }
        if (weighted_rank) {
            cands[c].count = n;                  // wcount keeps the value that ranked the template
        } else {
            cands[c].wcount = nw;                // count is already exact
        }
    }
}

__global__ void __launch_bounds__(kCandThreads) stage2_kernel(const TrackTables t, const float *__restrict__ rho,
                                                              int64_t stride, const float *__restrict__ w,
                                                              bsh_cand *__restrict__ cands, int n_cands)
{
    __shared__ float sh_p[kCandThreads / 32];
    const int c = blockIdx.x;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (c >= n_cands) return;
    const TemplateCoord tc = decode_template(t, cands[c].index);
    const TemplateConst k = template_const(t, tc);
    float pw = 0.0f;
    for (int i = threadIdx.x; i < t.n_sft; i += kCandThreads) {
        const int col = track_column(k, i, t.n_bins);
        if (col >= 0) {
            const float r = rho[(int64_t)i * stride + col];
            pw += (w ? w[i] : 1.0f) * r;
        }
    }
    pw = warp_sum(pw);
    if (lane == 0) sh_p[warp] = pw;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int q = 1; q < kCandThreads / 32; ++q) pw += sh_p[q];
        cands[c].power = pw;
        cands[c].flags |= 2u;
    }
}

// LARGE candidate lists (a fraction N_C of the bank, millions of candidates): one THREAD per candidate, the block's
// 256 candidates walk the SFTs together, so that row i of the power slab (or of the peakgram), D[.][i] and (cos, sin)[.][i]
// are fetched once per block and served to its threads by L1 -- with one block per candidate every gather pulls its own
// 32-byte sector through L2 (measured 2.4e11 gathers/s).  FP32 sums (R-20): partial sums over chunks of kRowChunk SFTs in
// SFT order, then the partials in chunk order.
constexpr int kRowChunk = 128;

// cs_t[i][p] = cs[p][i]: with the periods of one SFT contiguous (and D laid out [SFT][pixel]: dtable_kernel with R = n_pix),
// the table reads of a warp whose lanes hold different templates fall into a few cache lines per SFT instead of one each
__global__ void __launch_bounds__(256) transpose_cs_kernel(const double2 *__restrict__ cs, int n_P, int n_pad,
                                                           double2 *__restrict__ cs_t)
{
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (int64_t)n_P * n_pad) return;
    const int i = (int)(t / n_P), p = (int)(t % n_P);
    cs_t[t] = cs[(int64_t)p * n_pad + i];
}

#ifndef BSH_ROWS_MINB
#define BSH_ROWS_MINB 8        // 32 registers, 64 warps per SM: the kernels are latency-bound (measured on the N_C = 5 % list of config 2:
#endif                         // rescoring + stage 2 68 ms at 8 blocks per SM against 80 ms at the 5 the compiler picked; unroll 4 / 6 / 16: 84 / 89 / 89 ms)
#ifndef BSH_ROWS_UNROLL
#define BSH_ROWS_UNROLL 8
#endif
#define BSH_PRAGMA_(x) _Pragma(#x)
#define BSH_PRAGMA(x) BSH_PRAGMA_(x)
template <bool ECC>
__global__ void __launch_bounds__(256, BSH_ROWS_MINB) stage2_rows_kernel(const TrackTables t, const float *__restrict__ rho, int64_t stride,
                                                          const float *__restrict__ w, bsh_cand *__restrict__ cands, int n_cands)
{
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= n_cands) return;
    const TemplateCoord tc = decode_template(t, cands[c].index);
    const TemplateConst k = template_const(t, tc);
    float total = 0.0f;
    for (int i0 = 0; i0 < t.n_sft; i0 += kRowChunk) {
        const int i1 = i0 + kRowChunk < t.n_sft ? i0 + kRowChunk : t.n_sft;
        float part = 0.0f;
BSH_PRAGMA(unroll BSH_ROWS_UNROLL)
        for (int i = i0; i < i1; ++i) {                   // (unrolled: the loads of 8 SFTs are in flight together)
            const int col = track_column<ECC>(k, i, t.n_bins);
            const float r = __ldg(rho + (int64_t)i * stride + (col >= 0 ? col : 0));
            if (col >= 0) part += (w ? __ldg(w + i) : 1.0f) * r;
        }
        total += part;
    }
    cands[c].power = total;
    cands[c].flags |= 2u;
}

template <bool ECC>
__global__ void __launch_bounds__(256, BSH_ROWS_MINB) rescore_rows_kernel(const TrackTables t, const uint32_t *__restrict__ peak,
                                                           int words_per_row, const float *__restrict__ w, int weighted_rank,
                                                           bsh_cand *__restrict__ cands, int n_cands)
{
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= n_cands) return;
    const TemplateCoord tc = decode_template(t, cands[c].index);
    const TemplateConst k = template_const(t, tc);
    int n = 0;
    float total = 0.0f;
    for (int i0 = 0; i0 < t.n_sft; i0 += kRowChunk) {
        const int i1 = i0 + kRowChunk < t.n_sft ? i0 + kRowChunk : t.n_sft;
        float part = 0.0f;
BSH_PRAGMA(unroll BSH_ROWS_UNROLL)
        for (int i = i0; i < i1; ++i) {
            const int col = track_column<ECC>(k, i, t.n_bins);
            const uint32_t word = __ldg(peak + (int64_t)i * words_per_row + ((col >= 0 ? col : 0) >> 5));
            if (col >= 0 && ((word >> (col & 31)) & 1u)) {
                n += 1;
                part += w ? __ldg(w + i) : 1.0f;
            }
        }
        total += part;
    }
    if (weighted_rank) cands[c].count = n;
    else cands[c].wcount = total;
}

// stage-2 reorder by (power desc, index asc): pack to RawCand keys, sort, permute
__global__ void pack_power_keys_kernel(const bsh_cand *__restrict__ cands, int n, RawCand *__restrict__ keys)
{
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= n) return;
    RawCand rc;
    rc.index = cands[c].index;
    const float p = cands[c].power;
    // monotone map float -> uint32 (handles negative values although powers are non-negative)
    const uint32_t b = __float_as_uint(p);
    rc.key = (b & 0x80000000u) ? ~b : (b | 0x80000000u);
    rc.pad = (uint32_t)c;                 // source slot
    keys[c] = rc;
}

__global__ void permute_cands_kernel(const bsh_cand *__restrict__ src, const RawCand *__restrict__ keys, int n,
                                     bsh_cand *__restrict__ dst)
{
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= n) return;
    dst[c] = src[keys[c].pad];
}

}  // namespace bsh
