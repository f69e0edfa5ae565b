// bsh_pos.cuh -- stage-1 accumulation kernels over the POSITION TABLE (pre-shifted windows) for sm_100a.
//
// The funnel-shift kernels of bsh_kernels.cuh spend 4 of their ~15 integer-pipe operations per (pixel, binary template,
// SFT) triple on extracting a 96-bit window at an arbitrary bit offset.  Here the window of EVERY start position is
// precomputed once per patch (build_position_table_kernel: [N_pad][n_pos] entries of 16 bytes), streamed through shared
// memory in stages of kStageSfts SFTs by 1-D TMA bulk copies, and read with one 16-byte shared-memory load at
// row + position.  Blocks are 8 full warps; warp w of a block works on pixel group
// oct * WPB + w, so all warps share the staged table rows and the (cos, sin)(Omega_p t_i) rows, and the four SM
// sub-partitions carry the same number of warps.  There is no block-wide barrier in the SFT loop: a stage is refilled by
// whichever warp releases it last (shared-memory counter), and warps wait only on the stage's "full" mbarrier.
// Breaks of the rounded shift inside the f0 tile (R-7, ~1 % of triples) read the all-zero position and are appended,
// predicated, to a per-thread list in local memory; lists are resolved in bulk from the global tables.
//
//   PAPER.md L102 Eq. (15) track, L223 number count, L241-L247 "loop over the binary templates"; R-5, R-7.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <utility>

#include "bsh_kernels.cuh"

namespace bsh {

constexpr int kStageSfts = 16;        // SFTs per shared-memory stage (half an unrolled block of 32)
constexpr int kMaxStages = 6;
constexpr int kPosHeader = 128;       // full[kMaxStages] mbarriers + done[kMaxStages] counters
constexpr int kListCap = 120;         // deferred breaks per (thread, template or pixel); flushed when more than 88 are
                                      // pending (< 2^kFixPlanes windows per flush).  64 measured 25-30 % slower at 8000 SFTs:
                                      // a flush is a long latency-bound loop during which the block's other warps run
                                      // out of staged SFTs, so fewer and fuller flushes win
constexpr int kWarpsUnweighted = 8;   // warps per block = pixel groups per block
#ifndef BSH_W_UNROLL
#define BSH_W_UNROLL 16
#endif
constexpr int kWeightedUnroll = BSH_W_UNROLL;   // SFTs of a stage unrolled in the weighted kernel's inner loop
constexpr int kWarpsWeighted = 8;     // (4-warp blocks, 3 per SM, measured 25.5 ms against 22.1 ms on config 2)

// ---------------------------------------------------------------------------------------------------------------------
// Position table: ptab[i][p] = window words of SFT i starting at slab column (p - off_table), zero outside [0, K) and
// for the padding SFTs.  One thread per entry.
// ---------------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t row_word(const uint32_t *row, int row_words, int q)
{
    return (q >= 0 && q < row_words) ? row[q] : 0u;
}

__global__ void __launch_bounds__(256) build_position_table_kernel(const uint32_t *__restrict__ peak, int words_per_row,
                                                                   int n_sft, int n_pad, int n_bins, int n_pos,
                                                                   int off_table, int s_zero, uint4 *__restrict__ ptab)
{
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (int64_t)n_pad * n_pos) return;
    const int i = (int)(t / n_pos), p = (int)(t % n_pos);
    uint32_t v[3] = {0u, 0u, 0u};
    if (i < n_sft && p != s_zero) {
        const int row_words = (n_bins + 31) >> 5;
        const uint32_t *row = peak + (int64_t)i * words_per_row;
        const int c0 = p - off_table;                    // slab column of window bit 0 (may be negative)
        const int q0 = c0 >> 5, sh = c0 & 31;            // arithmetic shift: floor division
        uint32_t lo = row_word(row, row_words, q0);
#pragma unroll
        for (int w = 0; w < 3; ++w) {
            const uint32_t hi = row_word(row, row_words, q0 + w + 1);
            v[w] = __funnelshift_r(lo, hi, sh);
            lo = hi;
        }
    }
    ptab[t] = make_uint4(v[0], v[1], v[2], 0u);
}

// D table for the position kernels: dpos[oct][i][w][r] = v_i . n_pix / c (canonical order, R-5) for pixel
// (oct * WPB + w) * R + r; padding SFTs get 0, padding pixels repeat the last real pixel (never written out).
__global__ void __launch_bounds__(256) dtable_pos_kernel(const double *__restrict__ v_over_c, const double *__restrict__ nvec,
                                                         int n_sft, int n_pad, int n_pix, int n_oct, int WPB, int R,
                                                         double *__restrict__ dpos)
{
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t total = (int64_t)n_oct * n_pad * WPB * R;
    if (t >= total) return;
    const int r = (int)(t % R);
    const int w = (int)((t / R) % WPB);
    const int i = (int)((t / ((int64_t)R * WPB)) % n_pad);
    const int oct = (int)(t / ((int64_t)R * WPB * n_pad));
    int pix = (oct * WPB + w) * R + r;
    if (pix >= n_pix) pix = n_pix - 1;
    double D = 0.0;
    if (i < n_sft) {
        const double a = __dmul_rn(v_over_c[3 * i + 0], nvec[3 * pix + 0]);
        const double b = __dmul_rn(v_over_c[3 * i + 1], nvec[3 * pix + 1]);
        const double c = __dmul_rn(v_over_c[3 * i + 2], nvec[3 * pix + 2]);
        D = __dadd_rn(__dadd_rn(a, b), c);
    }
    dpos[t] = D;
}

struct PosParams {
    const uint4 *ptab;          // [n_pad][n_pos]
    const double2 *cs;          // [n_P][n_pad]  (cos, sin)(Omega_p t_i)
    const double *dpos;         // [n_oct][n_pad][WPB][R]
    const float *w_pad;         // [n_pad]
    const double *A;            // [n_ap][n_P]
    const double2 *casa;        // [n_P][n_tasc]
    const double2 *ke;          // [n_tasc] (e cos omega, e sin omega), or NULL (circular orbits)
    int n_pad, n_pos, n_chunks, n_stages;
    int n_pix, n_ap, n_P, n_tasc, n_f0;
    int j0, n_fj;               // f0 tile
    int n_groups, n_oct, n_aq, n_aq_tiles;
    double u0;                  // k_band0 + j0
    int off, s_max, s_zero;     // position coordinates (TrackConst)
    const Threshold *thr;
    RawCand *cand;
    unsigned int *cand_count;
    unsigned int cand_cap;
    void *counts_full;
};

struct PosCoord {
    int oct, ip, ia, it, warp, lane, group, n_active;
    bool active;                // this lane's (a_p, t_asc) pair exists
};

__device__ __forceinline__ PosCoord pos_coord(const PosParams &p, int WPB)
{
    PosCoord c;
    int b = blockIdx.x;
    const int tile = b % p.n_aq_tiles;
    b /= p.n_aq_tiles;
    c.ip = b % p.n_P;
    c.oct = b / p.n_P;
    c.warp = threadIdx.x >> 5;
    c.lane = threadIdx.x & 31;
    c.group = c.oct * WPB + c.warp;
    const int rest = p.n_groups - c.oct * WPB;
    c.n_active = rest < WPB ? rest : WPB;
    int aq = tile * 32 + c.lane;
    c.active = aq < p.n_aq;
    if (!c.active) aq = p.n_aq - 1;
    c.ia = aq / p.n_tasc;
    c.it = aq - c.ia * p.n_tasc;
    return c;
}

__device__ __forceinline__ TrackConst pos_track_const(const PosParams &p, const PosCoord &c)
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

// Shared-memory stage: position rows, (cos, sin) rows, D rows of the block's WPB pixel groups, weights.
template <int WPB, int R, bool WEIGHTED>
struct PosStage {
    int tab_bytes, cs_bytes, d_bytes, w_bytes, stride;
    __device__ __host__ PosStage(int n_pos)
    {
        tab_bytes = kStageSfts * n_pos * 16;
        cs_bytes = kStageSfts * 16;
        d_bytes = kStageSfts * WPB * R * 8;
        w_bytes = WEIGHTED ? kStageSfts * 4 : 0;
        stride = tab_bytes + cs_bytes + d_bytes + w_bytes;
    }
    __device__ __host__ int total(int n_stages) const { return kPosHeader + n_stages * stride; }
};

template <int WPB, int R, bool WEIGHTED>
__device__ __forceinline__ void pos_issue(const PosParams &p, const PosStage<WPB, R, WEIGHTED> &L, unsigned char *stage,
                                          uint64_t *bar, int chunk, int ip, int oct)
{
    const int64_t i0 = (int64_t)chunk * kStageSfts;
    mbar_expect_tx(bar, (uint32_t)L.stride);
    tma_bulk_g2s(stage, p.ptab + i0 * p.n_pos, (uint32_t)L.tab_bytes, bar);
    tma_bulk_g2s(stage + L.tab_bytes, p.cs + (int64_t)ip * p.n_pad + i0, (uint32_t)L.cs_bytes, bar);
    tma_bulk_g2s(stage + L.tab_bytes + L.cs_bytes, p.dpos + ((int64_t)oct * p.n_pad + i0) * (WPB * R), (uint32_t)L.d_bytes,
                 bar);
    if (WEIGHTED)
        tma_bulk_g2s(stage + L.tab_bytes + L.cs_bytes + L.d_bytes, p.w_pad + i0, (uint32_t)L.w_bytes, bar);
}

// A warp is done with `stage`: the warp that releases it last refills it with chunk c + n_stages.
template <int WPB, int R, bool WEIGHTED>
__device__ __forceinline__ void pos_release(const PosParams &p, const PosStage<WPB, R, WEIGHTED> &L, unsigned char *smem,
                                            int st, int c, const PosCoord &pc)
{
    __syncwarp();
    if (pc.lane == 0) {
        unsigned int *done = reinterpret_cast<unsigned int *>(smem + 8 * kMaxStages) + st;
        unsigned int old;
        asm volatile("atom.acq_rel.cta.shared.add.u32 %0, [%1], 1;" : "=r"(old) : "r"(smem_u32(done)) : "memory");
        if ((old + 1u) % (unsigned)pc.n_active == 0u && c + p.n_stages < p.n_chunks)
            pos_issue<WPB, R, WEIGHTED>(p, L, smem + kPosHeader + st * L.stride, reinterpret_cast<uint64_t *>(smem) + st,
                                        c + p.n_stages, pc.ip, pc.oct);
    }
}

// ---------------------------------------------------------------------------------------------------------------------
// Unweighted number count (L223): thread = one (a_p, t_asc) pair x 2 pixels x up to 32 NW f0 bins, bit-sliced carry-save
// counters (bsh_core.cuh).  One SFT of the unrolled block of 32: binary term once, then per pixel the position (or the
// zero position + a list entry on a break) and one 16-byte load pushed into the tree at compile-time slot K.
// ---------------------------------------------------------------------------------------------------------------------
template <int K, int NW, int HP, bool CLAMP>
__device__ __forceinline__ void pos_step_unweighted(const TrackConst &tc, const uint4 *tab, int n_pos, const double2 *cs,
                                                    const double2 *dd, Counter<NW, HP> (&cnt)[2],
                                                    uint16_t (&list)[2][kListCap], int (&npend)[2], int i_block)
{
    constexpr int kk = K % kStageSfts;
    const double2 c = cs[kk];
    const double B = binary_term(tc, c.x, c.y);
    const double2 d2 = dd[kk * kWarpsUnweighted];
    const double Dv[2] = {d2.x, d2.y};
#pragma unroll
    for (int r = 0; r < 2; ++r) {
        bool b;
        const int32_t s = track_position_deferred<CLAMP>(tc, Dv[r], B, b);
        if (b) {
            list[r][npend[r]] = (uint16_t)(i_block + K);
            npend[r] += 1;
        }
        push<K, NW, HP>(cnt[r], load_position<NW>(tab + kk * n_pos, s));
    }
}

template <int K0, int NW, int HP, bool CLAMP, int... Ks>
__device__ __forceinline__ void pos_half_unweighted(const TrackConst &tc, const uint4 *tab, int n_pos, const double2 *cs,
                                                    const double2 *dd, Counter<NW, HP> (&cnt)[2],
                                                    uint16_t (&list)[2][kListCap], int (&npend)[2], int i_block,
                                                    std::integer_sequence<int, Ks...>)
{
    (pos_step_unweighted<K0 + Ks, NW, HP, CLAMP>(tc, tab, n_pos, cs, dd, cnt, list, npend, i_block), ...);
}

// exact window of one deferred (pixel r, SFT i) from the global tables, added by ripple carry
template <int NW, int HP, bool CLAMP>
__device__ __forceinline__ void pos_fixup_unweighted(const PosParams &p, const TrackConst &tc, const PosCoord &pc, int r,
                                                     int i, Counter<NW, HP> &cnt)
{
    const double2 c = p.cs[(int64_t)pc.ip * p.n_pad + i];
    const double B = binary_term(tc, c.x, c.y);
    const double D = p.dpos[(((int64_t)pc.oct * p.n_pad + i) * kWarpsUnweighted + pc.warp) * 2 + r];
    add_window(cnt, track_window_pos<NW, CLAMP>(tc, p.ptab + (int64_t)i * p.n_pos, D, B));
}

template <int NW, int HP, bool CLAMP>
__global__ void __launch_bounds__(32 * kWarpsUnweighted, 2) stage1_unweighted_pos_kernel(const PosParams p)
{
    extern __shared__ __align__(128) unsigned char smem[];
    constexpr int WPB = kWarpsUnweighted;
    uint64_t *full = reinterpret_cast<uint64_t *>(smem);
    const PosStage<WPB, 2, false> L(p.n_pos);
    const PosCoord pc = pos_coord(p, WPB);
    const TrackConst tc = pos_track_const(p, pc);

    if (threadIdx.x == 0) {
        for (int s = 0; s < kMaxStages; ++s) {
            mbar_init(&full[s], 1);
            reinterpret_cast<unsigned int *>(smem + 8 * kMaxStages)[s] = 0u;
        }
        mbar_fence_init();
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        const int n0 = p.n_stages < p.n_chunks ? p.n_stages : p.n_chunks;
        for (int s = 0; s < n0; ++s)
            pos_issue<WPB, 2, false>(p, L, smem + kPosHeader + s * L.stride, &full[s], s, pc.ip, pc.oct);
    }
    if (pc.group >= p.n_groups) return;                  // whole warp: no pixel group (n_active excludes it)

    Counter<NW, HP> cnt[2];
    uint16_t list[2][kListCap];
    int npend[2] = {0, 0};
    cnt[0].clear();
    cnt[1].clear();

    int st = 0;
    uint32_t parity = 0u;
    const int n_blocks = p.n_chunks >> 1;                // n_pad is a multiple of 32
    for (int blk = 0; blk < n_blocks; ++blk) {
        const int i_block = blk * kBlock;
        {
            mbar_wait(&full[st], parity);
            const unsigned char *sp = smem + kPosHeader + st * L.stride;
            pos_half_unweighted<0, NW, HP, CLAMP>(tc, reinterpret_cast<const uint4 *>(sp), p.n_pos,
                                                  reinterpret_cast<const double2 *>(sp + L.tab_bytes),
                                                  reinterpret_cast<const double2 *>(sp + L.tab_bytes + L.cs_bytes) + pc.warp,
                                                  cnt, list, npend, i_block, std::make_integer_sequence<int, kStageSfts>{});
            pos_release<WPB, 2, false>(p, L, smem, st, 2 * blk, pc);
            if (++st == p.n_stages) { st = 0; parity ^= 1u; }
        }
        {
            mbar_wait(&full[st], parity);
            const unsigned char *sp = smem + kPosHeader + st * L.stride;
            pos_half_unweighted<kStageSfts, NW, HP, CLAMP>(
                tc, reinterpret_cast<const uint4 *>(sp), p.n_pos, reinterpret_cast<const double2 *>(sp + L.tab_bytes),
                reinterpret_cast<const double2 *>(sp + L.tab_bytes + L.cs_bytes) + pc.warp, cnt, list, npend, i_block,
                std::make_integer_sequence<int, kStageSfts>{});
            pos_release<WPB, 2, false>(p, L, smem, st, 2 * blk + 1, pc);
            if (++st == p.n_stages) { st = 0; parity ^= 1u; }
        }
        // resolve the deferred breaks when some list of the warp could overflow in the next block, and at the end
        const bool want = npend[0] > kListCap - kBlock || npend[1] > kListCap - kBlock;
        if (__any_sync(0xFFFFFFFFu, want) || blk + 1 == n_blocks) {
#pragma unroll
            for (int r = 0; r < 2; ++r) {
                for (int n = 0; n < npend[r]; ++n) pos_fixup_unweighted<NW, HP, CLAMP>(p, tc, pc, r, (int)list[r][n], cnt[r]);
                npend[r] = 0;
            }
        }
    }

    // epilogue: threshold in bit-sliced form, emit the (rare) survivors
    const int32_t tau = p.thr->tau_i;
#pragma unroll
    for (int r = 0; r < 2; ++r) {
        const int pix = pc.group * 2 + r;
        if (!pc.active || pix >= p.n_pix) continue;
        const uint64_t base =
            ((((uint64_t)pix * p.n_ap + pc.ia) * p.n_P + pc.ip) * p.n_tasc + pc.it) * (uint64_t)p.n_f0 + p.j0;
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
                emit_survivor(p.thr, p.cand, p.cand_count, p.cand_cap, base + 32 * w + b, (uint32_t)count_at(cnt[r], w, b));
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------------
// Weighted number count (L223, Eq. 22): thread = one (a_p, t_asc) pair x 1 pixel x NB f0 bins, one FP32 accumulator per
// bin.  Summation order (R-20): SFT order for the SFTs whose shift is constant across the tile; the deferred (break)
// SFTs are added when their list is flushed -- fixed by the launch geometry, hence run-to-run deterministic.
// ---------------------------------------------------------------------------------------------------------------------
template <int NW, int NB>
__device__ __forceinline__ void accumulate_bins(float (&acc)[NB], const Win<NW> &x, float wi)
{
#pragma unroll
    for (int j = 0; j < NB; ++j)
        if ((x.x[j >> 5] >> (j & 31)) & 1u) acc[j] += wi;
}

template <int NW, int NB, bool CLAMP>
__global__ void __launch_bounds__(32 * kWarpsWeighted, 2) stage1_weighted_pos_kernel(const PosParams p)
{
    extern __shared__ __align__(128) unsigned char smem[];
    constexpr int WPB = kWarpsWeighted;
    uint64_t *full = reinterpret_cast<uint64_t *>(smem);
    const PosStage<WPB, 1, true> L(p.n_pos);
    const PosCoord pc = pos_coord(p, WPB);
    const TrackConst tc = pos_track_const(p, pc);

    if (threadIdx.x == 0) {
        for (int s = 0; s < kMaxStages; ++s) {
            mbar_init(&full[s], 1);
            reinterpret_cast<unsigned int *>(smem + 8 * kMaxStages)[s] = 0u;
        }
        mbar_fence_init();
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        const int n0 = p.n_stages < p.n_chunks ? p.n_stages : p.n_chunks;
        for (int s = 0; s < n0; ++s)
            pos_issue<WPB, 1, true>(p, L, smem + kPosHeader + s * L.stride, &full[s], s, pc.ip, pc.oct);
    }
    if (pc.group >= p.n_groups) return;

    float acc[NB];
#pragma unroll
    for (int j = 0; j < NB; ++j) acc[j] = 0.0f;
    uint16_t list[kListCap];
    int npend = 0;

    int st = 0;
    uint32_t parity = 0u;
    for (int c = 0; c < p.n_chunks; ++c) {
        mbar_wait(&full[st], parity);
        const unsigned char *sp = smem + kPosHeader + st * L.stride;
        const uint4 *tab = reinterpret_cast<const uint4 *>(sp);
        const double2 *cs = reinterpret_cast<const double2 *>(sp + L.tab_bytes);
        const double *d = reinterpret_cast<const double *>(sp + L.tab_bytes + L.cs_bytes) + pc.warp;
        const float *wv = reinterpret_cast<const float *>(sp + L.tab_bytes + L.cs_bytes + L.d_bytes);
#pragma unroll(kWeightedUnroll)
        for (int k = 0; k < kStageSfts; ++k) {
            const double2 csk = cs[k];
            const double B = binary_term(tc, csk.x, csk.y);
            bool b;
            const int32_t s = track_position_deferred<CLAMP>(tc, d[k * WPB], B, b);
            if (b) {
                list[npend] = (uint16_t)(c * kStageSfts + k);
                npend += 1;
            }
            accumulate_bins<NW, NB>(acc, load_position<NW>(tab + k * p.n_pos, s), wv[k]);
        }
        pos_release<WPB, 1, true>(p, L, smem, st, c, pc);
        if (++st == p.n_stages) { st = 0; parity ^= 1u; }
        if (__any_sync(0xFFFFFFFFu, npend > kListCap - kStageSfts) || c + 1 == p.n_chunks) {
            for (int n = 0; n < npend; ++n) {
                const int i = (int)list[n];
                const double2 ci = p.cs[(int64_t)pc.ip * p.n_pad + i];
                const double B = binary_term(tc, ci.x, ci.y);
                const double D = p.dpos[((int64_t)pc.oct * p.n_pad + i) * WPB + pc.warp];
                accumulate_bins<NW, NB>(acc, track_window_pos<NW, CLAMP>(tc, p.ptab + (int64_t)i * p.n_pos, D, B),
                                        p.w_pad[i]);
            }
            npend = 0;
        }
    }

    const float tau = p.thr->tau_f;
    const int pix = pc.group;
    if (pc.active && pix < p.n_pix) {
        const uint64_t base =
            ((((uint64_t)pix * p.n_ap + pc.ia) * p.n_P + pc.ip) * p.n_tasc + pc.it) * (uint64_t)p.n_f0 + p.j0;
        float *out = p.counts_full ? reinterpret_cast<float *>(p.counts_full) + base : nullptr;
#pragma unroll
        for (int j = 0; j < NB; ++j) {
            if (j < p.n_fj) {
                if (out) out[j] = acc[j];
                if (acc[j] >= tau) {
                    emit_survivor(p.thr, p.cand, p.cand_count, p.cand_cap, base + j, __float_as_uint(acc[j]));
                }
            }
        }
    }
}

}  // namespace bsh
