// bsh_wpix.cuh -- stage-1 WEIGHTED number count ("the weighted sum of 1s and 0s", weights Eq. 22)
// with SKY PIXELS ON THE LANES, sm_100a.  One pass over the band: the track of a (pixel, binary template, SFT) triple is
// evaluated ONCE and serves all its f0 bins.
//
// The method's work is one FP32 add per accumulation (template x SFT); this kernel is built so that little else is
// issued:
//   * thread = 1 pixel x 1 binary template x ALL f0 bins of the tile (up to 90 FP32 accumulators in registers);
//     warp = one binary template x 32 neighbouring pixels; block = kWpixWarps templates of one period;
//   * the window of peakgram bits a triple needs is read with ONE shared-memory load from a position table whose entries
//     hold 6 bins per byte (bin j = bit j % 6 of byte j / 6): ptxas turns the six `if (bit) acc += w` of a byte into one
//     R2P (register byte -> predicates P0..P5) + 6 predicated FADD, no shifts, no masks.  (7 bins per byte would need all
//     seven predicate registers: ptxas then keeps one for the break flag and extracts every 7th bin with LOP3 + ISETP --
//     measured 143 instead of 124 lane-instructions per triple; 15 bytes x 6 bins are exactly the 90 bins of a band);
//   * the binary term B = A (C CA + S SA) of Eq. (15) (L102) is the same for the 32 lanes: lane l computes the one of SFT
//     l & 15 of the stage and the warp shares them through shared memory; the hot loop has 6 FP64 operations per triple;
//   * the position offset is folded into the rounding constant (an EVEN integer added to 1.5 2^52 leaves the tie rule of
//     R-1 unchanged), so the low word of the magic add IS the table position;
//   * breaks of the rounded shift inside the f0 tile (R-7, ~1 % of triples) read the all-zero position and are noted in
//     a bit mask; masks become per-thread lists that the whole block resolves TOGETHER (one block barrier per 32 SFTs):
//     a flush is a latency-bound loop over L2 reads, and a lone flushing warp would stall the others on the stage ring.
// FP32 summation order (R-20): SFT order for the SFTs whose shift is constant across the tile; the break SFTs of a flush
// period follow in SFT order when the lists are flushed.  Fixed by the launch geometry: deterministic run to run.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <utility>

#include "bsh_pix.cuh"

namespace bsh {

#ifndef BSH_WPIX_WARPS
#define BSH_WPIX_WARPS 12
#endif
#ifndef BSH_WPIX_BPS
#define BSH_WPIX_BPS 1
#endif
constexpr int kWpixBlocksPerSm = BSH_WPIX_BPS;       // resident blocks per SM the kernel is built for (measured on config 2: 1 x 12
                                                     // warps 15.90 ms, 2 x 6 warps 16.16 ms, 3 x 4 warps 15.66 ms -- but with 3 blocks
                                                     // the wide tables of configs 3 and 5 leave no room for two stages)
constexpr int kWpixWarps = BSH_WPIX_WARPS;           // warps (= binary templates) per block; one block per SM
constexpr int kWpixHeader = 128 + kWpixWarps * kStageSfts * 8;   // mbarriers + one B buffer per warp

// BSH_WPIX_ROLL 1: one copy of the 16-SFT stage code serves both halves of a block of 32 (same speed as two copies, half the
// code).  Rolling further (groups of 2 / 4 / 8 SFTs) measured 23.4 / 18.8 / 19.1 ms against 15.9 ms on config 2: the
// look-ahead across the whole stage hides the load and FP64 latencies.
// Also measured and rejected: 3 bins per byte in alternating bit triples (R2P masks 0x0e / 0x70 write disjoint predicates, so
// the next R2P can issue before the adds of the previous byte): 30 R2P per triple instead of 15, 17.1 ms.
#ifndef BSH_WPIX_ROLL
#define BSH_WPIX_ROLL 1
#endif
constexpr int kWpixBits = 6;
#ifndef BSH_WPIX_SHIFT
#define BSH_WPIX_SHIFT 1
#endif
constexpr int kWpixShift = BSH_WPIX_SHIFT;           // bin b of a byte sits in bit kWpixShift + b: with bits 1..6 every R2P has the
                                                     // mask 0x7e (ptxas never takes bit 0 of a register into an R2P: it tests
                                                     // it with LOP3 + ISETP), and P0 stays free for the break flag
__host__ __device__ constexpr int wpix_bins(int nbytes) { return kWpixBits * nbytes; }
__host__ __device__ constexpr int wpix_entry_bytes(int nbytes) { return nbytes <= 8 ? 8 : 16; }
// The staged table is POSITION-MAJOR: the record of position p holds the entries of the stage's kStageSfts SFTs, plus one
// entry of padding, so that (i) the address of (SFT kk, position s) is s * record + kk * entry -- one multiply-add per
// triple, the SFT part an instruction immediate -- and (ii) neighbouring positions start 4 (2) banks apart: the 8 lanes
// a 16-byte (8-byte: 16 lanes) shared-memory wavefront serves read neighbouring positions without bank conflicts.
__host__ __device__ constexpr int wpix_record_bytes(int eb) { return (kStageSfts + 1) * eb; }
// bytes of one stage of the table (n_pos records), rounded up to the 16 bytes a bulk copy moves
__host__ __device__ constexpr int64_t wpix_stage_tab_bytes(int n_pos, int eb) { return ((int64_t)n_pos * wpix_record_bytes(eb) + 15) & ~(int64_t)15; }

// 6-bins-per-byte position table: entry p of SFT i = the window STARTING at table position p (slab column p - off_table),
// bin j in bit (j % 6) of byte (j / 6); bits outside [0, K), the padding SFTs and position s_zero are zero.
template <int EB>
__global__ void __launch_bounds__(256) build_position7_table_kernel(const uint32_t *__restrict__ peak, int words_per_row,
                                                                    int n_sft, int n_pad, int n_bins, int n_pos,
                                                                    int off_table, int s_zero, unsigned char *__restrict__ tab)
{
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (int64_t)n_pad * n_pos) return;
    const int i = (int)(t / n_pos), p = (int)(t % n_pos);
    uint32_t v[4] = {0u, 0u, 0u, 0u};                    // 128 contiguous window bits
    if (i < n_sft && p != s_zero) {
        const int row_words = (n_bins + 31) >> 5;
        const uint32_t *row = peak + (int64_t)i * words_per_row;
        const int c0 = p - off_table;
        const int q0 = c0 >> 5, sh = c0 & 31;
        uint32_t lo = row_word(row, row_words, q0);
#pragma unroll
        for (int w = 0; w < 4; ++w) {
            const uint32_t hi = row_word(row, row_words, q0 + w + 1);
            v[w] = __funnelshift_r(lo, hi, sh);
            lo = hi;
        }
    }
    uint32_t out[4] = {0u, 0u, 0u, 0u};
#pragma unroll
    for (int q = 0; q < EB; ++q) {                       // byte q <- window bits [6 q, 6 q + 6)
        const int b = kWpixBits * q, w = b >> 5, s = b & 31;
        uint32_t bits = v[w] >> s;
        if (s > 32 - kWpixBits && w + 1 < 4) bits |= v[w + 1] << (32 - s);
        out[q >> 2] |= (bits & ((1u << kWpixBits) - 1u)) << (8 * (q & 3) + kWpixShift);
    }
    unsigned char *dst = tab + (int64_t)(i / kStageSfts) * wpix_stage_tab_bytes(n_pos, EB) + (int64_t)p * wpix_record_bytes(EB) +
                         (i % kStageSfts) * EB;
    if (EB == 8) *reinterpret_cast<uint2 *>(dst) = make_uint2(out[0], out[1]);
    else *reinterpret_cast<uint4 *>(dst) = make_uint4(out[0], out[1], out[2], out[3]);
    if (i % kStageSfts == 0) {                           // the record's padding entry
        if (EB == 8) *reinterpret_cast<uint2 *>(dst + kStageSfts * EB) = make_uint2(0u, 0u);
        else *reinterpret_cast<uint4 *>(dst + kStageSfts * EB) = make_uint4(0u, 0u, 0u, 0u);
    }
}

// address of entry (SFT i, position s) in the global table
template <int EB>
__device__ __forceinline__ const unsigned char *entry7(const unsigned char *tab, int n_pos, int i, int s)
{
    return tab + (int64_t)(i / kStageSfts) * wpix_stage_tab_bytes(n_pos, EB) + (int64_t)s * wpix_record_bytes(EB) + (i % kStageSfts) * EB;
}

struct WpixParams {
    const unsigned char *tab7;  // [n_pad / kStageSfts] stages of [n_pos] records (position-major, see wpix_record_bytes)
    const double2 *cs;          // [n_P][n_pad]  (cos, sin)(Omega_p t_i)
    const double *dpix;         // [n_pg][n_pad / 2][32][2]
    const float *w_pad;         // [n_pad]
    const double *A;            // [n_ap][n_P]
    const double2 *casa;        // [n_P][n_tasc]
    const double2 *ke;          // [n_tasc] (e cos omega, e sin omega), or NULL (circular orbits)
    int n_pad, n_pos, n_chunks, n_stages;
    int n_pix, n_ap, n_P, n_tasc, n_f0;
    int j0, n_fj;               // f0 tile
    int n_pg, n_aq, n_aq_tiles;
    double u0;                  // k_band0 + j0
    int off, s_max, s_zero;     // position coordinates (TrackConst)
    const Threshold *thr;
    RawCand *cand;
    unsigned int *cand_count;
    unsigned int cand_cap;
    void *counts_full;
};

struct WpixStage {
    int tab_bytes, cs_bytes, d_bytes, w_bytes, stride;
    __device__ __host__ WpixStage(int n_pos, int eb)
    {
        tab_bytes = (int)wpix_stage_tab_bytes(n_pos, eb);
        cs_bytes = kStageSfts * 16;
        d_bytes = kStageSfts * 32 * 8;
        w_bytes = kStageSfts * 4;
        stride = tab_bytes + cs_bytes + d_bytes + w_bytes;
    }
    __device__ __host__ int total(int n_stages) const { return kWpixHeader + n_stages * stride; }
};

__device__ __forceinline__ void wpix_issue(const WpixParams &p, const WpixStage &L, unsigned char *stage, uint64_t *bar, int chunk,
                                           int ip, int pg)
{
    const int64_t i0 = (int64_t)chunk * kStageSfts;
    mbar_expect_tx(bar, (uint32_t)L.stride);
    tma_bulk_g2s(stage, p.tab7 + (int64_t)chunk * L.tab_bytes, (uint32_t)L.tab_bytes, bar);
    tma_bulk_g2s(stage + L.tab_bytes, p.cs + (int64_t)ip * p.n_pad + i0, (uint32_t)L.cs_bytes, bar);
    tma_bulk_g2s(stage + L.tab_bytes + L.cs_bytes, p.dpix + ((int64_t)pg * p.n_pad + i0) * 32, (uint32_t)L.d_bytes, bar);
    tma_bulk_g2s(stage + L.tab_bytes + L.cs_bytes + L.d_bytes, p.w_pad + i0, (uint32_t)L.w_bytes, bar);
}

// A warp is done with `stage`: the warp that releases it last refills it with chunk c + n_stages.
__device__ __forceinline__ void wpix_release(const WpixParams &p, const WpixStage &L, unsigned char *smem, int st, int c, int lane,
                                             int ip, int pg)
{
    __syncwarp();
    if (lane == 0) {
        unsigned int *done = reinterpret_cast<unsigned int *>(smem + 8 * kMaxStages) + st;
        unsigned int old;
        asm volatile("atom.acq_rel.cta.shared.add.u32 %0, [%1], 1;" : "=r"(old) : "r"(smem_u32(done)) : "memory");
        if ((old + 1u) % (unsigned)kWpixWarps == 0u && c + p.n_stages < p.n_chunks)
            wpix_issue(p, L, smem + kWpixHeader + st * L.stride, reinterpret_cast<uint64_t *>(smem) + st, c + p.n_stages, ip, pg);
    }
}

template <int NBYTES>
struct Win7 {
    uint32_t x[wpix_entry_bytes(NBYTES) / 4];
};

template <int NBYTES>
__device__ __forceinline__ Win7<NBYTES> load7(const unsigned char *entry)
{
    Win7<NBYTES> w;
    if (wpix_entry_bytes(NBYTES) == 8) {
        const uint2 e = *reinterpret_cast<const uint2 *>(entry);
        w.x[0] = e.x; w.x[1] = e.y;
    } else {
        const uint4 e = *reinterpret_cast<const uint4 *>(entry);
        w.x[0] = e.x; w.x[1] = e.y; w.x[2 % (wpix_entry_bytes(NBYTES) / 4)] = e.z; w.x[3 % (wpix_entry_bytes(NBYTES) / 4)] = e.w;
    }
    return w;
}

// acc[j] += wi for every bin j whose bit is set: bin j = bit (kWpixShift + j % 6) of byte (j / 6)  (one R2P + 6 predicated
// FADD per byte).  (An inline-PTX form with the accumulators as read-write operands removes the ~2 register copies per
// triple ptxas adds here, but costs 3 spill accesses per triple: measured 17.2 ms against 15.9 ms on config 2.)
template <int NBYTES>
__device__ __forceinline__ void accumulate7(float (&acc)[kWpixBits * NBYTES], const Win7<NBYTES> &x, float wi)
{
#pragma unroll
    for (int q = 0; q < NBYTES; ++q) {
        const uint32_t word = x.x[q >> 2];
#pragma unroll
        for (int b = 0; b < kWpixBits; ++b)
            if (word & (1u << (8 * (q & 3) + kWpixShift + b))) acc[kWpixBits * q + b] += wi;
    }
}

struct WpixConst {
    double u0, uL;
    double magic;               // 1.5 2^52 + (off rounded down to even): the low word of fl(y + magic) is position - (off & 1)
    int32_t off, s_max, s_zero;
};

// One SFT (slot K of the block of 32; KK = its row in the stage).
template <int K, int NBYTES, bool CLAMP>
__device__ __forceinline__ void wpix_step(const WpixConst &k, const unsigned char *tab, const double *bwarp,
                                          const double2 *dpair, const float *wv, float (&acc)[kWpixBits * NBYTES], uint32_t &brk)
{
    constexpr int kk = K % kStageSfts;
    constexpr int EB = wpix_entry_bytes(NBYTES);
    const double2 d2 = dpair[(kk >> 1) * 32];
    const double D = (kk & 1) ? d2.y : d2.x;
    const double g = __dsub_rn(D, bwarp[kk]);
    const double m0 = __dadd_rn(__dmul_rn(k.u0, g), k.magic);         // low word = round(fl(u0 g)) + even offset (R-1)
    const double mL = __dadd_rn(__dmul_rn(k.uL, g), k.magic);
    int32_t s;                                                        // table position - (off & 1)
    if (!CLAMP) {
        asm("{\n\t"
            ".reg .pred p;\n\t"
            "setp.neu.f64 p, %2, %3;\n\t"
            "@p or.b32 %0, %0, %4;\n\t"
            "selp.b32 %1, %5, %6, p;\n\t"
            "}"
            : "+r"(brk), "=r"(s)
            : "d"(m0), "d"(mL), "n"(1u << K), "r"(k.s_zero - (k.off & 1)), "r"(__double2loint(m0)));
    } else {
        const int32_t odd = k.off & 1;
        const int32_t s0 = clamp_s(__double2loint(m0) + odd, k.s_max);
        const int32_t sL = clamp_s(__double2loint(mL) + odd, k.s_max);   // equal after clamping => every bin reads 0
        const bool b = s0 != sL;
        brk |= b ? (1u << K) : 0u;
        s = (b ? k.s_zero : s0) - odd;
    }
    const unsigned char *entry = tab + (ptrdiff_t)s * wpix_record_bytes(EB) + kk * EB;   // tab: record of position (off & 1)
    accumulate7<NBYTES>(acc, load7<NBYTES>(entry), wv[kk]);
}

template <int K0, int NBYTES, bool CLAMP, int... Ks>
__device__ __forceinline__ void wpix_half(const WpixConst &k, const unsigned char *tab, const double *bwarp,
                                          const double2 *dpair, const float *wv, float (&acc)[kWpixBits * NBYTES], uint32_t &brk,
                                          std::integer_sequence<int, Ks...>)
{
    (wpix_step<K0 + Ks, NBYTES, CLAMP>(k, tab, bwarp, dpair, wv, acc, brk), ...);
}

// Exact window (6-bins-per-byte) of a (pixel, template, SFT) whose rounded shift differs between the two ends of the f0
// tile (R-7), from the global table: one break -> blend of the two neighbouring positions at the
// break bin (estimated, then corrected on the canonical evaluation itself); otherwise every bin from its own position.
template <int NBYTES, bool CLAMP>
__device__ __noinline__ Win7<NBYTES> exact_window7(const TrackConst &tc, const unsigned char *tab, int n_pos, int i, double D,
                                                   double B)
{
    constexpr int EB = wpix_entry_bytes(NBYTES);
    constexpr int NWORDS = EB / 4;
    const double g = dsub(D, B);
    const double y0 = dmul(tc.u0, g);
    const int32_t r0 = round_int(y0);
    const int32_t s0 = tc.off + r0;
    const int32_t sL = tc.off + round_int(dmul(tc.uL, g));
    const int32_t d = sL - s0;
    Win7<NBYTES> out;
    if (!CLAMP && (d == 1 || d == -1)) {
        const float dist = (float)(((double)r0 + (d > 0 ? 0.5 : -0.5)) - y0);
        int j = (int)ceilf(fast_divide(dist, (float)g));
        j = j < 1 ? 1 : (j > tc.n_fj - 1 ? tc.n_fj - 1 : j);
        while (j > 1 && tc.off + round_int(dmul(dadd(tc.u0, (double)(j - 1)), g)) != s0) --j;
        while (j < tc.n_fj - 1 && tc.off + round_int(dmul(dadd(tc.u0, (double)j), g)) == s0) ++j;
        const Win7<NBYTES> a = load7<NBYTES>(entry7<EB>(tab, n_pos, i, s0));
        const Win7<NBYTES> b = load7<NBYTES>(entry7<EB>(tab, n_pos, i, sL));
        const int pos = 8 * (j / kWpixBits) + (j % kWpixBits) + kWpixShift;   // bit position of bin j; bins >= j take the second window
#pragma unroll
        for (int w = 0; w < NWORDS; ++w) {
            const int rel = pos - 32 * w;
            const uint32_t m = rel <= 0 ? 0xFFFFFFFFu : (rel >= 32 ? 0u : (0xFFFFFFFFu << rel));
            out.x[w] = (a.x[w] & ~m) | (b.x[w] & m);
        }
        return out;
    }
#pragma unroll
    for (int w = 0; w < NWORDS; ++w) out.x[w] = 0u;
    for (int j = 0; j < tc.n_fj; ++j) {
        int32_t sj = tc.off + round_int(dmul(dadd(tc.u0, (double)j), g));
        sj = clamp_s(sj, tc.s_max);                      // identity in the unclamped geometry (proven range)
        const int pos = 8 * (j / kWpixBits) + (j % kWpixBits) + kWpixShift;
        const uint32_t word = reinterpret_cast<const uint32_t *>(entry7<EB>(tab, n_pos, i, sj))[pos >> 5];
        const uint32_t bit = (word >> (pos & 31)) & 1u;
#pragma unroll
        for (int w = 0; w < NWORDS; ++w)
            if ((pos >> 5) == w) out.x[w] |= bit << (pos & 31);
    }
    return out;
}

template <int NBYTES, bool CLAMP>
__global__ void __launch_bounds__(32 * kWpixWarps, kWpixBlocksPerSm) stage1_weighted_pix_kernel(const WpixParams p)
{
    extern __shared__ __align__(128) unsigned char smem[];
    constexpr int NB = kWpixBits * NBYTES;
    constexpr int EB = wpix_entry_bytes(NBYTES);
    uint64_t *full = reinterpret_cast<uint64_t *>(smem);
    const WpixStage L(p.n_pos, EB);
    int b = blockIdx.x;
    const int tile = b % p.n_aq_tiles;
    b /= p.n_aq_tiles;
    const int ip = b % p.n_P;
    const int pg = b / p.n_P;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    double *bwarp = reinterpret_cast<double *>(smem + 128) + warp * kStageSfts;      // [16 SFTs] binary terms of this warp

    // the warp's binary template (an (a_p, t_asc) pair of period ip); a missing one repeats the last real pair
    int aq = tile * kWpixWarps + warp;
    const bool act = aq < p.n_aq;
    if (!act) aq = p.n_aq - 1;
    const int ia = aq / p.n_tasc, it = aq - ia * p.n_tasc;
    const double A_d = p.A[ia * p.n_P + ip];
    const double2 q_d = p.casa[ip * p.n_tasc + it];

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
        for (int s = 0; s < n0; ++s) wpix_issue(p, L, smem + kWpixHeader + s * L.stride, &full[s], s, ip, pg);
    }

    WpixConst kc;
    kc.u0 = p.u0;
    kc.uL = p.u0 + (double)(p.n_fj - 1);
    kc.off = p.off;
    kc.magic = kMagic + (double)(p.off & ~1);
    kc.s_max = p.s_max;
    kc.s_zero = p.s_zero;

    float acc[NB];
#pragma unroll
    for (int j = 0; j < NB; ++j) acc[j] = 0.0f;
    uint16_t list[kListCap];
    int npend = 0;

    int st = 0;
    uint32_t parity = 0u;
    const int n_blocks = p.n_chunks >> 1;                // n_pad is a multiple of 32
    for (int blk = 0; blk < n_blocks; ++blk) {
        uint32_t brk = 0u;
#if BSH_WPIX_ROLL
#pragma unroll 1
#else
#pragma unroll
#endif
        for (int half = 0; half < 2; ++half) {
            mbar_wait(&full[st], parity);
            const unsigned char *sp = smem + kWpixHeader + st * L.stride;
            {   // binary terms of this stage: B = fl(A fl(fl(C CA) + fl(S SA)))  (R-5), lane l the one of SFT l & 15
                const double2 c = reinterpret_cast<const double2 *>(sp + L.tab_bytes)[lane & (kStageSfts - 1)];
                double Bv;
                if (p.ke) {                              // eccentric grid (Eq. 14): the pair is re-read per stage (L1), so
                    const double2 ke_d = p.ke[it];       // that the circular search keeps its registers
                    Bv = __dmul_rn(A_d, orbit_bracket(c.x, c.y, q_d.x, q_d.y, ke_d.x, ke_d.y));
                } else {
                    Bv = __dmul_rn(A_d, __dadd_rn(__dmul_rn(c.x, q_d.x), __dmul_rn(c.y, q_d.y)));
                }
                __syncwarp();                            // the previous stage's readers are done with bwarp
                if (lane < kStageSfts) bwarp[lane] = Bv;
                __syncwarp();
            }
            const double2 *dpair = reinterpret_cast<const double2 *>(sp + L.tab_bytes + L.cs_bytes) + lane;
            const float *wv = reinterpret_cast<const float *>(sp + L.tab_bytes + L.cs_bytes + L.d_bytes);
            const unsigned char *tab = sp + (p.off & 1) * wpix_record_bytes(EB);
#if BSH_WPIX_ROLL
            uint32_t brk16 = 0u;                         // one copy of the stage's code for both halves of the block
            wpix_half<0, NBYTES, CLAMP>(kc, tab, bwarp, dpair, wv, acc, brk16, std::make_integer_sequence<int, kStageSfts>{});
            brk |= brk16 << (kStageSfts * half);
#else
            if (half == 0)
                wpix_half<0, NBYTES, CLAMP>(kc, tab, bwarp, dpair, wv, acc, brk, std::make_integer_sequence<int, kStageSfts>{});
            else
                wpix_half<kStageSfts, NBYTES, CLAMP>(kc, tab, bwarp, dpair, wv, acc, brk,
                                                     std::make_integer_sequence<int, kStageSfts>{});
#endif
            wpix_release(p, L, smem, st, 2 * blk + half, lane, ip, pg);
            if (++st == p.n_stages) { st = 0; parity ^= 1u; }
        }
        // note the SFTs whose shift broke inside the tile
        while (brk) {
            const int k = __ffs(brk) - 1;
            brk &= brk - 1;
            list[npend] = (uint16_t)(blk * kBlock + k);
            npend += 1;
        }
        // the whole block resolves its lists together, when one could overflow in the next block of SFTs, and at the end
        if (__syncthreads_or(npend > kListCap - kBlock) || blk + 1 == n_blocks) {
            TrackConst tc;
            tc.u0 = kc.u0; tc.uL = kc.uL; tc.magic = kMagic; tc.off = p.off; tc.s_max = p.s_max; tc.s_zero = p.s_zero;
            tc.n_fj = p.n_fj;
            const double2 ke_f = p.ke ? p.ke[it] : make_double2(0.0, 0.0);
            tc.A = A_d; tc.CA = q_d.x; tc.SA = q_d.y; tc.kap = ke_f.x; tc.eta = ke_f.y;
            for (int n = 0; n < npend; ++n) {
                const int i = (int)list[n];
                const double2 c = p.cs[(int64_t)ip * p.n_pad + i];
                const double B = binary_term(tc, c.x, c.y);
                const double D = p.dpix[((((int64_t)pg * (p.n_pad >> 1)) + (i >> 1)) * 32 + lane) * 2 + (i & 1)];
                const Win7<NBYTES> x = exact_window7<NBYTES, CLAMP>(tc, p.tab7, p.n_pos, i, D, B);
                accumulate7<NBYTES>(acc, x, p.w_pad[i]);
            }
            npend = 0;
        }
    }

    const float tau = p.thr->tau_f;
    const int pix = pg * 32 + lane;
    if (act && pix < p.n_pix) {
        const uint64_t base =
            ((((uint64_t)pix * p.n_ap + ia) * p.n_P + ip) * p.n_tasc + it) * (uint64_t)p.n_f0 + p.j0;
        float *out = p.counts_full ? reinterpret_cast<float *>(p.counts_full) + base : nullptr;
#pragma unroll
        for (int j = 0; j < NB; ++j) {
            if (j < p.n_fj) {
                if (out) out[j] = acc[j];
                if (acc[j] >= tau) {
                    emit_survivor_out_of_line(p.thr, p.cand, p.cand_count, p.cand_cap, base + j, __float_as_uint(acc[j]));
                }
            }
        }
    }
}

}  // namespace bsh
