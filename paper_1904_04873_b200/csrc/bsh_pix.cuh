// bsh_pix.cuh -- stage-1 unweighted accumulation kernel with SKY PIXELS ON THE LANES ("pixel-lane" mapping), sm_100a.
//
// The position-table kernel of bsh_pos.cuh puts 32 different binary templates on the lanes of a warp.  Their tracks are
// unrelated, so the 32 16-byte window reads of one (warp, SFT) scatter over the staged table row and the kernel is bound
// by shared-memory wavefronts (ncu: 5.2 wavefronts per LDS.128, l1tex data pipe 78 % busy).  Here a warp holds ONE
// pair of binary templates and 32 neighbouring sky pixels:
//   * the pixels of a patch are less than one frequency bin apart per pixel step (Eq. 34), so the 32 positions
//     of a warp fall into a handful of consecutive table entries: same entry -> broadcast, neighbours -> different
//     banks (ncu: 136 M -> 20 M bank conflicts); the window is read as LDS.64 + LDS.32 from a split table;
//   * the binary term B = A (C CA + S SA) of Eq. (15) (L102) is the same for all lanes.  Each lane computes ONE of the
//     warp's 2 x 16 values per stage and the warp shares them through shared memory, so the hot loop spends no FP64
//     work on it: g = D - B, y at both band ends, two rounding adds, one compare = 6 FP64 operations per (pixel,
//     template, SFT) triple;
//   * breaks of the rounded shift inside the f0 tile (R-7) are flagged by comparing the two magic-add results as
//     doubles (FP64 pipe, not the integer pipe) and recorded in a 32-bit mask per block of 32 SFTs;
//   * the bit-sliced counters are two-level: 5 + 2 planes in registers, the planes above in shared memory.
// Thread = 1 pixel x 2 templates x up to 32 NW f0 bins; block = 8 warps = 16 templates of one period, 32 pixels.
//
//   PAPER.md L102 Eq. (15) track, L223 number count, L241-L247 "loop over the binary templates"; R-5, R-7.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <utility>

#include "bsh_pos.cuh"

namespace bsh {

#ifndef BSH_PIX_WARPS
#define BSH_PIX_WARPS 8
#endif
constexpr int kPixWarps = BSH_PIX_WARPS;             // warps per block
constexpr int kPixTpl = 2;                           // binary templates per thread
constexpr int kPixTile = kPixWarps * kPixTpl;        // binary templates per block
constexpr int kPixWarpScratch = kStageSfts * kPixTpl * 8 + kPixTpl * 32;       // B buffer of one stage + template constants
constexpr int kPixHeader = 128 + kPixWarps * kPixWarpScratch;
constexpr int kPixMid = 2;                           // high planes kept in registers (the other HP - 2 live in shared
                                                     // memory); 3 and 4 measured 2 % and 5 % slower on config 2

// bytes of the shared-memory high planes of one block: (HP - kPixMid) planes x 2 templates x NW words x 256 threads
__host__ __device__ constexpr int pix_hi_bytes(int NW, int HP) { return (HP - kPixMid) * kPixTpl * NW * 32 * kPixWarps * 4; }

// D table for the pixel-lane kernel: dpix[pg][i / 2][lane][i & 1] = v_i . n_pix / c (canonical order, R-5) for pixel
// pg * 32 + lane; padding SFTs get 0, padding lanes repeat the last real pixel (never written out).  One LDS.128 per
// lane returns the values of two consecutive SFTs.
__global__ void __launch_bounds__(256) dtable_pix_kernel(const double *__restrict__ v_over_c, const double *__restrict__ nvec,
                                                         int n_sft, int n_pad, int n_pix, int n_pg,
                                                         double *__restrict__ dpix)
{
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t total = (int64_t)n_pg * n_pad * 32;
    if (t >= total) return;
    const int e = (int)(t & 1);
    const int lane = (int)((t >> 1) & 31);
    const int64_t q = t >> 6;
    const int half = n_pad >> 1;
    const int i = 2 * (int)(q % half) + e;
    const int pg = (int)(q / half);
    int pix = pg * 32 + lane;
    if (pix >= n_pix) pix = n_pix - 1;
    double D = 0.0;
    if (i < n_sft) {
        const double a = __dmul_rn(v_over_c[3 * i + 0], nvec[3 * pix + 0]);
        const double b = __dmul_rn(v_over_c[3 * i + 1], nvec[3 * pix + 1]);
        const double c = __dmul_rn(v_over_c[3 * i + 2], nvec[3 * pix + 2]);
        D = __dadd_rn(__dadd_rn(a, b), c);
    }
    dpix[t] = D;
}

// Position-major table staged by the pixel-lane kernel.  Per stage of kStageSfts SFTs, the RECORD of position p holds
//   [kStageSfts] (word 0, word 1) pairs (8 bytes each), then for NW = 3 [kStageSfts] words 2 (4 bytes each), then 8 bytes
//   of padding:  200 bytes (NW = 3) or 136 bytes (NW = 2).
// Why: (i) the address of (SFT kk, position s) is  base + s * record + kk * 8  -- ONE multiply-add per triple (IMAD, on
// the FMA pipe, which this kernel leaves idle) with the SFT part an instruction immediate, instead of the SEL + VIADD +
// 2 LEA of an SFT-major table (all on the half-rate integer pipe that the LOP3 counters saturate); (ii) a window is read
// as LDS.64 + LDS.32 (3 wavefronts; one LDS.128 would cost 4); (iii) 50 (34) words per record put the neighbouring
// positions a warp reads (Eq. 34: pixels of a patch are less than a bin apart) into different banks.
__host__ __device__ constexpr int pix_rec_bytes(int NW) { return NW >= 3 ? kStageSfts * 12 + 8 : kStageSfts * 8 + 8; }
__host__ __device__ constexpr int pix_stage_tab_bytes(int n_pos, int NW) { return (n_pos * pix_rec_bytes(NW) + 15) & ~15; }

__global__ void __launch_bounds__(256) pm_position_table_kernel(const uint4 *__restrict__ ptab, int n_pad, int n_pos, int NW,
                                                                unsigned char *__restrict__ out)
{
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (int64_t)n_pad * n_pos) return;
    const int i = (int)(t / n_pos), p = (int)(t % n_pos);
    const uint4 e = ptab[t];
    const int rec = pix_rec_bytes(NW);
    unsigned char *r = out + (int64_t)(i / kStageSfts) * pix_stage_tab_bytes(n_pos, NW) + (int64_t)p * rec;
    const int kk = i % kStageSfts;
    reinterpret_cast<uint2 *>(r)[kk] = make_uint2(e.x, e.y);
    if (NW >= 3) reinterpret_cast<uint32_t *>(r + kStageSfts * 8)[kk] = e.z;
    if (kk == 0) *reinterpret_cast<uint2 *>(r + rec - 8) = make_uint2(0u, 0u);
}

struct PixParams {
    const uint4 *ptab;          // [n_pad][n_pos]  (fix-ups)
    const unsigned char *split; // [n_pad / kStageSfts] stages of the position-major table (hot loop)
    const double2 *cs;          // [n_P][n_pad]  (cos, sin)(Omega_p t_i)
    const double *dpix;         // [n_pg][n_pad / 2][32][2]
    const double *A;            // [n_ap][n_P]
    const double2 *casa;        // [n_P][n_tasc]
    const double2 *ke;          // [n_tasc] (e cos omega, e sin omega), or NULL (circular orbits)
    int n_pad, n_pos, n_chunks, n_stages;
    int n_pix, n_ap, n_P, n_tasc, n_f0;
    int j0, n_fj;               // f0 tile
    int n_pg, n_aq, n_aq_tiles;
    double u0;                  // k_band0 + j0
    int off, s_max, s_zero;     // position coordinates (TrackConst)
    unsigned int one, zero;     // 1 and 0 (run-time constants the compiler cannot fold, see pix_step)
    const Threshold *thr;
    RawCand *cand;
    unsigned int *cand_count;
    unsigned int cand_cap;
    void *counts_full;
};

struct PixStage {
    int tab_bytes, cs_bytes, d_bytes, stride;
    __device__ __host__ PixStage(int n_pos, int NW)
    {
        tab_bytes = pix_stage_tab_bytes(n_pos, NW);
        cs_bytes = kStageSfts * 16;
        d_bytes = kStageSfts * 32 * 8;
        stride = tab_bytes + cs_bytes + d_bytes;
    }
    __device__ __host__ int total(int n_stages) const { return kPixHeader + n_stages * stride; }
};

__device__ __forceinline__ void pix_issue(const PixParams &p, const PixStage &L, unsigned char *stage, uint64_t *bar, int chunk,
                                          int ip, int pg)
{
    const int64_t i0 = (int64_t)chunk * kStageSfts;
    mbar_expect_tx(bar, (uint32_t)L.stride);
    tma_bulk_g2s(stage, p.split + (int64_t)chunk * L.tab_bytes, (uint32_t)L.tab_bytes, bar);
    tma_bulk_g2s(stage + L.tab_bytes, p.cs + (int64_t)ip * p.n_pad + i0, (uint32_t)L.cs_bytes, bar);
    tma_bulk_g2s(stage + L.tab_bytes + L.cs_bytes, p.dpix + ((int64_t)pg * p.n_pad + i0) * 32, (uint32_t)L.d_bytes, bar);
}

// A warp is done with `stage`: the warp that releases it last refills it with chunk c + n_stages.
__device__ __forceinline__ void pix_release(const PixParams &p, const PixStage &L, unsigned char *smem, int st, int c, int lane,
                                            int ip, int pg)
{
    __syncwarp();
    if (lane == 0) {
        unsigned int *done = reinterpret_cast<unsigned int *>(smem + 8 * kMaxStages) + st;
        unsigned int old;
        asm volatile("atom.acq_rel.cta.shared.add.u32 %0, [%1], 1;" : "=r"(old) : "r"(smem_u32(done)) : "memory");
        if ((old + 1u) % (unsigned)kPixWarps == 0u && c + p.n_stages < p.n_chunks)
            pix_issue(p, L, smem + kPixHeader + st * L.stride, reinterpret_cast<uint64_t *>(smem) + st, c + p.n_stages, ip, pg);
    }
}

// Per-thread constants of the hot loop (the binary-term constants live in shared memory, only the fix-ups need them).
struct PixConst {
    double u0, uL;
    double magic;               // 1.5 2^52 + (off rounded down to even): the low word of fl(y + magic) is position - (off & 1);
                                // an EVEN integer added to the rounding constant leaves the tie rule of R-1 unchanged
    int32_t off, s_max, s_zero;
    uint32_t rec;               // bytes per record of the staged table (in a register, so that the address is one IMAD)
    uint32_t s_zero_rel;        // s_zero - (off & 1)
    uint32_t one, zero;         // 1 and 0, opaque to the compiler (kernel parameters)
};

// Position (table entry) to read for one (pixel, template, SFT) and the break flag (R-7): the all-zero position on a
// break.  Clamped geometry only (the unclamped hot path is pix_step below).
__device__ __forceinline__ int32_t pix_position_clamped(const PixConst &k, double D, double B, bool &brk)
{
    const double g = __dsub_rn(D, B);
    const double m0 = __dadd_rn(__dmul_rn(k.u0, g), kMagic);         // low word = round(fl(u0 g)), R-1
    const double mL = __dadd_rn(__dmul_rn(k.uL, g), kMagic);
    const int32_t s0 = clamp_s(k.off + __double2loint(m0), k.s_max);
    const int32_t sL = clamp_s(k.off + __double2loint(mL), k.s_max); // equal after clamping => every bin reads 0
    brk = s0 != sL;
    return brk ? k.s_zero : s0;
}

// Window of SFT KK of the stage from the record at shared-memory address `rec_addr`.
template <int NW, int KK>
__device__ __forceinline__ Win<NW> pix_load(uint32_t rec_addr)
{
    Win<NW> w;
    asm volatile("ld.shared.v2.u32 {%0, %1}, [%2+%3];" : "=r"(w.x[0]), "=r"(w.x[1 % NW]) : "r"(rec_addr), "n"(KK * 8));
    if (NW > 2) asm volatile("ld.shared.u32 %0, [%1+%2];" : "=r"(w.x[2 % NW]) : "r"(rec_addr), "n"(kStageSfts * 8 + KK * 4));
    return w;
}

#ifndef BSH_PIX_SELMODE
#define BSH_PIX_SELMODE 0
#endif
#ifndef BSH_PIX_BRKMODE
#define BSH_PIX_BRKMODE 1
#endif
#if BSH_PIX_SELMODE == 1
#define BSH_PIX_SEL_ASM "@p mad.lo.s32 lo, lo, %13, %6;\n\t"
#else
#define BSH_PIX_SEL_ASM "@p mov.b32 lo, %6;\n\t"
#endif
#if BSH_PIX_BRKMODE == 1
#define BSH_PIX_BRK_ASM3 "@p mad.lo.u32 %3, %12, %7, %3;\n\t"
#else
#define BSH_PIX_BRK_ASM3 "@p or.b32 %3, %3, %7;\n\t"
#endif

// One SFT (slot K of the unrolled block of 32) for both templates of the thread.  base = shared-memory address of the
// record of position (off & 1) of the stage (unclamped) or of position 0 (clamped).
template <int K, int NW, int HP, bool CLAMP>
__device__ __forceinline__ void pix_step(const PixConst &k, uint32_t base, const double2 *bpair, const double2 *dpair,
                                         Counter<NW, kPixMid> (&cnt)[kPixTpl], uint32_t (&brk)[kPixTpl])
{
    constexpr int kk = K % kStageSfts;
    const double2 d2 = dpair[(kk >> 1) * 32];
    const double D = (kk & 1) ? d2.y : d2.x;
    const double2 b2 = bpair[kk];
    const double Bv[kPixTpl] = {b2.x, b2.y};
#pragma unroll
    for (int r = 0; r < kPixTpl; ++r) {
        Win<NW> w;
        if (!CLAMP) {
            // g = D - B, y at both band ends, rounding adds (the low word of m0 IS the table position), then ONE predicate
            // from the FP64 compare (equal doubles <=> equal roundings) drives the break mask and the position select; the
            // record address is one multiply-add.  6 FP64 + 1 FMA-pipe + 2 integer + 2 load instructions per triple.
            const double g = __dsub_rn(D, Bv[r]);
            const double m0 = __dadd_rn(__dmul_rn(k.u0, g), k.magic);
            const double mL = __dadd_rn(__dmul_rn(k.uL, g), k.magic);
            // The select, the mask update and the address are written as multiply-adds with the run-time constant
            // k.one (= 1): ptxas then issues them as IMAD on the FMA pipe instead of SEL / LOP3 / LEA on the integer
            // pipe, which the LOP3 counters need.
            if (NW > 2)
                asm volatile("{\n\t"
                             ".reg .pred p;\n\t"
                             ".reg .b32 lo, hi, a;\n\t"
                             "setp.neu.f64 p, %4, %5;\n\t"
                             "mov.b64 {lo, hi}, %4;\n\t"
                             BSH_PIX_SEL_ASM
                             BSH_PIX_BRK_ASM3
                             "mad.lo.s32 a, lo, %8, %9;\n\t"
                             "ld.shared.v2.u32 {%0, %1}, [a+%10];\n\t"
                             "ld.shared.u32 %2, [a+%11];\n\t"
                             "}"
                             : "=r"(w.x[0]), "=r"(w.x[1 % NW]), "=r"(w.x[2 % NW]), "+r"(brk[r])
                             : "d"(m0), "d"(mL), "r"(k.s_zero_rel), "n"(1u << K), "r"(k.rec), "r"(base), "n"(kk * 8),
                               "n"(kStageSfts * 8 + kk * 4), "r"(k.one), "r"(k.zero));
            else
                asm volatile("{\n\t"
                             ".reg .pred p;\n\t"
                             ".reg .b32 lo, hi, a;\n\t"
                             "setp.neu.f64 p, %3, %4;\n\t"
                             "mov.b64 {lo, hi}, %3;\n\t"
                             "@p mov.b32 lo, %5;\n\t"
                             "@p or.b32 %2, %2, %6;\n\t"
                             "mad.lo.s32 a, lo, %7, %8;\n\t"
                             "ld.shared.v2.u32 {%0, %1}, [a+%9];\n\t"
                             "}"
                             : "=r"(w.x[0]), "=r"(w.x[1 % NW]), "+r"(brk[r])
                             : "d"(m0), "d"(mL), "r"(k.s_zero_rel), "n"(1u << K), "r"(k.rec), "r"(base), "n"(kk * 8));
        } else {
            bool b;
            const int32_t s = pix_position_clamped(k, D, Bv[r], b);
            brk[r] |= b ? (1u << K) : 0u;
            w = pix_load<NW, kk>(base + (uint32_t)s * k.rec);
        }
        push<K, NW, kPixMid>(cnt[r], w);
    }
}

template <int K0, int NW, int HP, bool CLAMP, int... Ks>
__device__ __forceinline__ void pix_half(const PixConst &k, uint32_t base, const double2 *bpair, const double2 *dpair,
                                         Counter<NW, kPixMid> (&cnt)[kPixTpl], uint32_t (&brk)[kPixTpl],
                                         std::integer_sequence<int, Ks...>)
{
    (pix_step<K0 + Ks, NW, HP, CLAMP>(k, base, bpair, dpair, cnt, brk), ...);
}

#ifndef BSH_PIX_MINB
#define BSH_PIX_MINB (BSH_PIX_WARPS > 8 ? 1 : 2)
#endif
// ECC: the grid has an eccentricity axis (Eq. 14); a template parameter, so that the circular search (Eq. 15) carries none of
// its code (as a run-time branch it cost 2 % of the circular kernel's time)
template <int NW, int HP, bool CLAMP, bool ECC>
__global__ void __launch_bounds__(32 * kPixWarps, BSH_PIX_MINB) stage1_unweighted_pix_kernel(const PixParams p)
{
    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t *full = reinterpret_cast<uint64_t *>(smem);
    const PixStage L(p.n_pos, NW);
    int b = blockIdx.x;
    const int tile = b % p.n_aq_tiles;
    b /= p.n_aq_tiles;
    const int ip = b % p.n_P;
    const int pg = b / p.n_P;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    unsigned char *wscr = smem + 128 + warp * kPixWarpScratch;
    double *bbuf = reinterpret_cast<double *>(wscr);                           // [16 SFTs][2 templates]
    double *tcst = reinterpret_cast<double *>(wscr + kStageSfts * kPixTpl * 8); // [2 templates][A, CA, SA, -]

    // the warp's two binary templates (a_p, t_asc pairs of period ip); a missing one repeats the last real pair
    int ia[kPixTpl], it[kPixTpl];
    bool act[kPixTpl];
#pragma unroll
    for (int r = 0; r < kPixTpl; ++r) {
        int aq = tile * kPixTile + warp * kPixTpl + r;
        act[r] = aq < p.n_aq;
        if (!act[r]) aq = p.n_aq - 1;
        ia[r] = aq / p.n_tasc;
        it[r] = aq - ia[r] * p.n_tasc;
    }
    // lane l computes the binary term of template (l & 1) at SFT (l >> 1) of every stage
    const int rd = lane & 1;
    const double A_d = p.A[(rd ? ia[1] : ia[0]) * p.n_P + ip];
    const double2 q_d = p.casa[ip * p.n_tasc + (rd ? it[1] : it[0])];
    if (lane < kPixTpl) {
        tcst[lane * 4 + 0] = A_d;
        tcst[lane * 4 + 1] = q_d.x;
        tcst[lane * 4 + 2] = q_d.y;
    }

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
        for (int s = 0; s < n0; ++s) pix_issue(p, L, smem + kPixHeader + s * L.stride, &full[s], s, ip, pg);
    }

    PixConst kc;
    kc.u0 = p.u0;
    kc.uL = p.u0 + (double)(p.n_fj - 1);
    kc.off = p.off;
    kc.s_max = p.s_max;
    kc.s_zero = p.s_zero;
    kc.magic = kMagic + (double)(p.off & ~1);
    kc.rec = (uint32_t)pix_rec_bytes(NW);
    kc.s_zero_rel = (uint32_t)(p.s_zero - (p.off & 1));
    kc.one = p.one;
    kc.zero = p.zero;
    const uint32_t rec_shift = CLAMP ? 0u : (uint32_t)(p.off & 1) * kc.rec;

    // Counters: 5 low planes (carry-save tree over a block of 32 SFTs) + kPixMid planes in registers; the HP - kPixMid
    // planes above live in shared memory, [plane][template][word][thread].  A register counter wraps at most once in
    // 2^kPixMid blocks (one carry of weight 32 per block), so its carries-out are OR-ed into `over` and rippled into the
    // shared planes every 2^kPixMid-th block (and around every fix-up merge): 66 -> 42 counter registers, no spills at
    // any SFT count.
    constexpr int HS = HP - kPixMid;
    uint32_t *hs = reinterpret_cast<uint32_t *>(smem + kPixHeader + p.n_stages * L.stride) + threadIdx.x;
    constexpr int kHsStride = 32 * kPixWarps;
#pragma unroll
    for (int q = 0; q < HS * kPixTpl * NW; ++q) hs[q * kHsStride] = 0u;
    auto spill_over = [&](Counter<NW, kPixMid> &c, int r) {
#pragma unroll
        for (int w = 0; w < NW; ++w) {
            uint32_t carry = c.over[w];
#pragma unroll
            for (int q = 0; q < HS; ++q) {
                uint32_t *pl = hs + ((q * kPixTpl + r) * NW + w) * kHsStride;
                const uint32_t t = *pl;
                *pl = t ^ carry;
                carry = t & carry;
            }
            c.over[w] = 0u;
        }
    };

    Counter<NW, kPixMid> cnt[kPixTpl];
    uint16_t list[kPixTpl][kListCap];
    int npend[kPixTpl];
#pragma unroll
    for (int r = 0; r < kPixTpl; ++r) {
        cnt[r].clear();
        npend[r] = 0;
    }

    int st = 0;
    uint32_t parity = 0u;
    const int n_blocks = p.n_chunks >> 1;                // n_pad is a multiple of 32
    for (int blk = 0; blk < n_blocks; ++blk) {
        uint32_t brk[kPixTpl] = {0u, 0u};
#pragma unroll
        for (int half = 0; half < 2; ++half) {
            mbar_wait(&full[st], parity);
            const unsigned char *sp = smem + kPixHeader + st * L.stride;
            const double2 *cs = reinterpret_cast<const double2 *>(sp + L.tab_bytes);
            {   // binary terms of this stage: B = fl(A bracket)  (R-5, R-23), one per lane
                const double2 c = cs[lane >> 1];
                if (ECC) {                     // eccentric grid (Eq. 14): the pair is re-read per stage (L1), so
                    const double2 ke_d = p.ke[rd ? it[1] : it[0]];   // that the circular search keeps its registers
                    bbuf[lane] = __dmul_rn(A_d, orbit_bracket(c.x, c.y, q_d.x, q_d.y, ke_d.x, ke_d.y));
                } else {
                    bbuf[lane] = __dmul_rn(A_d, __dadd_rn(__dmul_rn(c.x, q_d.x), __dmul_rn(c.y, q_d.y)));
                }
                __syncwarp();                            // (the previous stage's readers passed the __syncwarp of pix_release)
            }
            const double2 *bpair = reinterpret_cast<const double2 *>(bbuf);
            const double2 *dpair = reinterpret_cast<const double2 *>(sp + L.tab_bytes + L.cs_bytes) + lane;
            const uint32_t base = smem_u32(sp) + rec_shift;
            if (half == 0)
                pix_half<0, NW, HP, CLAMP>(kc, base, bpair, dpair, cnt, brk, std::make_integer_sequence<int, kStageSfts>{});
            else
                pix_half<kStageSfts, NW, HP, CLAMP>(kc, base, bpair, dpair, cnt, brk,
                                                    std::make_integer_sequence<int, kStageSfts>{});
            pix_release(p, L, smem, st, 2 * blk + half, lane, ip, pg);
            if (++st == p.n_stages) { st = 0; parity ^= 1u; }
        }
        // note the SFTs whose shift broke inside the tile; resolve the lists when one could overflow, and at the end
        bool want = false;
#pragma unroll
        for (int r = 0; r < kPixTpl; ++r) {
            uint32_t m = brk[r];
            while (m) {
                const int k = __ffs(m) - 1;
                m &= m - 1;
                list[r][npend[r]] = (uint16_t)(blk * kBlock + k);
                npend[r] += 1;
            }
            want = want || npend[r] > kListCap - kBlock;
        }
        if (__any_sync(0xFFFFFFFFu, want) || blk + 1 == n_blocks) {
#pragma unroll
            for (int r = 0; r < kPixTpl; ++r) {
                TrackConst tc;
                tc.u0 = kc.u0; tc.uL = kc.uL; tc.magic = kMagic; tc.off = p.off; tc.s_max = p.s_max; tc.s_zero = p.s_zero;
                tc.n_fj = p.n_fj;
                tc.A = tcst[r * 4 + 0]; tc.CA = tcst[r * 4 + 1]; tc.SA = tcst[r * 4 + 2];
                const double2 ke_r = ECC ? p.ke[it[r]] : make_double2(0.0, 0.0);
                tc.kap = ke_r.x; tc.eta = ke_r.y;
                uint32_t tp[kFixPlanes][NW];
#pragma unroll
                for (int q = 0; q < kFixPlanes; ++q)
#pragma unroll
                    for (int w = 0; w < NW; ++w) tp[q][w] = 0u;
                for (int n = 0; n < npend[r]; ++n) {
                    const int i = (int)list[r][n];
                    const double2 c = p.cs[(int64_t)ip * p.n_pad + i];
                    const double B = binary_term(tc, c.x, c.y);
                    const double D = p.dpix[((((int64_t)pg * (p.n_pad >> 1)) + (i >> 1)) * 32 + lane) * 2 + (i & 1)];
                    fix_accumulate<NW>(tp, exact_window_pos<NW, CLAMP>(tc, p.ptab + (int64_t)i * p.n_pos, D, B));
                }
                spill_over(cnt[r], r);                   // `over` must be empty: the merge may carry out of plane 7
                fix_merge<NW, kPixMid>(cnt[r], tp);
                spill_over(cnt[r], r);
                npend[r] = 0;
            }
        }
        if ((blk & ((1 << kPixMid) - 1)) == (1 << kPixMid) - 1 || blk + 1 == n_blocks) {
#pragma unroll
            for (int r = 0; r < kPixTpl; ++r) spill_over(cnt[r], r);
        }
    }

    // epilogue: threshold in bit-sliced form, emit the (rare) survivors
    const int32_t tau = p.thr->tau_i;
    const int pix = pg * 32 + lane;
#pragma unroll
    for (int r = 0; r < kPixTpl; ++r) {
        if (!act[r] || pix >= p.n_pix) continue;
        Counter<NW, HP> full_cnt;                        // all 5 + HP planes of this template, for the comparisons below
#pragma unroll
        for (int w = 0; w < NW; ++w) {
#pragma unroll
            for (int l = 0; l < kLowPlanes; ++l) full_cnt.low[l][w] = cnt[r].low[l][w];
#pragma unroll
            for (int q = 0; q < kPixMid; ++q) full_cnt.hi[q][w] = cnt[r].hi[q][w];
#pragma unroll
            for (int q = 0; q < HS; ++q) full_cnt.hi[kPixMid + q][w] = hs[((q * kPixTpl + r) * NW + w) * kHsStride];
        }
        const uint64_t base =
            ((((uint64_t)pix * p.n_ap + ia[r]) * p.n_P + ip) * p.n_tasc + it[r]) * (uint64_t)p.n_f0 + p.j0;
        const Win<NW> ge = count_ge(full_cnt, tau);
        int32_t *out = p.counts_full ? reinterpret_cast<int32_t *>(p.counts_full) + base : nullptr;
#pragma unroll
        for (int w = 0; w < NW; ++w) {
            if (out) {
                for (int bb = 0; bb < 32; ++bb)
                    if (32 * w + bb < p.n_fj) out[32 * w + bb] = count_at(full_cnt, w, bb);
            }
            uint32_t m = ge.x[w] & valid_mask(p.n_fj, w);
            while (m) {
                const int bb = __ffs(m) - 1;
                m &= m - 1;
                emit_survivor(p.thr, p.cand, p.cand_count, p.cand_cap, base + 32 * w + bb, (uint32_t)count_at(full_cnt, w, bb));
            }
        }
    }
}

}  // namespace bsh
