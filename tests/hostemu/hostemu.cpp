// hostemu.cpp -- GPU-less emulation of the stage-1 accumulation kernels' per-thread logic (TEST CODE, never shipped in
// libbsh.so).  It runs the SAME header code the kernels run (csrc/bsh_core.cuh: canonical track, window extraction, break
// handling, carry-save counters, weighted accumulation; csrc/bsh_host.hpp: tables, table geometry), with plain loops in
// place of the CUDA grid and plain arrays in place of the TMA-staged shared memory.  It lets `-m "not gpu"` tests check
// the host logic and the kernel arithmetic against the oracle before any GPU time is spent.
// Build: g++ -O2 -std=c++17 -ffp-contract=off -shared -fPIC
#include <stdint.h>
#include <string.h>

#include <utility>
#include <vector>

#include "../../paper_1904_04873_b200/csrc/bsh_core.cuh"
#include "../../paper_1904_04873_b200/csrc/bsh_host.hpp"

using namespace bsh;

namespace {

struct Tables {
    std::vector<double> cs, casa, A, nv, dtab;
    std::vector<uint4> wtab;
    std::vector<float> w_pad;
    int n_pad;
};

// mirrors sft_step_unweighted / block_unweighted of bsh_kernels.cuh (R = 1): breaks read the zero window and set a bit
template <int K, int NW, int HP, bool CLAMP>
inline void step(const TrackConst &tc, const uint4 *wt, int n_entries, const double *cs, const double *d, Counter<NW, HP> &cnt,
                 uint32_t &brk)
{
    const double B = binary_term(tc, cs[2 * K], cs[2 * K + 1]);
    bool b;
    const Win<NW> x = track_window_deferred<NW, CLAMP>(tc, wt + K * n_entries, d[K], B, b);
    brk |= b ? (1u << K) : 0u;
    push<K, NW, HP>(cnt, x);
}

template <int NW, int HP, bool CLAMP, int... Ks>
inline void block(const TrackConst &tc, const uint4 *wt, int n_entries, const double *cs, const double *d, Counter<NW, HP> &cnt,
                  uint32_t &brk, std::integer_sequence<int, Ks...>)
{
    (step<Ks, NW, HP, CLAMP>(tc, wt, n_entries, cs, d, cnt, brk), ...);
}

// mirrors fixup_from_global: the exact window of a deferred SFT, added by ripple carry
template <int NW, int HP, bool CLAMP>
inline void fixup(const TrackConst &tc, const uint4 *wtab, int n_entries, const double *cs, const double *d, int i,
                  Counter<NW, HP> &cnt)
{
    const double B = binary_term(tc, cs[2 * i], cs[2 * i + 1]);
    add_window(cnt, track_window<NW, CLAMP>(tc, wtab + (size_t)i * n_entries, d[i], B));
}

template <int NW, int HP, bool CLAMP>
void run(int n_sft, int n_pix, int n_ap, int n_P, int n_tasc, int n_f0, int64_t k_band0, int64_t k_slab0, const Tables &T,
         const TableGeometry &tg, int weighted, int32_t *counts, float *wcounts)
{
    const int tile_bins = 32 * NW;
    for (int j0 = 0; j0 < n_f0; j0 += tile_bins) {
        const int n_fj = std::min(tile_bins, n_f0 - j0);
        for (int pix = 0; pix < n_pix; ++pix)
            for (int ip = 0; ip < n_P; ++ip)
                for (int ia = 0; ia < n_ap; ++ia)
                    for (int it = 0; it < n_tasc; ++it) {
                        TrackConst tc;
                        tc.u0 = (double)(k_band0 + j0);
                        tc.uL = tc.u0 + (double)(n_fj - 1);
                        tc.A = T.A[(size_t)ia * n_P + ip];
                        tc.CA = T.casa[((size_t)ip * n_tasc + it) * 2];
                        tc.SA = T.casa[((size_t)ip * n_tasc + it) * 2 + 1];
                        tc.kap = 0.0; tc.eta = 0.0;
                        tc.off = (int)(k_band0 - k_slab0) + j0 + tg.off_table;
                        tc.magic = kMagic + (double)tc.off;
                        tc.s_max = tg.s_max;
                        tc.s_zero = tg.s_zero;
                        tc.n_fj = n_fj;
                        const double *cs = T.cs.data() + (size_t)ip * T.n_pad * 2;
                        const double *d = T.dtab.data() + (size_t)pix * T.n_pad;
                        const uint64_t base = ((((uint64_t)pix * n_ap + ia) * n_P + ip) * n_tasc + it) * (uint64_t)n_f0 + j0;
                        if (!weighted) {
                            Counter<NW, HP> cnt;
                            cnt.clear();
                            // deferred-break list with a tiny capacity so that the bulk flush, the end flush and
                            // the list-full path of the kernel are all exercised
                            const int cap = 3;
                            int list[3], npend = 0;
                            for (int i0 = 0; i0 < T.n_pad; i0 += kBlock) {
                                uint32_t brk = 0u;
                                block<NW, HP, CLAMP>(tc, T.wtab.data() + (size_t)i0 * tg.n_entries, tg.n_entries, cs + 2 * i0,
                                                     d + i0, cnt, brk, std::make_integer_sequence<int, kBlock>{});
                                for (int k = 0; k < kBlock; ++k) {
                                    if (!((brk >> k) & 1u)) continue;
                                    if (npend < cap) list[npend++] = i0 + k;
                                    else fixup<NW, HP, CLAMP>(tc, T.wtab.data(), tg.n_entries, cs, d, i0 + k, cnt);
                                }
                                if (npend > 2 || i0 + kBlock >= T.n_pad) {
                                    for (int n = 0; n < npend; ++n)
                                        fixup<NW, HP, CLAMP>(tc, T.wtab.data(), tg.n_entries, cs, d, list[n], cnt);
                                    npend = 0;
                                }
                            }
                            // also exercise the bit-sliced threshold: count_ge must agree with the extracted counts
                            for (int w = 0; w < NW; ++w)
                                for (int b = 0; b < 32; ++b)
                                    if (32 * w + b < n_fj) counts[base + 32 * w + b] = count_at(cnt, w, b);
                            for (int tau : {0, 1, 7, 13, 40, 400, 1 << (kLowPlanes + HP)}) {
                                const Win<NW> ge = count_ge(cnt, tau);
                                for (int w = 0; w < NW; ++w)
                                    for (int b = 0; b < 32; ++b)
                                        if (32 * w + b < n_fj && ((ge.x[w] >> b) & 1u) != (uint32_t)(count_at(cnt, w, b) >= tau))
                                            counts[base + 32 * w + b] = -1;      // poison: test will fail
                            }
                        } else {
                            float acc[32 * NW];
                            for (int j = 0; j < 32 * NW; ++j) acc[j] = 0.f;
                            for (int i = 0; i < T.n_pad; ++i) {
                                const double B = binary_term(tc, cs[2 * i], cs[2 * i + 1]);
                                const Win<NW> x = track_window<NW, CLAMP>(tc, T.wtab.data() + (size_t)i * tg.n_entries, d[i], B);
                                accumulate_weighted<NW>(acc, x, T.w_pad[i]);
                            }
                            for (int j = 0; j < n_fj; ++j) wcounts[base + j] = acc[j];
                        }
                    }
    }
}

// mirrors stage1_unweighted_pix_kernel of bsh_pix.cuh for one (pixel, binary template): positions from the position
// table, breaks parked on the zero position and noted in a mask per block of 32 SFTs, masks -> list, lists resolved with
// exact_window_pos + the small fix-up accumulator (tiny list capacity so that bulk, overflow and end flushes all run)
template <int K, int NW, int HP, bool CLAMP>
inline void pix_step_emu(const TrackConst &tc, const uint4 *ptab, int n_pos, const double *cs, const double *d,
                         Counter<NW, HP> &cnt, uint32_t &brk)
{
    const double B = binary_term(tc, cs[2 * K], cs[2 * K + 1]);
    bool b;
    const int32_t s = track_position_deferred<CLAMP>(tc, d[K], B, b);
    brk |= b ? (1u << K) : 0u;
    push<K, NW, HP>(cnt, load_position<NW>(ptab + (size_t)K * n_pos, s));
}

template <int NW, int HP, bool CLAMP, int... Ks>
inline void pix_block_emu(const TrackConst &tc, const uint4 *ptab, int n_pos, const double *cs, const double *d,
                          Counter<NW, HP> &cnt, uint32_t &brk, std::integer_sequence<int, Ks...>)
{
    (pix_step_emu<Ks, NW, HP, CLAMP>(tc, ptab, n_pos, cs, d, cnt, brk), ...);
}

template <int NW, int HP, bool CLAMP>
void run_pix(int n_sft, int n_pix, int n_ap, int n_P, int n_tasc, int n_f0, int64_t k_band0, int64_t k_slab0, int n_bins,
             const uint32_t *peak, int words_per_row, const Tables &T, const TableGeometry &tg, int32_t *counts)
{
    const PosGeometry pg = pos_geometry(tg, n_bins, n_f0, NW);
    // position table (mirrors build_position_table_kernel)
    std::vector<uint4> ptab((size_t)T.n_pad * pg.n_pos, uint4{0, 0, 0, 0});
    const int row_words = (n_bins + 31) / 32;
    for (int i = 0; i < n_sft; ++i)
        for (int p = 0; p < pg.n_pos; ++p) {
            if (p == pg.s_zero) continue;
            const int c0 = p - pg.off_table;
            const int q0 = c0 >> 5, sh = c0 & 31;
            auto word = [&](int q) { return (q >= 0 && q < row_words) ? peak[(size_t)i * words_per_row + q] : 0u; };
            uint32_t v[3], lo = word(q0);
            for (int w = 0; w < 3; ++w) {
                const uint32_t hi = word(q0 + w + 1);
                v[w] = funnel_r(lo, hi, sh);
                lo = hi;
            }
            ptab[(size_t)i * pg.n_pos + p] = uint4{v[0], v[1], v[2], 0u};
        }
    const int tile_bins = 32 * NW;
    for (int j0 = 0; j0 < n_f0; j0 += tile_bins) {
        const int n_fj = std::min(tile_bins, n_f0 - j0);
        for (int pix = 0; pix < n_pix; ++pix)
            for (int ip = 0; ip < n_P; ++ip)
                for (int ia = 0; ia < n_ap; ++ia)
                    for (int it = 0; it < n_tasc; ++it) {
                        TrackConst tc;
                        tc.u0 = (double)(k_band0 + j0);
                        tc.uL = tc.u0 + (double)(n_fj - 1);
                        tc.A = T.A[(size_t)ia * n_P + ip];
                        tc.CA = T.casa[((size_t)ip * n_tasc + it) * 2];
                        tc.SA = T.casa[((size_t)ip * n_tasc + it) * 2 + 1];
                        tc.kap = 0.0; tc.eta = 0.0;
                        tc.off = (int)(k_band0 - k_slab0) + j0 + pg.off_table;
                        tc.magic = kMagic + (double)tc.off;
                        tc.s_max = pg.s_max;
                        tc.s_zero = pg.s_zero;
                        tc.n_fj = n_fj;
                        const double *cs = T.cs.data() + (size_t)ip * T.n_pad * 2;
                        const double *d = T.dtab.data() + (size_t)pix * T.n_pad;
                        const uint64_t base = ((((uint64_t)pix * n_ap + ia) * n_P + ip) * n_tasc + it) * (uint64_t)n_f0 + j0;
                        Counter<NW, HP> cnt;
                        cnt.clear();
                        const int cap = 5;
                        int list[5], npend = 0;
                        auto flush = [&]() {
                            uint32_t tp[kFixPlanes][NW];
                            for (int q = 0; q < kFixPlanes; ++q)
                                for (int w = 0; w < NW; ++w) tp[q][w] = 0u;
                            for (int n = 0; n < npend; ++n) {
                                const int i = list[n];
                                const double B = binary_term(tc, cs[2 * i], cs[2 * i + 1]);
                                fix_accumulate<NW>(tp, exact_window_pos<NW, CLAMP>(tc, ptab.data() + (size_t)i * pg.n_pos, d[i], B));
                            }
                            fix_merge<NW, HP>(cnt, tp);
                            npend = 0;
                        };
                        for (int i0 = 0; i0 < T.n_pad; i0 += kBlock) {
                            uint32_t brk = 0u;
                            pix_block_emu<NW, HP, CLAMP>(tc, ptab.data() + (size_t)i0 * pg.n_pos, pg.n_pos, cs + 2 * i0, d + i0,
                                                         cnt, brk, std::make_integer_sequence<int, kBlock>{});
                            for (int k = 0; k < kBlock; ++k) {
                                if (!((brk >> k) & 1u)) continue;
                                if (npend == cap) flush();
                                list[npend++] = i0 + k;
                            }
                            if (npend > 3 || i0 + kBlock >= T.n_pad) flush();
                        }
                        for (int w = 0; w < NW; ++w)
                            for (int b = 0; b < 32; ++b)
                                if (32 * w + b < n_fj) counts[base + 32 * w + b] = count_at(cnt, w, b);
                    }
    }
}

}  // namespace

extern "C" int emu_stage1(int n_sft, const double *t_mid, const double *v_over_c, double t_search_mid, int64_t k_slab0,
                          int n_bins, int64_t k_band0, int n_f0, int n_pix, const double *alpha, const double *delta, int n_ap,
                          const double *ap, int n_P, const double *P, int n_tasc, const double *tasc_frac,
                          const uint32_t *peak, int words_per_row, const float *w, int weighted, int force_clamp, int nw_force,
                          int32_t *counts, float *wcounts, int *info)
{
    Tables T;
    T.n_pad = pad_sfts(n_sft);
    build_binary_tables(n_sft, T.n_pad, t_mid, t_search_mid, n_P, P, n_tasc, tasc_frac, n_ap, ap, T.cs, T.casa, T.A);
    pixel_vectors(n_pix, alpha, delta, T.nv);
    const int NW = nw_force ? nw_force : (n_f0 <= 64 ? 2 : 3);
    const TableGeometry tg =
        table_geometry(n_sft, v_over_c, n_P, P, n_ap, ap, k_band0, k_slab0, n_f0, n_bins, NW, force_clamp != 0);
    // D table, canonical order (mirrors dtable_kernel, R = 1 layout)
    T.dtab.assign((size_t)n_pix * T.n_pad, 0.0);
    for (int pix = 0; pix < n_pix; ++pix)
        for (int i = 0; i < n_sft; ++i) {
            const double a = dmul(v_over_c[3 * i + 0], T.nv[3 * pix + 0]);
            const double b = dmul(v_over_c[3 * i + 1], T.nv[3 * pix + 1]);
            const double c = dmul(v_over_c[3 * i + 2], T.nv[3 * pix + 2]);
            T.dtab[(size_t)pix * T.n_pad + i] = dadd(dadd(a, b), c);
        }
    // window table (mirrors prep_table_kernel)
    const int row_words = (n_bins + 31) / 32, off_words = tg.off_table / 32;
    T.wtab.assign((size_t)T.n_pad * tg.n_entries, uint4{0, 0, 0, 0});
    T.w_pad.assign(T.n_pad, 0.f);
    for (int i = 0; i < n_sft; ++i) {
        for (int e = 0; e < tg.n_entries; ++e) {
            uint32_t v[4];
            for (int c = 0; c < 4; ++c) {
                const int wd = e + c - off_words;
                v[c] = (wd >= 0 && wd < row_words) ? peak[(size_t)i * words_per_row + wd] : 0u;
            }
            T.wtab[(size_t)i * tg.n_entries + e] = uint4{v[0], v[1], v[2], v[3]};
        }
        T.w_pad[i] = w ? w[i] : 1.0f;
    }
    if (info) { info[0] = tg.clamp; info[1] = tg.n_entries; info[2] = NW; info[3] = tg.s_max; }
    const int HP = n_sft < (1 << 11) ? 6 : 8;
#define RUN(NW_, HP_, CL_)                                                                                                \
    if (NW == NW_ && HP == HP_ && tg.clamp == CL_ && weighted == 2) {                                                     \
        run_pix<NW_, HP_, CL_>(n_sft, n_pix, n_ap, n_P, n_tasc, n_f0, k_band0, k_slab0, n_bins, peak, words_per_row, T, tg,  \
                               counts);                                                                                   \
        return 0;                                                                                                         \
    }                                                                                                                     \
    if (NW == NW_ && HP == HP_ && tg.clamp == CL_) {                                                                      \
        run<NW_, HP_, CL_>(n_sft, n_pix, n_ap, n_P, n_tasc, n_f0, k_band0, k_slab0, T, tg, weighted, counts, wcounts);    \
        return 0;                                                                                                         \
    }
    RUN(1, 6, false) RUN(1, 6, true) RUN(2, 6, false) RUN(2, 6, true) RUN(3, 6, false) RUN(3, 6, true)
    RUN(2, 8, false) RUN(2, 8, true) RUN(3, 8, false) RUN(3, 8, true)
    return -1;
}
