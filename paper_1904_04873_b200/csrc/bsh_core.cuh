// bsh_core.cuh -- per-thread arithmetic of the stage-1 accumulation: canonical track (R-5), window extraction from
// the staged peakgram, exact break handling across the f0 band (R-7), bit-sliced carry-save counters (unweighted) and
// FP32 accumulators (weighted), and the threshold epilogue.  Header-only, __host__ __device__, so the same logic can be
// exercised by the host-side emulation test (tests/hostemu) without a GPU.  Nothing here is shared with oracle/.
//
// PAPER.md L102 Eq. (15): f(t) = f0 [1 + v.n/c - a_p Omega cos(Omega (t - t_asc))]; the slab column of template j at
// SFT i is  k = m + j + r,  r = round(y) (nearest, ties to even),  y = fl(u_j g),  u_j = k_band0 + j,  g = fl(D - fl(A cphi)),
// cphi = fl(fl(C CA) + fl(S SA))  (R-5).  All FP64 operations are individually rounded (no FMA).
#pragma once
#include <stdint.h>
#include <math.h>

#if defined(__CUDACC__)
#define BSH_HD __host__ __device__ __forceinline__
#define BSH_HD_NOINLINE __host__ __device__ __noinline__
#else
#define BSH_HD inline
#define BSH_HD_NOINLINE
struct uint4 { uint32_t x, y, z, w; };
#endif

namespace bsh {

constexpr double kMagic = 6755399441055744.0;   // 1.5 * 2^52: fl(y + kMagic) carries round-to-nearest-even(y) in its low word
constexpr int kMaxWords = 3;                    // f0 bins per pass <= 96 (three 32-bit window words)
constexpr int kLowPlanes = 5;                   // carry-save levels = log2(SFTs per unrolled block)
constexpr int kBlock = 32;                      // SFTs per unrolled block

BSH_HD double dmul(double a, double b)
{
#ifdef __CUDA_ARCH__
    return __dmul_rn(a, b);
#else
    return a * b;                                // host translation units are built with -ffp-contract=off
#endif
}
BSH_HD double dadd(double a, double b)
{
#ifdef __CUDA_ARCH__
    return __dadd_rn(a, b);
#else
    return a + b;
#endif
}
BSH_HD double dsub(double a, double b)
{
#ifdef __CUDA_ARCH__
    return __dsub_rn(a, b);
#else
    return a - b;
#endif
}

// r = y rounded to the nearest integer, ties to even (IEEE-754 default rounding; R-1), |y| < 2^31: the
// low word of fl(y + 1.5 2^52) on the device (one FP64 add), nearbyint() on the host.
BSH_HD int32_t round_int(double y)
{
#ifdef __CUDA_ARCH__
    return __double2loint(__dadd_rn(y, kMagic));
#else
    return (int32_t)nearbyint(y);
#endif
}

// s = off + round(fl(u g))
BSH_HD int32_t shift_of(double u, double g, int32_t off) { return off + round_int(dmul(u, g)); }

BSH_HD uint32_t funnel_r(uint32_t lo, uint32_t hi, int sh)   // low 32 bits of ((hi:lo) >> (sh & 31))
{
#ifdef __CUDA_ARCH__
    return __funnelshift_r(lo, hi, sh);
#else
    return (uint32_t)(((((uint64_t)hi) << 32) | lo) >> (sh & 31));
#endif
}

BSH_HD uint32_t xor3(uint32_t a, uint32_t b, uint32_t c)
{
#ifdef __CUDA_ARCH__
    uint32_t r;
    asm("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(r) : "r"(a), "r"(b), "r"(c));
    return r;
#else
    return a ^ b ^ c;
#endif
}
BSH_HD uint32_t maj3(uint32_t a, uint32_t b, uint32_t c)
{
#ifdef __CUDA_ARCH__
    uint32_t r;
    asm("lop3.b32 %0, %1, %2, %3, 0xE8;" : "=r"(r) : "r"(a), "r"(b), "r"(c));
    return r;
#else
    return (a & b) | (a & c) | (b & c);
#endif
}

// ---------------------------------------------------------------------------------------------------------------------
// Per-thread constants of one (binary template, f0 tile).
// ---------------------------------------------------------------------------------------------------------------------
struct TrackConst {
    double u0, uL;      // k_band0 + j0  and  k_band0 + j0 + n_fj - 1
    double A;           // fl(a_p Omega)
    double CA, SA;      // cos / sin (Omega t_asc)  (host libm table values)
    double kap, eta;    // e cos(omega), e sin(omega) of the ELL1 track, Eq. (14) (0, 0: circular orbit, Eq. 15)
    double magic;       // kMagic + off
    int32_t off;        // m + j0 + table offset: s = off + r is the bit position of tile bin 0 in table coordinates
    int32_t s_max;      // clamp range [0, s_max] of s (table coordinates); only used by CLAMP variants
    int32_t s_zero;     // a table position whose NW-word window reads only zeros (deferred breaks park there)
    int32_t n_fj;       // f0 bins in this tile (<= 32 * NW)
};

template <int NW>
struct Win {
    uint32_t x[NW];
};

// Window table (built by the prep kernel): entry e of SFT i holds the four row words covering table bits
// [32 e, 32 e + 128); table bit b is slab column (b - table_offset), zero outside [0, K).  One 16-byte load gives the
// NW + 1 words a window starting at any bit of entry e needs.
template <int NW>
BSH_HD Win<NW> load_window(const uint4 *row_entries, int32_t s)
{
    const uint4 e = row_entries[s >> 5];
    Win<NW> w;
    w.x[0] = funnel_r(e.x, e.y, s);
    if (NW > 1) w.x[1 % NW] = funnel_r(e.y, e.z, s);
    if (NW > 2) w.x[2 % NW] = funnel_r(e.z, e.w, s);
    return w;
}

BSH_HD int32_t clamp_s(int32_t s, int32_t s_max) { return s < 0 ? 0 : (s > s_max ? s_max : s); }

// One table bit by absolute table position p; entries beyond the last one are read from its trailing words.
BSH_HD uint32_t table_bit(const uint4 *row_entries, int32_t p, int32_t e_last)
{
    const int32_t e = p >> 5;
    if (p < 0 || e > e_last + 3) return 0u;
    uint32_t word;
    if (e <= e_last) {
        word = row_entries[e].x;
    } else {
        const uint4 q = row_entries[e_last];
        const int k = e - e_last;
        word = k == 1 ? q.y : (k == 2 ? q.z : q.w);
    }
    return (word >> (p & 31)) & 1u;
}

// Exact window when the rounded shift is NOT the same at both ends of the f0 tile (R-7).  y_j = fl(u_j g) is monotone
// in j, so r_j is monotone; with |s_L - s_0| == 1 there is exactly one break, located by bisection on the canonical
// evaluation itself; otherwise (only possible for unphysically large |g| n_f) every bin is evaluated on its own.
template <int NW, bool CLAMP>
BSH_HD_NOINLINE Win<NW> break_window(const uint4 *row_entries, double g, double u0, double magic, int32_t off, int32_t n_fj,
                            int32_t s_max, int32_t s0, int32_t sL)
{
    Win<NW> out;
    const int32_t d = sL - s0;
    if (d == 1 || d == -1) {
        int lo = 0, hi = n_fj - 1;                       // shift(lo) == s0, shift(hi) == sL
        while (hi - lo > 1) {
            const int mid = (lo + hi) >> 1;
            const int32_t sm = shift_of(dadd(u0, (double)mid), g, off);
            if (sm == s0) lo = mid; else hi = mid;
        }
        const Win<NW> a = load_window<NW>(row_entries, CLAMP ? clamp_s(s0, s_max) : s0);
        const Win<NW> b = load_window<NW>(row_entries, CLAMP ? clamp_s(sL, s_max) : sL);
#pragma unroll
        for (int w = 0; w < NW; ++w) {
            const int rel = hi - 32 * w;                 // bins j >= hi take the second window
            const uint32_t m = rel <= 0 ? 0xFFFFFFFFu : (rel >= 32 ? 0u : (0xFFFFFFFFu << rel));
            out.x[w] = (a.x[w] & ~m) | (b.x[w] & m);
        }
        return out;
    }
#pragma unroll
    for (int w = 0; w < NW; ++w) out.x[w] = 0u;
    for (int j = 0; j < n_fj; ++j) {
        const int32_t sj = shift_of(dadd(u0, (double)j), g, off);
        const uint32_t bit = table_bit(row_entries, sj + j, s_max >> 5);
#pragma unroll
        for (int w = 0; w < NW; ++w)
            if ((j >> 5) == w) out.x[w] |= bit << (j & 31);
    }
    return out;
}

// The NW-word window of peakgram bits that the n_fj templates of this tile read at one SFT.
template <int NW, bool CLAMP>
BSH_HD Win<NW> track_window(const TrackConst &tc, const uint4 *row_entries, double D, double B)
{
    const double g = dsub(D, B);
    const int32_t s0 = shift_of(tc.u0, g, tc.off);
    const int32_t sL = shift_of(tc.uL, g, tc.off);
    if (s0 != sL) return break_window<NW, CLAMP>(row_entries, g, tc.u0, tc.magic, tc.off, tc.n_fj, tc.s_max, s0, sL);
    return load_window<NW>(row_entries, CLAMP ? clamp_s(s0, tc.s_max) : s0);
}

// Main-loop form of track_window(): when the rounded shift differs between the two ends of the f0 tile (a "break",
// ~1 % of (pixel, binary template, SFT) triples, R-7) the thread reads the all-zero window at s_zero instead and reports
// brk = true; the caller records the SFT and later adds the exact window (track_window + add_window).  This keeps the
// hot loop free of divergent code; the sum over SFTs is order-independent for the integer count.
template <int NW, bool CLAMP>
BSH_HD Win<NW> track_window_deferred(const TrackConst &tc, const uint4 *row_entries, double D, double B, bool &brk)
{
    const double g = dsub(D, B);
    const int32_t s0 = shift_of(tc.u0, g, tc.off);
    const int32_t sL = shift_of(tc.uL, g, tc.off);
    brk = s0 != sL;
    int32_t s = CLAMP ? clamp_s(s0, tc.s_max) : s0;
    s = brk ? tc.s_zero : s;
    return load_window<NW>(row_entries, s);
}

// The bracket of the binary term of Eq. (14) (L95-L98):  cos phi + kap cos 2 phi - eta sin 2 phi,  phi = Omega (t - t_asc),
// from the table values (C, S) = (cos, sin)(Omega t), (CA, SA) = (cos, sin)(Omega t_asc) with rounded +, -, * only
// (R-23):  cos phi = fl(fl(C CA) + fl(S SA)),  sin phi = fl(fl(S CA) - fl(C SA)),
// cos 2 phi = fl(fl(cos^2 phi) - fl(sin^2 phi)),  sin 2 phi = fl(fl(2 sin phi) cos phi),
// E = fl(fl(kap cos 2 phi) - fl(eta sin 2 phi)),  bracket = fl(cos phi + E).  kap = eta = 0 is Eq. (15): cos phi.
BSH_HD double orbit_bracket(double C, double S, double CA, double SA, double kap, double eta)
{
    const double cphi = dadd(dmul(C, CA), dmul(S, SA));
    if (kap == 0.0 && eta == 0.0) return cphi;
    const double sphi = dsub(dmul(S, CA), dmul(C, SA));
    const double cos2 = dsub(dmul(cphi, cphi), dmul(sphi, sphi));
    const double sin2 = dmul(dmul(2.0, sphi), cphi);
    const double E = dsub(dmul(kap, cos2), dmul(eta, sin2));
    return dadd(cphi, E);
}

BSH_HD double binary_term(const TrackConst &tc, double C, double S)   // B = fl(A bracket)
{
    return dmul(tc.A, orbit_bracket(C, S, tc.CA, tc.SA, tc.kap, tc.eta));
}

// ---------------------------------------------------------------------------------------------------------------------
// Pre-shifted window table ("position table"): entry p of SFT i holds the NW window words of a window STARTING at table
// position p (x, y, z = words 0..2; w unused), so the hot loop needs no funnel shift and no entry/bit split: one 16-byte
// load at row + p.  Position p is slab column (p - off_table) of tile bin 0; bits outside [0, K) are zero.  TrackConst
// is used unchanged: s = off + r is the position, [0, s_max] the clamp range, s_zero an all-zero position.
// ---------------------------------------------------------------------------------------------------------------------
template <int NW>
BSH_HD Win<NW> load_position(const uint4 *row_positions, int32_t s)
{
    const uint4 e = row_positions[s];
    Win<NW> w;
    w.x[0] = e.x;
    if (NW > 1) w.x[1 % NW] = e.y;
    if (NW > 2) w.x[2 % NW] = e.z;
    return w;
}

// Exact window of a break (R-7) from the position table: one break -> blend of the two neighbouring positions at the
// break bin (located on the canonical evaluation itself); several breaks -> every bin from its own position.
template <int NW, bool CLAMP>
BSH_HD_NOINLINE Win<NW> break_window_pos(const uint4 *row_positions, double g, double u0, double magic, int32_t off,
                                         int32_t n_fj, int32_t s_max, int32_t s0, int32_t sL)
{
    Win<NW> out;
    const int32_t d = sL - s0;
    if (d == 1 || d == -1) {
        int lo = 0, hi = n_fj - 1;                       // shift(lo) == s0, shift(hi) == sL
        while (hi - lo > 1) {
            const int mid = (lo + hi) >> 1;
            const int32_t sm = shift_of(dadd(u0, (double)mid), g, off);
            if (sm == s0) lo = mid; else hi = mid;
        }
        const Win<NW> a = load_position<NW>(row_positions, CLAMP ? clamp_s(s0, s_max) : s0);
        const Win<NW> b = load_position<NW>(row_positions, CLAMP ? clamp_s(sL, s_max) : sL);
#pragma unroll
        for (int w = 0; w < NW; ++w) {
            const int rel = hi - 32 * w;                 // bins j >= hi take the second window
            const uint32_t m = rel <= 0 ? 0xFFFFFFFFu : (rel >= 32 ? 0u : (0xFFFFFFFFu << rel));
            out.x[w] = (a.x[w] & ~m) | (b.x[w] & m);
        }
        return out;
    }
#pragma unroll
    for (int w = 0; w < NW; ++w) out.x[w] = 0u;
    for (int j = 0; j < n_fj; ++j) {
        int32_t sj = shift_of(dadd(u0, (double)j), g, off);
        sj = clamp_s(sj, s_max);                         // in the unclamped geometry this is the identity (proven range)
        const uint4 e = row_positions[sj];
        const uint32_t word = (j >> 5) == 0 ? e.x : ((j >> 5) == 1 ? e.y : e.z);
        const uint32_t bit = (word >> (j & 31)) & 1u;
#pragma unroll
        for (int w = 0; w < NW; ++w)
            if ((j >> 5) == w) out.x[w] |= bit << (j & 31);
    }
    return out;
}

template <int NW, bool CLAMP>
BSH_HD Win<NW> track_window_pos(const TrackConst &tc, const uint4 *row_positions, double D, double B)
{
    const double g = dsub(D, B);
    const int32_t s0 = shift_of(tc.u0, g, tc.off);
    const int32_t sL = shift_of(tc.uL, g, tc.off);
    if (s0 != sL) return break_window_pos<NW, CLAMP>(row_positions, g, tc.u0, tc.magic, tc.off, tc.n_fj, tc.s_max, s0, sL);
    return load_position<NW>(row_positions, CLAMP ? clamp_s(s0, tc.s_max) : s0);
}

// Hot-loop form: the position to read (the all-zero position on a break) and the break flag.
template <bool CLAMP>
BSH_HD int32_t track_position_deferred(const TrackConst &tc, double D, double B, bool &brk)
{
    const double g = dsub(D, B);
    int32_t s0 = shift_of(tc.u0, g, tc.off);
    int32_t sL = shift_of(tc.uL, g, tc.off);
    if (CLAMP) { s0 = clamp_s(s0, tc.s_max); sL = clamp_s(sL, tc.s_max); }   // equal after clamping => every bin reads 0
    brk = s0 != sL;
    return brk ? tc.s_zero : s0;
}

// ---------------------------------------------------------------------------------------------------------------------
// Unweighted: bit-sliced counter.  32 lanes of a word are 32 f0 bins; plane p holds bit p of each bin's count.
// Inputs arrive in blocks of 32 SFTs; within a block a carry-save adder tree (one full adder = 2 LOP3 per word) keeps
// planes 0..4 and emits one weight-32 carry per block, which is rippled into the HP high planes.
// ---------------------------------------------------------------------------------------------------------------------
template <int NW, int HP>
struct Counter {
    uint32_t low[kLowPlanes][NW];
    uint32_t hold[kLowPlanes][NW];
    uint32_t hi[HP][NW];
    uint32_t over[NW];                                   // carries out of the last high plane (weight 2^(5 + HP)); stays 0
                                                         // when HP covers the SFT count, else the kernel spills it
    BSH_HD void clear()
    {
#pragma unroll
        for (int w = 0; w < NW; ++w) {
            over[w] = 0u;
#pragma unroll
            for (int l = 0; l < kLowPlanes; ++l) { low[l][w] = 0u; hold[l][w] = 0u; }
#pragma unroll
            for (int p = 0; p < HP; ++p) hi[p][w] = 0u;
        }
    }
};

template <int K, int L, int NW, int HP>
BSH_HD void push_level(Counter<NW, HP> &c, Win<NW> &x)
{
    if constexpr (L == kLowPlanes) {
#pragma unroll
        for (int p = 0; p < HP; ++p)
#pragma unroll
            for (int w = 0; w < NW; ++w) {
                const uint32_t t = c.hi[p][w] & x.x[w];
                c.hi[p][w] ^= x.x[w];
                x.x[w] = t;
            }
#pragma unroll
        for (int w = 0; w < NW; ++w) c.over[w] |= x.x[w];
    } else if constexpr (((K >> L) & 1) == 0) {
#pragma unroll
        for (int w = 0; w < NW; ++w) c.hold[L][w] = x.x[w];
    } else {
#pragma unroll
        for (int w = 0; w < NW; ++w) {
            const uint32_t s = c.low[L][w], h = c.hold[L][w], v = x.x[w];
            c.low[L][w] = xor3(s, h, v);
            x.x[w] = maj3(s, h, v);
        }
        push_level<K, L + 1, NW, HP>(c, x);
    }
}

// K = position of this SFT inside its block of 32 (compile-time, so the tree is straight-line code)
template <int K, int NW, int HP>
BSH_HD void push(Counter<NW, HP> &c, Win<NW> x)
{
    push_level<K, 0, NW, HP>(c, x);
}

// Ripple-carry add of one window (one bit per bin) into the counter.  Only valid between blocks of kBlock SFTs, when
// no input is parked in the hold registers.
template <int NW, int HP>
BSH_HD void add_window(Counter<NW, HP> &c, Win<NW> x)
{
#pragma unroll
    for (int w = 0; w < NW; ++w) {
        uint32_t carry = x.x[w];
#pragma unroll
        for (int l = 0; l < kLowPlanes; ++l) {
            const uint32_t t = c.low[l][w] & carry;
            c.low[l][w] ^= carry;
            carry = t;
        }
#pragma unroll
        for (int p = 0; p < HP; ++p) {
            const uint32_t t = c.hi[p][w] & carry;
            c.hi[p][w] ^= carry;
            carry = t;
        }
    }
}

template <int NW, int HP>
BSH_HD uint32_t plane_word(const Counter<NW, HP> &c, int p, int w)
{
    return p < kLowPlanes ? c.low[p][w] : c.hi[p - kLowPlanes][w];
}

// mask of bins whose count >= tau (tau uniform).  Planes hold counts < 2^(5 + HP).
template <int NW, int HP>
BSH_HD Win<NW> count_ge(const Counter<NW, HP> &c, int32_t tau)
{
    Win<NW> ge;
    constexpr int NP = kLowPlanes + HP;
    if (tau <= 0) {
#pragma unroll
        for (int w = 0; w < NW; ++w) ge.x[w] = 0xFFFFFFFFu;
        return ge;
    }
    if (tau >= (1 << NP)) {
#pragma unroll
        for (int w = 0; w < NW; ++w) ge.x[w] = 0u;
        return ge;
    }
#pragma unroll
    for (int w = 0; w < NW; ++w) {
        uint32_t gt = 0u, eq = 0xFFFFFFFFu;
#pragma unroll
        for (int p = NP - 1; p >= 0; --p) {
            const uint32_t pl = plane_word(c, p, w);
            if ((tau >> p) & 1) {
                eq &= pl;
            } else {
                gt |= eq & pl;
                eq &= ~pl;
            }
        }
        ge.x[w] = gt | eq;
    }
    return ge;
}

// count of bin (32 w + b); w must be a compile-time constant at the call site (unrolled loop) so that the counter
// planes are only ever indexed statically and stay in registers.
template <int NW, int HP>
BSH_HD int32_t count_at(const Counter<NW, HP> &c, int w, int b)
{
    constexpr int NP = kLowPlanes + HP;
    int32_t n = 0;
#pragma unroll
    for (int p = 0; p < NP; ++p) n |= (int32_t)((plane_word(c, p, w) >> b) & 1u) << p;
    return n;
}

// ---------------------------------------------------------------------------------------------------------------------
// Lean resolution of deferred breaks (used by the pixel-lane kernel, bsh_pix.cuh; __host__ __device__ so that the host
// emulation test runs the same code).
// ---------------------------------------------------------------------------------------------------------------------
#ifndef BSH_FIX_SHORTCUT
#define BSH_FIX_SHORTCUT 1
#endif
BSH_HD float fast_divide(float a, float b)
{
#ifdef __CUDA_ARCH__
    return __fdividef(a, b);
#else
    return a / b;
#endif
}

// Exact window of a (pixel, template, SFT) whose rounded shift is not the same at both ends of the f0 tile (R-7).
// One break (|sL - s0| == 1): r_j is monotone in j, so there is one bin jb with shift(jb - 1) == s0, shift(jb) == sL.
// jb is estimated from the distance of fl(u0 g) to the half-integer it crosses (FP32 division) and then corrected on
// the canonical evaluation itself -- the estimate only saves work, the result is exact.  More breaks (unphysical
// |g| n_f) or clamped positions: the generic per-bin routine of bsh_core.cuh.
template <int NW, bool CLAMP>
BSH_HD Win<NW> exact_window_pos(const TrackConst &tc, const uint4 *row_positions, double D, double B)
{
    const double g = dsub(D, B);
    const double y0 = dmul(tc.u0, g);
    const int32_t r0 = round_int(y0);
    const int32_t s0 = tc.off + r0;
    const int32_t sL = shift_of(tc.uL, g, tc.off);
    const int32_t d = sL - s0;
    if (CLAMP || (d != 1 && d != -1)) return track_window_pos<NW, CLAMP>(tc, row_positions, D, B);
    const float dist = (float)(((double)r0 + (d > 0 ? 0.5 : -0.5)) - y0);     // signed distance to the crossed half-integer
    const float t = fast_divide(dist, (float)g);         // the crossing in units of j: y_j = y_0 + j g up to 1e-14
    int j = (int)ceilf(t);
    // Error of t against the true crossing of the canonical y_j = fl(fl(u_0 + j) g), in bins of j (|t| < 2^7):
    //   FP32: the two conversions and the division, __fdividef being good to 2 ulp: (1 + 1 + 2) 6e-8 2^7 < 4e-5;
    //   FP64: y_0 and y_j each carry a rounding of <= |y| 2^-53, and so does forming dist; divided by |g| that is
    //         <= 3 u 2^-53 < 1e-6 for u < 2^32 (validate() in bsh_api.cu enforces k_band0 + n_f0 < 2^32).
    // Together < 5e-5, a twentieth of the guard: when t lies further than 1e-3 from an integer, ceil(t) IS the first bin
    // with the new shift and the canonical re-evaluation is skipped (99.8 % of breaks); otherwise it is re-evaluated.
    const bool sure = BSH_FIX_SHORTCUT && fabsf(t - rintf(t)) > 1e-3f && j >= 1 && j <= tc.n_fj - 1;
    if (!sure) {
        j = j < 1 ? 1 : (j > tc.n_fj - 1 ? tc.n_fj - 1 : j);
        while (j > 1 && shift_of(dadd(tc.u0, (double)(j - 1)), g, tc.off) != s0) --j;
        while (j < tc.n_fj - 1 && shift_of(dadd(tc.u0, (double)j), g, tc.off) == s0) ++j;
    }
    const Win<NW> a = load_position<NW>(row_positions, s0);
    const Win<NW> b = load_position<NW>(row_positions, sL);
    Win<NW> out;
#pragma unroll
    for (int w = 0; w < NW; ++w) {
        const int rel = j - 32 * w;                      // bins >= j take the second window
        const uint32_t m = rel <= 0 ? 0xFFFFFFFFu : (rel >= 32 ? 0u : (0xFFFFFFFFu << rel));
        out.x[w] = (a.x[w] & ~m) | (b.x[w] & m);
    }
    return out;
}

// The deferred windows of one flush are first summed in a small bit-sliced accumulator (kFixPlanes planes, ripple
// carry: 2 kFixPlanes LOP per word and window instead of 2 (5 + HP)), which is then added to the counter once.
constexpr int kFixPlanes = 7;                            // up to 127 windows per flush (kListCap = 120)

template <int NW>
BSH_HD void fix_accumulate(uint32_t (&tp)[kFixPlanes][NW], const Win<NW> &x)
{
#pragma unroll
    for (int w = 0; w < NW; ++w) {
        uint32_t carry = x.x[w];
#pragma unroll
        for (int q = 0; q < kFixPlanes; ++q) {
            const uint32_t t = tp[q][w] & carry;
            tp[q][w] ^= carry;
            carry = t;
        }
    }
}

template <int NW, int HP>
BSH_HD void fix_merge(Counter<NW, HP> &c, const uint32_t (&tp)[kFixPlanes][NW])
{
    static_assert(kLowPlanes + HP >= kFixPlanes, "counter narrower than the fix-up accumulator");
#pragma unroll
    for (int w = 0; w < NW; ++w) {
        uint32_t carry = 0u;
#pragma unroll
        for (int q = 0; q < kLowPlanes + HP; ++q) {
            uint32_t &pl = q < kLowPlanes ? c.low[q < kLowPlanes ? q : 0][w] : c.hi[q < kLowPlanes ? 0 : q - kLowPlanes][w];
            const uint32_t a = pl, b = q < kFixPlanes ? tp[q < kFixPlanes ? q : 0][w] : 0u;
            pl = xor3(a, b, carry);
            carry = maj3(a, b, carry);
        }
        c.over[w] |= carry;
    }
}

BSH_HD uint32_t valid_mask(int n_fj, int w)
{
    const int rel = n_fj - 32 * w;
    return rel >= 32 ? 0xFFFFFFFFu : (rel <= 0 ? 0u : ((1u << rel) - 1u));
}

// ---------------------------------------------------------------------------------------------------------------------
// Weighted: one FP32 accumulator per f0 bin, sequential in SFT order (R-20).
// ---------------------------------------------------------------------------------------------------------------------
template <int NW>
BSH_HD void accumulate_weighted(float (&acc)[32 * NW], const Win<NW> &x, float wi)
{
#pragma unroll
    for (int w = 0; w < NW; ++w)
#pragma unroll
        for (int b = 0; b < 32; ++b)
            if ((x.x[w] >> b) & 1u) acc[32 * w + b] += wi;
}

// Candidate record appended by the accumulation kernels and consumed by the selection kernels (16 bytes).
struct RawCand {
    uint64_t index;
    uint32_t key;       // count, or the bit pattern of the non-negative FP32 weighted count (monotone as uint32)
    uint32_t pad;
};

}  // namespace bsh
