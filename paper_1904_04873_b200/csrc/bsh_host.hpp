// bsh_host.hpp -- host-side (plain C++) pieces of the stage-1/2 setup: the cos/sin tables of DESIGN.md R-5 (the only
// transcendental evaluations of the whole path, by libm), the pixel unit vectors, and the geometry of the window table.
// Used by bsh_api.cu and by the GPU-less host emulation test (tests/hostemu).  Shares nothing with oracle/.
#pragma once
#include <math.h>
#include <stdint.h>

#include <algorithm>
#include <vector>

namespace bsh {

constexpr int kHostChunk = 64;     // SFT padding granularity (= kChunk of the kernels)

inline int pad_sfts(int n) { return (n + kHostChunk - 1) / kHostChunk * kHostChunk; }

// cs[p][i] = (cos, sin)(Omega_p t_i) for i < n_sft, (0, 0) for the padding SFTs;  casa[p][q] = (cos, sin)(Omega_p t_asc),
// t_asc = t_search_mid + frac_q P_p (Eq. 35);  A[a][p] = a_p Omega_p;  Omega_p = (2 pi) / P_p (L61).
// Eccentric grids (Eq. 14; n_ecc > 0): the kernels see ONE combined axis tq = q n_ecc + e of n_tasc n_ecc entries -- casa is
// replicated over e, and ke[tq] = (e cos omega, e sin omega)_e -- so the template index keeps its R-11 form with the
// eccentricity pair between t_asc and f0.
inline void build_binary_tables(int n_sft, int n_pad, const double *t_mid, double t_search_mid, int n_P, const double *P,
                                int n_tasc, const double *tasc_frac, int n_ap, const double *ap, std::vector<double> &cs,
                                std::vector<double> &casa, std::vector<double> &A, int n_ecc = 0,
                                const double *ecosw = nullptr, const double *esinw = nullptr,
                                std::vector<double> *ke = nullptr)
{
    const int ne = n_ecc > 0 ? n_ecc : 1;
    cs.assign((size_t)n_P * n_pad * 2, 0.0);
    casa.assign((size_t)n_P * n_tasc * ne * 2, 0.0);
    A.assign((size_t)n_ap * n_P, 0.0);
    if (ke) {
        ke->assign((size_t)n_tasc * ne * 2, 0.0);
        for (int q = 0; q < n_tasc; ++q)
            for (int e = 0; e < n_ecc; ++e) {
                (*ke)[((size_t)q * ne + e) * 2 + 0] = ecosw[e];
                (*ke)[((size_t)q * ne + e) * 2 + 1] = esinw[e];
            }
    }
    const double two_pi = 2.0 * M_PI;
    for (int p = 0; p < n_P; ++p) {
        const double Pp = P[p];
        const double Om = two_pi / Pp;
        for (int i = 0; i < n_sft; ++i) {
            const double arg = Om * t_mid[i];
            cs[((size_t)p * n_pad + i) * 2 + 0] = cos(arg);
            cs[((size_t)p * n_pad + i) * 2 + 1] = sin(arg);
        }
        for (int q = 0; q < n_tasc; ++q) {
            const double fp = tasc_frac[q] * Pp;
            const double ta = t_search_mid + fp;
            const double arg = Om * ta;
            const double ca = cos(arg), sa = sin(arg);
            for (int e = 0; e < ne; ++e) {
                casa[(((size_t)p * n_tasc + q) * ne + e) * 2 + 0] = ca;
                casa[(((size_t)p * n_tasc + q) * ne + e) * 2 + 1] = sa;
            }
        }
        for (int a = 0; a < n_ap; ++a) A[(size_t)a * n_P + p] = ap[a] * Om;
    }
}

// n = (cos d cos a, cos d sin a, sin d)
inline void pixel_vectors(int n_pix, const double *alpha, const double *delta, std::vector<double> &nv)
{
    nv.resize((size_t)n_pix * 3);
    for (int p = 0; p < n_pix; ++p) {
        const double cd = cos(delta[p]);
        nv[3 * p + 0] = cd * cos(alpha[p]);
        nv[3 * p + 1] = cd * sin(alpha[p]);
        nv[3 * p + 2] = sin(delta[p]);
    }
}

// Geometry of the window table for a slab of n_bins columns and windows of NW words.
//   clamp == false: proven that every window of every template lies inside the slab; table coordinates = slab columns.
//   clamp == true : table coordinates = slab column + off_table, with NW + 1 zero words in front and one behind, and the
//                   start position clamped to [0, s_max] (a clamped window reads only zeros).
//   s_zero: a table position whose window is all zero in both geometries (the first words of the clamped table; one
//           extra all-zero entry behind the row otherwise): where the accumulation kernels park deferred breaks.
struct TableGeometry {
    bool clamp;
    int off_table, s_max, n_entries, s_zero;
};

inline TableGeometry table_geometry(int n_sft, const double *v_over_c, int n_P, const double *P, int n_ap, const double *ap,
                                    int64_t k_band0, int64_t k_slab0, int n_f0, int n_bins, int NW, bool force_clamp,
                                    double ecc_max = 0.0 /* max |e cos w| + |e sin w| of the grid (Eq. 14) */)
{
    double vmax = 0;
    for (int i = 0; i < n_sft; ++i) {
        const double *v = v_over_c + 3 * (size_t)i;
        vmax = std::max(vmax, sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]));
    }
    double pmin = P[0], apmax = 0;
    for (int p = 0; p < n_P; ++p) pmin = std::min(pmin, P[p]);
    for (int a = 0; a < n_ap; ++a) apmax = std::max(apmax, fabs(ap[a]));
    const double amax = apmax * 2.0 * M_PI / pmin * (1.0 + ecc_max);   // |cos phi + k cos 2 phi - h sin 2 phi| <= 1 + |k| + |h|
    // |r| <= |y| + 1/2 rounded, |y| <= u_max (|v|/c + a_p Omega); generous relative slack for the rounded operations
    const double rmax = floor((double)(k_band0 + n_f0) * (vmax * 1.000001 + amax * 1.000001) + 0.5) + 1.0;
    const int64_t m = k_band0 - k_slab0;
    TableGeometry g;
    g.clamp = force_clamp || !((double)m - rmax >= 0.0 && (double)(m + n_f0 - 1) + rmax <= (double)(n_bins - 1));
    const int row_words = (n_bins + 31) / 32;
    if (g.clamp) {
        g.off_table = 32 * (NW + 1);
        g.s_max = g.off_table + 32 * row_words;
        g.n_entries = (g.s_max >> 5) + 1;
        g.s_zero = 0;
    } else {
        g.off_table = 0;
        g.s_max = n_bins - 1;
        g.n_entries = (g.s_max >> 5) + 2;
        g.s_zero = 32 * (g.n_entries - 1);
    }
    return g;
}

// Geometry of the position table (pre-shifted windows, bsh_core.cuh) derived from the window-table geometry `tg`:
//   clamp == false: position = slab column of tile bin 0, valid range [0, K - w_min] (w_min = narrowest f0 tile);
//                   one extra all-zero position behind it (s_zero).
//   clamp == true : position = slab column + 32 NW, clamped to [0, K + 32 NW]; both ends are all-zero windows.
struct PosGeometry {
    int off_table, s_max, n_pos, s_zero;
};

inline PosGeometry pos_geometry(const TableGeometry &tg, int n_bins, int n_f0, int NW, int tile_bins = 0)
{
    PosGeometry g;
    if (tg.clamp) {
        g.off_table = 32 * NW;
        g.s_max = n_bins + 32 * NW;
        g.n_pos = g.s_max + 1;
        g.s_zero = 0;
    } else {
        const int tile = tile_bins > 0 ? tile_bins : 32 * NW;
        const int w_min = n_f0 <= tile ? n_f0 : ((n_f0 % tile) ? (n_f0 % tile) : tile);
        g.off_table = 0;
        g.s_max = n_bins - w_min;
        g.s_zero = g.s_max + 1;
        g.n_pos = g.s_max + 2;
    }
    return g;
}

inline int pick_threads_per_block(int n_aq)
{
    int best = 64;
    double best_eff = 0;
    for (int t = 256; t >= 64; t -= 32) {
        const int tiles = (n_aq + t - 1) / t;
        const double eff = (double)n_aq / ((double)tiles * t);
        if (eff > best_eff + 1e-9) { best_eff = eff; best = t; }
    }
    return best;
}

}  // namespace bsh
