/*
 * bsh_oracle.c -- plain CPU ORACLE for the BinarySkyHough hot path.  TEST INFRASTRUCTURE ONLY.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may build, load or
 * call this file.  It shares no code, header, table or constant with the CUDA path (paper_1904_04873_b200/csrc);
 * it is written from /root/reference/PAPER.md alone:
 *
 *   peakgram      PAPER.md L176  (section IV.A): bin -> 1 if rho > rho_th (= 1.6), else 0
 *   track         PAPER.md L102  Eq. (15):  f(t) = f0 + f0 v(t).n/c - f0 a_p Omega cos[Omega (t - t_asc)],
 *                 and, for small eccentricity (ELL1), L95-L98 Eq. (14): the two further terms
 *                 - f0 a_p Omega e cos(omega) cos[2 Omega (t - t_asc)] + f0 a_p Omega e sin(omega) sin[2 Omega (t - t_asc)],
 *                 Omega = 2 pi / P (L61), a_p in seconds (L70), t_asc range Eq. (35),
 *                 f0 lattice delta f = 1/T_c (Eq. 33); bin = round((f - f_slab_start) T)  (BASELINE.json)
 *   stage 1       PAPER.md L223  (section IV.C): number count n = weighted sum of 1s and 0s along the track
 *   toplist       PAPER.md L217, L225-L229: keep the best templates of the region, ordered by the statistic
 *   stage 2       PAPER.md L227-L229 Eq. (26): P = sum of weighted normalised powers along the exact track
 *
 * Everything is FP64 (weights and powers are read as the FP32 inputs they are, then widened), compiled with
 * -ffp-contract=off so no multiply-add is fused.  Loops are literal: for template: for SFT.
 *
 * Two track modes (readings R-1, R-5):
 *   DIRECT     Eq. (15) exactly as printed, one libm cos per (template, SFT).
 *   CANONICAL  the same quantity with the operations fixed in an order that uses only table values of libm
 *              cos/sin (of Omega t_i and Omega t_asc) plus rounded +,-,* : the form in which bit-exactness
 *              against another implementation is a meaningful demand.  y = u_j * g, g = D - A*cphi.
 * tests/test_oracle_pins.py checks DIRECT == CANONICAL except at flagged near-ties, and pins both to
 * independent evaluations (50-digit mpmath brute force, a_p = 0 limit, column sums, binomial statistics,
 * injected-signal recovery).  No function here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#ifndef M_PI
#define M_PI 3.14159265358979323846
#endif

typedef struct {
    int32_t n_sft;            /* N */
    double t_sft;             /* T: SFT length = coherent time T_c, seconds; bin width 1/T (Eq. 33) */
    const double *t_mid;      /* [N] SFT mid-times, seconds (L176: "calculated at the mid-time of each SFT") */
    const double *v_over_c;   /* [N][3] detector velocity / c */
    double t_search_mid;      /* t_mid of Eq. (35) */
    int64_t k_slab0;          /* absolute bin of slab column 0 */
    int32_t n_bins;           /* K: slab columns */
    int64_t k_band0;          /* absolute bin of f0 lattice point j = 0 */
    int32_t n_f0;
    int32_t n_pix;
    const double *alpha, *delta;
    int32_t n_ap;   const double *ap;          /* seconds */
    int32_t n_P;    const double *P;           /* seconds */
    int32_t n_tasc; const double *tasc_frac;   /* t_asc = t_search_mid + frac * P, frac in [-1/2, 1/2) */
    int32_t n_ecc;  const double *ecosw, *esinw;  /* SURVEY NEXT-3, Eq. (14): [n_ecc] pairs (e cos omega, e sin omega);
                                                  n_ecc = 0: circular orbits, Eq. (15) */
} orc_problem;

static inline int n_ecc_eff(const orc_problem *pb) { return pb->n_ecc > 0 ? pb->n_ecc : 1; }
static inline double ecc_k(const orc_problem *pb, int ie) { return pb->n_ecc > 0 ? pb->ecosw[ie] : 0.0; }
static inline double ecc_h(const orc_problem *pb, int ie) { return pb->n_ecc > 0 ? pb->esinw[ie] : 0.0; }

enum { ORC_DIRECT = 0, ORC_CANONICAL = 1 };

int orc_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ---------------------------------------------------------------------------------------------------------
 * Peakgram.  Strict '>' in FP32 (R-8); NaN compares false -> 0.  Bit k of row i is bit (k & 31)
 * of word (k >> 5), least-significant bit first; pad bits are zero.
 * ------------------------------------------------------------------------------------------------------- */
void orc_peakgram(const float *rho, int32_t n_sft, int32_t n_bins, float rho_th, uint32_t *peak, int32_t words_per_row)
{
    for (int32_t i = 0; i < n_sft; ++i) {
        uint32_t *row = peak + (size_t)i * words_per_row;
        for (int32_t wd = 0; wd < words_per_row; ++wd) row[wd] = 0u;
        for (int32_t k = 0; k < n_bins; ++k)
            if (rho[(size_t)i * n_bins + k] > rho_th) row[k >> 5] |= 1u << (k & 31);
    }
}

/* ---------------------------------------------------------------------------------------------------------
 * Track, DIRECT mode: Eq. (15) as printed, then bin = round((f - f_slab_start) * T)   (R-1: to the nearest integer,
 * ties to even -- IEEE-754 round-to-nearest, nearbyint() in the default rounding mode).
 * Returns the slab column (may lie outside [0, K): such an SFT contributes nothing, R-6).
 * If x_out != NULL it receives x, the unrounded bin coordinate (for near-tie flagging).
 * ------------------------------------------------------------------------------------------------------- */
int64_t orc_track_direct(const orc_problem *pb, int pix, int ia, int ip, int it, int ie, int j, int i, double *x_out)
{
    const double T = pb->t_sft;
    const double alpha = pb->alpha[pix], delta = pb->delta[pix];
    const double nx = cos(delta) * cos(alpha), ny = cos(delta) * sin(alpha), nz = sin(delta);
    const double *v = pb->v_over_c + 3 * (size_t)i;
    const double v_dot_n = v[0] * nx + v[1] * ny + v[2] * nz;           /* v(t).n / c */
    const double f0 = (double)(pb->k_band0 + j) / T;                    /* lattice, Eq. (33) */
    const double P = pb->P[ip];
    const double Omega = 2.0 * M_PI / P;                                /* L61 */
    const double t_asc = pb->t_search_mid + pb->tasc_frac[it] * P;      /* Eq. (35) */
    const double a_p = pb->ap[ia];
    double f = f0 + f0 * v_dot_n - f0 * a_p * Omega * cos(Omega * (pb->t_mid[i] - t_asc));         /* Eq. (15) */
    if (pb->n_ecc > 0) {                                                /* Eq. (14): the O(e) terms of the ELL1 model */
        const double ecw = pb->ecosw[ie], esw = pb->esinw[ie];
        f = f - f0 * a_p * Omega * ecw * cos(2.0 * Omega * (pb->t_mid[i] - t_asc))
              + f0 * a_p * Omega * esw * sin(2.0 * Omega * (pb->t_mid[i] - t_asc));
    }
    const double f_slab = (double)pb->k_slab0 / T;
    const double x = (f - f_slab) * T;
    if (x_out) *x_out = x;
    return (int64_t)nearbyint(x);
}

/* ---------------------------------------------------------------------------------------------------------
 * Track, CANONICAL mode (R-5).  Same quantity, written x = (k_band0 - k_slab0) + j + y with
 *   y = u_j * g,  u_j = k_band0 + j  (= f0_j * T, an exact integer),  g = v.n/c - a_p Omega cos[Omega(t - t_asc)]
 * and cos[Omega(t - t_asc)] = cos(Omega t) cos(Omega t_asc) + sin(Omega t) sin(Omega t_asc).
 * Every operation below is one rounded FP64 operation in the order written.
 * Eccentric tracks (Eq. 14; R-23): g = v.n/c - A [cos phi + k cos 2 phi - h sin 2 phi], k = e cos(omega),
 * h = e sin(omega), phi = Omega (t - t_asc), with sin phi = S CA - C SA and the double angle from cos phi, sin phi:
 * cos 2 phi = cos^2 phi - sin^2 phi, sin 2 phi = 2 sin phi cos phi (rounded +, -, * only; k = h = 0 gives Eq. (15)
 * bit for bit).
 * ------------------------------------------------------------------------------------------------------- */
static void unit_vector(double alpha, double delta, double n[3])
{
    const double cd = cos(delta);
    n[0] = cd * cos(alpha);
    n[1] = cd * sin(alpha);
    n[2] = sin(delta);
}

static double canon_D(const double *v, const double n[3])
{
    const double a = v[0] * n[0];
    const double b = v[1] * n[1];
    const double c = v[2] * n[2];
    const double ab = a + b;
    return ab + c;
}

static int64_t canon_bin(const orc_problem *pb, double D, double A, double C, double S, double CA, double SA, double k,
                         double h, int j, double *y_out)
{
    const double cc = C * CA;
    const double ss = S * SA;
    const double cphi = cc + ss;
    double bracket = cphi;
    if (k != 0.0 || h != 0.0) {
        const double sc = S * CA;
        const double cs = C * SA;
        const double sphi = sc - cs;
        const double c2a = cphi * cphi;
        const double s2a = sphi * sphi;
        const double cos2 = c2a - s2a;
        const double two_s = 2.0 * sphi;
        const double sin2 = two_s * cphi;
        const double kc = k * cos2;
        const double hs = h * sin2;
        const double E = kc - hs;
        bracket = cphi + E;
    }
    const double B = A * bracket;
    const double g = D - B;
    const double u = (double)(pb->k_band0 + j);
    const double y = u * g;
    if (y_out) *y_out = y;
    const int64_t r = (int64_t)nearbyint(y);             /* R-1: nearest integer, ties to even */
    return (pb->k_band0 - pb->k_slab0) + j + r;
}

int64_t orc_track_canonical(const orc_problem *pb, int pix, int ia, int ip, int it, int ie, int j, int i, double *y_out)
{
    double n[3];
    unit_vector(pb->alpha[pix], pb->delta[pix], n);
    const double D = canon_D(pb->v_over_c + 3 * (size_t)i, n);
    const double P = pb->P[ip];
    const double two_pi = 2.0 * M_PI;
    const double Omega = two_pi / P;
    const double A = pb->ap[ia] * Omega;
    const double fp = pb->tasc_frac[it] * P;
    const double ta = pb->t_search_mid + fp;
    const double arg_t = Omega * pb->t_mid[i];
    const double arg_a = Omega * ta;
    return canon_bin(pb, D, A, cos(arg_t), sin(arg_t), cos(arg_a), sin(arg_a), ecc_k(pb, ie), ecc_h(pb, ie), j, y_out);
}

/* one full track (all SFTs) of one template, either mode */
void orc_track(const orc_problem *pb, int mode, int pix, int ia, int ip, int it, int ie, int j, int64_t *k_out,
               double *aux_out)
{
    for (int i = 0; i < pb->n_sft; ++i) {
        double aux;
        k_out[i] = (mode == ORC_DIRECT) ? orc_track_direct(pb, pix, ia, ip, it, ie, j, i, &aux)
                                        : orc_track_canonical(pb, pix, ia, ip, it, ie, j, i, &aux);
        if (aux_out) aux_out[i] = aux;
    }
}

/* template linear index (R-11): f0 fastest, then the eccentricity pair (one value when the grid is circular) */
static inline uint64_t tmpl_index(const orc_problem *pb, int pix, int ia, int ip, int it, int ie, int j)
{
    return (((((uint64_t)pix * pb->n_ap + ia) * pb->n_P + ip) * pb->n_tasc + it) * n_ecc_eff(pb) + ie) * pb->n_f0 + j;
}

void orc_decode_index(const orc_problem *pb, uint64_t idx, int32_t *out6)
{
    out6[5] = (int32_t)(idx % pb->n_f0);      idx /= pb->n_f0;        /* j   */
    out6[4] = (int32_t)(idx % n_ecc_eff(pb)); idx /= n_ecc_eff(pb);   /* ie  */
    out6[3] = (int32_t)(idx % pb->n_tasc);    idx /= pb->n_tasc;      /* it  */
    out6[2] = (int32_t)(idx % pb->n_P);       idx /= pb->n_P;         /* ip  */
    out6[1] = (int32_t)(idx % pb->n_ap);      idx /= pb->n_ap;        /* ia  */
    out6[0] = (int32_t)idx;                                           /* pix */
}

static inline int peak_bit(const uint32_t *peak, int32_t words_per_row, int32_t n_bins, int i, int64_t k)
{
    if (k < 0 || k >= n_bins) return 0;                         /* R-6: outside the slab contributes 0 */
    return (peak[(size_t)i * words_per_row + (k >> 5)] >> (k & 31)) & 1u;
}

/* ---------------------------------------------------------------------------------------------------------
 * Stage 1: for every template, n = sum_i bit[i][k_i], n_w = sum_i w_i bit[i][k_i] (FP64).
 * count_out / wcount_out: [n_templates] in R-11 order; either may be NULL.  w may be NULL (then n_w = n).
 * DIRECT mode is the literal double loop.  CANONICAL mode hoists the loop-invariant table values
 * (cos/sin of Omega t_i per period, D per pixel) out of the inner loops; the per-accumulation arithmetic is
 * canon_bin() unchanged, and tests assert it equals orc_track_canonical() call by call.
 * ------------------------------------------------------------------------------------------------------- */
void orc_stage1(const orc_problem *pb, int mode, const uint32_t *peak, int32_t words_per_row, const float *w,
                int32_t *count_out, double *wcount_out, int n_threads)
{
    const int N = pb->n_sft;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
    if (mode == ORC_DIRECT) {
        const long n_outer = (long)pb->n_pix * pb->n_ap * pb->n_P * pb->n_tasc * n_ecc_eff(pb);
#pragma omp parallel for schedule(dynamic, 4)
        for (long o = 0; o < n_outer; ++o) {
            long r = o;
            const int ie = (int)(r % n_ecc_eff(pb)); r /= n_ecc_eff(pb);
            const int it = (int)(r % pb->n_tasc); r /= pb->n_tasc;
            const int ip = (int)(r % pb->n_P);    r /= pb->n_P;
            const int ia = (int)(r % pb->n_ap);   r /= pb->n_ap;
            const int pix = (int)r;
            for (int j = 0; j < pb->n_f0; ++j) {
                int32_t n = 0;
                double nw = 0.0;
                for (int i = 0; i < N; ++i) {
                    const int64_t k = orc_track_direct(pb, pix, ia, ip, it, ie, j, i, NULL);
                    if (peak_bit(peak, words_per_row, pb->n_bins, i, k)) {
                        n += 1;
                        nw += w ? (double)w[i] : 1.0;
                    }
                }
                const uint64_t idx = tmpl_index(pb, pix, ia, ip, it, ie, j);
                if (count_out) count_out[idx] = n;
                if (wcount_out) wcount_out[idx] = nw;
            }
        }
        return;
    }
    /* CANONICAL */
    const double two_pi = 2.0 * M_PI;
    double *Dtab = (double *)malloc(sizeof(double) * (size_t)pb->n_pix * N);
    for (int pix = 0; pix < pb->n_pix; ++pix) {
        double n[3];
        unit_vector(pb->alpha[pix], pb->delta[pix], n);
        for (int i = 0; i < N; ++i) Dtab[(size_t)pix * N + i] = canon_D(pb->v_over_c + 3 * (size_t)i, n);
    }
    for (int ip = 0; ip < pb->n_P; ++ip) {
        const double P = pb->P[ip];
        const double Omega = two_pi / P;
        double *Ct = (double *)malloc(sizeof(double) * N), *St = (double *)malloc(sizeof(double) * N);
        for (int i = 0; i < N; ++i) {
            const double arg = Omega * pb->t_mid[i];
            Ct[i] = cos(arg);
            St[i] = sin(arg);
        }
        const long n_outer = (long)pb->n_pix * pb->n_ap * pb->n_tasc * n_ecc_eff(pb);
#pragma omp parallel for schedule(dynamic, 4)
        for (long o = 0; o < n_outer; ++o) {
            long r = o;
            const int ie = (int)(r % n_ecc_eff(pb)); r /= n_ecc_eff(pb);
            const int it = (int)(r % pb->n_tasc); r /= pb->n_tasc;
            const int ia = (int)(r % pb->n_ap);   r /= pb->n_ap;
            const int pix = (int)r;
            const double A = pb->ap[ia] * Omega;
            const double fp = pb->tasc_frac[it] * P;
            const double ta = pb->t_search_mid + fp;
            const double arg_a = Omega * ta;
            const double CA = cos(arg_a), SA = sin(arg_a);
            const double *D = Dtab + (size_t)pix * N;
            for (int j = 0; j < pb->n_f0; ++j) {
                int32_t n = 0;
                double nw = 0.0;
                for (int i = 0; i < N; ++i) {
                    const int64_t k = canon_bin(pb, D[i], A, Ct[i], St[i], CA, SA, ecc_k(pb, ie), ecc_h(pb, ie), j, NULL);
                    if (peak_bit(peak, words_per_row, pb->n_bins, i, k)) {
                        n += 1;
                        nw += w ? (double)w[i] : 1.0;
                    }
                }
                const uint64_t idx = tmpl_index(pb, pix, ia, ip, it, ie, j);
                if (count_out) count_out[idx] = n;
                if (wcount_out) wcount_out[idx] = nw;
            }
        }
        free(Ct);
        free(St);
    }
    free(Dtab);
}

/* ---------------------------------------------------------------------------------------------------------
 * DIRECT vs CANONICAL over a whole grid: counts the accumulations where the two modes give different bins and
 * how many of those are NOT flagged as near-ties (|x + 1/2 - nearest integer| < tol in either mode).
 * out[0] = accumulations compared, out[1] = disagreements, out[2] = unflagged disagreements, out[3] = flagged.
 * ------------------------------------------------------------------------------------------------------- */
void orc_compare_modes(const orc_problem *pb, double tol, int64_t *out)
{
    int64_t n_cmp = 0, n_dis = 0, n_unfl = 0, n_flag = 0;
    const long n_outer = (long)pb->n_pix * pb->n_ap * pb->n_P * pb->n_tasc * n_ecc_eff(pb);
    const int64_t m = pb->k_band0 - pb->k_slab0;
#pragma omp parallel for schedule(dynamic, 4) reduction(+ : n_cmp, n_dis, n_unfl, n_flag)
    for (long o = 0; o < n_outer; ++o) {
        long r = o;
        const int ie = (int)(r % n_ecc_eff(pb)); r /= n_ecc_eff(pb);
        const int it = (int)(r % pb->n_tasc); r /= pb->n_tasc;
        const int ip = (int)(r % pb->n_P);    r /= pb->n_P;
        const int ia = (int)(r % pb->n_ap);   r /= pb->n_ap;
        const int pix = (int)r;
        for (int j = 0; j < pb->n_f0; ++j)
            for (int i = 0; i < pb->n_sft; ++i) {
                double x, y;
                const int64_t kd = orc_track_direct(pb, pix, ia, ip, it, ie, j, i, &x);
                const int64_t kc = orc_track_canonical(pb, pix, ia, ip, it, ie, j, i, &y);
                const double xd = x + 0.5, xc = (double)(m + j) + y + 0.5;
                const int flagged = fabs(xd - nearbyint(xd)) < tol || fabs(xc - nearbyint(xc)) < tol;
                n_cmp += 1;
                n_flag += flagged;
                if (kd != kc) {
                    n_dis += 1;
                    if (!flagged) n_unfl += 1;
                }
            }
    }
    out[0] = n_cmp; out[1] = n_dis; out[2] = n_unfl; out[3] = n_flag;
}

/* ---------------------------------------------------------------------------------------------------------
 * Score an explicit list of templates (used for sampled parity at full size and for stage 2):
 *   count  = sum_i bit[i][k_i]                    (NULL to skip; needs peak)
 *   wcount = sum_i w_i bit[i][k_i]                (NULL to skip)
 *   power  = sum_i w_i rho[i][k_i], Eq. (26)      (NULL to skip; needs rho [N][K] row-major FP32)
 * w == NULL means unit weights.  All sums FP64 in SFT order.
 * ------------------------------------------------------------------------------------------------------- */
void orc_score(const orc_problem *pb, int mode, const uint64_t *idx, int64_t n_idx, const uint32_t *peak,
               int32_t words_per_row, const float *rho, const float *w, int32_t *count, double *wcount, double *power,
               int n_threads)
{
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t c = 0; c < n_idx; ++c) {
        int32_t t6[6];
        orc_decode_index(pb, idx[c], t6);
        int32_t n = 0;
        double nw = 0.0, pw = 0.0;
        for (int i = 0; i < pb->n_sft; ++i) {
            const int64_t k = (mode == ORC_DIRECT)
                                  ? orc_track_direct(pb, t6[0], t6[1], t6[2], t6[3], t6[4], t6[5], i, NULL)
                                  : orc_track_canonical(pb, t6[0], t6[1], t6[2], t6[3], t6[4], t6[5], i, NULL);
            const double wi = w ? (double)w[i] : 1.0;
            if (peak && peak_bit(peak, words_per_row, pb->n_bins, i, k)) {
                n += 1;
                nw += wi;
            }
            if (rho && k >= 0 && k < pb->n_bins) pw += wi * (double)rho[(size_t)i * pb->n_bins + k];
        }
        if (count) count[c] = n;
        if (wcount) wcount[c] = nw;
        if (power) power[c] = pw;
    }
}

/* Stage 2, Eq. (26) (L227): the power statistic of each candidate along its exact track. */
void orc_stage2(const orc_problem *pb, int mode, const uint64_t *idx, int64_t n_idx, const float *rho, const float *w,
                double *power, int n_threads)
{
    orc_score(pb, mode, idx, n_idx, NULL, 0, rho, w, NULL, NULL, power, n_threads);
}

/* ---------------------------------------------------------------------------------------------------------
 * Toplist (L217, L225-L229): full sort of all n values by (value descending, index ascending) (R-11), keep k.
 * ------------------------------------------------------------------------------------------------------- */
typedef struct { double v; uint64_t i; } orc_pair;

static int cmp_pair(const void *a, const void *b)
{
    const orc_pair *x = (const orc_pair *)a, *y = (const orc_pair *)b;
    if (x->v > y->v) return -1;
    if (x->v < y->v) return 1;
    if (x->i < y->i) return -1;
    if (x->i > y->i) return 1;
    return 0;
}

int64_t orc_toplist(const double *values, int64_t n, int64_t k, uint64_t *idx_out)
{
    orc_pair *p = (orc_pair *)malloc(sizeof(orc_pair) * (size_t)(n > 0 ? n : 1));
    for (int64_t i = 0; i < n; ++i) { p[i].v = values[i]; p[i].i = (uint64_t)i; }
    qsort(p, (size_t)n, sizeof(orc_pair), cmp_pair);
    const int64_t kk = k < n ? k : n;
    for (int64_t i = 0; i < kk; ++i) idx_out[i] = p[i].i;
    free(p);
    return kk;
}

/* ---------------------------------------------------------------------------------------------------------
 * Front end, Eq. (20)-(21): complex SFT bins -> normalised power
 *     rho_Jk = |x_Jk|^2 / <n_Jk>^2,
 * "<n_Jk>^2 is usually estimated with a running median over a number of frequency bins (usually 101 bins are used)".
 * The paper prints no formula for the estimate; reading R-22:
 *   - input: n_raw complex bins per SFT (FP32 re, im interleaved, as SFT files store them); the slab column k is raw bin
 *     k + h, h = (window - 1) / 2, so every output bin has a full window and there is no edge rule:
 *     K = n_raw - window + 1 columns ("wing" bins on both sides are the caller's, as the SFT reader supplies them);
 *   - power    p_q   = fl32(fl32(re re) + fl32(im im))                     (FP32, no FMA: the kernel's precision)
 *   - median   med_k = the (h + 1)-th smallest of p_k .. p_{k + window - 1} (a selection: exact; NaN ranks above +inf)
 *   - noise    n2_k  = fl32(med_k / bias)         bias = E[median of `window` iid Exp(1) draws] = sum_{i=h+1}^{window} 1/i
 *                                                 (the median of exponential noise power is NOT its mean; for window -> inf
 *                                                  the factor is ln 2.  Passed in as an FP32 number.)
 *   - rho_k          = fl32(p_{k + h} / n2_k)
 * Written as literally as that: copy the window, sort it, take the middle.
 * ------------------------------------------------------------------------------------------------------- */
double orc_median_bias(int32_t window)
{
    const int h = (window - 1) / 2;
    double s = 0.0;
    for (int i = window; i >= h + 1; --i) s += 1.0 / (double)i;      /* E of the (h+1)-th order statistic of Exp(1) */
    return s;
}

static int cmp_float_nan_last(const void *a, const void *b)
{
    const float x = *(const float *)a, y = *(const float *)b;
    const int xn = x != x, yn = y != y;
    if (xn || yn) return xn - yn;                                   /* NaN above everything */
    return (x > y) - (x < y);
}

void orc_normalise(const float *sft, int32_t n_sft, int32_t n_raw, int32_t window, float bias, float *rho)
{
    const int h = (window - 1) / 2;
    const int K = n_raw - window + 1;
    float *p = (float *)malloc(sizeof(float) * (size_t)n_raw);
    float *win = (float *)malloc(sizeof(float) * (size_t)window);
    for (int32_t J = 0; J < n_sft; ++J) {
        const float *row = sft + 2 * (size_t)J * n_raw;
        for (int q = 0; q < n_raw; ++q) {
            const float re = row[2 * q], im = row[2 * q + 1];
            const float rr = re * re;
            const float ii = im * im;
            p[q] = rr + ii;                                         /* |x|^2, Eq. (20) numerator */
        }
        for (int k = 0; k < K; ++k) {
            memcpy(win, p + k, sizeof(float) * (size_t)window);
            qsort(win, (size_t)window, sizeof(float), cmp_float_nan_last);
            const float med = win[h];                               /* running median, L171 */
            const float n2 = med / bias;                            /* <n>^2 estimate, Eq. (21) */
            rho[(size_t)J * K + k] = p[k + h] / n2;                 /* Eq. (20) */
        }
    }
    free(p);
    free(win);
}

/* ---------------------------------------------------------------------------------------------------------
 * Post-processing of the toplists, section V.E, L385-L407.
 *
 * A candidate is a point p = (f, x, y, a_p, Omega, t_asc) (x, y: "cartesian ecliptical coordinates projected into the
 * ecliptical plane", L397) with a significance s and the parameter resolutions delta = (df, dtheta, dtheta, da_p, dOmega,
 * dt_asc) AT that point.  Distance, Eq. (44), "given as a number of bins"; "we use a mean of the resolution at both
 * points" (L399):
 *     d^2(a, b) = sum_k [ (p_k(a) - p_k(b)) / ((delta_k(a) + delta_k(b)) / 2) ]^2        k in the order of Eq. (44)
 * (R-25: plain differences, no wrap of t_asc modulo P; every operation one rounded FP64 operation in the order
 * written, the six squares added left to right.)
 *   coincidences (step 1, L387-L393): all pairs (a in list A, b in list B) with d < window; per pair the centroid
 *       "average locations in parameter space weighted by significance" and the summed significance (R-25).
 *   clusters (step 2, L401-L403): "analyzing the distance of each template from all other templates, and keeping a list of
 *       indices of members with distances below the threshold ... if a template was already in a cluster its newly
 *       generated cluster and the old one will be joined" = connected components of the graph d < window.  The label of a
 *       cluster is the smallest index of its members.  Option B (L403): members further than prune_window from the
 *       cluster's top template (largest significance, smallest index among equals) are removed (label -1).
 *   centroids (step 3, L405): significance-weighted average of the members, summed significance; the most significant
 *       cluster is the one kept per band.
 * ------------------------------------------------------------------------------------------------------- */
#define ORC_NPAR 6

double orc_distance2(const double *pa, const double *ra, const double *pb, const double *rb)
{
    double d2 = 0.0;
    for (int k = 0; k < ORC_NPAR; ++k) {
        const double sum = ra[k] + rb[k];
        const double res = 0.5 * sum;                      /* mean of the resolutions at both points, L399 */
        const double diff = pa[k] - pb[k];
        const double q = diff / res;
        const double sq = q * q;
        d2 = d2 + sq;                                      /* Eq. (44) */
    }
    return d2;
}

/* step 1: pairs in (a, b) lexicographic order; returns the number found (writes at most max_pairs) */
int64_t orc_coincidences(int32_t na, const double *pa, const double *ra, const double *sa, int32_t nb, const double *pb,
                         const double *rb, const double *sb, double window, int64_t max_pairs, int32_t *pair_a,
                         int32_t *pair_b, double *centroid, double *pair_sig)
{
    int64_t n = 0;
    const double w2 = window * window;
    for (int32_t a = 0; a < na; ++a)
        for (int32_t b = 0; b < nb; ++b) {
            const double d2 = orc_distance2(pa + ORC_NPAR * (size_t)a, ra + ORC_NPAR * (size_t)a, pb + ORC_NPAR * (size_t)b,
                                            rb + ORC_NPAR * (size_t)b);
            if (!(d2 < w2)) continue;
            if (n < max_pairs) {
                pair_a[n] = a;
                pair_b[n] = b;
                const double s = sa[a] + sb[b];
                pair_sig[n] = s;
                for (int k = 0; k < ORC_NPAR; ++k) {
                    const double wa = sa[a] * pa[ORC_NPAR * (size_t)a + k];
                    const double wb = sb[b] * pb[ORC_NPAR * (size_t)b + k];
                    centroid[ORC_NPAR * n + k] = (wa + wb) / s;
                }
            }
            n += 1;
        }
    return n;
}

/* steps 2 and 3.  label[n]; per cluster (in increasing label order): root, centroid[6], summed significance, members.
 * Returns the number of clusters; *best = position (in that order) of the most significant cluster, -1 if none. */
int32_t orc_cluster(int32_t n, const double *p, const double *r, const double *s, double window, double prune_window,
                    int32_t *label, int32_t *root, double *centroid, double *cluster_sig, int32_t *n_members, int32_t *best)
{
    const double w2 = window * window;
    for (int32_t i = 0; i < n; ++i) label[i] = i;                       /* every template starts as its own cluster */
    for (int32_t i = 0; i < n; ++i)
        for (int32_t j = 0; j < n; ++j) {
            if (j == i) continue;
            const double d2 = orc_distance2(p + ORC_NPAR * (size_t)i, r + ORC_NPAR * (size_t)i, p + ORC_NPAR * (size_t)j,
                                            r + ORC_NPAR * (size_t)j);
            if (d2 < w2 && label[i] != label[j]) {                      /* join the two clusters (L401) */
                const int32_t keep = label[i] < label[j] ? label[i] : label[j];
                const int32_t drop = label[i] < label[j] ? label[j] : label[i];
                for (int32_t m = 0; m < n; ++m)
                    if (label[m] == drop) label[m] = keep;
            }
        }
    if (prune_window > 0.0) {                                           /* option B, L403 */
        const double pw2 = prune_window * prune_window;
        int32_t *top = (int32_t *)malloc(sizeof(int32_t) * (size_t)(n > 0 ? n : 1));
        for (int32_t c = 0; c < n; ++c) {
            top[c] = -1;
            for (int32_t m = 0; m < n; ++m)
                if (label[m] == c && (top[c] < 0 || s[m] > s[top[c]])) top[c] = m;
        }
        for (int32_t m = 0; m < n; ++m) {
            const int32_t t = top[label[m]];
            const double d2 = orc_distance2(p + ORC_NPAR * (size_t)m, r + ORC_NPAR * (size_t)m, p + ORC_NPAR * (size_t)t,
                                            r + ORC_NPAR * (size_t)t);
            if (!(d2 < pw2) && m != t) label[m] = -(label[m] + 2);      /* marked; resolved below (labels stay readable) */
        }
        for (int32_t m = 0; m < n; ++m)
            if (label[m] < 0) label[m] = -1;
        free(top);
    }
    int32_t nc = 0;
    *best = -1;
    for (int32_t c = 0; c < n; ++c) {                                   /* clusters in increasing label order */
        double ssum = 0.0, acc[ORC_NPAR] = {0, 0, 0, 0, 0, 0};
        int32_t members = 0;
        for (int32_t m = 0; m < n; ++m)
            if (label[m] == c) {
                members += 1;
                ssum = ssum + s[m];
                for (int k = 0; k < ORC_NPAR; ++k) acc[k] = acc[k] + s[m] * p[ORC_NPAR * (size_t)m + k];
            }
        if (members == 0) continue;
        root[nc] = c;
        n_members[nc] = members;
        cluster_sig[nc] = ssum;
        for (int k = 0; k < ORC_NPAR; ++k) centroid[ORC_NPAR * (size_t)nc + k] = acc[k] / ssum;   /* L405 */
        if (*best < 0 || ssum > cluster_sig[*best]) *best = nc;
        nc += 1;
    }
    return nc;
}
