/*
 * bsh_tier2.c -- TIER-2 CPU REFERENCE for stage 1 (SURVEY.md section 8(c) "coverage plan").  TEST INFRASTRUCTURE ONLY.
 *
 * The plain oracle (bsh_oracle.c: one track evaluation per (template, SFT)) cannot run the full grids of the large
 * configurations (2.8e11 - 1.3e13 accumulations).  This is a second, separately written CPU implementation that is fast
 * enough to score EVERY template of configs 2, 4 and a patch of 5 in seconds to minutes on the host cores:
 *   - table driven: v.n/c per (pixel, SFT), (cos, sin)(Omega t) per (period, SFT), (cos, sin)(Omega t_asc) per (period, t_asc);
 *   - one evaluation of g = v.n/c - a_p Omega [...] per (pixel, binary template, SFT), shared by all f0 bins: y_j = u_j g is
 *     monotone in j, so when the rounded shift is the same at both ends of the band it is the same in between and the
 *     peakgram bytes of the band are added with one vector loop; otherwise every bin is evaluated on its own (no bisection,
 *     no blend: the simplest exact fallback);
 *   - OpenMP over (pixel, binary template).
 * It must equal the plain oracle's CANONICAL mode BIT FOR BIT on every grid the plain oracle can run (tests/test_tier2.py);
 * the chain   plain oracle == tier 2 (sub-grids)   and   tier 2 == GPU (full grids)   is what the parity tests assert.
 * Same canonical operation order as DESIGN.md R-5 / R-23, retyped here: it shares no code with bsh_oracle.c nor with the
 * CUDA path (paper_1904_04873_b200/csrc).   PAPER.md L102 Eq. (15), L95-L98 Eq. (14), L223.
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

typedef struct {                      /* same plain-data layout as orc_problem (filled by oracle/__init__.py) */
    int32_t n_sft;
    double t_sft;
    const double *t_mid;
    const double *v_over_c;
    double t_search_mid;
    int64_t k_slab0;
    int32_t n_bins;
    int64_t k_band0;
    int32_t n_f0;
    int32_t n_pix;
    const double *alpha, *delta;
    int32_t n_ap;   const double *ap;
    int32_t n_P;    const double *P;
    int32_t n_tasc; const double *tasc_frac;
    int32_t n_ecc;  const double *ecosw, *esinw;
} t2_problem;

/* counts [n_templates] int32 and/or wcounts [n_templates] double (either may be NULL), R-11 order. */
void t2_stage1(const t2_problem *pb, const uint32_t *peak, int32_t words_per_row, const float *w, int32_t *counts,
               double *wcounts, int n_threads)
{
    const int N = pb->n_sft, K = pb->n_bins, NF = pb->n_f0;
    const int ne = pb->n_ecc > 0 ? pb->n_ecc : 1;
    const int64_t m = pb->k_band0 - pb->k_slab0;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
    /* peakgram as bytes, each row padded with zeros so that any in-range shift reads inside the row */
    const int64_t PAD = (int64_t)NF + 64;
    const int64_t RW = K + 2 * PAD;
    uint8_t *bits = (uint8_t *)calloc((size_t)N * RW, 1);
    for (int i = 0; i < N; ++i)
        for (int k = 0; k < K; ++k)
            bits[(size_t)i * RW + PAD + k] = (uint8_t)((peak[(size_t)i * words_per_row + (k >> 5)] >> (k & 31)) & 1u);
    /* tables */
    double *D = (double *)malloc(sizeof(double) * (size_t)pb->n_pix * N);
    for (int pix = 0; pix < pb->n_pix; ++pix) {
        const double cd = cos(pb->delta[pix]);
        const double nx = cd * cos(pb->alpha[pix]), ny = cd * sin(pb->alpha[pix]), nz = sin(pb->delta[pix]);
        for (int i = 0; i < N; ++i) {
            const double *v = pb->v_over_c + 3 * (size_t)i;
            const double a = v[0] * nx, b = v[1] * ny, c = v[2] * nz;
            const double ab = a + b;
            D[(size_t)pix * N + i] = ab + c;
        }
    }
    double *C = (double *)malloc(sizeof(double) * (size_t)pb->n_P * N), *S = (double *)malloc(sizeof(double) * (size_t)pb->n_P * N);
    double *Om = (double *)malloc(sizeof(double) * pb->n_P);
    const double two_pi = 2.0 * M_PI;
    for (int ip = 0; ip < pb->n_P; ++ip) {
        Om[ip] = two_pi / pb->P[ip];
        for (int i = 0; i < N; ++i) {
            const double arg = Om[ip] * pb->t_mid[i];
            C[(size_t)ip * N + i] = cos(arg);
            S[(size_t)ip * N + i] = sin(arg);
        }
    }
    const double u0 = (double)pb->k_band0, uL = (double)(pb->k_band0 + NF - 1);
    const int64_t n_outer = (int64_t)pb->n_pix * pb->n_ap * pb->n_P * pb->n_tasc * ne;
#pragma omp parallel
    {
        int32_t *cnt = (int32_t *)malloc(sizeof(int32_t) * NF);
        double *wc = (double *)malloc(sizeof(double) * NF);
#pragma omp for schedule(dynamic, 16)
        for (int64_t o = 0; o < n_outer; ++o) {
            int64_t r = o;
            const int ie = (int)(r % ne);          r /= ne;
            const int it = (int)(r % pb->n_tasc);  r /= pb->n_tasc;
            const int ip = (int)(r % pb->n_P);     r /= pb->n_P;
            const int ia = (int)(r % pb->n_ap);    r /= pb->n_ap;
            const int pix = (int)r;
            const double A = pb->ap[ia] * Om[ip];
            const double fp = pb->tasc_frac[it] * pb->P[ip];
            const double ta = pb->t_search_mid + fp;
            const double arg_a = Om[ip] * ta;
            const double CA = cos(arg_a), SA = sin(arg_a);
            const double kap = pb->n_ecc > 0 ? pb->ecosw[ie] : 0.0, eta = pb->n_ecc > 0 ? pb->esinw[ie] : 0.0;
            const int ecc = kap != 0.0 || eta != 0.0;
            const double *Dp = D + (size_t)pix * N, *Cp = C + (size_t)ip * N, *Sp = S + (size_t)ip * N;
            for (int j = 0; j < NF; ++j) { cnt[j] = 0; wc[j] = 0.0; }
            for (int i = 0; i < N; ++i) {
                const double cc = Cp[i] * CA, ss = Sp[i] * SA;
                const double cphi = cc + ss;
                double br = cphi;
                if (ecc) {
                    const double sc = Sp[i] * CA, cs = Cp[i] * SA;
                    const double sphi = sc - cs;
                    const double c2 = cphi * cphi, s2 = sphi * sphi;
                    const double cos2 = c2 - s2;
                    const double ts = 2.0 * sphi;
                    const double sin2 = ts * cphi;
                    const double kc = kap * cos2, hs = eta * sin2;
                    const double E = kc - hs;
                    br = cphi + E;
                }
                const double B = A * br;
                const double g = Dp[i] - B;
                const double y0 = u0 * g, yL = uL * g;
                const int64_t r0 = (int64_t)nearbyint(y0), rL = (int64_t)nearbyint(yL);
                const uint8_t *row = bits + (size_t)i * RW + PAD;
                const double wi = w ? (double)w[i] : 1.0;
                if (r0 == rL) {                                   /* the whole band has this shift (monotone y_j) */
                    int64_t s = m + r0;                           /* slab column of bin j = 0 */
                    if (s < -PAD) s = -PAD;                       /* entirely outside the slab: reads only padding zeros */
                    if (s > K + PAD - NF) s = K + PAD - NF;
                    const uint8_t *src = row + s;
                    if (wcounts) {
                        for (int j = 0; j < NF; ++j) {
                            cnt[j] += src[j];
                            if (src[j]) wc[j] += wi;
                        }
                    } else {
                        for (int j = 0; j < NF; ++j) cnt[j] += src[j];
                    }
                } else {                                          /* the shift changes inside the band: bin by bin */
                    for (int j = 0; j < NF; ++j) {
                        const double u = (double)(pb->k_band0 + j);
                        const double y = u * g;
                        const int64_t k = m + j + (int64_t)nearbyint(y);
                        if (k >= 0 && k < K && row[k]) {
                            cnt[j] += 1;
                            wc[j] += wi;
                        }
                    }
                }
            }
            const uint64_t base = (uint64_t)o * (uint64_t)NF;     /* R-11: f0 fastest, then ie, it, ip, ia, pix */
            if (counts) memcpy(counts + base, cnt, sizeof(int32_t) * NF);
            if (wcounts) memcpy(wcounts + base, wc, sizeof(double) * NF);
        }
        free(cnt);
        free(wc);
    }
    free(bits); free(D); free(C); free(S); free(Om);
}
