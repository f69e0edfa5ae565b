/*
 * bsh.h -- C ABI of the B200-native BinarySkyHough hot path (Covas & Sintes, arXiv:1904.04873).
 *
 * Citations are lines of /root/reference/PAPER.md ("L123") with the section / equation they fall in, or DESIGN.md
 * readings ("R-5").  The library computes, for every template of a sky patch x template grid,
 *
 *   peakgram   bit[i][k] = rho[i][k] > rho_th                                   L176 (sec. IV.A), rho_th = 1.6
 *   track      k_i = round((f(t_i) - f_slab_start) T),                          BASELINE.json north_star
 *              f(t) = f0 [1 + v(t).n/c - a_p Omega cos(Omega (t - t_asc))]      L102 Eq. (15), Omega = 2 pi / P (L61)
 *   stage 1    n = sum_i bit[i][k_i],  n_w = sum_i w_i bit[i][k_i]              L223 (sec. IV.C) "number count"
 *   toplist    the topk templates of the patch by the stage-1 statistic         L217, L225-L229
 *   stage 2    P = sum_i w_i rho[i][k_i] along the same track                   L227 Eq. (26)
 *
 * Conventions
 *   - Every function returns int: BSH_OK (0) or a negative error code.  Nothing throws; bsh_last_error(ctx) returns a
 *     description of the last failure on that context (valid until the next call on it).
 *   - Pointer prefixes:  d_ = DEVICE memory owned by the caller, never freed or retained by the library beyond the
 *     call unless stated;  h_ = HOST memory, read (or written) during the call only.
 *   - All device work is enqueued on the CUDA stream given to bsh_create().  Functions documented "asynchronous"
 *     return before the work completes; the caller synchronises that stream before reading results.
 *   - There is no CPU fallback: without a CUDA device bsh_create() fails with BSH_ECUDA.
 *   - Template linear index (R-11): ((((pix * n_ap + ia) * n_P + ip) * n_tasc + it) * n_f0 + j, f0 fastest; with an
 *     eccentricity axis: (((((pix * n_ap + ia) * n_P + ip) * n_tasc + it) * n_ecc + ie) * n_f0 + j.
 *   - Ordering everywhere: (statistic descending, template index ascending).
 */
#ifndef BSH_H_
#define BSH_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define BSH_OK        0
#define BSH_EINVAL   -1   /* bad size / null pointer / inconsistent arguments (nothing was launched)            */
#define BSH_ENOMEM   -2   /* device or host allocation failed                                                    */
#define BSH_ECUDA    -3   /* a CUDA runtime call or kernel failed (message in bsh_last_error)                    */
#define BSH_ESMALL   -4   /* an output buffer is too small (e.g. words_per_row * 32 < n_bins)                    */
#define BSH_ESTATE   -5   /* call order violated (e.g. bsh_stage1_collect without bsh_stage1_launch), or the threshold   */
                          /* search of the toplist gave up after 24 accumulation passes; message in bsh_last_error */
#define BSH_ELIMIT   -6   /* a list is longer than the fixed scratch of bsh_post_coincidences_static holds               */

/* mode bits for stage 1 */
#define BSH_UNWEIGHTED 0  /* rank by the integer number count n                                   (L223)         */
#define BSH_WEIGHTED   1  /* rank by n_w = sum w_i bit, FP32 accumulation in SFT order            (L223, Eq. 22) */
#define BSH_NAIVE      16 /* diagnostic: one thread per template, one track evaluation per (template, SFT), global-
                             memory gathers.  Same results; exists to cross-check the tiled kernels at full size. */

/* bsh_set_option(): DIAGNOSTIC switches, so that the tests can reach every kernel family and both table geometries
 * on any input.  Production leaves the defaults (the library picks the family from the problem shape). */
#define BSH_OPT_KERNEL_FAMILY      1   /* one of BSH_FAMILY_*                                                      */
#define BSH_OPT_FORCE_CLAMP        2   /* 1: use the clamped table geometry even when no track can leave the slab  */
#define BSH_OPT_PIXELS_PER_THREAD  3   /* window-table family only: 0 = auto, 1, 2                                 */
#define BSH_FAMILY_AUTO        0
#define BSH_FAMILY_PIXEL_LANE  1       /* sky pixels on the lanes (bsh_pix.cuh)                                    */
#define BSH_FAMILY_TEMPLATE_LANE 2     /* binary templates on the lanes, position table (bsh_pos.cuh)              */
#define BSH_FAMILY_WINDOW      3       /* binary templates on the lanes, funnel-shift window table (wide slabs)    */

/* bsh_stats.kernel_variant / 1000: the accumulation kernel that ran.  A separate numbering from BSH_FAMILY_* on purpose:
 * a family is what the caller may ask for, a kernel id says what was launched (the pixel-lane family has two kernels). */
#define BSH_KERNEL_WINDOW         0    /* funnel-shift window table           (BSH_FAMILY_WINDOW)                          */
#define BSH_KERNEL_TEMPLATE_LANE  1    /* position table, templates on lanes  (BSH_FAMILY_TEMPLATE_LANE)                   */
#define BSH_KERNEL_PIXEL_LANE     2    /* unweighted pixel-lane kernel        (BSH_FAMILY_PIXEL_LANE, BSH_UNWEIGHTED)      */
#define BSH_KERNEL_PIXEL_LANE_W   3    /* weighted pixel-lane kernel          (BSH_FAMILY_PIXEL_LANE, BSH_WEIGHTED)        */

typedef struct bsh_ctx bsh_ctx;

/* One SFT set.  Stage 1 and stage 2 may be given different sets (the paper's stage 2 adds half-overlapped SFTs,
 * L233); all five BASELINE.json configs use the same set for both. */
typedef struct {
    int32_t       n_sft;         /* N >= 1                                                                       */
    double        t_sft;         /* T = T_c, seconds; the bin width is 1/T (Eq. 33)                        */
    const double *h_t_mid;       /* [N] SFT mid-times in seconds relative to any reference epoch (R-2); the same  */
                                 /*     epoch as t_search_mid.  Keep |Omega t| moderate (epoch near the data).    */
    const double *h_v_over_c;    /* [N][3] detector velocity / c at t_mid, equatorial frame; one row per SFT, so  */
                                 /*     several detectors are simply more rows                                    */
    const float  *d_w;           /* [N] per-SFT weights (Eq. 22), caller-normalised (R-9); NULL = all 1     */
    int64_t       k_slab0;       /* absolute frequency-bin index (f * T) of column 0 of the slab                  */
    int32_t       n_bins;        /* K = slab columns                                                              */
    double        t_search_mid;  /* t_mid of Eq. (35) (L305)                                                      */
} bsh_sfts;

/* One sky patch x template grid. */
typedef struct {
    int32_t n_pix;  const double *h_alpha, *h_delta;  /* [n_pix] right ascension / declination, radians           */
    int64_t k_band0;                                  /* f0_j = (k_band0 + j) / T, j = 0 .. n_f0-1 (R-3); requires */
    int32_t n_f0;                                     /*   k_slab0 <= k_band0 <= k_slab0 + 2^24, k_band0 + n_f0 < 2^32 */
    int32_t n_ap;   const double *h_ap;               /* [n_ap]  projected semi-major axis, light-seconds (L70)    */
    int32_t n_P;    const double *h_P;                /* [n_P]   orbital period, seconds                           */
    int32_t n_tasc; const double *h_tasc_frac;        /* [n_tasc] t_asc = t_search_mid + frac * P (Eq. 35, R-13)   */
    /* Eccentric orbits (ELL1 model, Eq. 14): n_ecc pairs (e cos omega, e sin omega); the track is
     * f(t) = f0 [1 + v.n/c - a_p Omega (cos phi + ecosw cos 2 phi - esinw sin 2 phi)], phi = Omega (t - t_asc), as Eq. (14)
     * prints it (readings R-23, R-24).  n_ecc = 0 (pointers ignored): circular orbits, Eq. (15).                          */
    int32_t n_ecc;  const double *h_ecosw, *h_esinw;  /* [n_ecc]                                                     */
} bsh_grid;

/* Toplist / candidate record (24 bytes). */
typedef struct {
    uint64_t index;    /* template linear index                                                                    */
    int32_t  count;    /* n   = sum_i bit                    (exact)                                               */
    float    wcount;   /* n_w = sum_i w_i bit                (FP32; = count when d_w is NULL)                       */
    float    power;    /* P   = sum_i w_i rho, Eq. (26)      (filled by bsh_stage2_power; 0 before)                */
    uint32_t flags;    /* bit 0: filled by stage 1; bit 1: power filled                                            */
} bsh_cand;

/* Diagnostics of the most recent calls on a context (all times in milliseconds, from CUDA events on the stream). */
typedef struct {
    float    peakgram_ms;        /* bsh_build_peakgram kernel                                                      */
    float    stage1_setup_ms;    /* window table, D table, threshold (device side)                                 */
    float    stage1_kernel_ms;   /* the accumulation kernel(s) of the last bsh_stage1_* (all passes)               */
    float    stage1_select_ms;   /* candidate sort + toplist rescoring                                             */
    float    stage2_ms;          /* bsh_stage2_power kernels                                                       */
    int64_t  n_templates;        /* templates of the last stage-1 call                                             */
    int64_t  n_accumulations;    /* n_templates * n_sft                                                            */
    int64_t  n_candidates;       /* templates that passed the in-kernel threshold                                  */
    double   threshold;          /* final in-kernel threshold (count or weighted count)                            */
    int32_t  n_passes;           /* accumulation passes (1 unless the threshold had to be moved)                   */
    int32_t  kernel_variant;     /* kernel * 1000 + words * 100 + pixels_per_thread * 10 + clamp; kernel = one of the  */
                                 /* BSH_KERNEL_* ids below (which accumulation kernel RAN; not a BSH_FAMILY_* request) */
    int32_t  threads_per_block;  /* of the accumulation kernel                                                     */
    int32_t  grid_blocks;        /* of the accumulation kernel                                                     */
    int64_t  launches;           /* kernels launched by this context since creation                                */
    float    host_tables_ms;     /* host time spent building cos/sin tables in the last call (0 when cached)       */
    float    frontend_ms;        /* bsh_normalise_peakgram kernel                                                  */
} bsh_stats;

/* On-chip peak rates of the context's device, MEASURED by bsh_measure_peaks() with microbenchmark kernels (32 warps
 * per SM on every SM, volatile inline PTX, timed with clock64 per block).  They are the denominators of
 * the roofline fractions of the stage-1 accumulation kernels, which are bound on chip and not by HBM. */
typedef struct {
    int32_t n_sm;                          /* multiprocessors                                                     */
    double  sm_clock_mhz;                  /* SM clock during the measurement (clock64 against globaltimer)       */
    double  issue_warp_inst_per_clk_smsp;  /* 1 LOP3 : 3 FADD stream: warp instructions per clock per scheduler   */
                                           /*   (SM sub-partition); lanes/clk/SM = 128 x this                     */
    double  lop3_lanes_per_clk_sm;         /* integer-ALU pipe (bit-sliced counters)                              */
    double  fadd_lanes_per_clk_sm;         /* predicated FP32 add (weighted number count, L223)                   */
    double  dadd_lanes_per_clk_sm;         /* FP64 add, no FMA (canonical track, R-5)                             */
    double  dmul_lanes_per_clk_sm;         /* FP64 multiply                                                       */
    double  lds32_bytes_per_clk_sm;        /* conflict-free shared-memory loads: LDS.32 / LDS.64 / LDS.128        */
    double  lds64_bytes_per_clk_sm;
    double  lds128_bytes_per_clk_sm;
} bsh_peaks;

/* Create a context bound to `device` and to `cuda_stream` (a cudaStream_t; NULL = legacy default stream).
 * The context owns scratch memory (tables, candidate buffer), grown on demand and freed by bsh_destroy. */
int bsh_create(bsh_ctx **out, int device, void *cuda_stream);
int bsh_destroy(bsh_ctx *ctx);
const char *bsh_last_error(const bsh_ctx *ctx);
int bsh_get_stats(bsh_ctx *ctx, bsh_stats *out);     /* synchronises the stream to read event timers */
int bsh_version(void);
int bsh_set_option(bsh_ctx *ctx, int32_t option, int32_t value);   /* BSH_EINVAL for an unknown option / value      */
int bsh_measure_peaks(bsh_ctx *ctx, bsh_peaks *h_out);             /* ~50 ms of device time; synchronous            */

/* Peakgram (L176): d_peak[i][k >> 5] bit (k & 31) = (d_rho[i * rho_row_stride + k] > rho_th), strict '>' in FP32,
 * NaN -> 0 (R-8); pad bits of each row are zero.  d_rho: [n_sft][rho_row_stride] FP32, rho_row_stride >= n_bins
 * (elements).  d_peak: [n_sft][words_per_row] uint32, words_per_row >= ceil(n_bins / 32) (else BSH_ESMALL); words
 * beyond ceil(n_bins / 32) are zeroed.  Asynchronous. */
int bsh_build_peakgram(bsh_ctx *ctx, const float *d_rho, int32_t n_sft, int32_t n_bins, int64_t rho_row_stride,
                       float rho_th, uint32_t *d_peak, int32_t words_per_row);

/* Front end (L167-L176, Eq. 20-21): complex SFT bins -> normalised powers -> peakgram, one fused kernel.
 *     rho_Jk = |x_Jk|^2 / <n_Jk>^2,   <n_Jk>^2 = running median of |x|^2 over `window` bins / median_bias   (reading R-22)
 *   d_sft        [n_sft][sft_row_stride] complex bins, FP32 (re, im) interleaved (8 bytes per bin, 8-byte aligned),
 *                sft_row_stride >= n_raw (in complex elements); raw bin q of row J is d_sft[2 (J stride + q)], [.. + 1]
 *   n_raw        raw bins per row = K + window - 1: slab column k is raw bin k + (window - 1) / 2, so every column has a
 *                full window (the caller supplies (window - 1) / 2 wing bins on each side; there is no edge rule)
 *   window       odd, 1 <= window <= n_raw <= 2048; the paper uses 101
 *   median_bias  E[median of `window` iid Exp(1) draws] (bsh_median_bias(window); -> ln 2 for large windows): the median of
 *                exponentially distributed noise power is not its mean, dividing by it makes <rho> = 1 in noise (L439)
 *   d_rho        [n_sft][rho_row_stride] FP32 normalised powers, K = n_raw - window + 1 columns written per row; may be NULL
 *   d_peak       [n_sft][words_per_row] bit-packed (rho > rho_th), layout as bsh_build_peakgram; may be NULL (not both)
 * Arithmetic (FP32, each operation rounded once, no FMA): p = fl(fl(re re) + fl(im im)); med = the ((window + 1) / 2)-th
 * smallest p of the window (exact selection; NaN ranks above +inf); n2 = fl(med / bias); rho = fl(p / n2).  Asynchronous. */
int bsh_normalise_peakgram(bsh_ctx *ctx, const float *d_sft, int32_t n_sft, int32_t n_raw, int64_t sft_row_stride,
                           int32_t window, float median_bias, float rho_th, float *d_rho, int64_t rho_row_stride,
                           uint32_t *d_peak, int32_t words_per_row);
double bsh_median_bias(int32_t window);    /* sum_{i = (window + 1) / 2}^{window} 1 / i; host function                     */

/* Stage 1 (L223, L241-L247): number count of every template of `grid` along its Eq. (15) track through the
 * peakgram, and the per-patch toplist (L217, L225).
 *   d_peak          [n_sft][words_per_row] as written by bsh_build_peakgram for this SFT set
 *   mode            BSH_UNWEIGHTED or BSH_WEIGHTED (needs sfts->d_w), optionally | BSH_NAIVE
 *   topk            entries wanted, 1 <= topk <= 2^27 (BSH_EINVAL beyond the candidate buffer)
 *   d_top           [topk] records, best first; entries beyond *h_n_top are zeroed
 *   h_n_top         receives min(topk, n_templates)
 *   d_counts_full   optional dump of the ranking statistic of EVERY template (int32 counts in BSH_UNWEIGHTED mode,
 *                   float weighted counts in BSH_WEIGHTED mode), [n_templates]; NULL in production
 * A track leaving the slab is not an error: that SFT contributes 0 (R-6).
 * Toplist selection: the accumulation kernels emit the templates at or above a threshold guessed from noise moments of the
 * peakgram into a candidate buffer (2^20 entries, more for topk > 2^17), which is then sorted.  When the data are not noise-
 * like and fewer than topk or more than the buffer holds pass, the accumulation is repeated with a corrected threshold
 * (bsh_stats.n_passes > 1): lowered in doubling steps, or raised to the topk-th value of the overflowed buffer.  When the
 * templates tied AT the cut value alone overflow the buffer (all-zero or constant peakgram rows, very few SFTs), the ties
 * are admitted in template-index order up to a limit found by a few more passes, so the result is still exactly the
 * (statistic desc, index asc) toplist.  Grids that fit the buffer are emitted whole and never need this.
 * bsh_stage1_hough = bsh_stage1_launch + bsh_stage1_collect; it returns with d_top complete (stream synchronised).
 * bsh_stage1_launch is asynchronous (no host synchronisation); bsh_stage1_collect synchronises the stream, runs the
 * selection, and leaves the toplist writes enqueued on the stream (h_n_top is final on return).  The wcount of every
 * toplist entry is re-scored in a fixed order that does not depend on the accumulation kernel, the two orders given at
 * bsh_stage2_power (block per entry up to 65536 entries, thread per entry beyond).  Between launch and
 * collect the caller may enqueue work on OTHER contexts/streams (this is how config 5 overlaps two patches).
 * The host arrays inside `sfts` and `grid` are read during launch only; the DEVICE buffers d_peak, sfts->d_w and
 * d_counts_full are read / written until bsh_stage1_collect returns (toplist rescoring and threshold retries) and must stay
 * valid until then.  Other calls on the same context between launch and collect are allowed (their tables use the other
 * cache slot). */
int bsh_stage1_hough(bsh_ctx *ctx, const uint32_t *d_peak, int32_t words_per_row, const bsh_sfts *sfts,
                     const bsh_grid *grid, int32_t mode, int32_t topk, bsh_cand *d_top, int32_t *h_n_top,
                     void *d_counts_full);
int bsh_stage1_launch(bsh_ctx *ctx, const uint32_t *d_peak, int32_t words_per_row, const bsh_sfts *sfts,
                      const bsh_grid *grid, int32_t mode, int32_t topk, void *d_counts_full);
int bsh_stage1_collect(bsh_ctx *ctx, bsh_cand *d_top, int32_t *h_n_top);

/* Stage 2 (Eq. 26): power[c] = sum_i w_i rho[i][k_i] along the track of d_cands[c].index over the SFT set
 * `sfts`, written into d_cands[c].power.  If sort_by_power != 0 the records are then reordered by (power desc, index asc).
 * FP32 summation order (R-20; deterministic run to run, but it DEPENDS ON THE LIST LENGTH):
 *   n_cands <= 65536   one 128-thread block per candidate: thread t sums the products of SFTs t, t + 128, ... in order, then
 *                      a fixed xor-shuffle tree per warp, then the four warp partials in warp order;
 *   n_cands  > 65536   one thread per candidate: partial sums over chunks of 128 consecutive SFTs in SFT order, then the
 *                      partials in chunk order.
 * The power of one template can therefore differ in its last bits between a short and a long list (both are within the
 * 1e-5 relative tolerance of the FP64 sum); the same holds for the wcount that bsh_stage1_collect re-scores.
 * d_rho: [n_sft][rho_row_stride] FP32.  Asynchronous. */
int bsh_stage2_power(bsh_ctx *ctx, const float *d_rho, int64_t rho_row_stride, const bsh_sfts *sfts,
                     const bsh_grid *grid, bsh_cand *d_cands, int32_t n_cands, int32_t sort_by_power);

/* Whole patch from HOST buffers (the end-to-end call): copies h_rho [n_sft][n_bins] and h_w [n_sft] (may be NULL) to
 * the device, builds the peakgram, runs stage 1 and stage 2 (sorted by power) and copies the toplist back into
 * h_top [topk].  sfts->d_w is ignored (h_w is used).  Synchronous. */
int bsh_search_patch_host(bsh_ctx *ctx, const float *h_rho, const float *h_w, float rho_th, const bsh_sfts *sfts,
                          const bsh_grid *grid, int32_t mode, int32_t topk, bsh_cand *h_top, int32_t *h_n_top);

/* Post-processing of the toplists (section V.E).  A candidate set: n points
 * p = (f, x, y, a_p, Omega, t_asc) (x, y: ecliptic coordinates projected into the ecliptic plane, L397), the parameter
 * resolutions at each point in the same order (delta f, delta theta, delta theta, delta a_p, delta Omega, delta t_asc:
 * Eq. 30-33), and a significance per point.  Distance (Eq. 44, "a mean of the resolution at both points" L399):
 *     d^2(a, b) = sum_k [ (p_k(a) - p_k(b)) / ((delta_k(a) + delta_k(b)) / 2) ]^2
 * in FP64, one rounding per operation, the six squares added in the order of Eq. (44) (reading R-25: plain differences,
 * t_asc is not wrapped modulo P).  Both calls are synchronous; n <= 32768. */
typedef struct {
    int32_t       n;
    const double *d_param;   /* [n][6] */
    const double *d_res;     /* [n][6], all > 0 */
    const double *d_sig;     /* [n]    */
} bsh_candset;

/* Step 1 (L387-L393): every pair (a in A, b in B) with d(a, b) < window, in (a, b) lexicographic order: indices, the
 * significance-weighted centroid [6] and the summed significance of each pair.  At most max_pairs are written;
 * *h_n_pairs receives the number found (may exceed max_pairs: call again with larger buffers). */
int bsh_post_coincidences(bsh_ctx *ctx, const bsh_candset *a, const bsh_candset *b, double window, int64_t max_pairs,
                          int32_t *d_pair_a, int32_t *d_pair_b, double *d_centroid, double *d_pair_sig, int64_t *h_n_pairs);

/* bsh_post_coincidences without any allocation -- for callers that must not, or cannot, allocate device memory.
 *
 * Who that is.  bsh_post_coincidences keeps its work area (the bit matrix "pair (a, b) is closer than the window", the
 * per-row pair counts and their prefix sums) in cudaMalloc'ed buffers that its context grows on demand.  That is wrong
 * for three kinds of user of this library:
 *   - a search job that has handed the whole of the GPU's memory to a pool of its own (a framework's caching allocator, a
 *     batch scheduler's fixed per-job share of a GPU that several jobs use): the library's own cudaMalloc then fails, or
 *     takes memory the job was promised;
 *   - the follow-up stage of a sweep that still has stage-1 kernels of other sky patches running on other streams:
 *     cudaMalloc and cudaFree make the whole device wait, so a growing work area stalls every one of those patches;
 *   - a monitoring / low-latency consumer of the toplists that has to answer in bounded time: an allocation takes an
 *     unbounded time and can fail at a moment when nothing can be done about it.
 * This call therefore takes no bsh_ctx (creating one allocates events and pinned memory) and calls no cudaMalloc, cudaFree,
 * cudaMallocHost or any other allocating routine: inputs and outputs are the caller's, and the work area is ONE array that is
 * part of the loaded library image on every GPU, BSH_STATIC_SCRATCH_BYTES (about 8.1 MiB) per GPU from the moment the
 * library is loaded there until the process exits, whether or not this call is ever made.
 *
 * Limit.  a->n <= BSH_STATIC_MAX_CANDS and b->n <= BSH_STATIC_MAX_CANDS (8192; the paper's final toplists hold 5000
 * candidates, L496).  Longer lists are refused with BSH_ELIMIT before anything is launched -- use
 * bsh_post_coincidences for those.
 *
 * Arguments and results are those of bsh_post_coincidences (same kernels, same operation order: the pair list, centroids
 * and significances are bit-identical), except:
 *   device, cuda_stream   the GPU and the cudaStream_t (NULL = legacy default stream) to run on, in place of the context
 *   h_err, err_len        optional caller's buffer that receives a NUL-terminated description when the result is not
 *                         BSH_OK (h_err may be NULL)
 * Synchronous: the stream is synchronised before the call returns.
 *
 * First call on each device: it looks up the device address of the work area (cudaGetSymbolAddress; this also makes the
 * CUDA runtime load the library's device code onto that GPU if nothing did so before) and remembers it.  Make that first
 * call during set-up, before any stream capture is begun; later calls on that device do no look-up.
 *
 * Sharing.  Every call on a device -- from any stream and any host thread of the process -- uses the same work area, and
 * the area keeps what the previous call left in it (the call clears the part that has to start at zero, the row counts;
 * everything else it reads it has first overwritten itself).  Two calls whose kernels can be on the same GPU at the same
 * time therefore corrupt each other's results: the caller runs them one after the other.  (Calls on different GPUs, and
 * calls in different processes, do not share anything.) */
#define BSH_STATIC_MAX_CANDS     8192
#define BSH_STATIC_SCRATCH_BYTES (65792 + 32768 + 8192 * (8192 / 32) * 4)
int bsh_post_coincidences_static(int device, void *cuda_stream, const bsh_candset *a, const bsh_candset *b, double window,
                                 int64_t max_pairs, int32_t *d_pair_a, int32_t *d_pair_b, double *d_centroid,
                                 double *d_pair_sig, int64_t *h_n_pairs, char *h_err, int32_t err_len);

/* Steps 2-3 (L401-L405): clusters = connected components of the graph d < window; d_label[i] = smallest index of the
 * members of i's cluster.  prune_window > 0 (option B, L403): members at that distance or further from the cluster's top
 * template (largest significance, smallest index among equals) are removed, d_label = -1.  Per cluster, in increasing
 * label order ([n] arrays, *h_n_clusters entries written): d_root (the label), d_centroid [6] (significance-weighted
 * average of the members, taken in index order), d_cluster_sig (summed significance), d_n_members.  *h_best = position
 * of the most significant cluster (first among equals), the one kept per 0.1 Hz band (L405); -1 when n = 0. */
int bsh_post_cluster(bsh_ctx *ctx, const bsh_candset *c, double window, double prune_window, int32_t *d_label,
                     int32_t *d_root, double *d_centroid, double *d_cluster_sig, int32_t *d_n_members,
                     int32_t *h_n_clusters, int32_t *h_best);

/* Template index helpers (R-11).  Pure host functions.  The first pair is for circular grids (n_ecc = 0; on an eccentric
 * grid it addresses pair ie = 0 / drops ie); the _ecc pair carries the eccentricity index. */
uint64_t bsh_template_index(const bsh_grid *grid, int32_t pix, int32_t ia, int32_t ip, int32_t it, int32_t j);
void     bsh_template_decode(const bsh_grid *grid, uint64_t index, int32_t *pix, int32_t *ia, int32_t *ip,
                             int32_t *it, int32_t *j);
uint64_t bsh_template_index_ecc(const bsh_grid *grid, int32_t pix, int32_t ia, int32_t ip, int32_t it, int32_t ie, int32_t j);
void     bsh_template_decode_ecc(const bsh_grid *grid, uint64_t index, int32_t *pix, int32_t *ia, int32_t *ip,
                                 int32_t *it, int32_t *ie, int32_t *j);

#ifdef __cplusplus
}
#endif
#endif /* BSH_H_ */
