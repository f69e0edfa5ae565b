// bsh_api.cu -- C ABI (include/bsh.h) of the B200-native BinarySkyHough hot path: context, host-side table building
// (the only place transcendentals are evaluated, R-5), kernel selection and launch, candidate selection.
// Build: nvcc -O3 -std=c++17 -gencode arch=compute_100a,code=sm_100a -lineinfo -Xcompiler -fPIC,-ffp-contract=off -shared
#include <cuda_runtime.h>
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <string.h>

#include <algorithm>
#include <chrono>
#include <mutex>
#include <string>
#include <vector>

#include "../../include/bsh.h"
#include "bsh_host.hpp"
#include "bsh_kernels.cuh"
#include "bsh_pos.cuh"
#include "bsh_pix.cuh"
#include "bsh_wpix.cuh"
#include "bsh_peaks.cuh"
#include "bsh_frontend.cuh"
#include "bsh_post.cuh"
#include "bsh_sort.cuh"

using namespace bsh;

namespace {

constexpr unsigned int kCandCap = 1u << 20;      // candidate buffer entries (16 MB)
constexpr int kMaxPasses = 24;               // accumulation passes per call, all phases of the threshold search together
constexpr int32_t kMaxTopk = 1 << 27;            // bsh.h: 1 <= topk <= 2^27 (also the largest candidate buffer)

struct DevBuf {
    void *p = nullptr;
    size_t bytes = 0;
};

struct TableCache {                   // cos/sin tables of one (SFT set, binary grid); content-addressed
    bool valid = false;
    uint64_t stamp = 0;
    std::vector<double> t_mid, v, P, tasc, ap, ecw, esw;
    double t_sft = 0, t_search_mid = 0;
    int n_sft = 0, n_pad = 0, n_P = 0, n_tasc = 0, n_ap = 0, n_ecc = 0;
    DevBuf d_v, d_cs, d_casa, d_A, d_ke, d_cs_t;
    bool have_cs_t = false;
};

struct Pending {                      // state between bsh_stage1_launch and bsh_stage1_collect
    bool active = false;
    int mode = 0, topk = 0;
    void *d_counts_full = nullptr;
    const uint32_t *d_peak = nullptr;
    int words_per_row = 0;
    const float *d_w = nullptr;
    int cache_slot = 0;
    int n_sft = 0, n_pad = 0, n_bins = 0, n_pix = 0, n_ap = 0, n_P = 0, n_tasc = 0, n_f0 = 0;
    int64_t k_band0 = 0, k_slab0 = 0;
    uint64_t n_templates = 0;
    bool emit_all = false, clamp = false;
    int tile_bins = 96;               // f0 bins per accumulation pass (<= 32 NW)
    unsigned int cand_cap = kCandCap; // candidate buffer entries of this call (grows with topk: fraction-N_C toplists, L225)
    int R = 2, NW = 3, HP = 6, n_entries = 0, off_table = 0, s_max = 0, s_zero = 0, list_cap = 0, tpb = 256, n_groups = 0, n_aq_tiles = 0;
    double frac = 0;
    int passes = 0;
    // threshold search of bsh_stage1_collect (passes after the first run with a host-given threshold)
    bool fixed = false;               // false: the noise-model threshold of threshold_kernel (first pass)
    double tau = 0;                   // the threshold of the pass in flight (integer-valued in unweighted mode)
    double lo_tau = 0;                // the last threshold with too many survivors ...
    uint64_t lo_n = 0;                // ... and how many there were
    double step_dn = 0.75;
    int phase = 0;                    // 0: search on tau; 1: count the templates above the tie value; 2: search on tie_limit
    uint64_t tie_limit = ~0ull, lim_lo = 0, lim_hi = 0, n_above = 0;
    uint32_t tie_key = 0;
    // position-table kernels (bsh_pos.cuh)
    bool use_pos = false;
    int pos_off = 0, pos_s_max = 0, pos_s_zero = 0, n_pos = 0, n_stages = 0, n_oct = 0, pos_groups = 0, pos_smem = 0;
    // pixel-lane kernel (bsh_pix.cuh)
    bool use_pix = false;
    int n_pg = 0, pix_stages = 0, pix_smem = 0;
    // weighted pixel-lane kernel (bsh_wpix.cuh)
    bool use_wpix = false;
    int wpix_nbytes = 0, wpix_stages = 0, wpix_smem = 0;
};

}  // namespace

struct bsh_ctx {
    int device = 0;
    cudaStream_t stream = nullptr;
    std::string err;
    TableCache cache[2];
    uint64_t stamp = 0;
    DevBuf wtab, w_pad, stats, thr, dtab, nvec, cand, cand_count, keys, tmp_cands, dtab2, nvec2, ptab, dpos, dpix, psplit, tab7;
    DevBuf h_rho, h_w, h_peak, h_top;                  // device staging of bsh_search_patch_host
    unsigned int *pinned_count = nullptr;
    cudaEvent_t ev[12] = {};
    Pending pend;
    int opt_family = BSH_FAMILY_AUTO, opt_force_clamp = 0, opt_pixels_per_thread = 0;   // bsh_set_option
    DevBuf peak_samples;
    DevBuf post_adj, post_cnt, post_off, post_tmp;
    DevBuf radix_hist;
    bsh_stats st = {};
    bool have_front = false;
    bool have_pk = false, have_setup = false, have_kernel = false, have_select = false, have_s2 = false;
    float kernel_ms_extra = 0.f;
};

namespace {

int fail(bsh_ctx *ctx, int code, const char *fmt, ...)
{
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    if (ctx) ctx->err = buf;
    return code;
}

#define CK(call)                                                                                              \
    do {                                                                                                      \
        cudaError_t e_ = (call);                                                                              \
        if (e_ != cudaSuccess)                                                                                \
            return fail(ctx, e_ == cudaErrorMemoryAllocation ? BSH_ENOMEM : BSH_ECUDA, "%s failed: %s (%s:%d)", \
                        #call, cudaGetErrorString(e_), __FILE__, __LINE__);                                   \
    } while (0)

int ensure(bsh_ctx *ctx, DevBuf &b, size_t bytes)
{
    if (b.bytes >= bytes && b.p) return BSH_OK;
    if (b.p) {
        CK(cudaStreamSynchronize(ctx->stream));
        CK(cudaFree(b.p));
        b.p = nullptr;
        b.bytes = 0;
    }
    const size_t want = std::max<size_t>(bytes + bytes / 4, 256);
    CK(cudaMalloc(&b.p, want));
    b.bytes = want;
    return BSH_OK;
}

// the ABI calls run on the context's device and leave the caller's current device as they found it
struct DeviceGuard {
    int prev = -1;
    explicit DeviceGuard(int dev)
    {
        if (cudaGetDevice(&prev) != cudaSuccess) prev = -1;
        if (prev != dev) cudaSetDevice(dev);
    }
    ~DeviceGuard()
    {
        if (prev >= 0) cudaSetDevice(prev);
    }
    DeviceGuard(const DeviceGuard &) = delete;
    DeviceGuard &operator=(const DeviceGuard &) = delete;
};

#define TRY(expr)                  \
    do {                           \
        int rc_ = (expr);          \
        if (rc_ != BSH_OK) return rc_; \
    } while (0)

inline void count_launch(bsh_ctx *ctx, int n = 1) { ctx->st.launches += n; }

static_assert(kHostChunk == kChunk, "SFT padding granularity");

// ---------------------------------------------------------------------------------------------------------------------
// Host tables (R-5).  The only transcendental evaluations of the whole path: libm cos/sin of Omega_p t_i and
// Omega_p t_asc, and of the pixel angles.  Cached by content: a sweep over sky patches reuses them.
// ---------------------------------------------------------------------------------------------------------------------
inline int n_ecc_of(const bsh_grid *g) { return g->n_ecc > 0 ? g->n_ecc : 0; }
inline int n_tq_of(const bsh_grid *g) { return g->n_tasc * (g->n_ecc > 0 ? g->n_ecc : 1); }   // combined (t_asc, eccentricity) axis

// the grid as the kernels see it: the eccentricity axis folded into the t_asc axis (bsh_host.hpp, build_binary_tables)
inline bsh_grid kernel_grid(const bsh_grid *g)
{
    bsh_grid k = *g;
    k.n_tasc = n_tq_of(g);
    k.n_ecc = 0;
    return k;
}

double ecc_max_of(const bsh_grid *g)
{
    double m = 0.0;
    for (int e = 0; e < n_ecc_of(g); ++e) m = std::max(m, fabs(g->h_ecosw[e]) + fabs(g->h_esinw[e]));
    return m;
}

int validate(bsh_ctx *ctx, const bsh_sfts *s, const bsh_grid *g)
{
    if (!s || !g) return fail(ctx, BSH_EINVAL, "null sfts/grid");
    if (s->n_sft < 1 || !(s->t_sft > 0) || !s->h_t_mid || !s->h_v_over_c || s->n_bins < 1)
        return fail(ctx, BSH_EINVAL, "bad SFT set (n_sft=%d, t_sft=%g, n_bins=%d)", s->n_sft, s->t_sft, s->n_bins);
    if (g->n_pix < 1 || g->n_f0 < 1 || g->n_ap < 1 || g->n_P < 1 || g->n_tasc < 1 || !g->h_alpha || !g->h_delta ||
        !g->h_ap || !g->h_P || !g->h_tasc_frac)
        return fail(ctx, BSH_EINVAL, "bad grid");
    if (g->k_band0 < s->k_slab0) return fail(ctx, BSH_EINVAL, "k_band0 < k_slab0");
    // k_band0 + n_f0 < 2^32: the break fix-up of bsh_core.cuh (exact_window_pos) estimates the break bin from
    // y_0 + j g, which differs from the canonical fl(fl(u_0 + j) g) by up to u 2^-52 bins of j; below 2^32 that is
    // < 1e-6, far inside its 1e-3 guard (R-7).  2^32 bins is 4.8 MHz at T = 900 s.
    if (g->k_band0 - s->k_slab0 > (1 << 24) || g->k_band0 + g->n_f0 >= (1ll << 32))
        return fail(ctx, BSH_EINVAL, "band offset out of range (k_band0 - k_slab0 <= 2^24, k_band0 + n_f0 < 2^32)");
    for (int p = 0; p < g->n_P; ++p)
        if (!(g->h_P[p] > 0)) return fail(ctx, BSH_EINVAL, "P[%d] <= 0", p);
    if (g->n_ecc < 0 || (g->n_ecc > 0 && (!g->h_ecosw || !g->h_esinw))) return fail(ctx, BSH_EINVAL, "bad eccentricity axis");
    for (int e = 0; e < n_ecc_of(g); ++e)
        if (!(fabs(g->h_ecosw[e]) + fabs(g->h_esinw[e]) < 1.0)) return fail(ctx, BSH_EINVAL, "eccentricity pair %d out of range", e);
    if ((int64_t)g->n_tasc * std::max(1, g->n_ecc) > (1 << 24)) return fail(ctx, BSH_EINVAL, "t_asc x eccentricity axis too long");
    return BSH_OK;
}

int get_tables(bsh_ctx *ctx, const bsh_sfts *s, const bsh_grid *g, int *slot_out)
{
    const int N = s->n_sft;
    for (int k = 0; k < 2; ++k) {
        TableCache &c = ctx->cache[k];
        if (c.valid && c.n_sft == N && c.n_P == g->n_P && c.n_tasc == g->n_tasc && c.n_ap == g->n_ap &&
            c.n_ecc == n_ecc_of(g) && (c.n_ecc == 0 || (!memcmp(c.ecw.data(), g->h_ecosw, sizeof(double) * c.n_ecc) &&
                                                         !memcmp(c.esw.data(), g->h_esinw, sizeof(double) * c.n_ecc))) &&
            c.t_sft == s->t_sft && c.t_search_mid == s->t_search_mid &&
            !memcmp(c.t_mid.data(), s->h_t_mid, sizeof(double) * N) &&
            !memcmp(c.v.data(), s->h_v_over_c, sizeof(double) * 3 * N) &&
            !memcmp(c.P.data(), g->h_P, sizeof(double) * g->n_P) &&
            !memcmp(c.tasc.data(), g->h_tasc_frac, sizeof(double) * g->n_tasc) &&
            !memcmp(c.ap.data(), g->h_ap, sizeof(double) * g->n_ap)) {
            c.stamp = ++ctx->stamp;
            *slot_out = k;
            ctx->st.host_tables_ms = 0.f;
            return BSH_OK;
        }
    }
    const auto t0 = std::chrono::steady_clock::now();
    int k = (!ctx->cache[0].valid || (ctx->cache[1].valid && ctx->cache[0].stamp < ctx->cache[1].stamp)) ? 0 : 1;
    if (ctx->pend.active && ctx->pend.cache_slot == k) k ^= 1;     // a launched, uncollected stage 1 still reads its slot
    TableCache &c = ctx->cache[k];
    c.valid = false;
    c.have_cs_t = false;
    const int n_pad = pad_sfts(N);
    c.t_mid.assign(s->h_t_mid, s->h_t_mid + N);
    c.v.assign(s->h_v_over_c, s->h_v_over_c + 3 * (size_t)N);
    c.P.assign(g->h_P, g->h_P + g->n_P);
    c.tasc.assign(g->h_tasc_frac, g->h_tasc_frac + g->n_tasc);
    c.ap.assign(g->h_ap, g->h_ap + g->n_ap);
    c.t_sft = s->t_sft;
    c.t_search_mid = s->t_search_mid;
    c.n_sft = N; c.n_pad = n_pad; c.n_P = g->n_P; c.n_tasc = g->n_tasc; c.n_ap = g->n_ap; c.n_ecc = n_ecc_of(g);
    c.ecw.assign(g->h_ecosw, g->h_ecosw + c.n_ecc);
    c.esw.assign(g->h_esinw, g->h_esinw + c.n_ecc);

    std::vector<double> cs, casa, A, ke;
    build_binary_tables(N, n_pad, s->h_t_mid, s->t_search_mid, g->n_P, g->h_P, g->n_tasc, g->h_tasc_frac, g->n_ap, g->h_ap, cs,
                        casa, A, c.n_ecc, g->h_ecosw, g->h_esinw, &ke);
    TRY(ensure(ctx, c.d_ke, sizeof(double) * ke.size()));
    CK(cudaMemcpyAsync(c.d_ke.p, ke.data(), sizeof(double) * ke.size(), cudaMemcpyHostToDevice, ctx->stream));
    TRY(ensure(ctx, c.d_v, sizeof(double) * 3 * (size_t)N));
    TRY(ensure(ctx, c.d_cs, sizeof(double) * cs.size()));
    TRY(ensure(ctx, c.d_casa, sizeof(double) * casa.size()));
    TRY(ensure(ctx, c.d_A, sizeof(double) * A.size()));
    CK(cudaMemcpyAsync(c.d_v.p, c.v.data(), sizeof(double) * 3 * (size_t)N, cudaMemcpyHostToDevice, ctx->stream));
    CK(cudaMemcpyAsync(c.d_cs.p, cs.data(), sizeof(double) * cs.size(), cudaMemcpyHostToDevice, ctx->stream));
    CK(cudaMemcpyAsync(c.d_casa.p, casa.data(), sizeof(double) * casa.size(), cudaMemcpyHostToDevice, ctx->stream));
    CK(cudaMemcpyAsync(c.d_A.p, A.data(), sizeof(double) * A.size(), cudaMemcpyHostToDevice, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));          // the std::vectors above go out of scope
    c.valid = true;
    c.stamp = ++ctx->stamp;
    *slot_out = k;
    ctx->st.host_tables_ms =
        std::chrono::duration<float, std::milli>(std::chrono::steady_clock::now() - t0).count();
    return BSH_OK;
}

// pixel unit vectors (host libm) -> device; D table on the device
int build_dtable(bsh_ctx *ctx, const bsh_grid *g, const TableCache &c, int R, DevBuf &nvec_buf, DevBuf &dtab_buf)
{
    std::vector<double> nv;
    pixel_vectors(g->n_pix, g->h_alpha, g->h_delta, nv);
    const int n_groups = (g->n_pix + R - 1) / R;
    TRY(ensure(ctx, nvec_buf, sizeof(double) * nv.size()));
    TRY(ensure(ctx, dtab_buf, sizeof(double) * (size_t)n_groups * c.n_pad * R));
    CK(cudaMemcpyAsync(nvec_buf.p, nv.data(), sizeof(double) * nv.size(), cudaMemcpyHostToDevice, ctx->stream));
    const int64_t total = (int64_t)n_groups * c.n_pad * R;
    dtable_kernel<<<(unsigned)((total + 255) / 256), 256, 0, ctx->stream>>>(
        (const double *)c.d_v.p, (const double *)nvec_buf.p, c.n_sft, c.n_pad, g->n_pix, n_groups, R, (double *)dtab_buf.p);
    count_launch(ctx);
    CK(cudaGetLastError());
    return BSH_OK;
}

// transposed (cos, sin) table of a cache slot, built on first use by the large-list kernels
int ensure_cs_t(bsh_ctx *ctx, TableCache &c)
{
    if (c.have_cs_t) return BSH_OK;
    const int64_t n = (int64_t)c.n_P * c.n_pad;
    TRY(ensure(ctx, c.d_cs_t, sizeof(double) * 2 * (size_t)n));
    transpose_cs_kernel<<<(unsigned)((n + 255) / 256), 256, 0, ctx->stream>>>((const double2 *)c.d_cs.p, c.n_P, c.n_pad,
                                                                            (double2 *)c.d_cs_t.p);
    count_launch(ctx);
    CK(cudaGetLastError());
    c.have_cs_t = true;
    return BSH_OK;
}

TrackTables make_track_tables(const TableCache &c, const bsh_sfts *s, const bsh_grid *g, const double *dtab, int R)
{
    TrackTables t;
    t.cs = (const double2 *)c.d_cs.p;
    t.dtab = dtab;
    t.A = (const double *)c.d_A.p;
    t.casa = (const double2 *)c.d_casa.p;
    t.ke = c.n_ecc > 0 ? (const double2 *)c.d_ke.p : nullptr;
    t.cs_t = nullptr;
    t.n_pad = c.n_pad;
    t.R = R;
    t.n_pix = g->n_pix; t.n_ap = g->n_ap; t.n_P = g->n_P; t.n_tasc = g->n_tasc; t.n_f0 = g->n_f0;
    t.k_band0 = g->k_band0;
    t.m = (int)(g->k_band0 - s->k_slab0);
    t.n_bins = s->n_bins;
    t.n_sft = s->n_sft;
    return t;
}

// ---------------------------------------------------------------------------------------------------------------------
// accumulation-kernel dispatch
// ---------------------------------------------------------------------------------------------------------------------
template <typename K, typename P>
int launch_stage1(bsh_ctx *ctx, K kernel, const P &p, int tpb, int grid, int smem)
{
    CK(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    kernel<<<grid, tpb, smem, ctx->stream>>>(p);
    count_launch(ctx);
    CK(cudaGetLastError());
    return BSH_OK;
}

#define UNW_CASE(NW_, HP_, R_, CL_)                                                                                   \
    if (pd.NW == NW_ && pd.HP == HP_ && pd.R == R_ && pd.clamp == CL_)                                                \
        return launch_stage1(ctx, stage1_unweighted_kernel<NW_, HP_, R_, CL_>, p, pd.tpb, grid,                       \
                             StageLayout<R_, false>(pd.n_entries).total() + R_ * pd.list_cap * pd.tpb * 2);

int dispatch_unweighted(bsh_ctx *ctx, const Pending &pd, const Stage1Params &p, int grid)
{
    UNW_CASE(3, 6, 2, false)
#ifndef BSH_MINIMAL                                  /* tuning builds instantiate only the config-2 kernels */
    UNW_CASE(2, 6, 2, false) UNW_CASE(2, 6, 2, true) UNW_CASE(3, 6, 2, true)
    UNW_CASE(2, 8, 2, false) UNW_CASE(2, 8, 2, true) UNW_CASE(3, 8, 2, false) UNW_CASE(3, 8, 2, true)
    UNW_CASE(2, 11, 2, false) UNW_CASE(2, 11, 2, true) UNW_CASE(3, 11, 2, false) UNW_CASE(3, 11, 2, true)
    UNW_CASE(2, 6, 1, false) UNW_CASE(3, 6, 1, false) UNW_CASE(2, 8, 1, false) UNW_CASE(3, 8, 1, false)
    UNW_CASE(2, 6, 1, true) UNW_CASE(3, 6, 1, true) UNW_CASE(2, 8, 1, true) UNW_CASE(3, 8, 1, true)
    UNW_CASE(2, 11, 1, false) UNW_CASE(3, 11, 1, false) UNW_CASE(2, 11, 1, true) UNW_CASE(3, 11, 1, true)
#endif
    return fail(ctx, BSH_EINVAL, "no unweighted kernel for NW=%d HP=%d R=%d clamp=%d", pd.NW, pd.HP, pd.R, (int)pd.clamp);
}

#define W_CASE(NW_, CL_)                                                                               \
    if (pd.NW == NW_ && pd.clamp == CL_)                                                               \
        return launch_stage1(ctx, stage1_weighted_kernel<NW_, CL_>, p, pd.tpb, grid,                   \
                             StageLayout<1, true>(pd.n_entries).total());

int dispatch_weighted(bsh_ctx *ctx, const Pending &pd, const Stage1Params &p, int grid)
{
    W_CASE(3, false)
#ifndef BSH_MINIMAL
    W_CASE(2, false) W_CASE(2, true) W_CASE(3, true)
#endif
    return fail(ctx, BSH_EINVAL, "no weighted kernel for NW=%d", pd.NW);
}

#define UNW_POS_CASE(NW_, HP_, CL_)                                                                   \
    if (pd.NW == NW_ && pd.HP == HP_ && pd.clamp == CL_)                                              \
        return launch_stage1(ctx, stage1_unweighted_pos_kernel<NW_, HP_, CL_>, p, 32 * kWarpsUnweighted, grid, pd.pos_smem);

int dispatch_unweighted_pos(bsh_ctx *ctx, const Pending &pd, const PosParams &p, int grid)
{
    UNW_POS_CASE(3, 6, false)
#ifndef BSH_MINIMAL
    UNW_POS_CASE(2, 6, false) UNW_POS_CASE(2, 6, true) UNW_POS_CASE(3, 6, true)
    UNW_POS_CASE(2, 8, false) UNW_POS_CASE(2, 8, true) UNW_POS_CASE(3, 8, false) UNW_POS_CASE(3, 8, true)
    UNW_POS_CASE(2, 11, false) UNW_POS_CASE(2, 11, true) UNW_POS_CASE(3, 11, false) UNW_POS_CASE(3, 11, true)
#endif
    return fail(ctx, BSH_EINVAL, "no unweighted position kernel for NW=%d HP=%d clamp=%d", pd.NW, pd.HP, (int)pd.clamp);
}

#define UNW_PIX_CASE(NW_, HP_, CL_)                                                                   \
    if (pd.NW == NW_ && pd.HP == HP_ && pd.clamp == CL_)                                              \
        return p.ke ? launch_stage1(ctx, stage1_unweighted_pix_kernel<NW_, HP_, CL_, true>, p, 32 * kPixWarps, grid, pd.pix_smem) \
                    : launch_stage1(ctx, stage1_unweighted_pix_kernel<NW_, HP_, CL_, false>, p, 32 * kPixWarps, grid, pd.pix_smem);

int dispatch_unweighted_pix(bsh_ctx *ctx, const Pending &pd, const PixParams &p, int grid)
{
    UNW_PIX_CASE(3, 6, false)
#ifndef BSH_MINIMAL
    UNW_PIX_CASE(2, 6, false) UNW_PIX_CASE(2, 6, true) UNW_PIX_CASE(3, 6, true)
    UNW_PIX_CASE(2, 8, false) UNW_PIX_CASE(2, 8, true) UNW_PIX_CASE(3, 8, false) UNW_PIX_CASE(3, 8, true)
    UNW_PIX_CASE(2, 11, false) UNW_PIX_CASE(2, 11, true) UNW_PIX_CASE(3, 11, false) UNW_PIX_CASE(3, 11, true)
#endif
    return fail(ctx, BSH_EINVAL, "no unweighted pixel-lane kernel for NW=%d HP=%d clamp=%d", pd.NW, pd.HP, (int)pd.clamp);
}

#define W_POS_CASE(NW_, NB_, CL_)                                                                     \
    if (pd.NW == NW_ && nb == NB_ && pd.clamp == CL_)                                                 \
        return launch_stage1(ctx, stage1_weighted_pos_kernel<NW_, NB_, CL_>, p, 32 * kWarpsWeighted, grid, pd.pos_smem);

int dispatch_weighted_pos(bsh_ctx *ctx, const Pending &pd, const PosParams &p, int grid)
{
    const int nb = pd.NW == 2 ? (pd.tile_bins <= 48 ? 48 : 64) : (p.n_fj <= 90 ? 90 : 96);
    W_POS_CASE(3, 90, false) W_POS_CASE(2, 48, false)
#ifndef BSH_MINIMAL
    W_POS_CASE(2, 64, false) W_POS_CASE(2, 64, true) W_POS_CASE(3, 90, true) W_POS_CASE(2, 48, true)
    W_POS_CASE(3, 96, false) W_POS_CASE(3, 96, true)
#endif
    return fail(ctx, BSH_EINVAL, "no weighted position kernel for NW=%d", pd.NW);
}

#define W_PIX_CASE(NBYTES_, CL_)                                                                      \
    if (pd.wpix_nbytes == NBYTES_ && pd.clamp == CL_)                                                 \
        return launch_stage1(ctx, stage1_weighted_pix_kernel<NBYTES_, CL_>, p, 32 * kWpixWarps, grid, pd.wpix_smem);

int dispatch_weighted_pix(bsh_ctx *ctx, const Pending &pd, const WpixParams &p, int grid)
{
    W_PIX_CASE(15, false) W_PIX_CASE(8, false)
#ifndef BSH_MINIMAL
    W_PIX_CASE(15, true) W_PIX_CASE(8, true)
#endif
    return fail(ctx, BSH_EINVAL, "no weighted pixel-lane kernel for %d bytes clamp=%d", pd.wpix_nbytes, (int)pd.clamp);
}

// one accumulation pass over all f0 tiles with the current threshold shift
int run_pass(bsh_ctx *ctx)
{
    Pending &pd = ctx->pend;
    const TableCache &c = ctx->cache[pd.cache_slot];
    const bool weighted = (pd.mode & BSH_WEIGHTED) != 0;
    CK(cudaMemsetAsync(ctx->cand_count.p, 0, sizeof(unsigned int), ctx->stream));
    threshold_kernel<<<1, 1, 0, ctx->stream>>>((const double *)ctx->stats.p, pd.frac, pd.emit_all ? 1 : 0, pd.fixed ? 1 : 0,
                                               (int32_t)std::max(-1.0e9, std::min(1.0e9, pd.tau)), (float)pd.tau, pd.tie_key,
                                               pd.tie_limit, (Threshold *)ctx->thr.p);
    count_launch(ctx);
    CK(cudaEventRecord(ctx->ev[2], ctx->stream));
    if (pd.mode & BSH_NAIVE) {
        bsh_sfts s = {};
        s.n_sft = pd.n_sft; s.k_slab0 = pd.k_slab0; s.n_bins = pd.n_bins;
        bsh_grid g = {};
        g.n_pix = pd.n_pix; g.n_ap = pd.n_ap; g.n_P = pd.n_P; g.n_tasc = pd.n_tasc; g.n_f0 = pd.n_f0; g.k_band0 = pd.k_band0;
        const TrackTables t = make_track_tables(c, &s, &g, (const double *)ctx->dtab.p, pd.R);
        const uint64_t blocks = (pd.n_templates + 255) / 256;
        if (blocks > 0x7FFFFFFFull) return fail(ctx, BSH_EINVAL, "naive kernel: too many templates");
        stage1_naive_kernel<<<(unsigned)blocks, 256, 0, ctx->stream>>>(
            t, pd.d_peak, pd.words_per_row, pd.d_w, weighted ? 1 : 0, pd.n_templates, (const Threshold *)ctx->thr.p,
            (RawCand *)ctx->cand.p, (unsigned int *)ctx->cand_count.p, pd.cand_cap, pd.d_counts_full);
        count_launch(ctx);
        CK(cudaGetLastError());
        ctx->st.grid_blocks = (int)blocks;
        ctx->st.threads_per_block = 256;
    } else if (pd.use_wpix && weighted) {
        const int tile_bins = pd.tile_bins;
        for (int j0 = 0; j0 < pd.n_f0; j0 += tile_bins) {
            WpixParams p;
            p.tab7 = (const unsigned char *)ctx->tab7.p;
            p.cs = (const double2 *)c.d_cs.p;
            p.dpix = (const double *)ctx->dpix.p;
            p.w_pad = (const float *)ctx->w_pad.p;
            p.A = (const double *)c.d_A.p;
            p.casa = (const double2 *)c.d_casa.p;
            p.ke = c.n_ecc > 0 ? (const double2 *)c.d_ke.p : nullptr;
            p.n_pad = pd.n_pad; p.n_pos = pd.n_pos; p.n_chunks = pd.n_pad / kStageSfts; p.n_stages = pd.wpix_stages;
            p.n_pix = pd.n_pix; p.n_ap = pd.n_ap; p.n_P = pd.n_P; p.n_tasc = pd.n_tasc; p.n_f0 = pd.n_f0;
            p.j0 = j0; p.n_fj = std::min(tile_bins, pd.n_f0 - j0);
            p.n_pg = pd.n_pg; p.n_aq = pd.n_ap * pd.n_tasc; p.n_aq_tiles = (p.n_aq + kWpixWarps - 1) / kWpixWarps;
            p.u0 = (double)(pd.k_band0 + j0);
            p.off = (int)(pd.k_band0 - pd.k_slab0) + j0 + pd.pos_off;
            p.s_max = pd.pos_s_max;
            p.s_zero = pd.pos_s_zero;
            p.thr = (const Threshold *)ctx->thr.p;
            p.cand = (RawCand *)ctx->cand.p;
            p.cand_count = (unsigned int *)ctx->cand_count.p;
            p.cand_cap = pd.cand_cap;
            p.counts_full = pd.d_counts_full;
            const int64_t grid = (int64_t)pd.n_pg * pd.n_P * p.n_aq_tiles;
            if (grid > 0x7FFFFFFFll) return fail(ctx, BSH_EINVAL, "grid too large");
            ctx->st.grid_blocks = (int)grid;
            ctx->st.threads_per_block = 32 * kWpixWarps;
            TRY(dispatch_weighted_pix(ctx, pd, p, (int)grid));
        }
    } else if (pd.use_pix && !weighted) {
        const int tile_bins = pd.tile_bins;
        for (int j0 = 0; j0 < pd.n_f0; j0 += tile_bins) {
            PixParams p;
            p.ptab = (const uint4 *)ctx->ptab.p;
            p.cs = (const double2 *)c.d_cs.p;
            p.dpix = (const double *)ctx->dpix.p;
            p.split = (const unsigned char *)ctx->psplit.p;
            p.one = 1u;
            p.zero = 0u;
            p.A = (const double *)c.d_A.p;
            p.casa = (const double2 *)c.d_casa.p;
            p.ke = c.n_ecc > 0 ? (const double2 *)c.d_ke.p : nullptr;
            p.n_pad = pd.n_pad; p.n_pos = pd.n_pos; p.n_chunks = pd.n_pad / kStageSfts; p.n_stages = pd.pix_stages;
            p.n_pix = pd.n_pix; p.n_ap = pd.n_ap; p.n_P = pd.n_P; p.n_tasc = pd.n_tasc; p.n_f0 = pd.n_f0;
            p.j0 = j0; p.n_fj = std::min(tile_bins, pd.n_f0 - j0);
            p.n_pg = pd.n_pg; p.n_aq = pd.n_ap * pd.n_tasc; p.n_aq_tiles = (p.n_aq + kPixTile - 1) / kPixTile;
            p.u0 = (double)(pd.k_band0 + j0);
            p.off = (int)(pd.k_band0 - pd.k_slab0) + j0 + pd.pos_off;
            p.s_max = pd.pos_s_max;
            p.s_zero = pd.pos_s_zero;
            p.thr = (const Threshold *)ctx->thr.p;
            p.cand = (RawCand *)ctx->cand.p;
            p.cand_count = (unsigned int *)ctx->cand_count.p;
            p.cand_cap = pd.cand_cap;
            p.counts_full = pd.d_counts_full;
            const int64_t grid = (int64_t)pd.n_pg * pd.n_P * p.n_aq_tiles;
            if (grid > 0x7FFFFFFFll) return fail(ctx, BSH_EINVAL, "grid too large");
            ctx->st.grid_blocks = (int)grid;
            ctx->st.threads_per_block = 32 * kPixWarps;
            TRY(dispatch_unweighted_pix(ctx, pd, p, (int)grid));
        }
    } else if (pd.use_pos) {
        const int tile_bins = pd.tile_bins;
        for (int j0 = 0; j0 < pd.n_f0; j0 += tile_bins) {
            PosParams p;
            p.ptab = (const uint4 *)ctx->ptab.p;
            p.cs = (const double2 *)c.d_cs.p;
            p.dpos = (const double *)ctx->dpos.p;
            p.w_pad = (const float *)ctx->w_pad.p;
            p.A = (const double *)c.d_A.p;
            p.casa = (const double2 *)c.d_casa.p;
            p.ke = c.n_ecc > 0 ? (const double2 *)c.d_ke.p : nullptr;
            p.n_pad = pd.n_pad; p.n_pos = pd.n_pos; p.n_chunks = pd.n_pad / kStageSfts; p.n_stages = pd.n_stages;
            p.n_pix = pd.n_pix; p.n_ap = pd.n_ap; p.n_P = pd.n_P; p.n_tasc = pd.n_tasc; p.n_f0 = pd.n_f0;
            p.j0 = j0; p.n_fj = std::min(tile_bins, pd.n_f0 - j0);
            p.n_groups = pd.pos_groups; p.n_oct = pd.n_oct; p.n_aq = pd.n_ap * pd.n_tasc; p.n_aq_tiles = (p.n_aq + 31) / 32;
            p.u0 = (double)(pd.k_band0 + j0);
            p.off = (int)(pd.k_band0 - pd.k_slab0) + j0 + pd.pos_off;
            p.s_max = pd.pos_s_max;
            p.s_zero = pd.pos_s_zero;
            p.thr = (const Threshold *)ctx->thr.p;
            p.cand = (RawCand *)ctx->cand.p;
            p.cand_count = (unsigned int *)ctx->cand_count.p;
            p.cand_cap = pd.cand_cap;
            p.counts_full = pd.d_counts_full;
            const int64_t grid = (int64_t)pd.n_oct * pd.n_P * p.n_aq_tiles;
            if (grid > 0x7FFFFFFFll) return fail(ctx, BSH_EINVAL, "grid too large");
            ctx->st.grid_blocks = (int)grid;
            ctx->st.threads_per_block = 32 * (weighted ? kWarpsWeighted : kWarpsUnweighted);
            TRY(weighted ? dispatch_weighted_pos(ctx, pd, p, (int)grid) : dispatch_unweighted_pos(ctx, pd, p, (int)grid));
        }
    } else {
        const int tile_bins = pd.tile_bins;
        for (int j0 = 0; j0 < pd.n_f0; j0 += tile_bins) {
            Stage1Params p;
            p.wtab = (const uint4 *)ctx->wtab.p;
            p.cs = (const double2 *)c.d_cs.p;
            p.dtab = (const double *)ctx->dtab.p;
            p.w_pad = (const float *)ctx->w_pad.p;
            p.A = (const double *)c.d_A.p;
            p.casa = (const double2 *)c.d_casa.p;
            p.ke = c.n_ecc > 0 ? (const double2 *)c.d_ke.p : nullptr;
            p.n_pad = pd.n_pad; p.n_entries = pd.n_entries; p.n_chunks = pd.n_pad / kChunk;
            p.n_pix = pd.n_pix; p.n_ap = pd.n_ap; p.n_P = pd.n_P; p.n_tasc = pd.n_tasc; p.n_f0 = pd.n_f0;
            p.j0 = j0; p.n_fj = std::min(tile_bins, pd.n_f0 - j0);
            p.n_groups = pd.n_groups; p.n_aq = pd.n_ap * pd.n_tasc; p.n_aq_tiles = pd.n_aq_tiles;
            p.u0 = (double)(pd.k_band0 + j0);
            p.off = (int)(pd.k_band0 - pd.k_slab0) + j0 + pd.off_table;
            p.s_max = pd.s_max;
            p.s_zero = pd.s_zero;
            p.list_cap = pd.list_cap;
            p.thr = (const Threshold *)ctx->thr.p;
            p.cand = (RawCand *)ctx->cand.p;
            p.cand_count = (unsigned int *)ctx->cand_count.p;
            p.cand_cap = pd.cand_cap;
            p.counts_full = pd.d_counts_full;
            const int64_t grid = (int64_t)pd.n_groups * pd.n_P * pd.n_aq_tiles;
            if (grid > 0x7FFFFFFFll) return fail(ctx, BSH_EINVAL, "grid too large");
            ctx->st.grid_blocks = (int)grid;
            ctx->st.threads_per_block = pd.tpb;
            TRY(weighted ? dispatch_weighted(ctx, pd, p, (int)grid) : dispatch_unweighted(ctx, pd, p, (int)grid));
        }
    }
    CK(cudaEventRecord(ctx->ev[3], ctx->stream));
    pd.passes += 1;
    return BSH_OK;
}

// sort the first n candidates of ctx->cand (buffer has room for the power-of-two padding)
int sort_candidates(bsh_ctx *ctx, RawCand *buf, unsigned int n)
{
    if (n <= 1) return BSH_OK;
    unsigned int n2 = 1;
    while (n2 < n) n2 <<= 1;
    if (n2 > n) {
        pad_candidates_kernel<<<(n2 - n + 255) / 256, 256, 0, ctx->stream>>>(buf, n, n2);
        count_launch(ctx);
    }
    const unsigned int tiles = (n2 + kSortTile - 1) / kSortTile;
    const unsigned int k_local = std::min<unsigned int>(n2, kSortTile);
    bitonic_tile_kernel<<<tiles, 1024, 0, ctx->stream>>>(buf, n2, 2u, k_local);
    count_launch(ctx);
    for (unsigned int k = kSortTile * 2; k <= n2; k <<= 1) {
        for (unsigned int j = k >> 1; j >= (unsigned)kSortTile; j >>= 1) {
            bitonic_global_kernel<<<(n2 / 2 + 255) / 256, 256, 0, ctx->stream>>>(buf, n2, k, j);
            count_launch(ctx);
        }
        bitonic_tile_kernel<<<tiles, 1024, 0, ctx->stream>>>(buf, n2, k, k);
        count_launch(ctx);
    }
    CK(cudaGetLastError());
    return BSH_OK;
}

constexpr unsigned int kRadixMin = 1u << 16;      // above this many records the radix sort replaces the bitonic network

// Large lists: stable LSD radix sort by (key desc, index asc), one pass per byte of the composite key in
// which the records differ.  buf and tmp hold n records each; *out = the buffer that ends up sorted.  Synchronises once.
int radix_sort_candidates(bsh_ctx *ctx, RawCand *buf, RawCand *tmp, unsigned int n, RawCand **out)
{
    *out = buf;
    if (n <= 1) return BSH_OK;
    const unsigned int n_tiles = (n + kRadixTile - 1) / kRadixTile;
    TRY(ensure(ctx, ctx->radix_hist, 64 + (size_t)256 * n_tiles * 4));
    unsigned int *d_diff = (unsigned int *)ctx->radix_hist.p;
    unsigned int *d_hist = d_diff + 16;
    CK(cudaMemsetAsync(d_diff, 0, 12, ctx->stream));
    radix_diff_kernel<<<std::min(1024u, (n + 255) / 256), 256, 0, ctx->stream>>>(buf, n, d_diff);
    count_launch(ctx);
    CK(cudaMemcpyAsync(ctx->pinned_count + 10, d_diff, 12, cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    const uint64_t di = (uint64_t)ctx->pinned_count[10] | ((uint64_t)ctx->pinned_count[11] << 32);
    const uint32_t dk = ctx->pinned_count[12];
    RawCand *src = buf, *dst = tmp;
    for (int pass = 0; pass < 12; ++pass) {
        const bool varies = pass < 8 ? ((di >> (8 * pass)) & 255u) != 0 : ((dk >> (8 * (pass - 8))) & 255u) != 0;
        if (!varies) continue;
        radix_hist_kernel<<<n_tiles, kRadixThreads, 0, ctx->stream>>>(src, n, pass, n_tiles, d_hist);
        radix_scan_kernel<<<1, 1024, 0, ctx->stream>>>(d_hist, 256u * n_tiles);
        radix_scatter_kernel<<<n_tiles, kRadixThreads, 0, ctx->stream>>>(src, n, pass, n_tiles, d_hist, dst);
        count_launch(ctx, 3);
        std::swap(src, dst);
    }
    CK(cudaGetLastError());
    *out = src;
    return BSH_OK;
}

}  // namespace

namespace {

template <int OP>
int run_peak(bsh_ctx *ctx, int n_sm, int iters, std::vector<PeakSample> &host, double *ops_per_clk_sm, double *mhz)
{
    PeakSample *d = (PeakSample *)ctx->peak_samples.p;
    uint32_t *sink = (uint32_t *)((char *)ctx->peak_samples.p + sizeof(PeakSample) * (size_t)n_sm);
    for (int rep = 0; rep < 2; ++rep) {                  // the first launch warms the instruction cache and the clocks
        peak_kernel<OP><<<n_sm, kPeakThreads, 0, ctx->stream>>>(iters, (uint32_t)(rep + 1), sink, d);
        count_launch(ctx);
    }
    CK(cudaGetLastError());
    CK(cudaMemcpyAsync(host.data(), d, sizeof(PeakSample) * (size_t)n_sm, cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    std::vector<double> cyc(n_sm), f(n_sm);
    for (int b = 0; b < n_sm; ++b) {
        cyc[b] = (double)host[b].cycles;
        f[b] = host[b].ns ? 1e3 * (double)host[b].cycles / (double)host[b].ns : 0.0;
    }
    std::sort(cyc.begin(), cyc.end());
    std::sort(f.begin(), f.end());
    *ops_per_clk_sm = (double)kPeakThreads * iters * kPeakUnroll / cyc[n_sm / 2];
    if (mhz) *mhz = f[n_sm / 2];
    return BSH_OK;
}

}  // namespace

// =====================================================================================================================
// C ABI
// =====================================================================================================================
extern "C" {

int bsh_version(void) { return 200; }

int bsh_create(bsh_ctx **out, int device, void *cuda_stream)
{
    if (!out) return BSH_EINVAL;
    *out = nullptr;
    int n_dev = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess || n_dev < 1 || device < 0 || device >= n_dev) return BSH_ECUDA;
    bsh_ctx *ctx = new (std::nothrow) bsh_ctx();
    if (!ctx) return BSH_ENOMEM;
    ctx->device = device;
    ctx->stream = (cudaStream_t)cuda_stream;
    const DeviceGuard device_guard(device);
    for (auto &e : ctx->ev)
        if (cudaEventCreate(&e) != cudaSuccess) { delete ctx; return BSH_ECUDA; }
    if (cudaMallocHost((void **)&ctx->pinned_count, 64) != cudaSuccess) { delete ctx; return BSH_ENOMEM; }
    *out = ctx;
    return BSH_OK;
}

int bsh_destroy(bsh_ctx *ctx)
{
    if (!ctx) return BSH_EINVAL;
    const DeviceGuard device_guard(ctx->device);
    cudaStreamSynchronize(ctx->stream);
    DevBuf *bufs[] = {&ctx->wtab, &ctx->w_pad, &ctx->stats, &ctx->thr, &ctx->dtab, &ctx->nvec, &ctx->cand, &ctx->cand_count,
                      &ctx->keys, &ctx->tmp_cands, &ctx->dtab2, &ctx->nvec2, &ctx->ptab, &ctx->dpos, &ctx->dpix, &ctx->psplit, &ctx->tab7, &ctx->h_rho, &ctx->h_w, &ctx->h_peak, &ctx->h_top, &ctx->peak_samples,
                      &ctx->post_adj, &ctx->post_cnt, &ctx->post_off, &ctx->post_tmp, &ctx->radix_hist};
    for (DevBuf *b : bufs)
        if (b->p) cudaFree(b->p);
    for (auto &c : ctx->cache) {
        DevBuf *cb[] = {&c.d_v, &c.d_cs, &c.d_casa, &c.d_A, &c.d_ke, &c.d_cs_t};
        for (DevBuf *b : cb)
            if (b->p) cudaFree(b->p);
    }
    for (auto &e : ctx->ev)
        if (e) cudaEventDestroy(e);
    if (ctx->pinned_count) cudaFreeHost(ctx->pinned_count);
    delete ctx;
    return BSH_OK;
}

const char *bsh_last_error(const bsh_ctx *ctx) { return ctx ? ctx->err.c_str() : "null context"; }

int bsh_get_stats(bsh_ctx *ctx, bsh_stats *out)
{
    if (!ctx || !out) return BSH_EINVAL;
    const DeviceGuard device_guard(ctx->device);
    CK(cudaStreamSynchronize(ctx->stream));
    float ms = 0.f;
    if (ctx->have_pk && cudaEventElapsedTime(&ms, ctx->ev[8], ctx->ev[9]) == cudaSuccess) ctx->st.peakgram_ms = ms;
    if (ctx->have_setup && cudaEventElapsedTime(&ms, ctx->ev[0], ctx->ev[1]) == cudaSuccess) ctx->st.stage1_setup_ms = ms;
    if (ctx->have_kernel && cudaEventElapsedTime(&ms, ctx->ev[2], ctx->ev[3]) == cudaSuccess)
        ctx->st.stage1_kernel_ms = ms + ctx->kernel_ms_extra;
    if (ctx->have_select && cudaEventElapsedTime(&ms, ctx->ev[4], ctx->ev[5]) == cudaSuccess) ctx->st.stage1_select_ms = ms;
    if (ctx->have_s2 && cudaEventElapsedTime(&ms, ctx->ev[6], ctx->ev[7]) == cudaSuccess) ctx->st.stage2_ms = ms;
    if (ctx->have_front && cudaEventElapsedTime(&ms, ctx->ev[10], ctx->ev[11]) == cudaSuccess) ctx->st.frontend_ms = ms;
    *out = ctx->st;
    return BSH_OK;
}

int bsh_set_option(bsh_ctx *ctx, int32_t option, int32_t value)
{
    if (!ctx) return BSH_EINVAL;
    switch (option) {
    case BSH_OPT_KERNEL_FAMILY:
        if (value < BSH_FAMILY_AUTO || value > BSH_FAMILY_WINDOW) return fail(ctx, BSH_EINVAL, "unknown kernel family %d", value);
        ctx->opt_family = value;
        return BSH_OK;
    case BSH_OPT_FORCE_CLAMP:
        ctx->opt_force_clamp = value != 0;
        return BSH_OK;
    case BSH_OPT_PIXELS_PER_THREAD:
        if (value < 0 || value > 2) return fail(ctx, BSH_EINVAL, "pixels per thread must be 0 (auto), 1 or 2");
        ctx->opt_pixels_per_thread = value;
        return BSH_OK;
    default:
        return fail(ctx, BSH_EINVAL, "unknown option %d", option);
    }
}

int bsh_measure_peaks(bsh_ctx *ctx, bsh_peaks *h_out)
{
    if (!ctx || !h_out) return BSH_EINVAL;
    const DeviceGuard device_guard(ctx->device);
    cudaDeviceProp prop;
    CK(cudaGetDeviceProperties(&prop, ctx->device));
    const int n_sm = prop.multiProcessorCount;
    TRY(ensure(ctx, ctx->peak_samples, sizeof(PeakSample) * (size_t)n_sm + 64));
    std::vector<PeakSample> host(n_sm);
    bsh_peaks pk = {};
    pk.n_sm = n_sm;
    double mhz[4] = {0, 0, 0, 0}, v = 0;
    TRY(run_peak<kOpLop3>(ctx, n_sm, 1000, host, &pk.lop3_lanes_per_clk_sm, &mhz[0]));
    TRY(run_peak<kOpFadd>(ctx, n_sm, 1000, host, &pk.fadd_lanes_per_clk_sm, &mhz[1]));
    TRY(run_peak<kOpDadd>(ctx, n_sm, 500, host, &pk.dadd_lanes_per_clk_sm, &mhz[2]));
    TRY(run_peak<kOpDmul>(ctx, n_sm, 500, host, &pk.dmul_lanes_per_clk_sm, nullptr));
    TRY(run_peak<kOpMixed>(ctx, n_sm, 1000, host, &v, &mhz[3]));
    pk.issue_warp_inst_per_clk_smsp = v / 32.0 / 4.0;
    TRY(run_peak<kOpLds32>(ctx, n_sm, 500, host, &v, nullptr));
    pk.lds32_bytes_per_clk_sm = 4.0 * v;
    TRY(run_peak<kOpLds64>(ctx, n_sm, 500, host, &v, nullptr));
    pk.lds64_bytes_per_clk_sm = 8.0 * v;
    TRY(run_peak<kOpLds128>(ctx, n_sm, 250, host, &v, nullptr));
    pk.lds128_bytes_per_clk_sm = 16.0 * v;
    std::sort(mhz, mhz + 4);
    pk.sm_clock_mhz = 0.5 * (mhz[1] + mhz[2]);
    *h_out = pk;
    return BSH_OK;
}

int bsh_build_peakgram(bsh_ctx *ctx, const float *d_rho, int32_t n_sft, int32_t n_bins, int64_t rho_row_stride,
                       float rho_th, uint32_t *d_peak, int32_t words_per_row)
{
    if (!ctx) return BSH_EINVAL;
    if (!d_rho || !d_peak || n_sft < 1 || n_bins < 1 || rho_row_stride < n_bins)
        return fail(ctx, BSH_EINVAL, "bsh_build_peakgram: bad arguments");
    if ((int64_t)words_per_row * 32 < n_bins) return fail(ctx, BSH_ESMALL, "words_per_row * 32 < n_bins");
    const DeviceGuard device_guard(ctx->device);
    CK(cudaEventRecord(ctx->ev[8], ctx->stream));
    const bool vec4 = (rho_row_stride % 4 == 0) && ((uintptr_t)d_rho % 16 == 0);
    if (vec4) {
        const int segs = (words_per_row + 3) / 4;
        const int64_t warps = (int64_t)n_sft * segs;
        peakgram_vec4_kernel<<<(unsigned)((warps + 7) / 8), 256, 0, ctx->stream>>>(d_rho, n_sft, n_bins, rho_row_stride,
                                                                                    rho_th, d_peak, words_per_row);
    } else {
        const int64_t warps = (int64_t)n_sft * words_per_row;
        peakgram_scalar_kernel<<<(unsigned)((warps + 7) / 8), 256, 0, ctx->stream>>>(d_rho, n_sft, n_bins, rho_row_stride,
                                                                                      rho_th, d_peak, words_per_row);
    }
    count_launch(ctx);
    CK(cudaGetLastError());
    CK(cudaEventRecord(ctx->ev[9], ctx->stream));
    ctx->have_pk = true;
    return BSH_OK;
}

double bsh_median_bias(int32_t window)
{
    if (window < 1) return 0.0;
    double s = 0.0;                                       // expectation of the middle order statistic of `window` Exp(1) draws
    for (int i = (window + 1) / 2; i <= window; ++i) s += 1.0 / (double)i;
    return s;
}

int bsh_normalise_peakgram(bsh_ctx *ctx, const float *d_sft, int32_t n_sft, int32_t n_raw, int64_t sft_row_stride,
                           int32_t window, float median_bias, float rho_th, float *d_rho, int64_t rho_row_stride,
                           uint32_t *d_peak, int32_t words_per_row)
{
    if (!ctx) return BSH_EINVAL;
    if (!d_sft || (!d_rho && !d_peak) || n_sft < 1 || n_raw < 1 || sft_row_stride < n_raw)
        return fail(ctx, BSH_EINVAL, "bsh_normalise_peakgram: bad arguments");
    if (window < 1 || (window & 1) == 0 || window > n_raw) return fail(ctx, BSH_EINVAL, "window must be odd and <= n_raw");
    if (n_raw > kFrontMaxRaw) return fail(ctx, BSH_EINVAL, "n_raw > %d: split the band", kFrontMaxRaw);
    if (!(median_bias > 0.f)) return fail(ctx, BSH_EINVAL, "median_bias must be positive");
    if ((uintptr_t)d_sft % 8 != 0) return fail(ctx, BSH_EINVAL, "d_sft must be 8-byte aligned");
    const int K = n_raw - window + 1;
    if (d_rho && rho_row_stride < K) return fail(ctx, BSH_EINVAL, "rho_row_stride < n_raw - window + 1");
    if (d_peak && (int64_t)words_per_row * 32 < K) return fail(ctx, BSH_ESMALL, "words_per_row * 32 < n_raw - window + 1");
    const DeviceGuard device_guard(ctx->device);
    const size_t smem = front_smem_bytes(n_raw);
    if (smem > 48 * 1024)
        CK(cudaFuncSetAttribute(normalise_peakgram_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    CK(cudaEventRecord(ctx->ev[10], ctx->stream));
    normalise_peakgram_kernel<<<(unsigned)n_sft, kFrontThreads, smem, ctx->stream>>>(
        (const float2 *)d_sft, n_raw, sft_row_stride, window, median_bias, rho_th, d_rho, rho_row_stride, d_peak,
        words_per_row);
    count_launch(ctx);
    CK(cudaGetLastError());
    CK(cudaEventRecord(ctx->ev[11], ctx->stream));
    ctx->have_front = true;
    return BSH_OK;
}

int bsh_stage1_launch(bsh_ctx *ctx, const uint32_t *d_peak, int32_t words_per_row, const bsh_sfts *sfts,
                      const bsh_grid *grid, int32_t mode, int32_t topk, void *d_counts_full)
{
    if (!ctx) return BSH_EINVAL;
    TRY(validate(ctx, sfts, grid));
    if (!d_peak || topk < 1) return fail(ctx, BSH_EINVAL, "bsh_stage1: null peakgram or topk < 1");
    if (topk > kMaxTopk) return fail(ctx, BSH_EINVAL, "bsh_stage1: topk = %d is beyond the documented maximum of 2^27", topk);
    if ((int64_t)words_per_row * 32 < sfts->n_bins) return fail(ctx, BSH_ESMALL, "words_per_row * 32 < n_bins");
    if ((mode & BSH_WEIGHTED) && !sfts->d_w) return fail(ctx, BSH_EINVAL, "BSH_WEIGHTED needs sfts->d_w");
    if (mode & ~(BSH_WEIGHTED | BSH_NAIVE)) return fail(ctx, BSH_EINVAL, "unknown mode bits");
    const DeviceGuard device_guard(ctx->device);
    ctx->pend.active = false;

    Pending pd;
    pd.mode = mode; pd.topk = topk; pd.d_counts_full = d_counts_full; pd.d_peak = d_peak;
    pd.words_per_row = words_per_row; pd.d_w = sfts->d_w;
    pd.n_sft = sfts->n_sft; pd.n_bins = sfts->n_bins; pd.n_pix = grid->n_pix; pd.n_ap = grid->n_ap; pd.n_P = grid->n_P;
    const bsh_grid kg = kernel_grid(grid);             // eccentricity axis folded into the t_asc axis
    const double ecc_max = ecc_max_of(grid);
    pd.n_tasc = kg.n_tasc; pd.n_f0 = grid->n_f0; pd.k_band0 = grid->k_band0; pd.k_slab0 = sfts->k_slab0;
    pd.n_templates = (uint64_t)grid->n_pix * grid->n_ap * grid->n_P * kg.n_tasc * (uint64_t)grid->n_f0;
    const bool weighted = (mode & BSH_WEIGHTED) != 0;

    TRY(get_tables(ctx, sfts, grid, &pd.cache_slot));
    const TableCache &c = ctx->cache[pd.cache_slot];
    pd.n_pad = c.n_pad;

    // kernel shape
    pd.NW = grid->n_f0 <= 64 ? 2 : 3;
    pd.R = weighted ? 1 : 2;
    pd.tile_bins = 32 * pd.NW;
    // weighted count: one FP32 accumulator per bin lives in registers; 90 of them spill (ncu: 0.2 local-memory accesses
    // per accumulation), so a band of 65..96 bins is done as two passes of half the bins (two-word windows)
    if (weighted && grid->n_f0 > 64 && grid->n_f0 <= 96) {
        pd.NW = 2;
        pd.tile_bins = (grid->n_f0 + 1) / 2;
    }
    // weighted pixel-lane kernel (bsh_wpix.cuh): one pass over tiles of <= 90 bins (15 bytes of 6 bins; 8 bytes for <= 48)
    pd.n_pg = (grid->n_pix + 31) / 32;
    const bool lanes_ok = 10 * grid->n_pix >= 6 * 32 * pd.n_pg;
    const int fam = ctx->opt_family;
    bool try_wpix = weighted && !(mode & BSH_NAIVE) && ((fam == BSH_FAMILY_AUTO && lanes_ok) || fam == BSH_FAMILY_PIXEL_LANE);
    if (try_wpix) {
#ifndef BSH_WPIX_MAXBINS
#define BSH_WPIX_MAXBINS 90
#endif
        const int n_tiles = (grid->n_f0 + BSH_WPIX_MAXBINS - 1) / BSH_WPIX_MAXBINS;
        const int tile = (grid->n_f0 + n_tiles - 1) / n_tiles;
        const int nbytes = tile <= 48 ? 8 : 15, nw = nbytes == 8 ? 2 : 3;
        const TableGeometry tgw = table_geometry(sfts->n_sft, sfts->h_v_over_c, grid->n_P, grid->h_P, grid->n_ap, grid->h_ap,
                                                 grid->k_band0, sfts->k_slab0, grid->n_f0, sfts->n_bins, nw,
                                                 ctx->opt_force_clamp != 0, ecc_max);
        const PosGeometry pgw = pos_geometry(tgw, sfts->n_bins, grid->n_f0, nw, tile);
        const WpixStage ws(pgw.n_pos, wpix_entry_bytes(nbytes));
        const int stages = std::min(kMaxStages, ((226 * 1024) / kWpixBlocksPerSm - 2048 - kWpixHeader) / ws.stride);
        if (stages >= 2) {
            pd.use_wpix = true;
            pd.tile_bins = tile; pd.wpix_nbytes = nbytes; pd.NW = nw;
            pd.wpix_stages = std::max(1, std::min(stages, pd.n_pad / kStageSfts));
            pd.wpix_smem = ws.total(pd.wpix_stages);
        }
    }
    if (!weighted && (ctx->opt_pixels_per_thread == 1 || ctx->opt_pixels_per_thread == 2)) pd.R = ctx->opt_pixels_per_thread;
    pd.HP = sfts->n_sft < (1 << 11) ? 6 : (sfts->n_sft < (1 << 13) ? 8 : 11);
    if (sfts->n_sft >= (1 << 16)) return fail(ctx, BSH_EINVAL, "n_sft >= 65536 not supported");
    const TableGeometry tg = table_geometry(sfts->n_sft, sfts->h_v_over_c, grid->n_P, grid->h_P, grid->n_ap, grid->h_ap,
                                            grid->k_band0, sfts->k_slab0, grid->n_f0, sfts->n_bins, pd.NW,
                                            ctx->opt_force_clamp != 0, ecc_max);
    pd.clamp = tg.clamp; pd.off_table = tg.off_table; pd.s_max = tg.s_max; pd.n_entries = tg.n_entries;
    pd.s_zero = tg.s_zero;
    const int n_aq = grid->n_ap * kg.n_tasc;
    pd.tpb = pick_threads_per_block(n_aq);
    pd.n_aq_tiles = (n_aq + pd.tpb - 1) / pd.tpb;
    pd.list_cap = 48;
    pd.n_groups = (grid->n_pix + pd.R - 1) / pd.R;
    {   // position-table kernels when 2+ stages of the table fit in shared memory (else the funnel-shift kernels)
        const PosGeometry pg = pos_geometry(tg, sfts->n_bins, grid->n_f0, pd.NW, pd.tile_bins);
        pd.pos_off = pg.off_table; pd.pos_s_max = pg.s_max; pd.pos_s_zero = pg.s_zero; pd.n_pos = pg.n_pos;
        const int wpb = weighted ? kWarpsWeighted : kWarpsUnweighted;
        const int stride = weighted ? PosStage<kWarpsWeighted, 1, true>(pg.n_pos).stride
                                    : PosStage<kWarpsUnweighted, 2, false>(pg.n_pos).stride;
        const int budgets[3] = {112 * 1024, 112 * 1024, 224 * 1024};                          // 2 / 2 / 1 blocks per SM
        const int pix_one = kPixWarps > 8 ? 224 * 1024 : 113 * 1024;                          // blocks of > 8 warps own an SM
        const int pix_budgets[3] = {pix_one, pix_one, 224 * 1024};                            // (228 KB - 1 KB per block) / 2
        pd.n_stages = 0;
        for (int b = 0; b < 3 && pd.n_stages < 2; ++b) pd.n_stages = std::min(kMaxStages, (budgets[b] - kPosHeader) / stride);
        pd.use_pos = pd.n_stages >= 2 && fam != BSH_FAMILY_WINDOW && !(mode & BSH_NAIVE);
        pd.n_stages = std::min(pd.n_stages, pd.n_pad / kStageSfts);
        pd.pos_groups = weighted ? grid->n_pix : (grid->n_pix + 1) / 2;
        pd.n_oct = (pd.pos_groups + wpb - 1) / wpb;
        pd.pos_smem = kPosHeader + pd.n_stages * stride;
        // pixel-lane kernel (unweighted): pixels on the lanes pay off when most of the 32 lanes of a group are used
        const PixStage ps(pg.n_pos, pd.NW);
        pd.pix_stages = 0;
        const int hi_bytes = pix_hi_bytes(pd.NW, pd.HP);                                    // shared-memory high planes
        for (int b = 1; b < 3 && pd.pix_stages < 2; ++b)
            pd.pix_stages = std::min(4, (pix_budgets[b] - kPixHeader - hi_bytes) / ps.stride);  // (2..6 stages measure alike)
        pd.use_pix = !weighted && pd.pix_stages >= 2 && (lanes_ok || fam == BSH_FAMILY_PIXEL_LANE) &&
                     (fam == BSH_FAMILY_AUTO || fam == BSH_FAMILY_PIXEL_LANE) && !(mode & BSH_NAIVE);
        pd.pix_stages = std::max(1, std::min(pd.pix_stages, pd.n_pad / kStageSfts));
        pd.pix_smem = kPixHeader + pd.pix_stages * ps.stride + hi_bytes;
    }
    // Toplists as large as a fraction N_C of the bank (L225: 5-10 % of all templates go to stage 2) need a larger
    // candidate buffer and a tighter first guess of the threshold (1.3 k instead of 8 k expected survivors).
    pd.cand_cap = kCandCap;
    if ((uint64_t)topk > kCandCap / 8) {
        const uint64_t need = std::min<uint64_t>(pd.n_templates, 4ull * (uint64_t)topk);
        while (pd.cand_cap < need && pd.cand_cap < (1u << 27)) pd.cand_cap <<= 1;
    }
    if (std::min<uint64_t>((uint64_t)topk, pd.n_templates) > pd.cand_cap)
        return fail(ctx, BSH_EINVAL, "topk = %d exceeds the candidate buffer (%u entries)", topk, pd.cand_cap);
    pd.emit_all = pd.n_templates <= pd.cand_cap;
    pd.frac = (double)std::max<int64_t>(8ll * topk, 4096) / (double)pd.n_templates;
    if ((uint64_t)topk > kCandCap / 8) pd.frac = (1.3 * (double)topk + 4096.0) / (double)pd.n_templates;
    if (pd.frac >= 0.25) pd.frac = (uint64_t)topk > kCandCap / 8 ? std::min(pd.frac, 0.45) : 0.25;
    pd.passes = 0;

    // device scratch
    TRY(ensure(ctx, ctx->wtab, (size_t)pd.n_pad * pd.n_entries * 16));
    TRY(ensure(ctx, ctx->w_pad, (size_t)pd.n_pad * 4));
    TRY(ensure(ctx, ctx->stats, 16));
    TRY(ensure(ctx, ctx->thr, sizeof(Threshold)));
    TRY(ensure(ctx, ctx->cand, (size_t)pd.cand_cap * sizeof(RawCand)));
    TRY(ensure(ctx, ctx->cand_count, 16));

    CK(cudaEventRecord(ctx->ev[0], ctx->stream));
    CK(cudaMemsetAsync(ctx->stats.p, 0, 16, ctx->stream));
    prep_table_kernel<<<(pd.n_pad + 255) / 256, 256, 0, ctx->stream>>>(
        d_peak, words_per_row, sfts->n_sft, pd.n_pad, sfts->n_bins, pd.n_entries, pd.off_table / 32,
        weighted ? sfts->d_w : nullptr, (uint4 *)ctx->wtab.p, (float *)ctx->w_pad.p, (double *)ctx->stats.p);
    count_launch(ctx);
    CK(cudaGetLastError());
    TRY(build_dtable(ctx, grid, c, pd.R, ctx->nvec, ctx->dtab));
    if (pd.use_wpix) {
        const int eb = wpix_entry_bytes(pd.wpix_nbytes);
        const int64_t n_ent = (int64_t)pd.n_pad * pd.n_pos;
        TRY(ensure(ctx, ctx->tab7, (size_t)(pd.n_pad / kStageSfts) * (size_t)wpix_stage_tab_bytes(pd.n_pos, eb)));
        TRY(ensure(ctx, ctx->dpix, sizeof(double) * (size_t)pd.n_pg * pd.n_pad * 32));
        if (eb == 8)
            build_position7_table_kernel<8><<<(unsigned)((n_ent + 255) / 256), 256, 0, ctx->stream>>>(
                d_peak, words_per_row, sfts->n_sft, pd.n_pad, sfts->n_bins, pd.n_pos, pd.pos_off, pd.pos_s_zero,
                (unsigned char *)ctx->tab7.p);
        else
            build_position7_table_kernel<16><<<(unsigned)((n_ent + 255) / 256), 256, 0, ctx->stream>>>(
                d_peak, words_per_row, sfts->n_sft, pd.n_pad, sfts->n_bins, pd.n_pos, pd.pos_off, pd.pos_s_zero,
                (unsigned char *)ctx->tab7.p);
        count_launch(ctx);
        const int64_t n_d = (int64_t)pd.n_pg * pd.n_pad * 32;
        dtable_pix_kernel<<<(unsigned)((n_d + 255) / 256), 256, 0, ctx->stream>>>(
            (const double *)c.d_v.p, (const double *)ctx->nvec.p, c.n_sft, pd.n_pad, grid->n_pix, pd.n_pg,
            (double *)ctx->dpix.p);
        count_launch(ctx);
        CK(cudaGetLastError());
    } else if (pd.use_pix) {
        TRY(ensure(ctx, ctx->ptab, (size_t)pd.n_pad * pd.n_pos * 16));
        TRY(ensure(ctx, ctx->dpix, sizeof(double) * (size_t)pd.n_pg * pd.n_pad * 32));
        const int64_t n_ent = (int64_t)pd.n_pad * pd.n_pos;
        build_position_table_kernel<<<(unsigned)((n_ent + 255) / 256), 256, 0, ctx->stream>>>(
            d_peak, words_per_row, sfts->n_sft, pd.n_pad, sfts->n_bins, pd.n_pos, pd.pos_off, pd.pos_s_zero,
            (uint4 *)ctx->ptab.p);
        count_launch(ctx);
        TRY(ensure(ctx, ctx->psplit, (size_t)(pd.n_pad / kStageSfts) * (size_t)pix_stage_tab_bytes(pd.n_pos, pd.NW)));
        pm_position_table_kernel<<<(unsigned)((n_ent + 255) / 256), 256, 0, ctx->stream>>>(
            (const uint4 *)ctx->ptab.p, pd.n_pad, pd.n_pos, pd.NW, (unsigned char *)ctx->psplit.p);
        count_launch(ctx);
        const int64_t n_d = (int64_t)pd.n_pg * pd.n_pad * 32;
        dtable_pix_kernel<<<(unsigned)((n_d + 255) / 256), 256, 0, ctx->stream>>>(
            (const double *)c.d_v.p, (const double *)ctx->nvec.p, c.n_sft, pd.n_pad, grid->n_pix, pd.n_pg,
            (double *)ctx->dpix.p);
        count_launch(ctx);
        CK(cudaGetLastError());
    } else if (pd.use_pos) {
        const int wpb = weighted ? kWarpsWeighted : kWarpsUnweighted, R = weighted ? 1 : 2;
        TRY(ensure(ctx, ctx->ptab, (size_t)pd.n_pad * pd.n_pos * 16));
        TRY(ensure(ctx, ctx->dpos, sizeof(double) * (size_t)pd.n_oct * pd.n_pad * wpb * R));
        const int64_t n_ent = (int64_t)pd.n_pad * pd.n_pos;
        build_position_table_kernel<<<(unsigned)((n_ent + 255) / 256), 256, 0, ctx->stream>>>(
            d_peak, words_per_row, sfts->n_sft, pd.n_pad, sfts->n_bins, pd.n_pos, pd.pos_off, pd.pos_s_zero,
            (uint4 *)ctx->ptab.p);
        count_launch(ctx);
        const int64_t n_d = (int64_t)pd.n_oct * pd.n_pad * wpb * R;
        dtable_pos_kernel<<<(unsigned)((n_d + 255) / 256), 256, 0, ctx->stream>>>(
            (const double *)c.d_v.p, (const double *)ctx->nvec.p, c.n_sft, pd.n_pad, grid->n_pix, pd.n_oct, wpb, R,
            (double *)ctx->dpos.p);
        count_launch(ctx);
        CK(cudaGetLastError());
    }
    CK(cudaEventRecord(ctx->ev[1], ctx->stream));
    ctx->have_setup = true;

    ctx->pend = pd;
    ctx->kernel_ms_extra = 0.f;
    TRY(run_pass(ctx));
    ctx->have_kernel = true;
    CK(cudaMemcpyAsync(ctx->pinned_count, ctx->cand_count.p, sizeof(unsigned int), cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaMemcpyAsync(ctx->pinned_count + 4, ctx->thr.p, kThresholdHostBytes, cudaMemcpyDeviceToHost, ctx->stream));
    ctx->pend.active = true;

    ctx->st.n_templates = (int64_t)pd.n_templates;
    ctx->st.n_accumulations = (int64_t)pd.n_templates * sfts->n_sft;
    ctx->st.kernel_variant = 1000 * (pd.use_wpix ? BSH_KERNEL_PIXEL_LANE_W : pd.use_pix ? BSH_KERNEL_PIXEL_LANE : pd.use_pos ? BSH_KERNEL_TEMPLATE_LANE : BSH_KERNEL_WINDOW) + pd.NW * 100 + pd.R * 10 + (pd.clamp ? 1 : 0);
    return BSH_OK;
}

int bsh_stage1_collect(bsh_ctx *ctx, bsh_cand *d_top, int32_t *h_n_top)
{
    if (!ctx) return BSH_EINVAL;
    if (!ctx->pend.active) return fail(ctx, BSH_ESTATE, "bsh_stage1_collect without a pending bsh_stage1_launch");
    if (!d_top || !h_n_top) return fail(ctx, BSH_EINVAL, "null d_top / h_n_top");
    const DeviceGuard device_guard(ctx->device);
    Pending &pd = ctx->pend;
    const bool weighted = (pd.mode & BSH_WEIGHTED) != 0;
    const uint64_t want = std::min<uint64_t>((uint64_t)pd.topk, pd.n_templates);
    unsigned int n_cand = 0;
    Threshold thr = {};
    // Threshold search.  The first pass used the noise-model threshold.  Too few survivors (< topk) or too many (> the
    // candidate buffer) happen when the data are not what the model assumes (lines, notched bands, constant rows).  Then:
    //   too few    lower tau by steps that double (0.75, 1.5, 3 ... model sigmas), not below 0 (both statistics are >= 0).
    //   too many   the buffer holds cand_cap of the survivors; its topk-th largest value T_b has at least topk templates at
    //              or above it, so tau = T_b cannot give too few and normally lands in range at once.  T_b equal to the
    //              threshold itself means that the templates AT that value alone overflow the buffer -- massive ties at
    //              the cut (notched band, constant rows, very few SFTs):
    //   phase 1    count the templates above the tie value T (one pass at the next representable threshold);
    //   phase 2    tau = T, and of the ties only those with template index < tie_limit are emitted; search on tie_limit
    //              (first guess from the tie density, then regula falsi / bisection).  The buffer then holds everything
    //              above T and the lowest-index ties, which contains the (value desc, index asc) toplist.
    for (;;) {
        CK(cudaStreamSynchronize(ctx->stream));
        n_cand = ctx->pinned_count[0];
        memcpy(&thr, ctx->pinned_count + 4, kThresholdHostBytes);
        if (!pd.fixed) pd.tau = weighted ? (double)thr.tau_f : (double)thr.tau_i;
        const bool too_few = n_cand < want, too_many = n_cand > pd.cand_cap;
        if (!too_few && !too_many) break;
        if (pd.passes >= kMaxPasses)
            return fail(ctx, BSH_ESTATE, "candidate selection did not converge after %d passes (%u candidates for topk %d at "
                                         "threshold %g, phase %d)", pd.passes, n_cand, pd.topk, pd.tau, pd.phase);
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, ctx->ev[2], ctx->ev[3]) == cudaSuccess) ctx->kernel_ms_extra += ms;
        const double sigma = (double)thr.sigma, mean = (double)thr.mean;
        const double unit = sigma > 0.0 ? sigma : (weighted ? std::max(fabs(mean) * 0.01, 1.0e-3) : 1.0);
        auto next_up = [&](double t) { return weighted ? (double)nextafterf((float)t, INFINITY) : t + 1.0; };
        bool start_ties = false;
        if (pd.phase == 1 && too_many) pd.phase = 0;                  // not ties after all: an ordinary overflow
        if (pd.phase == 0 && too_many) {
            TRY(ensure(ctx, ctx->keys, (size_t)pd.cand_cap * sizeof(RawCand)));
            RawCand *by_value = nullptr;
            TRY(radix_sort_candidates(ctx, (RawCand *)ctx->cand.p, (RawCand *)ctx->keys.p, pd.cand_cap, &by_value));
            CK(cudaMemcpyAsync(ctx->pinned_count + 2, &by_value[want - 1].key, 4, cudaMemcpyDeviceToHost, ctx->stream));
            CK(cudaStreamSynchronize(ctx->stream));
            const uint32_t kb = ctx->pinned_count[2];
            float fb;
            memcpy(&fb, &kb, 4);
            const double t_b = weighted ? (double)fb : (double)kb;
            pd.lo_tau = std::max(pd.tau, 0.0);
            pd.lo_n = n_cand;
            if (t_b > pd.lo_tau) {
                pd.tau = t_b;
            } else {
                pd.phase = 1;
                pd.tau = next_up(pd.lo_tau);
            }
        } else if (pd.phase == 0) {                                   // too few
            double t = weighted ? (double)(float)(pd.tau - pd.step_dn * unit) : floor(pd.tau - pd.step_dn * unit);
            if (t >= pd.tau) t = weighted ? (double)nextafterf((float)pd.tau, -INFINITY) : pd.tau - 1.0;
            if (pd.tau <= 0.0)
                return fail(ctx, BSH_ESTATE, "fewer than topk = %d of the %llu templates pass a threshold of zero", pd.topk,
                            (unsigned long long)pd.n_templates);
            pd.tau = t > 0.0 ? t : 0.0;
            pd.step_dn *= 2.0;
        } else if (pd.phase == 1) {                                   // this pass ran just above the tie value: too few
            pd.n_above = n_cand;
            start_ties = true;
        } else {                                                      // phase 2: this pass ran with pd.tie_limit
            if (too_few) pd.lim_lo = pd.tie_limit; else pd.lim_hi = pd.tie_limit;
            const double got = (double)n_cand - (double)pd.n_above;   // ties below the limit
            const double need = 1.5 * (double)(want - pd.n_above) + 64.0;
            double guess = got > 0.0 ? (double)pd.tie_limit * need / got : (double)pd.tie_limit * 16.0;
            const double lo = (double)pd.lim_lo, hi = (double)pd.lim_hi;
            if (!(guess > lo + 0.05 * (hi - lo) && guess < hi - 0.05 * (hi - lo))) guess = 0.5 * (lo + hi);
            if (pd.lim_hi - pd.lim_lo <= 1)
                return fail(ctx, BSH_ESTATE, "tie-limit search collapsed at %llu (%u candidates for topk %d)",
                            (unsigned long long)pd.tie_limit, n_cand, pd.topk);
            pd.tie_limit = std::min<uint64_t>(pd.lim_hi - 1, std::max<uint64_t>(pd.lim_lo + 1, (uint64_t)guess));
        }
        pd.fixed = true;
        if (start_ties) {
            pd.phase = 2;
            pd.tau = pd.lo_tau;
            const float tf = (float)pd.lo_tau;
            uint32_t key;
            if (weighted) memcpy(&key, &tf, 4); else key = (uint32_t)(int32_t)pd.lo_tau;
            pd.tie_key = key;
            pd.lim_lo = 0;
            pd.lim_hi = pd.n_templates;
            const double n_tie = (double)pd.lo_n - (double)pd.n_above;            // templates AT the tie value
            const double need = 1.5 * (double)(want - pd.n_above) + 64.0;
            pd.tie_limit = (uint64_t)std::min((double)pd.n_templates - 1.0, std::max(1.0, (double)pd.n_templates * need / std::max(n_tie, 1.0)));
        }
        TRY(run_pass(ctx));
        CK(cudaMemcpyAsync(ctx->pinned_count, ctx->cand_count.p, sizeof(unsigned int), cudaMemcpyDeviceToHost, ctx->stream));
        CK(cudaMemcpyAsync(ctx->pinned_count + 4, ctx->thr.p, kThresholdHostBytes, cudaMemcpyDeviceToHost, ctx->stream));
    }
    ctx->st.n_candidates = n_cand;
    ctx->st.threshold = weighted ? (double)thr.tau_f : (double)thr.tau_i;
    ctx->st.n_passes = pd.passes;

    CK(cudaEventRecord(ctx->ev[4], ctx->stream));
    RawCand *sorted = (RawCand *)ctx->cand.p;
    if (n_cand > kRadixMin) {
        TRY(ensure(ctx, ctx->keys, (size_t)pd.cand_cap * sizeof(RawCand)));
        TRY(radix_sort_candidates(ctx, (RawCand *)ctx->cand.p, (RawCand *)ctx->keys.p, n_cand, &sorted));
    } else if (n_cand > (unsigned)kSortTile && (uint64_t)n_cand > want) {
        // only the candidates at or above the k-th largest key take part in the sort (ties at the cut included)
        TRY(ensure(ctx, ctx->keys, (size_t)pd.cand_cap * sizeof(RawCand)));
        select_cut_kernel<<<1, 1024, 0, ctx->stream>>>((const RawCand *)ctx->cand.p, n_cand, (unsigned int)want,
                                                       (RawCand *)ctx->keys.p, (unsigned int *)ctx->cand_count.p + 1);
        count_launch(ctx);
        CK(cudaMemcpyAsync(ctx->pinned_count + 1, (unsigned int *)ctx->cand_count.p + 1, sizeof(unsigned int),
                           cudaMemcpyDeviceToHost, ctx->stream));
        CK(cudaStreamSynchronize(ctx->stream));
        const unsigned int n_sel = ctx->pinned_count[1];
        if (n_sel < want || n_sel > n_cand) return fail(ctx, BSH_ECUDA, "toplist pre-selection kept %u of %u", n_sel, n_cand);
        sorted = (RawCand *)ctx->keys.p;
        TRY(sort_candidates(ctx, sorted, n_sel));
    } else {
        TRY(sort_candidates(ctx, sorted, n_cand));
    }
    const int n_keep = (int)want;
    finalize_top_kernel<<<(pd.topk + 255) / 256, 256, 0, ctx->stream>>>(sorted, n_keep, pd.topk, weighted ? 1 : 0, d_top);
    count_launch(ctx);
    {
        const TableCache &c = ctx->cache[pd.cache_slot];
        bsh_sfts s = {};
        s.n_sft = pd.n_sft; s.k_slab0 = pd.k_slab0; s.n_bins = pd.n_bins;
        bsh_grid g = {};
        g.n_pix = pd.n_pix; g.n_ap = pd.n_ap; g.n_P = pd.n_P; g.n_tasc = pd.n_tasc; g.n_f0 = pd.n_f0; g.k_band0 = pd.k_band0;
        TrackTables t = make_track_tables(c, &s, &g, (const double *)ctx->dtab.p, pd.R);
        if ((unsigned)n_keep > kRadixMin) {
            TRY(ensure_cs_t(ctx, ctx->cache[pd.cache_slot]));
            t.cs_t = (const double2 *)c.d_cs_t.p;
            if (t.ke)
                rescore_rows_kernel<true><<<(n_keep + 255) / 256, 256, 0, ctx->stream>>>(t, pd.d_peak, pd.words_per_row, pd.d_w,
                                                                                         weighted ? 1 : 0, d_top, n_keep);
            else
                rescore_rows_kernel<false><<<(n_keep + 255) / 256, 256, 0, ctx->stream>>>(t, pd.d_peak, pd.words_per_row, pd.d_w,
                                                                                          weighted ? 1 : 0, d_top, n_keep);
        } else
            rescore_kernel<<<n_keep, kCandThreads, 0, ctx->stream>>>(t, pd.d_peak, pd.words_per_row, pd.d_w,
                                                                              weighted ? 1 : 0, d_top, n_keep);
        count_launch(ctx);
    }
    CK(cudaGetLastError());
    CK(cudaEventRecord(ctx->ev[5], ctx->stream));
    ctx->have_select = true;
    *h_n_top = n_keep;
    pd.active = false;
    return BSH_OK;
}

int bsh_stage1_hough(bsh_ctx *ctx, const uint32_t *d_peak, int32_t words_per_row, const bsh_sfts *sfts,
                     const bsh_grid *grid, int32_t mode, int32_t topk, bsh_cand *d_top, int32_t *h_n_top,
                     void *d_counts_full)
{
    if (!ctx) return BSH_EINVAL;
    if (!d_top || !h_n_top) return fail(ctx, BSH_EINVAL, "null d_top / h_n_top");
    TRY(bsh_stage1_launch(ctx, d_peak, words_per_row, sfts, grid, mode, topk, d_counts_full));
    TRY(bsh_stage1_collect(ctx, d_top, h_n_top));
    CK(cudaStreamSynchronize(ctx->stream));
    return BSH_OK;
}

int bsh_stage2_power(bsh_ctx *ctx, const float *d_rho, int64_t rho_row_stride, const bsh_sfts *sfts,
                     const bsh_grid *grid, bsh_cand *d_cands, int32_t n_cands, int32_t sort_by_power)
{
    if (!ctx) return BSH_EINVAL;
    TRY(validate(ctx, sfts, grid));
    if (!d_rho || !d_cands || n_cands < 0 || rho_row_stride < sfts->n_bins)
        return fail(ctx, BSH_EINVAL, "bsh_stage2_power: bad arguments");
    if (n_cands == 0) return BSH_OK;
    const DeviceGuard device_guard(ctx->device);
    int slot = 0;
    TRY(get_tables(ctx, sfts, grid, &slot));
    const TableCache &c = ctx->cache[slot];
    CK(cudaEventRecord(ctx->ev[6], ctx->stream));
    const bool rows = (unsigned)n_cands > kRadixMin;       // large lists: D laid out [SFT][pixel], (cos, sin) transposed
    const int R2 = rows ? grid->n_pix : 1;
    TRY(build_dtable(ctx, grid, c, R2, ctx->nvec2, ctx->dtab2));
    const bsh_grid kg = kernel_grid(grid);
    TrackTables t = make_track_tables(c, sfts, &kg, (const double *)ctx->dtab2.p, R2);
    if (rows) {
        TRY(ensure_cs_t(ctx, ctx->cache[slot]));
        t.cs_t = (const double2 *)c.d_cs_t.p;
    }
    if (rows && t.ke)
        stage2_rows_kernel<true><<<(n_cands + 255) / 256, 256, 0, ctx->stream>>>(t, d_rho, rho_row_stride, sfts->d_w, d_cands, n_cands);
    else if (rows)
        stage2_rows_kernel<false><<<(n_cands + 255) / 256, 256, 0, ctx->stream>>>(t, d_rho, rho_row_stride, sfts->d_w, d_cands, n_cands);
    else
        stage2_kernel<<<(unsigned)n_cands, kCandThreads, 0, ctx->stream>>>(t, d_rho, rho_row_stride, sfts->d_w, d_cands, n_cands);
    count_launch(ctx);
    CK(cudaGetLastError());
    if (sort_by_power && n_cands > 1) {
        unsigned int n2 = 1;
        while (n2 < (unsigned)n_cands) n2 <<= 1;
        const bool large = (unsigned)n_cands > kRadixMin;
        TRY(ensure(ctx, ctx->keys, (size_t)n2 * sizeof(RawCand) * (large ? 2 : 1)));
        TRY(ensure(ctx, ctx->tmp_cands, (size_t)n_cands * sizeof(bsh_cand)));
        pack_power_keys_kernel<<<(n_cands + 255) / 256, 256, 0, ctx->stream>>>(d_cands, n_cands, (RawCand *)ctx->keys.p);
        count_launch(ctx);
        RawCand *order = (RawCand *)ctx->keys.p;
        if (large) TRY(radix_sort_candidates(ctx, (RawCand *)ctx->keys.p, (RawCand *)ctx->keys.p + n2, (unsigned)n_cands, &order));
        else TRY(sort_candidates(ctx, (RawCand *)ctx->keys.p, (unsigned)n_cands));
        CK(cudaMemcpyAsync(ctx->tmp_cands.p, d_cands, (size_t)n_cands * sizeof(bsh_cand), cudaMemcpyDeviceToDevice,
                           ctx->stream));
        permute_cands_kernel<<<(n_cands + 255) / 256, 256, 0, ctx->stream>>>((const bsh_cand *)ctx->tmp_cands.p,
                                                                            (const RawCand *)order, n_cands, d_cands);
        count_launch(ctx);
        CK(cudaGetLastError());
    }
    CK(cudaEventRecord(ctx->ev[7], ctx->stream));
    ctx->have_s2 = true;
    return BSH_OK;
}

int bsh_search_patch_host(bsh_ctx *ctx, const float *h_rho, const float *h_w, float rho_th, const bsh_sfts *sfts,
                          const bsh_grid *grid, int32_t mode, int32_t topk, bsh_cand *h_top, int32_t *h_n_top)
{
    if (!ctx) return BSH_EINVAL;
    TRY(validate(ctx, sfts, grid));
    if (!h_rho || !h_top || !h_n_top || topk < 1) return fail(ctx, BSH_EINVAL, "bsh_search_patch_host: bad arguments");
    if (topk > kMaxTopk) return fail(ctx, BSH_EINVAL, "bsh_search_patch_host: topk = %d is beyond the documented maximum of 2^27", topk);
    if ((mode & BSH_WEIGHTED) && !h_w) return fail(ctx, BSH_EINVAL, "BSH_WEIGHTED needs h_w");
    const DeviceGuard device_guard(ctx->device);
    const int N = sfts->n_sft, K = sfts->n_bins, W = (K + 31) / 32;
    TRY(ensure(ctx, ctx->h_rho, sizeof(float) * (size_t)N * K));
    TRY(ensure(ctx, ctx->h_w, sizeof(float) * (size_t)N));
    TRY(ensure(ctx, ctx->h_peak, sizeof(uint32_t) * (size_t)N * W));
    TRY(ensure(ctx, ctx->h_top, sizeof(bsh_cand) * (size_t)topk));
    CK(cudaMemcpyAsync(ctx->h_rho.p, h_rho, sizeof(float) * (size_t)N * K, cudaMemcpyHostToDevice, ctx->stream));
    if (h_w) CK(cudaMemcpyAsync(ctx->h_w.p, h_w, sizeof(float) * (size_t)N, cudaMemcpyHostToDevice, ctx->stream));
    bsh_sfts s = *sfts;
    s.d_w = h_w ? (const float *)ctx->h_w.p : nullptr;
    TRY(bsh_build_peakgram(ctx, (const float *)ctx->h_rho.p, N, K, K, rho_th, (uint32_t *)ctx->h_peak.p, W));
    TRY(bsh_stage1_launch(ctx, (const uint32_t *)ctx->h_peak.p, W, &s, grid, mode, topk, nullptr));
    TRY(bsh_stage1_collect(ctx, (bsh_cand *)ctx->h_top.p, h_n_top));
    TRY(bsh_stage2_power(ctx, (const float *)ctx->h_rho.p, K, &s, grid, (bsh_cand *)ctx->h_top.p, *h_n_top, 1));
    CK(cudaMemcpyAsync(h_top, ctx->h_top.p, sizeof(bsh_cand) * (size_t)topk, cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    return BSH_OK;
}

static int check_candset(bsh_ctx *ctx, const bsh_candset *c, const char *what)
{
    if (!c || c->n < 0 || c->n > 32768 || (c->n > 0 && (!c->d_param || !c->d_res || !c->d_sig)))
        return fail(ctx, BSH_EINVAL, "%s: bad candidate set", what);
    return BSH_OK;
}

int bsh_post_coincidences(bsh_ctx *ctx, const bsh_candset *a, const bsh_candset *b, double window, int64_t max_pairs,
                          int32_t *d_pair_a, int32_t *d_pair_b, double *d_centroid, double *d_pair_sig, int64_t *h_n_pairs)
{
    if (!ctx) return BSH_EINVAL;
    TRY(check_candset(ctx, a, "bsh_post_coincidences"));
    TRY(check_candset(ctx, b, "bsh_post_coincidences"));
    if (!h_n_pairs || max_pairs < 0 || !(window > 0.0) || (max_pairs > 0 && (!d_pair_a || !d_pair_b || !d_centroid || !d_pair_sig)))
        return fail(ctx, BSH_EINVAL, "bsh_post_coincidences: bad arguments");
    *h_n_pairs = 0;
    if (a->n == 0 || b->n == 0) return BSH_OK;
    const DeviceGuard device_guard(ctx->device);
    const int words = (b->n + 31) / 32;
    TRY(ensure(ctx, ctx->post_adj, (size_t)a->n * words * 4));
    TRY(ensure(ctx, ctx->post_cnt, (size_t)a->n * 4));
    TRY(ensure(ctx, ctx->post_off, (size_t)(a->n + 1) * 8));
    CK(cudaMemsetAsync(ctx->post_cnt.p, 0, (size_t)a->n * 4, ctx->stream));
    const int64_t warps = (int64_t)a->n * words;
    post_adjacency_kernel<<<(unsigned)((warps + 7) / 8), 256, 0, ctx->stream>>>(
        a->n, a->d_param, a->d_res, b->n, b->d_param, b->d_res, window * window, 0, words, (uint32_t *)ctx->post_adj.p,
        (int32_t *)ctx->post_cnt.p);
    post_scan_kernel<<<1, 1024, 0, ctx->stream>>>(a->n, (const int32_t *)ctx->post_cnt.p, (int64_t *)ctx->post_off.p);
    post_pairs_kernel<<<(a->n + 255) / 256, 256, 0, ctx->stream>>>(
        a->n, words, (const uint32_t *)ctx->post_adj.p, (const int64_t *)ctx->post_off.p, a->d_param, a->d_sig, b->d_param,
        b->d_sig, max_pairs, d_pair_a, d_pair_b, d_centroid, d_pair_sig);
    count_launch(ctx, 3);
    CK(cudaGetLastError());
    CK(cudaMemcpyAsync(h_n_pairs, (const int64_t *)ctx->post_off.p + a->n, 8, cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    return BSH_OK;
}

int bsh_post_cluster(bsh_ctx *ctx, const bsh_candset *c, double window, double prune_window, int32_t *d_label,
                     int32_t *d_root, double *d_centroid, double *d_cluster_sig, int32_t *d_n_members,
                     int32_t *h_n_clusters, int32_t *h_best)
{
    if (!ctx) return BSH_EINVAL;
    TRY(check_candset(ctx, c, "bsh_post_cluster"));
    if (!h_n_clusters || !h_best || !(window > 0.0)) return fail(ctx, BSH_EINVAL, "bsh_post_cluster: bad arguments");
    *h_n_clusters = 0;
    *h_best = -1;
    const int n = c->n;
    if (n == 0) return BSH_OK;
    if (!d_label || !d_root || !d_centroid || !d_cluster_sig || !d_n_members) return fail(ctx, BSH_EINVAL, "bsh_post_cluster: null output");
    const DeviceGuard device_guard(ctx->device);
    const int words = (n + 31) / 32;
    TRY(ensure(ctx, ctx->post_adj, (size_t)n * words * 4));
    // scratch: [flag + (n_clusters, best)] | top [n] | members_by_label [n] | sig_by_label [n] | cen_by_label [6 n]
    TRY(ensure(ctx, ctx->post_tmp, 64 + (size_t)n * (4 + 4 + 8 + 8 * kNPar)));
    int *d_flag = (int *)ctx->post_tmp.p;
    int32_t *d_top = (int32_t *)((char *)ctx->post_tmp.p + 64);
    int32_t *d_mem = d_top + n;
    double *d_sigl = (double *)((char *)ctx->post_tmp.p + 64 + (size_t)n * 8);
    double *d_cenl = d_sigl + n;
    const int64_t warps = (int64_t)n * words;
    post_adjacency_kernel<<<(unsigned)((warps + 7) / 8), 256, 0, ctx->stream>>>(
        n, c->d_param, c->d_res, n, c->d_param, c->d_res, window * window, 1, words, (uint32_t *)ctx->post_adj.p, nullptr);
    post_iota_kernel<<<(n + 255) / 256, 256, 0, ctx->stream>>>(n, d_label);
    count_launch(ctx, 2);
    for (int iter = 0; iter < n + 2; ++iter) {               // min-label propagation: at most (diameter + 1) sweeps
        CK(cudaMemsetAsync(d_flag, 0, 4, ctx->stream));
        post_propagate_kernel<<<(n + 255) / 256, 256, 0, ctx->stream>>>(n, words, (const uint32_t *)ctx->post_adj.p, d_label,
                                                                       d_flag);
        count_launch(ctx);
        CK(cudaMemcpyAsync(ctx->pinned_count + 8, d_flag, 4, cudaMemcpyDeviceToHost, ctx->stream));
        CK(cudaStreamSynchronize(ctx->stream));
        if (ctx->pinned_count[8] == 0) break;
    }
    if (prune_window > 0.0) {
        post_top_kernel<<<(n + 255) / 256, 256, 0, ctx->stream>>>(n, d_label, c->d_sig, d_top);
        post_prune_kernel<<<(n + 255) / 256, 256, 0, ctx->stream>>>(n, c->d_param, c->d_res, d_top,
                                                                   prune_window * prune_window, d_label);
        count_launch(ctx, 2);
    }
    post_centroid_kernel<<<(n + 127) / 128, 128, 0, ctx->stream>>>(n, c->d_param, c->d_sig, d_label, d_cenl, d_sigl, d_mem);
    post_compact_kernel<<<1, 1024, 0, ctx->stream>>>(n, d_cenl, d_sigl, d_mem, d_root, d_centroid, d_cluster_sig, d_n_members,
                                                     (int32_t *)d_flag + 2);
    count_launch(ctx, 2);
    CK(cudaGetLastError());
    CK(cudaMemcpyAsync(ctx->pinned_count + 8, (int32_t *)d_flag + 2, 8, cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    *h_n_clusters = (int32_t)ctx->pinned_count[8];
    *h_best = (int32_t)ctx->pinned_count[9];
    return BSH_OK;
}

uint64_t bsh_template_index_ecc(const bsh_grid *g, int32_t pix, int32_t ia, int32_t ip, int32_t it, int32_t ie, int32_t j)
{
    const uint64_t ne = g->n_ecc > 0 ? (uint64_t)g->n_ecc : 1u;
    return (((((uint64_t)pix * g->n_ap + ia) * g->n_P + ip) * g->n_tasc + it) * ne + ie) * (uint64_t)g->n_f0 + j;
}

uint64_t bsh_template_index(const bsh_grid *g, int32_t pix, int32_t ia, int32_t ip, int32_t it, int32_t j)
{
    return bsh_template_index_ecc(g, pix, ia, ip, it, 0, j);
}

void bsh_template_decode_ecc(const bsh_grid *g, uint64_t idx, int32_t *pix, int32_t *ia, int32_t *ip, int32_t *it, int32_t *ie,
                             int32_t *j)
{
    const uint64_t ne = g->n_ecc > 0 ? (uint64_t)g->n_ecc : 1u;
    const int32_t jj = (int32_t)(idx % (uint64_t)g->n_f0);   idx /= (uint64_t)g->n_f0;
    const int32_t ee = (int32_t)(idx % ne);                  idx /= ne;
    if (ie) *ie = ee;
    bsh_grid k = *g;
    k.n_ecc = 0;
    k.n_f0 = 1;
    bsh_template_decode(&k, idx, pix, ia, ip, it, nullptr);
    if (j) *j = jj;
}

void bsh_template_decode(const bsh_grid *g, uint64_t idx, int32_t *pix, int32_t *ia, int32_t *ip, int32_t *it, int32_t *j)
{
    if (g->n_ecc > 0) { bsh_template_decode_ecc(g, idx, pix, ia, ip, it, nullptr, j); return; }
    const int32_t jj = (int32_t)(idx % (uint64_t)g->n_f0);   idx /= (uint64_t)g->n_f0;
    const int32_t tt = (int32_t)(idx % (uint64_t)g->n_tasc); idx /= (uint64_t)g->n_tasc;
    const int32_t pp = (int32_t)(idx % (uint64_t)g->n_P);    idx /= (uint64_t)g->n_P;
    const int32_t aa = (int32_t)(idx % (uint64_t)g->n_ap);   idx /= (uint64_t)g->n_ap;
    if (pix) *pix = (int32_t)idx;
    if (ia) *ia = aa;
    if (ip) *ip = pp;
    if (it) *it = tt;
    if (j) *j = jj;
}

}  // extern "C"

// =====================================================================================================================
// bsh_post_coincidences_static: step 1 of the post-processing with its work area in the library image (include/bsh.h says
// for whom and why).  Nothing below allocates: no cudaMalloc / cudaFree / cudaMallocHost, no std::string or std::vector.
// =====================================================================================================================
namespace {

constexpr int kStaticMaxCands = BSH_STATIC_MAX_CANDS;
constexpr int kStaticMaxDevices = 64;
// layout of the work area (every part on a 256-byte boundary):  prefix sums [n_a + 1] int64 | row counts [n_a] int32 |
// bit matrix [n_a][ceil(n_b / 32)] uint32
constexpr size_t kStaticOffBytes = ((size_t)(kStaticMaxCands + 1) * 8 + 255) / 256 * 256;
constexpr size_t kStaticCntBytes = (size_t)kStaticMaxCands * 4;
constexpr size_t kStaticAdjBytes = (size_t)kStaticMaxCands * (kStaticMaxCands / 32) * 4;
static_assert(kStaticOffBytes + kStaticCntBytes + kStaticAdjBytes == (size_t)BSH_STATIC_SCRATCH_BYTES, "bsh.h states the size");
static_assert(kStaticCntBytes % 256 == 0 && kStaticMaxCands % 32 == 0, "alignment of the parts");

// One copy per GPU that loads this library, for the life of the process.  In HOST code the name `g_static_scratch` is only
// a handle for the runtime's symbol calls, not a device address: the kernels are given the pointer cudaGetSymbolAddress
// returns for the current device (static_scratch_of below), never the name.
static __device__ __align__(256) unsigned char g_static_scratch[BSH_STATIC_SCRATCH_BYTES];

std::mutex g_static_mutex;
unsigned char *g_static_ptr[kStaticMaxDevices] = {};      // device address of g_static_scratch on each GPU, once looked up

int static_fail(char *h_err, int32_t err_len, int code, const char *fmt, ...)
{
    if (h_err && err_len > 0) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(h_err, (size_t)err_len, fmt, ap);
        va_end(ap);
    }
    return code;
}

// `device` must be the current device.  The first call per device does the look-up; the answer never changes afterwards.
int static_scratch_of(int device, unsigned char **out, char *h_err, int32_t err_len)
{
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_ptr[device]) {
        void *p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_static_scratch);
        if (e != cudaSuccess || !p)
            return static_fail(h_err, err_len, BSH_ECUDA, "bsh_post_coincidences_static: cudaGetSymbolAddress on device %d failed: %s",
                               device, cudaGetErrorString(e));
        g_static_ptr[device] = (unsigned char *)p;
    }
    *out = g_static_ptr[device];
    return BSH_OK;
}

#define CKS(call)                                                                                                  \
    do {                                                                                                           \
        cudaError_t e_ = (call);                                                                                   \
        if (e_ != cudaSuccess)                                                                                     \
            return static_fail(h_err, err_len, BSH_ECUDA, "bsh_post_coincidences_static: %s failed: %s", #call,   \
                               cudaGetErrorString(e_));                                                            \
    } while (0)

bool static_candset_ok(const bsh_candset *c) { return c && c->n >= 0 && (c->n == 0 || (c->d_param && c->d_res && c->d_sig)); }

}  // namespace

extern "C" int bsh_post_coincidences_static(int device, void *cuda_stream, const bsh_candset *a, const bsh_candset *b,
                                            double window, int64_t max_pairs, int32_t *d_pair_a, int32_t *d_pair_b,
                                            double *d_centroid, double *d_pair_sig, int64_t *h_n_pairs, char *h_err,
                                            int32_t err_len)
{
    if (h_err && err_len > 0) h_err[0] = 0;
    if (!static_candset_ok(a) || !static_candset_ok(b))
        return static_fail(h_err, err_len, BSH_EINVAL, "bsh_post_coincidences_static: bad candidate set");
    if (!h_n_pairs || max_pairs < 0 || !(window > 0.0) || (max_pairs > 0 && (!d_pair_a || !d_pair_b || !d_centroid || !d_pair_sig)))
        return static_fail(h_err, err_len, BSH_EINVAL, "bsh_post_coincidences_static: bad arguments");
    *h_n_pairs = 0;
    if (a->n > kStaticMaxCands || b->n > kStaticMaxCands)
        return static_fail(h_err, err_len, BSH_ELIMIT,
                           "bsh_post_coincidences_static: lists of %d and %d candidates, the fixed work area holds at most %d "
                           "per list (BSH_STATIC_MAX_CANDS); use bsh_post_coincidences for longer lists",
                           a->n, b->n, kStaticMaxCands);
    int n_dev = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess || n_dev < 1 || device < 0 || device >= n_dev || device >= kStaticMaxDevices)
        return static_fail(h_err, err_len, BSH_ECUDA, "bsh_post_coincidences_static: no CUDA device %d", device);
    if (a->n == 0 || b->n == 0) return BSH_OK;
    const DeviceGuard device_guard(device);
    unsigned char *scratch = nullptr;
    TRY(static_scratch_of(device, &scratch, h_err, err_len));
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    int64_t *d_off = (int64_t *)scratch;
    int32_t *d_cnt = (int32_t *)(scratch + kStaticOffBytes);
    uint32_t *d_adj = (uint32_t *)(scratch + kStaticOffBytes + kStaticCntBytes);
    const int words = (b->n + 31) / 32;
    // the work area still holds the previous call's contents: the row counts are accumulated with atomicAdd and must start
    // at zero; d_adj [n_a][words] and d_off [n_a + 1] are written in full by the kernels below before they are read
    CKS(cudaMemsetAsync(d_cnt, 0, (size_t)a->n * 4, stream));
    const int64_t warps = (int64_t)a->n * words;
    post_adjacency_kernel<<<(unsigned)((warps + 7) / 8), 256, 0, stream>>>(a->n, a->d_param, a->d_res, b->n, b->d_param, b->d_res,
                                                                          window * window, 0, words, d_adj, d_cnt);
    post_scan_kernel<<<1, 1024, 0, stream>>>(a->n, d_cnt, d_off);
    post_pairs_kernel<<<(a->n + 255) / 256, 256, 0, stream>>>(a->n, words, d_adj, d_off, a->d_param, a->d_sig, b->d_param, b->d_sig,
                                                             max_pairs, d_pair_a, d_pair_b, d_centroid, d_pair_sig);
    CKS(cudaGetLastError());
    CKS(cudaMemcpyAsync(h_n_pairs, d_off + a->n, 8, cudaMemcpyDeviceToHost, stream));
    CKS(cudaStreamSynchronize(stream));
    return BSH_OK;
}
