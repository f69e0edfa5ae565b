"""Parity of the CUDA path (through the C ABI) against the CPU oracle.  All tests here need a B200: -m gpu.

Bars (BASELINE.json north_star): tracks, unweighted counts and unweighted toplists bit-exact against the oracle's
CANONICAL mode; weighted counts and the stage-2 power within 1e-5 relative (FP32 accumulate vs FP64 oracle); weighted /
power toplists identical except for ties within that tolerance at the cut.
"""
import dataclasses
import math

import numpy as np
import pytest

import oracle
import synth

pytestmark = pytest.mark.gpu

RTOL = 1e-5


@pytest.fixture(scope="module")
def bsh():
    import paper_1904_04873_b200 as b
    return b


@pytest.fixture(scope="module")
def torch():
    import torch
    return torch


@pytest.fixture()
def ctx(bsh):
    c = bsh.Context(0)
    yield c
    c.close()


def dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def gpu_stage1(bsh, torch, ctx, wl, mode, topk=None, full=True, rho=None):
    rho = wl.rho if rho is None else rho
    d_rho = dev(torch, rho)
    d_w = dev(torch, wl.w)
    d_peak = ctx.build_peakgram(d_rho, 1.6)
    weighted = bool(mode & bsh.BSH_WEIGHTED)
    counts = None
    if full:
        counts = torch.full((wl.n_templates,), -7, dtype=torch.float32 if weighted else torch.int32, device="cuda")
    d_top, n_top = ctx.stage1_hough(d_peak, wl, mode=mode, topk=topk, d_w=d_w, counts_full=counts)
    return dict(d_rho=d_rho, d_w=d_w, d_peak=d_peak, counts=None if counts is None else counts.cpu().numpy(),
                top=ctx.records(d_top, n_top), d_top=d_top, n_top=n_top)


def check_unweighted_toplist(top, counts_all, k):
    """identical toplist: (count desc, index asc) of ALL counts, by a numpy lexsort"""
    want = np.lexsort((np.arange(counts_all.size), -counts_all.astype(np.int64)))[:k]
    assert np.array_equal(top["index"], want.astype(np.uint64))
    assert np.array_equal(top["count"], counts_all[want])


def check_float_toplist(idx_got, values_ref, k, rtol=RTOL):
    """same set as the reference top-k except for entries within rtol of the k-th value"""
    order = np.lexsort((np.arange(values_ref.size), -values_ref))
    want = set(order[:k].tolist())
    got = set(int(i) for i in idx_got)
    assert len(got) == min(k, values_ref.size)
    cut = values_ref[order[min(k, values_ref.size) - 1]]
    for i in want ^ got:
        assert abs(values_ref[i] - cut) <= rtol * abs(cut), (i, values_ref[i], cut)


def check_toplist_complete(torch, d_counts, top, k, weighted):
    """No better template was dropped: against the FULL dump of the ranking statistic (on the device, O(n), library ops
    only): every template above the cut value is in the toplist, and the entries AT the cut are the lowest indices
    (unweighted: exactly; weighted: inside the 1e-5 band of the k-th value)."""
    vals = top["wcount"] if weighted else top["count"]
    assert len(set(int(i) for i in top["index"][:k])) == k, "a template appears twice in the toplist"
    cut = vals[k - 1]
    d_cut = torch.tensor(cut, dtype=d_counts.dtype, device=d_counts.device)
    if weighted:
        lo, hi = cut * (1 - RTOL), cut * (1 + RTOL)
        above = torch.nonzero(d_counts > hi).flatten().cpu().numpy()
        assert set(above.tolist()) <= set(int(i) for i in top["index"])
        n_ge = int((d_counts >= lo).sum())
        assert n_ge >= k
        got = d_counts[torch.from_numpy(top["index"].astype(np.int64)).to(d_counts.device)].cpu().numpy()
        assert np.array_equal(got, vals) and np.all(got >= lo)
    else:
        above = torch.nonzero(d_counts > d_cut).flatten().cpu().numpy()
        n_above = above.size
        assert n_above < k and n_above == int((vals > cut).sum())
        assert np.array_equal(np.sort(top["index"][:n_above].astype(np.int64)), above)
        at = torch.nonzero(d_counts == d_cut).flatten()[:k - n_above].cpu().numpy()
        assert np.array_equal(top["index"][n_above:k].astype(np.int64), at)


# ------------------------------------------------------------------------------------------------------------
# peakgram
# ------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n,k", [(1, 1), (3, 31), (5, 32), (7, 33), (64, 63), (50, 172), (9, 257), (2000, 172), (8000, 252)])
def test_peakgram_bit_exact(bsh, torch, ctx, n, k):
    rng = np.random.default_rng(n * 1000 + k)
    rho = rng.standard_exponential((n, k)).astype(np.float32)
    rho[0, 0] = np.float32(1.6)
    if k > 2:
        rho[0, 1] = np.nextafter(np.float32(1.6), np.float32(2))
        rho[0, 2] = np.nan
    want = oracle.peakgram(rho)
    got = ctx.build_peakgram(dev(torch, rho), 1.6).cpu().numpy().view(np.uint32)
    assert np.array_equal(got, want)
    # strided input (row stride > K) and a wider output buffer
    wide = np.zeros((n, k + 5), np.float32)
    wide[:, :k] = rho
    d_wide = dev(torch, wide)
    out = torch.full((n, want.shape[1] + 2), -1, dtype=torch.int32, device="cuda")
    got2 = ctx.build_peakgram(d_wide[:, :k], 1.6, out=out).cpu().numpy().view(np.uint32)
    assert np.array_equal(got2[:, :want.shape[1]], want) and not got2[:, want.shape[1]:].any()


def test_empty_and_bad_arguments_are_rejected(bsh, torch, ctx):
    wl = synth.config1()
    d_rho = dev(torch, wl.rho)
    d_peak = ctx.build_peakgram(d_rho)
    small = torch.empty((wl.n_sft, 1), dtype=torch.int32, device="cuda")
    with pytest.raises(bsh.BshError):
        ctx.build_peakgram(d_rho, out=small)                         # words_per_row * 32 < n_bins
    with pytest.raises(bsh.BshError):
        ctx.stage1_hough(d_peak, wl, mode=bsh.BSH_WEIGHTED, d_w=None)  # weighted without weights
    with pytest.raises(bsh.BshError):
        ctx.stage1_hough(d_peak, wl, topk=0)
    bad = dataclasses.replace(wl, k_band0=wl.k_slab0 - 1)
    with pytest.raises(bsh.BshError):
        ctx.stage1_hough(d_peak, bad)
    far = dataclasses.replace(wl, k_band0=(1 << 32) - wl.n_f0, k_slab0=(1 << 32) - wl.n_f0 - 9)
    with pytest.raises(bsh.BshError, match="2\\^32"):
        ctx.stage1_hough(d_peak, far)                                  # band beyond the range the break fix-up is proven on (R-7)
    with pytest.raises(bsh.BshError):
        ctx._pending = (None, 4)                                       # collect without a pending launch
        ctx.stage1_collect()
    # topk beyond the documented 2^27 is refused before anything is sized from it, even on a grid this small (the
    # output pointers are never touched, so small dummies do)
    import ctypes as C
    pb = bsh.binding._Problem(wl, None)
    dummy = torch.zeros(64, dtype=torch.uint8, device="cuda")
    n_top = C.c_int32(-5)
    for topk in ((1 << 27) + 1, 2**31 - 1):
        rc = ctx.lib.bsh_stage1_hough(ctx._ctx, C.c_void_p(d_peak.data_ptr()), C.c_int32(d_peak.shape[1]), C.byref(pb.sfts),
                                      C.byref(pb.grid), C.c_int32(0), C.c_int32(topk), C.c_void_p(dummy.data_ptr()),
                                      C.byref(n_top), None)
        assert rc == -1 and b"2^27" in ctx.lib.bsh_last_error(ctx._ctx)
        rho = np.ascontiguousarray(wl.rho, np.float32)
        host_top = np.zeros(4, bsh.CAND_DTYPE)
        rc = ctx.lib.bsh_search_patch_host(ctx._ctx, C.c_void_p(rho.ctypes.data), None, C.c_float(1.6), C.byref(pb.sfts),
                                           C.byref(pb.grid), C.c_int32(0), C.c_int32(topk), C.c_void_p(host_top.ctypes.data),
                                           C.byref(n_top))
        assert rc == -1 and b"2^27" in ctx.lib.bsh_last_error(ctx._ctx) and not host_top["index"].any()
    got, n = ctx.stage1_hough(d_peak, wl, topk=1 << 20)                  # far more than the 1620 templates: still fine
    assert n == 1620


# ------------------------------------------------------------------------------------------------------------
# config 1 (both pixels): everything, element by element
# ------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("pixel", ["ecliptic", "pole"])
@pytest.mark.parametrize("naive", [False, True])
def test_config1_full_parity(bsh, torch, ctx, pixel, naive):
    wl = synth.config1(pixel=pixel)
    pk = oracle.peakgram(wl.rho)
    want_n, want_w = oracle.stage1(wl, pk, wl.w, mode=oracle.CANONICAL)
    extra = bsh.BSH_NAIVE if naive else 0
    # unweighted
    r = gpu_stage1(bsh, torch, ctx, wl, bsh.BSH_UNWEIGHTED | extra)
    assert np.array_equal(r["d_peak"].cpu().numpy().view(np.uint32), pk)
    assert np.array_equal(r["counts"], want_n)
    assert r["n_top"] == 10
    check_unweighted_toplist(r["top"], want_n, 10)
    assert np.allclose(r["top"]["wcount"], want_w[r["top"]["index"].astype(np.int64)], rtol=RTOL, atol=0)
    # stage 2 on that toplist
    ctx.stage2_power(r["d_rho"], wl, r["d_top"], r["n_top"], d_w=r["d_w"], sort_by_power=True)
    recs = ctx.records(r["d_top"], r["n_top"])
    want_p = oracle.stage2(wl, recs["index"], wl.rho, wl.w, mode=oracle.CANONICAL)
    assert np.allclose(recs["power"], want_p, rtol=RTOL, atol=0)
    assert set(recs["index"].tolist()) == set(r["top"]["index"].tolist())
    order = np.lexsort((recs["index"], -recs["power"]))
    assert np.array_equal(order, np.arange(len(recs)))
    assert (recs["flags"] == 3).all()
    # weighted
    r = gpu_stage1(bsh, torch, ctx, wl, bsh.BSH_WEIGHTED | extra)
    assert np.allclose(r["counts"], want_w, rtol=RTOL, atol=0)
    check_float_toplist(r["top"]["index"], want_w, 10)
    assert np.array_equal(r["top"]["count"], want_n[r["top"]["index"].astype(np.int64)])
    assert np.allclose(r["top"]["wcount"], want_w[r["top"]["index"].astype(np.int64)], rtol=RTOL, atol=0)


def test_topk_larger_than_template_count(bsh, torch, ctx):
    wl = synth.noise_workload(seed=3, n_sft=40, n_f0=5, margin=20, f_band_start=100.0, n_pix_side=1, ap=(10.0,),
                              P_days=(15.0,), n_t=2, topk=64)
    pk = oracle.peakgram(wl.rho)
    want_n, _ = oracle.stage1(wl, pk, None)
    r = gpu_stage1(bsh, torch, ctx, wl, bsh.BSH_UNWEIGHTED, topk=64)
    assert r["n_top"] == wl.n_templates == 10
    check_unweighted_toplist(r["top"], want_n, 64)
    rest = ctx.records(r["d_top"])[10:]
    assert not rest["flags"].any() and not rest["index"].any()


# ------------------------------------------------------------------------------------------------------------
# ragged sizes: several SFT chunks + tail, several f0 tiles + tail, odd pixel counts, both table variants
# ------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n_sft,n_f0,margin,f0,side", [(1, 1, 3, 50.0, 1), (33, 7, 12, 80.0, 1), (64, 90, 30, 120.0, 2),
                                                        (200, 96, 45, 150.0, 3), (130, 97, 45, 150.0, 2),
                                                        (70, 200, 60, 200.0, 1), (2100, 64, 50, 180.0, 1)])
def test_ragged_sizes(bsh, torch, ctx, n_sft, n_f0, margin, f0, side):
    wl = synth.noise_workload(seed=n_sft + n_f0, n_sft=n_sft, n_f0=n_f0, margin=margin, f_band_start=f0, n_pix_side=side,
                              ap=(10.0, 40.0), P_days=(15.0, 31.0), n_t=3, topk=7)
    pk = oracle.peakgram(wl.rho)
    want_n, want_w = oracle.stage1(wl, pk, wl.w, mode=oracle.CANONICAL)
    for family in (bsh.BSH_FAMILY_AUTO, bsh.BSH_FAMILY_TEMPLATE_LANE, bsh.BSH_FAMILY_WINDOW):
        ctx.set_option(bsh.BSH_OPT_KERNEL_FAMILY, family)
        for force_clamp in (False, True):
            ctx.set_option(bsh.BSH_OPT_FORCE_CLAMP, int(force_clamp))
            for ppt in ((1, 2) if family == bsh.BSH_FAMILY_WINDOW else (0,)):
                ctx.set_option(bsh.BSH_OPT_PIXELS_PER_THREAD, ppt)
                r = gpu_stage1(bsh, torch, ctx, wl, bsh.BSH_UNWEIGHTED)
                assert np.array_equal(r["counts"], want_n), (family, force_clamp, ppt)
                check_unweighted_toplist(r["top"], want_n, 7)
            ctx.set_option(bsh.BSH_OPT_PIXELS_PER_THREAD, 0)
            r = gpu_stage1(bsh, torch, ctx, wl, bsh.BSH_WEIGHTED)
            assert np.allclose(r["counts"], want_w, rtol=RTOL, atol=0), (family, force_clamp)
            check_float_toplist(r["top"]["index"], want_w, 7)


def test_multiple_breaks_per_band_fallback(bsh, torch, ctx):
    wl = synth.noise_workload(seed=77, n_sft=96, n_f0=90, margin=40, f_band_start=150.0, n_pix_side=1,
                              ap=(2500.0, 6000.0), P_days=(15.0,), n_t=4)
    pk = oracle.peakgram(wl.rho)
    want_n, _ = oracle.stage1(wl, pk, None, mode=oracle.CANONICAL)
    r = gpu_stage1(bsh, torch, ctx, wl, bsh.BSH_UNWEIGHTED)
    assert np.array_equal(r["counts"], want_n)


# ------------------------------------------------------------------------------------------------------------
# the pixel-lane kernel (bsh_pix.cuh) forced on small and ragged problems: partly filled pixel groups (1, 9, 36 pixels),
# several f0 tiles with a ragged last one, SFT counts off the 32-block, both table geometries, the multi-break fallback
# ------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n_sft,n_f0,margin,f0,side", [(1, 1, 3, 50.0, 1), (33, 7, 12, 80.0, 3), (64, 90, 30, 120.0, 6),
                                                        (130, 97, 45, 150.0, 6), (70, 200, 60, 200.0, 3),
                                                        (2100, 64, 50, 180.0, 6), (8200, 33, 45, 150.0, 3)])
def test_pixel_lane_kernel_ragged(bsh, torch, ctx, n_sft, n_f0, margin, f0, side):
    wl = synth.noise_workload(seed=1000 + n_sft + n_f0, n_sft=n_sft, n_f0=n_f0, margin=margin, f_band_start=f0,
                              n_pix_side=side, ap=(10.0, 40.0), P_days=(15.0, 31.0), n_t=3, topk=7)
    pk = oracle.peakgram(wl.rho)
    want_n, want_w = oracle.stage1(wl, pk, wl.w, mode=oracle.CANONICAL)
    ctx.set_option(bsh.BSH_OPT_KERNEL_FAMILY, bsh.BSH_FAMILY_PIXEL_LANE)
    for force_clamp in (False, True):
        ctx.set_option(bsh.BSH_OPT_FORCE_CLAMP, int(force_clamp))
        r = gpu_stage1(bsh, torch, ctx, wl, bsh.BSH_UNWEIGHTED)
        assert ctx.stats()["kernel_variant"] // 1000 == 2, "the pixel-lane kernel did not run"
        assert np.array_equal(r["counts"], want_n), force_clamp
        check_unweighted_toplist(r["top"], want_n, 7)
        r = gpu_stage1(bsh, torch, ctx, wl, bsh.BSH_WEIGHTED)
        # (a clamped table of a 320-column slab does not fit two shared-memory stages: the template-lane kernel runs)
        wide = force_clamp and n_f0 == 200
        assert ctx.stats()["kernel_variant"] // 1000 == (1 if wide else 3), "the weighted pixel-lane kernel did not run"
        assert np.allclose(r["counts"], want_w, rtol=RTOL, atol=0), force_clamp
        check_float_toplist(r["top"]["index"], want_w, 7)


def test_pixel_lane_kernel_multiple_breaks(bsh, torch, ctx):
    wl = synth.noise_workload(seed=78, n_sft=96, n_f0=90, margin=40, f_band_start=150.0, n_pix_side=2,
                              ap=(2500.0, 6000.0), P_days=(15.0,), n_t=4)
    pk = oracle.peakgram(wl.rho)
    want_n, _ = oracle.stage1(wl, pk, None, mode=oracle.CANONICAL)
    ctx.set_option(bsh.BSH_OPT_KERNEL_FAMILY, bsh.BSH_FAMILY_PIXEL_LANE)
    r = gpu_stage1(bsh, torch, ctx, wl, bsh.BSH_UNWEIGHTED)
    assert ctx.stats()["kernel_variant"] // 1000 == 2
    assert np.array_equal(r["counts"], want_n)
    _, want_w = oracle.stage1(wl, pk, wl.w, mode=oracle.CANONICAL)
    r = gpu_stage1(bsh, torch, ctx, wl, bsh.BSH_WEIGHTED)
    assert ctx.stats()["kernel_variant"] // 1000 == 3
    assert np.allclose(r["counts"], want_w, rtol=RTOL, atol=0)


# ------------------------------------------------------------------------------------------------------------
# config 2: a complete sub-grid element by element, then the full grid in the bench's launch configuration
# ------------------------------------------------------------------------------------------------------------
def test_config2_subgrid_element_by_element(bsh, torch, ctx):
    wl = synth.config2()
    rng = np.random.default_rng(2)
    sub = wl.subgrid(ia=np.sort(rng.choice(20, 3, replace=False)), ip=np.sort(rng.choice(30, 4, replace=False)),
                     it=np.sort(rng.choice(40, 3, replace=False)))
    pk = oracle.peakgram(wl.rho)
    want_n, want_w = oracle.stage1(sub, pk, wl.w, mode=oracle.CANONICAL)        # 64 pix x 36 b x 90 f0 x 2000 SFTs
    r = gpu_stage1(bsh, torch, ctx, sub, bsh.BSH_UNWEIGHTED, topk=1000)
    assert np.array_equal(r["counts"], want_n)
    check_unweighted_toplist(r["top"], want_n, 1000)
    r = gpu_stage1(bsh, torch, ctx, sub, bsh.BSH_WEIGHTED, topk=1000)
    assert np.allclose(r["counts"], want_w, rtol=RTOL, atol=0)
    check_float_toplist(r["top"]["index"], want_w, 1000)


def _sampled_full_size_checks(bsh, torch, ctx, wl, weighted, n_sample=3000):
    """Full grid: (a) toplist entries re-scored one by one by the oracle; (b) a seeded sample of ALL templates re-scored by
    the oracle against the full dump; (c) the toplist is the true top-k of the dump (torch sort, a library routine);
    (d) stage-2 power of the toplist against the oracle."""
    mode = bsh.BSH_WEIGHTED if weighted else bsh.BSH_UNWEIGHTED
    r = gpu_stage1(bsh, torch, ctx, wl, mode, topk=wl.topk)
    st = ctx.stats()
    pk = oracle.peakgram(wl.rho)
    top = r["top"]
    assert r["n_top"] == wl.topk
    assert len(set(int(i) for i in top["index"])) == wl.topk, "a template appears twice in the toplist"
    n_o, w_o, _ = oracle.score(wl, top["index"], peak=pk, w=wl.w)
    assert np.array_equal(top["count"], n_o)
    assert np.allclose(top["wcount"], w_o, rtol=RTOL, atol=0)
    rng = np.random.default_rng(123)
    idx = rng.integers(0, wl.n_templates, n_sample).astype(np.uint64)
    n_s, w_s, _ = oracle.score(wl, idx, peak=pk, w=wl.w)
    got = r["counts"][idx.astype(np.int64)]
    if weighted:
        assert np.allclose(got, w_s, rtol=RTOL, atol=0)
    else:
        assert np.array_equal(got, n_s)
    # (c) toplist == top-k of the dump
    d_counts = torch.from_numpy(r["counts"]).cuda()
    if weighted:
        vals, order = torch.sort(d_counts, descending=True, stable=True)
        cut = float(vals[wl.topk - 1])
        got_set = set(int(i) for i in top["index"])
        want_set = set(order[:wl.topk].cpu().numpy().tolist())
        for i in got_set ^ want_set:
            assert abs(float(r["counts"][i]) - cut) <= RTOL * cut
        assert np.all(np.diff(top["wcount"]) <= 0)
    else:
        vals, order = torch.sort(d_counts, descending=True, stable=True)
        assert np.array_equal(top["index"], order[:wl.topk].cpu().numpy().astype(np.uint64))
        assert np.array_equal(top["count"], vals[:wl.topk].cpu().numpy())
    # (d) stage 2
    ctx.stage2_power(r["d_rho"], wl, r["d_top"], r["n_top"], d_w=r["d_w"], sort_by_power=True)
    recs = ctx.records(r["d_top"], r["n_top"])
    p_o = oracle.stage2(wl, recs["index"], wl.rho, wl.w)
    assert np.allclose(recs["power"], p_o, rtol=RTOL, atol=0)
    assert np.all(np.diff(recs["power"]) <= 0)
    return r, st


def test_config2_full_size_unweighted(bsh, torch, ctx):
    wl = synth.config2()
    r, st = _sampled_full_size_checks(bsh, torch, ctx, wl, weighted=False)
    assert st["n_templates"] == 138_240_000 and st["n_accumulations"] == 276_480_000_000
    # the tiled kernel and the one-thread-per-template diagnostic kernel agree on every one of the 1.38e8 counts
    rn = gpu_stage1(bsh, torch, ctx, wl, bsh.BSH_UNWEIGHTED | bsh.BSH_NAIVE, topk=wl.topk)
    assert np.array_equal(rn["counts"], r["counts"])
    assert np.array_equal(rn["top"]["index"], r["top"]["index"])
    # noise statistics of the full dump: Binomial(2000, e^-1.6) up to the sample's peak fraction
    # The mean count over all templates is a WEIGHTED mean of this realisation's peakgram bits (each (row, column) weighted
    # by how many tracks visit it; a track visits one of >= n_f0 = 90 columns of a row), so it scatters around the closed
    # form N e^-1.6 (L439) with a standard deviation of at most sqrt(N p (1 - p) / n_f0) = 1.9 counts: allow 4 sigma.
    p = math.exp(-1.6)
    assert abs(r["counts"].mean() - wl.n_sft * p) < 4.0 * math.sqrt(wl.n_sft * p * (1 - p) / wl.n_f0)
    assert abs(r["counts"].std() / math.sqrt(wl.n_sft * p * (1 - p)) - 1) < 0.05
    check_toplist_complete(torch, torch.from_numpy(r["counts"]).cuda(), r["top"], wl.topk, weighted=False)


def test_config2_full_grid_against_the_tier2_cpu_reference(bsh, torch, ctx):
    """Every one of the 1.38e8 templates of config 2, both counts, against the tier-2 CPU reference (oracle/bsh_tier2.c),
    which equals the plain oracle bit for bit wherever the plain oracle can run (tests/test_tier2.py): the chain
    plain oracle == tier 2 == GPU of SURVEY.md 8(c)."""
    wl = synth.config2()
    pk = oracle.peakgram(wl.rho)
    n_ref, w_ref = oracle.tier2_stage1(wl, pk, wl.w, want_wcount=True)
    r = gpu_stage1(bsh, torch, ctx, wl, bsh.BSH_UNWEIGHTED, topk=wl.topk)
    assert np.array_equal(r["counts"], n_ref)
    check_unweighted_toplist(r["top"], n_ref, wl.topk)
    rw = gpu_stage1(bsh, torch, ctx, wl, bsh.BSH_WEIGHTED, topk=wl.topk)
    assert np.allclose(rw["counts"], w_ref, rtol=RTOL, atol=0)
    check_float_toplist(rw["top"]["index"], w_ref, wl.topk)


def test_config3_slice_config4_and_config5_patch_against_the_tier2_cpu_reference(bsh, torch, ctx):
    """Full grids of a config-4 patch and a config-5 patch, and a 10 % slice (4 of the 40 a_p values) of the full-size
    config-3 run -- integer counts and the FP32 weighted counts of the headline mode -- against the tier-2 CPU reference."""
    # config 3: the GPU runs the FULL grid in the bench launch configuration; the slice of its dump is compared
    wl = synth.config3()
    pk = oracle.peakgram(wl.rho)
    ia = [0, 13, 26, 39]
    n_ref = oracle.tier2_stage1(wl.subgrid(ia=ia), pk)
    d_rho, d_w = dev(torch, wl.rho), dev(torch, wl.w)
    d_peak = ctx.build_peakgram(d_rho, 1.6)
    d_counts = torch.full((wl.n_templates,), -7, dtype=torch.int32, device="cuda")
    ctx.stage1_hough(d_peak, wl, mode=bsh.BSH_UNWEIGHTED, topk=wl.topk, d_w=d_w, counts_full=d_counts)
    per_ap = len(wl.P) * len(wl.tasc_frac) * wl.n_f0
    got = d_counts.view(wl.n_pix, len(wl.ap), per_ap)[:, ia, :].contiguous().view(-1).cpu().numpy()
    assert np.array_equal(got, n_ref)
    del d_counts, got
    # the headline mode at the headline size: the WEIGHTED FP32 counts of the same full-size run, one a_p value of the
    # grid (4.1e7 templates, every one compared) against the tier-2 reference's FP64 weighted counts (its FP64 weighted
    # path is ~10x slower than its integer one: a 4-value slice would double the run time of the whole GPU suite)
    ia = [26]
    _, w_ref = oracle.tier2_stage1(wl.subgrid(ia=ia), pk, wl.w, want_wcount=True)
    d_wcounts = torch.full((wl.n_templates,), -7.0, dtype=torch.float32, device="cuda")
    ctx.stage1_hough(d_peak, wl, mode=bsh.BSH_WEIGHTED, topk=wl.topk, d_w=d_w, counts_full=d_wcounts)
    assert ctx.stats()["kernel_variant"] // 1000 == 3, "the weighted pixel-lane kernel did not run"
    got_w = d_wcounts.view(wl.n_pix, len(wl.ap), per_ap)[:, ia, :].contiguous().view(-1).cpu().numpy()
    del d_wcounts
    assert got_w.shape == w_ref.shape and np.allclose(got_w, w_ref, rtol=RTOL, atol=0)
    del got_w, w_ref
    # config 4, patch 0 (with its injection), from |x|^2
    c4 = synth.config4()
    inj = c4.injections[0]
    bins = [oracle.track(c4.patch_workload(i.patch, None), i.pix, i.ia, i.ip, i.it, i.j, mode=oracle.DIRECT) for i in c4.injections]
    rho = c4.deposit(bins)
    wl4 = c4.patch_workload(inj.patch, rho)
    r = gpu_stage1(bsh, torch, ctx, wl4, bsh.BSH_UNWEIGHTED, topk=1000)
    assert np.array_equal(r["counts"], oracle.tier2_stage1(wl4, oracle.peakgram(rho)))
    # config 5, one patch at high declination
    c5 = synth.config5()
    wl5 = c5.patch_workload(15)
    r = gpu_stage1(bsh, torch, ctx, wl5, bsh.BSH_UNWEIGHTED, topk=1000, rho=c5.base.rho)
    assert np.array_equal(r["counts"], oracle.tier2_stage1(wl5, oracle.peakgram(c5.base.rho)))


def test_config2_full_size_weighted(bsh, torch, ctx):
    _sampled_full_size_checks(bsh, torch, ctx, synth.config2(), weighted=True)


def test_config3_full_size_weighted(bsh, torch, ctx):
    """BASELINE.json configs[2]: 1.66e9 templates, 8000 SFTs, weighted FP32 counts."""
    wl = synth.config3()
    r, st = _sampled_full_size_checks(bsh, torch, ctx, wl, weighted=True, n_sample=1500)
    assert st["n_templates"] == 1_658_880_000


def test_config3_full_size_unweighted_toplist(bsh, torch, ctx):
    """All 1.66e9 integer counts dumped: the toplist is complete (nothing above the cut is missing, ties at the cut are
    the lowest indices), its entries equal the oracle's re-score, and a seeded sample of the dump equals the oracle."""
    wl = synth.config3()
    d_rho, d_w = dev(torch, wl.rho), dev(torch, wl.w)
    d_peak = ctx.build_peakgram(d_rho, 1.6)
    d_counts = torch.full((wl.n_templates,), -7, dtype=torch.int32, device="cuda")
    d_top, n_top = ctx.stage1_hough(d_peak, wl, mode=bsh.BSH_UNWEIGHTED, topk=wl.topk, d_w=d_w, counts_full=d_counts)
    top = ctx.records(d_top, n_top)
    pk = oracle.peakgram(wl.rho)
    n_o, w_o, _ = oracle.score(wl, top["index"], peak=pk, w=wl.w)
    assert np.array_equal(top["count"], n_o)
    assert np.all(np.diff(top["count"].astype(np.int64)) <= 0)
    ties = np.diff(top["count"].astype(np.int64)) == 0
    assert np.all(np.diff(top["index"].astype(np.int64))[ties] > 0)
    check_toplist_complete(torch, d_counts, top, wl.topk, weighted=False)
    idx = np.random.default_rng(321).integers(0, wl.n_templates, 1500)
    n_s, _, _ = oracle.score(wl, idx.astype(np.uint64), peak=pk, w=None)
    assert np.array_equal(d_counts[torch.from_numpy(idx).cuda()].cpu().numpy(), n_s)


# ------------------------------------------------------------------------------------------------------------
# config 4: injected signals are recovered as the loudest candidate of their patch
# ------------------------------------------------------------------------------------------------------------
def test_config4_signal_recovery(bsh, torch, ctx):
    c4 = synth.config4()
    bins = []
    for inj in c4.injections:
        wl_p = c4.patch_workload(inj.patch, None)
        bins.append(oracle.track(wl_p, inj.pix, inj.ia, inj.ip, inj.it, inj.j, mode=oracle.DIRECT))
    rho = c4.deposit(bins)
    pk = oracle.peakgram(rho)
    rng = np.random.default_rng(44)
    for inj in c4.injections:
        wl = c4.patch_workload(inj.patch, rho)
        r = gpu_stage1(bsh, torch, ctx, wl, bsh.BSH_UNWEIGHTED, topk=1000, full=True)
        want = oracle.encode_index(wl, inj.pix, inj.ia, inj.ip, inj.it, inj.j)
        assert int(r["top"]["index"][0]) == want, inj.patch
        # completeness of the toplist against the full dump, and a sample of the dump against the oracle
        check_toplist_complete(torch, torch.from_numpy(r["counts"]).cuda(), r["top"], 1000, weighted=False)
        idx = rng.integers(0, wl.n_templates, 200)
        n_s, _, _ = oracle.score(wl, idx.astype(np.uint64), peak=pk, w=None)
        assert np.array_equal(r["counts"][idx], n_s)
        n_o, _, _ = oracle.score(wl, r["top"]["index"], peak=pk, w=None)
        assert np.array_equal(r["top"]["count"], n_o)
        p_sig = 0.29568
        assert abs(r["top"]["count"][0] - wl.n_sft * p_sig) < 5 * math.sqrt(wl.n_sft * p_sig * (1 - p_sig))
        ctx.stage2_power(r["d_rho"], wl, r["d_top"], r["n_top"], d_w=None, sort_by_power=True)
        recs = ctx.records(r["d_top"], r["n_top"])
        assert int(recs["index"][0]) == want
        p_o = oracle.stage2(wl, recs["index"][:50], rho, None)
        assert np.allclose(recs["power"][:50], p_o, rtol=RTOL, atol=0)


# ------------------------------------------------------------------------------------------------------------
# config 5: patches streamed on two CUDA streams (two contexts), shared peakgram
# ------------------------------------------------------------------------------------------------------------
def test_config5_two_streams(bsh, torch):
    c5 = synth.config5()
    # 16 of the 256 patches: every declination band of the 16 x 16 tiling (index = i_alpha * 16 + i_delta), varying alpha
    patches = [((5 * d + 3) % 16) * 16 + d for d in range(16)]
    assert len({p % 16 for p in patches}) == 16 and 100 not in patches
    patches[6] = 100
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    ctxs = [bsh.Context(0, stream=s) for s in streams]
    d_rho = dev(torch, c5.base.rho)
    torch.cuda.synchronize()
    with torch.cuda.stream(streams[0]):
        d_peak = ctxs[0].build_peakgram(d_rho)
    torch.cuda.synchronize()
    pk = oracle.peakgram(c5.base.rho)
    assert np.array_equal(d_peak.cpu().numpy().view(np.uint32), pk)
    results, wls, keep = {}, {}, {}
    pending = [None, None]
    for n, ip in enumerate(patches + [None, None]):
        s = n % 2
        if pending[s] is not None:                              # collect the patch launched two steps ago on this stream
            jp = pending[s]
            with torch.cuda.stream(streams[s]):
                d_top, n_top = ctxs[s].stage1_collect()
                ctxs[s].stage2_power(d_rho, wls[jp], d_top, n_top, d_w=keep[jp], sort_by_power=True)
            results[jp] = (d_top, n_top)
            pending[s] = None
        if ip is not None:
            wls[ip] = c5.patch_workload(ip)
            with torch.cuda.stream(streams[s]):
                keep[ip] = dev(torch, wls[ip].w)
                ctxs[s].stage1_launch(d_peak, wls[ip], mode=bsh.BSH_UNWEIGHTED, topk=1000, d_w=keep[ip])
            pending[s] = ip
    torch.cuda.synchronize()
    for ip in patches:
        d_top, n_top = results[ip]
        recs = ctxs[0].records(d_top, n_top)
        assert n_top == 1000
        n_o, w_o, p_o = oracle.score(wls[ip], recs["index"], peak=pk, rho=c5.base.rho, w=wls[ip].w)
        assert np.array_equal(recs["count"], n_o)
        assert np.allclose(recs["wcount"], w_o, rtol=RTOL, atol=0)
        assert np.allclose(recs["power"], p_o, rtol=RTOL, atol=0)
        assert np.all(np.diff(recs["power"]) <= 0)
    # same patch on one stream gives the same toplist; with the full dump: the streamed toplists are complete
    for ip in (100, patches[0], patches[15]):
        with torch.cuda.stream(streams[0]):
            d_counts = torch.full((wls[ip].n_templates,), -7, dtype=torch.int32, device="cuda")
            d_top, n_top = ctxs[0].stage1_hough(d_peak, wls[ip], topk=1000, d_w=keep[ip], counts_full=d_counts)
            top1 = ctxs[0].records(d_top, n_top).copy()
            ctxs[0].stage2_power(d_rho, wls[ip], d_top, n_top, d_w=keep[ip], sort_by_power=True)
        torch.cuda.synchronize()
        assert np.array_equal(ctxs[0].records(d_top, n_top), ctxs[0].records(results[ip][0], 1000))
        check_toplist_complete(torch, d_counts, top1, 1000, weighted=False)
        idx = np.random.default_rng(ip).integers(0, wls[ip].n_templates, 200)
        n_s, _, _ = oracle.score(wls[ip], idx.astype(np.uint64), peak=pk, w=None)
        assert np.array_equal(d_counts[torch.from_numpy(idx).cuda()].cpu().numpy(), n_s)
    for c in ctxs:
        c.close()


# ------------------------------------------------------------------------------------------------------------
# the host-buffer end-to-end call
# ------------------------------------------------------------------------------------------------------------
def test_search_patch_host_end_to_end(bsh, torch, ctx):
    wl = synth.config1(pixel="pole")
    recs, n_top = ctx.search_patch_host(wl.rho, wl.w, wl, mode=bsh.BSH_UNWEIGHTED, topk=10)
    pk = oracle.peakgram(wl.rho)
    want_n, want_w = oracle.stage1(wl, pk, wl.w)
    want_idx = oracle.toplist(want_n.astype(np.float64), 10)
    assert n_top == 10 and set(recs["index"].tolist()) == set(want_idx.tolist())
    p_o = oracle.stage2(wl, recs["index"], wl.rho, wl.w)
    assert np.allclose(recs["power"], p_o, rtol=RTOL, atol=0)
    assert np.array_equal(recs["count"], want_n[recs["index"].astype(np.int64)])
    assert np.all(np.diff(recs["power"]) <= 0)
    st = ctx.stats()
    assert st["launches"] > 0 and st["n_templates"] == 1620


@pytest.mark.parametrize("weighted", [False, True])
def test_search_patch_host_at_config2_size(bsh, torch, ctx, weighted):
    """The call `e2e` times in bench.py, at the size it is timed at: record by record against the device-buffer path,
    and every record against the oracle's re-score."""
    wl = synth.config2()
    mode = bsh.BSH_WEIGHTED if weighted else bsh.BSH_UNWEIGHTED
    recs, n_top = ctx.search_patch_host(wl.rho, wl.w, wl, mode=mode, topk=wl.topk)
    assert n_top == wl.topk
    r = gpu_stage1(bsh, torch, ctx, wl, mode, topk=wl.topk, full=False)
    ctx.stage2_power(r["d_rho"], wl, r["d_top"], r["n_top"], d_w=r["d_w"], sort_by_power=True)
    dev_recs = ctx.records(r["d_top"], r["n_top"])
    assert np.array_equal(recs, dev_recs)
    n_o, w_o, p_o = oracle.score(wl, recs["index"], peak=oracle.peakgram(wl.rho), rho=wl.rho, w=wl.w)
    assert np.array_equal(recs["count"], n_o)
    assert np.allclose(recs["wcount"], w_o, rtol=RTOL, atol=0)
    assert np.allclose(recs["power"], p_o, rtol=RTOL, atol=0)
    assert np.all(np.diff(recs["power"]) <= 0)


def test_ties_round_to_even_on_the_gpu(bsh, torch, ctx):
    """R-1: exact half-integer bin coordinates (synth.tie_workload): every kernel family rounds them like the oracle."""
    wl = synth.tie_workload()
    pk = oracle.peakgram(wl.rho)
    want_n, want_w = oracle.stage1(wl, pk, wl.w, mode=oracle.CANONICAL)
    for env in ((bsh.BSH_FAMILY_AUTO, 0), (bsh.BSH_FAMILY_PIXEL_LANE, 0), (bsh.BSH_FAMILY_TEMPLATE_LANE, 0),
                (bsh.BSH_FAMILY_WINDOW, 0), (bsh.BSH_FAMILY_AUTO, 1), (bsh.BSH_FAMILY_PIXEL_LANE, 1)):
        ctx.set_option(bsh.BSH_OPT_KERNEL_FAMILY, env[0])
        ctx.set_option(bsh.BSH_OPT_FORCE_CLAMP, env[1])
        r = gpu_stage1(bsh, torch, ctx, wl, bsh.BSH_UNWEIGHTED)
        assert np.array_equal(r["counts"], want_n), env
        r = gpu_stage1(bsh, torch, ctx, wl, bsh.BSH_WEIGHTED)
        assert np.allclose(r["counts"], want_w, rtol=RTOL, atol=0), env
    ctx.set_option(bsh.BSH_OPT_KERNEL_FAMILY, bsh.BSH_FAMILY_AUTO)
    ctx.set_option(bsh.BSH_OPT_FORCE_CLAMP, 0)
    r = gpu_stage1(bsh, torch, ctx, wl, bsh.BSH_UNWEIGHTED | bsh.BSH_NAIVE)
    assert np.array_equal(r["counts"], want_n)


def test_stage2_on_half_overlapped_sft_set(bsh, torch, ctx):
    """PAPER.md L233 / SURVEY NEXT-1: stage 2 re-scores the stage-1 toplist on a DIFFERENT SFT set (the stage-1 SFTs plus
    a set shifted by T/2: 2 N rows, other velocities, powers and weights), same templates."""
    wl = synth.noise_workload(seed=501, n_sft=300, n_f0=90, margin=45, f_band_start=150.0, n_pix_side=6,
                              ap=(10.0, 25.0, 40.0), P_days=(15.0, 31.0), n_t=4, topk=200)
    wl2 = synth.overlapped_stage2_set(wl, seed=502)
    assert wl2.n_sft == 2 * wl.n_sft and wl2.t_search_mid == wl.t_search_mid
    r = gpu_stage1(bsh, torch, ctx, wl, bsh.BSH_UNWEIGHTED, topk=200, full=False)
    d_rho2, d_w2 = dev(torch, wl2.rho), dev(torch, wl2.w)
    ctx.stage2_power(d_rho2, wl2, r["d_top"], 200, d_w=d_w2, sort_by_power=True)
    torch.cuda.synchronize()
    recs = ctx.records(r["d_top"], 200)
    want = oracle.stage2(wl2, recs["index"], wl2.rho, wl2.w)
    assert np.allclose(recs["power"], want, rtol=RTOL, atol=0)
    assert np.all(np.diff(recs["power"]) <= 0), "sorted by power, best first"
    assert set(recs["index"].tolist()) == set(r["top"]["index"].tolist()), "same candidates, new order"


def test_fraction_nc_toplist_and_stage2(bsh, torch, ctx):
    """PAPER.md L225-L233 / SURVEY NEXT-1: the toplist is a FRACTION N_C = 5 % of all templates of the patch (here 5.6e5 of
    1.1e7, beyond the default candidate buffer), and stage 2 re-scores all of them on the half-overlapped SFT set.
    The full count dump is checked against the oracle on sampled templates; the toplist must be exactly the top-k of the
    dump by (count desc, index asc); powers are checked against the oracle on sampled candidates."""
    wl = synth.noise_workload(seed=601, n_sft=500, n_f0=90, margin=45, f_band_start=150.0, n_pix_side=8,
                              ap=tuple(np.linspace(10.0, 40.0, 8)), P_days=tuple(np.linspace(15.0, 45.0, 12)), n_t=20,
                              topk=10)
    assert wl.n_templates == 64 * 8 * 12 * 20 * 90
    k = int(0.05 * wl.n_templates)
    assert k > (1 << 20) // 2
    r = gpu_stage1(bsh, torch, ctx, wl, bsh.BSH_UNWEIGHTED, topk=k, full=True)
    assert r["n_top"] == k
    dump = r["counts"]
    rng = np.random.default_rng(5)
    pk = oracle.peakgram(wl.rho)
    sample = np.unique(rng.integers(0, wl.n_templates, 3000)).astype(np.uint64)
    want_n, _, _ = oracle.score(wl, sample, peak=pk, w=wl.w)
    assert np.array_equal(dump[sample.astype(np.int64)], want_n)
    want_top = np.lexsort((np.arange(dump.size), -dump.astype(np.int64)))[:k]
    assert np.array_equal(r["top"]["index"].astype(np.int64), want_top)
    assert np.array_equal(r["top"]["count"], dump[want_top])
    # stage 2 on all N_C candidates, on the half-overlapped set
    wl2 = synth.overlapped_stage2_set(wl, seed=602)
    d_rho2, d_w2 = dev(torch, wl2.rho), dev(torch, wl2.w)
    ctx.stage2_power(d_rho2, wl2, r["d_top"], k, d_w=d_w2, sort_by_power=True)
    torch.cuda.synchronize()
    recs = ctx.records(r["d_top"], k)
    assert np.all(np.diff(recs["power"]) <= 0)
    assert np.array_equal(np.sort(recs["index"]), np.sort(r["top"]["index"]))
    pick = np.unique(np.concatenate([np.arange(200), rng.integers(0, k, 2000)]))
    want_p = oracle.stage2(wl2, recs["index"][pick], wl2.rho, wl2.w)
    assert np.allclose(recs["power"][pick], want_p, rtol=RTOL, atol=0)


# ------------------------------------------------------------------------------------------------------------
# boundary extras: diagnostic options, measured peaks, state between launch and collect
# ------------------------------------------------------------------------------------------------------------
def test_set_option_validates(bsh, torch, ctx):
    with pytest.raises(bsh.BshError):
        ctx.set_option(99, 1)
    with pytest.raises(bsh.BshError):
        ctx.set_option(bsh.BSH_OPT_KERNEL_FAMILY, 7)
    with pytest.raises(bsh.BshError):
        ctx.set_option(bsh.BSH_OPT_PIXELS_PER_THREAD, 3)
    ctx.set_option(bsh.BSH_OPT_KERNEL_FAMILY, bsh.BSH_FAMILY_AUTO)


def test_outputs_live_on_the_contexts_device_and_stream(bsh, torch, ctx):
    """Every buffer the binding hands to the library is allocated on the context's device under the context's stream
    (ADVICE r2): a context bound to a side stream, used while torch's current stream is the default one, returns the same
    results as the default-stream context, on the right device."""
    side = torch.cuda.Stream()
    c2 = bsh.Context(0, stream=side)
    try:
        wl = synth.config1()
        d_rho = dev(torch, wl.rho)
        torch.cuda.synchronize()
        want = ctx.build_peakgram(d_rho)
        got = c2.build_peakgram(d_rho)
        side.synchronize()
        assert got.device == d_rho.device and torch.equal(got, want)
        cl = synth.candidate_list(3, n_background=200)
        d = tuple(torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (cl.param, cl.res, cl.sig))
        torch.cuda.synchronize()
        a, b = ctx.post_cluster(d, 3.0), c2.post_cluster(d, 3.0)
        assert all(torch.equal(a[k], b[k]) for k in ("label", "root", "centroid", "significance", "n_members")) and a["best"] == b["best"]
        assert b["label"].device.index == 0
        pa, pb = ctx.post_coincidences(d, d, 3.0), c2.post_coincidences(d, d, 3.0)
        assert all(torch.equal(x, y) for x, y in zip(pa, pb)) and pb[0].device.index == 0
        top_a, n_a = ctx.stage1_hough(want, wl)
        top_b, n_b = c2.stage1_hough(got, wl)
        side.synchronize()
        assert n_a == n_b and torch.equal(top_a, top_b)
    finally:
        c2.close()


def test_measured_peaks_are_plausible(bsh, torch, ctx):
    """bsh_measure_peaks: every rate must sit between half and 1.05x of the guide's unit counts for sm_100 (per SM and
    clock: 128 FP32 lanes, 64 integer-ALU lanes, 128 B of shared memory, one warp instruction per scheduler)."""
    pk = ctx.measure_peaks()
    assert pk["n_sm"] == torch.cuda.get_device_properties(0).multi_processor_count
    assert 1000 < pk["sm_clock_mhz"] < 2200
    assert 0.5 < pk["issue_warp_inst_per_clk_smsp"] <= 1.02
    assert 32 < pk["lop3_lanes_per_clk_sm"] <= 134
    assert 64 < pk["fadd_lanes_per_clk_sm"] <= 134
    assert 8 < pk["dadd_lanes_per_clk_sm"] <= 68 and 8 < pk["dmul_lanes_per_clk_sm"] <= 68
    for k in ("lds32_bytes_per_clk_sm", "lds64_bytes_per_clk_sm", "lds128_bytes_per_clk_sm"):
        assert 64 < pk[k] <= 134, (k, pk[k])


def test_foreign_sft_sets_between_launch_and_collect(bsh, torch, ctx):
    """The table cache holds two (SFT set, grid) entries; a launched, uncollected stage 1 must keep its entry while
    stage 2 runs on two OTHER SFT sets in between (the LRU slot could be the pending call's)."""
    wl = synth.noise_workload(seed=701, n_sft=300, n_f0=90, margin=45, f_band_start=150.0, n_pix_side=6,
                              ap=(10.0, 25.0, 40.0), P_days=(15.0, 31.0), n_t=4, topk=50)
    pk = oracle.peakgram(wl.rho)
    want_n, want_w = oracle.stage1(wl, pk, wl.w, mode=oracle.CANONICAL)
    d_rho, d_w = dev(torch, wl.rho), dev(torch, wl.w)
    d_peak = ctx.build_peakgram(d_rho)
    # a first toplist to feed the foreign stage-2 calls
    d_top0, n0 = ctx.stage1_hough(d_peak, wl, topk=50, d_w=d_w)
    others = [synth.overlapped_stage2_set(wl, seed=s) for s in (702, 703)]
    counts = torch.full((wl.n_templates,), -7, dtype=torch.int32, device="cuda")
    ctx.stage1_launch(d_peak, wl, mode=bsh.BSH_UNWEIGHTED, topk=50, d_w=d_w, counts_full=counts)
    for o in others:                                           # two different SFT sets: both cache slots are wanted
        d_r, d_ww = dev(torch, o.rho), dev(torch, o.w)
        ctx.stage2_power(d_r, o, d_top0, n0, d_w=d_ww, sort_by_power=False)
    d_top, n_top = ctx.stage1_collect()
    torch.cuda.synchronize()
    assert np.array_equal(counts.cpu().numpy(), want_n)
    top = ctx.records(d_top, n_top)
    check_unweighted_toplist(top, want_n, 50)
    assert np.allclose(top["wcount"], want_w[top["index"].astype(np.int64)], rtol=RTOL, atol=0)
