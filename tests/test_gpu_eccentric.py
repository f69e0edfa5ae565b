"""Eccentric (ELL1) tracks on the GPU (Eq. 14; R-23, R-24) against the oracle's
CANONICAL mode: counts bit-exact, weighted counts / powers within 1e-5, toplists identical.  Needs a B200: -m gpu."""
import dataclasses

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


def run(bsh, torch, ctx, wl, mode, topk=None):
    d_rho = torch.from_numpy(wl.rho).cuda()
    d_w = torch.from_numpy(wl.w).cuda()
    d_peak = ctx.build_peakgram(d_rho, 1.6)
    weighted = bool(mode & bsh.BSH_WEIGHTED)
    counts = torch.full((wl.n_templates,), -7, dtype=torch.float32 if weighted else torch.int32, device="cuda")
    d_top, n_top = ctx.stage1_hough(d_peak, wl, mode=mode, topk=topk, d_w=d_w, counts_full=counts)
    ctx.stage2_power(d_rho, wl, d_top, n_top, d_w=d_w, sort_by_power=False)
    torch.cuda.synchronize()
    return counts.cpu().numpy(), ctx.records(d_top, n_top)


def check_all(bsh, torch, ctx, wl, want_n, want_w, k, tag):
    n, top = run(bsh, torch, ctx, wl, bsh.BSH_UNWEIGHTED, topk=k)
    assert np.array_equal(n, want_n), tag
    order = np.lexsort((np.arange(want_n.size), -want_n.astype(np.int64)))[:k]
    assert np.array_equal(top["index"], order.astype(np.uint64)), tag
    assert np.array_equal(top["count"], want_n[order]), tag
    assert np.allclose(top["wcount"], want_w[order], rtol=RTOL, atol=0), tag
    assert np.allclose(top["power"], oracle.stage2(wl, top["index"], wl.rho, wl.w), rtol=RTOL, atol=0), tag
    w, topw = run(bsh, torch, ctx, wl, bsh.BSH_WEIGHTED, topk=k)
    assert np.allclose(w, want_w, rtol=RTOL, atol=0), tag
    cut = np.sort(want_w)[::-1][k - 1]
    for i in set(int(i) for i in topw["index"]) ^ set(np.lexsort((np.arange(want_w.size), -want_w))[:k].tolist()):
        assert abs(want_w[i] - cut) <= RTOL * cut, tag
    assert np.array_equal(topw["count"], want_n[topw["index"].astype(np.int64)]), tag


@pytest.mark.parametrize("pixel", ["ecliptic", "pole"])
def test_config1_eccentric_every_kernel_family(bsh, torch, ctx, pixel):
    """Config 1 with seven eccentricity pairs (one of them circular): 11 340 templates, one pixel -> the template-lane and
    funnel-shift kernels, the diagnostic kernel, rescoring and stage 2; some tracks leave the slab (R-6)."""
    wl = synth.eccentric(synth.config1(pixel=pixel))
    pk = oracle.peakgram(wl.rho)
    want_n, want_w = oracle.stage1(wl, pk, wl.w, mode=oracle.CANONICAL)
    for family in (bsh.BSH_FAMILY_AUTO, bsh.BSH_FAMILY_PIXEL_LANE, bsh.BSH_FAMILY_TEMPLATE_LANE, bsh.BSH_FAMILY_WINDOW):
        ctx.set_option(bsh.BSH_OPT_KERNEL_FAMILY, family)
        check_all(bsh, torch, ctx, wl, want_n, want_w, 10, (pixel, family))
    ctx.set_option(bsh.BSH_OPT_KERNEL_FAMILY, bsh.BSH_FAMILY_AUTO)
    n, _ = run(bsh, torch, ctx, wl, bsh.BSH_UNWEIGHTED | bsh.BSH_NAIVE, topk=10)
    assert np.array_equal(n, want_n)
    # the circular pair of the eccentric grid is the circular grid, bit for bit
    base = synth.config1(pixel=pixel)
    n0, _ = run(bsh, torch, ctx, base, bsh.BSH_UNWEIGHTED, topk=10)
    assert np.array_equal(n.reshape(1, 3, 3, 4, 7, 45)[:, :, :, :, 0, :].ravel(), n0)
    for idx in (0, 46, 7 * 45 + 3, wl.n_templates - 1):
        t6 = bsh.binding.template_decode_ecc(wl, idx)
        assert t6 == oracle.decode_index(wl, idx) and bsh.binding.template_index_ecc(wl, *t6) == idx


@pytest.mark.parametrize("side,n_sft,margin", [(8, 200, 60), (6, 96, 60), (8, 130, 30)])
def test_pixel_lane_kernels_eccentric(bsh, torch, ctx, side, n_sft, margin):
    """Patches of 36 / 64 pixels: the pixel-lane kernels (unweighted and weighted), whose warps compute the binary term --
    now with the two Eq. (14) terms -- once per (template, SFT).  margin 60: no track leaves the slab (unclamped table);
    margin 30: the clamped geometry."""
    wl = synth.eccentric(synth.noise_workload(seed=3 * side + n_sft, n_sft=n_sft, n_f0=90, margin=margin, f_band_start=150.0,
                                              n_pix_side=side, ap=(10.0, 40.0), P_days=(15.0, 31.0), n_t=3, topk=40),
                         e_max=0.08, n_e=1, n_omega=3)
    assert wl.n_ecc == 4
    pk = oracle.peakgram(wl.rho)
    want_n, want_w = oracle.stage1(wl, pk, wl.w, mode=oracle.CANONICAL)
    ctx.set_option(bsh.BSH_OPT_KERNEL_FAMILY, bsh.BSH_FAMILY_PIXEL_LANE)    # (36 pixels fill 56 % of two lane groups: forced)
    for force_clamp in (False, True):
        ctx.set_option(bsh.BSH_OPT_FORCE_CLAMP, int(force_clamp))
        check_all(bsh, torch, ctx, wl, want_n, want_w, 40, (side, n_sft, force_clamp))
        assert ctx.stats()["kernel_variant"] // 1000 == 3
    # eccentricity moves the counts: the e != 0 slices differ from the circular one
    cube = want_n.reshape(side * side, 2, 2, 3, 4, 90)
    assert not np.array_equal(cube[..., 1, :], cube[..., 0, :])


def test_eccentric_grid_rejects_bad_pairs(bsh, torch, ctx):
    wl = synth.eccentric(synth.config1())
    bad = dataclasses.replace(wl, ecosw=np.array([0.9]), esinw=np.array([0.3]))
    d_rho = torch.from_numpy(wl.rho).cuda()
    d_peak = ctx.build_peakgram(d_rho, 1.6)
    with pytest.raises(bsh.BshError):
        ctx.stage1_hough(d_peak, bad, mode=bsh.BSH_UNWEIGHTED, topk=10)


def test_eccentric_large_toplist_paths(bsh, torch, ctx):
    """A toplist of 100 000 entries on an eccentric grid: the radix sort and the one-thread-per-candidate rescoring / stage-2
    kernels (the large-list path of SURVEY NEXT-1) with the Eq. (14) terms compiled in."""
    wl = synth.eccentric(synth.noise_workload(seed=21, n_sft=200, n_f0=90, margin=60, f_band_start=150.0, n_pix_side=8,
                                              ap=(10.0, 40.0), P_days=(15.0, 31.0), n_t=3, topk=100_000),
                         e_max=0.08, n_e=1, n_omega=3)
    assert wl.n_templates == 64 * 2 * 2 * 3 * 4 * 90
    pk = oracle.peakgram(wl.rho)
    want_n, want_w = oracle.stage1(wl, pk, wl.w, mode=oracle.CANONICAL)
    n, top = run(bsh, torch, ctx, wl, bsh.BSH_UNWEIGHTED, topk=100_000)
    assert np.array_equal(n, want_n)
    order = np.lexsort((np.arange(want_n.size), -want_n.astype(np.int64)))[:100_000]
    assert np.array_equal(top["index"], order.astype(np.uint64))
    assert np.array_equal(top["count"], want_n[order])
    assert np.allclose(top["wcount"], want_w[order], rtol=RTOL, atol=0)
    assert np.allclose(top["power"], oracle.stage2(wl, top["index"], wl.rho, wl.w), rtol=RTOL, atol=0)
    w, topw = run(bsh, torch, ctx, wl, bsh.BSH_WEIGHTED, topk=100_000)
    assert np.array_equal(topw["count"], want_n[topw["index"].astype(np.int64)])
    assert np.all(np.diff(topw["wcount"]) <= 0)
    assert np.allclose(w, want_w, rtol=RTOL, atol=0)                                  # every weighted count of the grid
    assert np.allclose(topw["wcount"], want_w[topw["index"].astype(np.int64)], rtol=RTOL, atol=0)
    assert len(set(int(i) for i in topw["index"])) == 100_000
    # the weighted toplist is the top 100 000 of the oracle's weighted counts up to ties within the tolerance at the cut
    cut = np.sort(want_w)[::-1][100_000 - 1]
    assert set(np.nonzero(want_w > cut * (1 + RTOL))[0].tolist()) <= set(int(i) for i in topw["index"])
    assert np.all(want_w[topw["index"].astype(np.int64)] >= cut * (1 - RTOL))
