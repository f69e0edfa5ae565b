"""The threshold search of the per-patch top-k (bsh_stage1_collect): inputs that are NOT what the
noise model of the first-pass threshold assumes, on grids larger than the candidate buffer (2^20 entries), so that the
"take everything" shortcut is off and the search has to run:

  too many survivors   a band of set columns in every row (an instrumental line, L407): far more than 2^20 templates clear
                       the noise-derived threshold;
  too few survivors    columns that no track visits are full of peaks: the model's mean is too high;
  massive ties         an all-zero peakgram (a notched band) and an all-ones one (constant rows): every template, or more
                       templates than the buffer holds, has exactly the k-th value, and the toplist is decided by the
                       template index alone (count desc, index asc) -- the tie-limit phase.

In every case the full dump of counts equals the tier-2 CPU reference (bit-exact; weighted 1e-5), the toplist is the
lexsort of those counts, and stats.n_passes shows that the search was entered.  Needs a B200: -m gpu."""
import dataclasses

import numpy as np
import pytest

import oracle
import synth

pytestmark = pytest.mark.gpu
RTOL = 1e-5
TOPK = 1000


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


def base_workload(n_sft=128):
    wl = synth.noise_workload(seed=5, n_sft=n_sft, n_f0=90, margin=60, f_band_start=150.0, span_days=20.0, n_pix_side=8,
                              ap=np.linspace(10.0, 40.0, 8), P_days=np.linspace(15.0, 45.0, 10), n_t=10, topk=TOPK)
    assert wl.n_templates == 4_608_000 > (1 << 20)
    return wl


def with_rho(wl, rho):
    return dataclasses.replace(wl, rho=np.ascontiguousarray(rho, np.float32))


def run(bsh, torch, ctx, wl, mode, topk=TOPK):
    d_rho = torch.from_numpy(wl.rho).cuda()
    d_w = torch.from_numpy(wl.w).cuda()
    d_peak = ctx.build_peakgram(d_rho, 1.6)
    weighted = bool(mode & bsh.BSH_WEIGHTED)
    counts = torch.full((wl.n_templates,), -7, dtype=torch.float32 if weighted else torch.int32, device="cuda")
    d_top, n_top = ctx.stage1_hough(d_peak, wl, mode=mode, topk=topk, d_w=d_w, counts_full=counts)
    st = ctx.stats()
    ctx.stage2_power(d_rho, wl, d_top, n_top, d_w=d_w, sort_by_power=False)
    torch.cuda.synchronize()
    assert n_top == topk
    return counts.cpu().numpy(), ctx.records(d_top, n_top), st


def check(bsh, torch, ctx, wl, min_passes, modes=("unweighted", "weighted"), topk=TOPK, naive=False):
    pk = oracle.peakgram(wl.rho)
    want_n, want_w = oracle.tier2_stage1(wl, pk, wl.w, want_wcount=True)
    out = {}
    for name in modes:
        weighted = name == "weighted"
        mode = (bsh.BSH_WEIGHTED if weighted else bsh.BSH_UNWEIGHTED) | (bsh.BSH_NAIVE if naive else 0)
        got, top, st = run(bsh, torch, ctx, wl, mode, topk)
        assert st["n_passes"] >= min_passes, (name, st["n_passes"])
        assert topk <= st["n_candidates"] <= max(1 << 20, 4 * topk)
        assert len(set(int(i) for i in top["index"])) == topk
        idx = top["index"].astype(np.int64)
        assert np.array_equal(top["count"], want_n[idx])
        assert np.allclose(top["wcount"], want_w[idx], rtol=RTOL, atol=0)
        assert np.allclose(top["power"], oracle.stage2(wl, top["index"], wl.rho, wl.w), rtol=RTOL, atol=0)
        if weighted:
            assert np.allclose(got, want_w, rtol=RTOL, atol=0)
            assert np.all(np.diff(top["wcount"]) <= 0)
            cut = np.sort(want_w)[::-1][topk - 1]
            above = np.nonzero(want_w > cut * (1 + RTOL))[0]
            assert set(above.tolist()) <= set(idx.tolist())
            assert np.all(want_w[idx] >= cut * (1 - RTOL))
            if np.all(got == got[0]):                                # all tied in FP32 too: the index alone decides
                assert np.array_equal(idx, np.arange(topk))              # (equal FP64 sums can differ in their last FP32
                                                                         # bit with the order of the additions, R-20)
        else:
            assert np.array_equal(got, want_n)
            order = np.lexsort((np.arange(want_n.size), -want_n.astype(np.int64)))[:topk]
            assert np.array_equal(idx, order)
        out[name] = st
    return out, want_n


@pytest.mark.parametrize("line_cols", [10, 40])
def test_too_many_survivors_a_line_in_every_row(bsh, torch, ctx, line_cols):
    wl = base_workload()
    rho = wl.rho.copy()
    c0 = wl.n_bins // 2
    rho[:, c0:c0 + line_cols] = 50.0
    st, want_n = check(bsh, torch, ctx, with_rho(wl, rho), min_passes=2)
    assert want_n.max() == wl.n_sft                                     # templates that stay on the line all the time
    assert st["unweighted"]["threshold"] > 40
    assert all(v["n_passes"] <= 4 for v in st.values())                 # one step from the overflowed buffer, not a walk
    print("passes:", {k: (v["n_passes"], v["threshold"], v["n_candidates"]) for k, v in st.items()})


def test_too_few_survivors_peaks_where_no_track_goes(bsh, torch, ctx):
    wl = base_workload()
    rho = wl.rho.copy()
    rho[:, :15] = 50.0
    rho[:, -15:] = 50.0
    st, _ = check(bsh, torch, ctx, with_rho(wl, rho), min_passes=2)
    print("passes:", {k: (v["n_passes"], v["threshold"], v["n_candidates"]) for k, v in st.items()})


@pytest.mark.parametrize("value", [0.0, 50.0])
def test_massive_ties_constant_peakgram(bsh, torch, ctx, value):
    """All-zero (every count 0) and all-ones rows (every count = the SFTs the track spends inside the slab, here all of
    them): the toplist is the lowest template indices.  Before round 3 this ended in BSH_ESTATE after 12 passes."""
    wl = base_workload(n_sft=64)
    st, want_n = check(bsh, torch, ctx, with_rho(wl, np.full_like(wl.rho, value)), min_passes=2)
    assert want_n.min() == want_n.max() == (0 if value == 0.0 else 64)
    assert st["unweighted"]["n_passes"] <= 4 and st["weighted"]["n_passes"] <= 4


def test_massive_ties_below_a_few_louder_templates(bsh, torch, ctx):
    """Eight SFT rows carry a peak in a column that few tracks reach, everything else is empty: 389 templates score 1 or 2
    and 4.6e6 are tied at zero; top-1000 = the louder ones in order, then the 611 lowest-index zeros.  Zero is too low a
    threshold, one is too high, and the tie-limit phase finishes the job -- for both statistics (the weighted one ties
    at 0.0f exactly), and also through the one-thread-per-template diagnostic kernel."""
    wl = base_workload(n_sft=64)
    rho = np.zeros_like(wl.rho)
    rho[::8, 36] = 50.0
    wl2 = with_rho(wl, rho)
    st, want_n = check(bsh, torch, ctx, wl2, min_passes=3)
    n_loud = int((want_n > 0).sum())
    assert 0 < n_loud < TOPK, n_loud
    for name in ("unweighted", "weighted"):
        assert st[name]["threshold"] == 0 and st[name]["n_candidates"] < 4 * TOPK and st[name]["n_passes"] <= 10
    print("passes:", {k: v["n_passes"] for k, v in st.items()})
    check(bsh, torch, ctx, wl2, min_passes=3, modes=("unweighted",), naive=True)
