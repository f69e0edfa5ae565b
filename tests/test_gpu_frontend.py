"""Front end on the GPU against the oracle: complex SFT bins -> running-median normalised power -> peakgram
(Eq. 20-21; R-22).  FP32 arithmetic with single roundings on both sides and an exact
selection for the median, so rho and the peak bits are compared BIT FOR BIT.  Needs a B200: -m gpu."""
import math

import numpy as np
import pytest

import oracle
import synth

pytestmark = pytest.mark.gpu


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


def same_floats(a, b):
    """bit-identical up to the payload of NaNs"""
    return a.shape == b.shape and np.array_equal(np.isnan(a), np.isnan(b)) and np.array_equal(a[~np.isnan(a)], b[~np.isnan(b)])


def run_front(torch, ctx, x, window, **kw):
    d_x = torch.from_numpy(np.ascontiguousarray(x)).cuda()
    d_rho, d_peak = ctx.normalise_peakgram(d_x, window=window, **kw)
    torch.cuda.synchronize()
    return (None if d_rho is None else d_rho.cpu().numpy(),
            None if d_peak is None else d_peak.cpu().numpy().view(np.uint32))


@pytest.mark.parametrize("n,n_raw,window", [(1, 101, 101), (3, 102, 101), (5, 150, 101), (33, 304, 101), (64, 352, 101),
                                            (7, 40, 3), (4, 64, 1), (2, 33, 33), (9, 133, 101), (3, 2048, 101), (2, 1000, 999),
                                            (2000, 272, 101), (8000, 352, 101)])
def test_frontend_bit_exact(bsh, torch, ctx, n, n_raw, window):
    x = synth.raw_sft_bins(100 + n, n, n_raw)
    rho, peak = run_front(torch, ctx, x, window)
    want = oracle.normalise(x, window)
    assert same_floats(rho, want)
    assert np.array_equal(peak, oracle.peakgram(want))
    assert abs(bsh.binding.median_bias(window) - oracle.median_bias(window)) < 1e-15


def test_frontend_special_values_strides_and_outputs(bsh, torch, ctx):
    x = synth.raw_sft_bins(3, 12, 140)
    x[0, 5] = np.nan                                      # NaN power ranks above everything
    x[1, 20:90] = 0                                       # zero medians: 0/0 and p/0
    x[2, 7] = np.inf
    x[3, :] = 3 + 4j                                      # constant power: rho = bias
    x[4, ::2] *= np.complex64(1e-22)                      # subnormal powers
    x[5, 60] = np.complex64(1e19 + 1e19j)                 # |x|^2 overflows to +inf
    want = oracle.normalise(x, 101)
    rho, peak = run_front(torch, ctx, x, 101)
    assert same_floats(rho, want)
    assert np.array_equal(peak, oracle.peakgram(want))
    # strided input rows (a view into a wider array), and either output alone
    wide = np.zeros((12, 200), np.complex64)
    wide[:, 30:170] = x
    d_wide = torch.from_numpy(wide).cuda()
    d_rho, d_peak = ctx.normalise_peakgram(d_wide[:, 30:170], window=101)
    assert same_floats(d_rho.cpu().numpy(), want)
    d_rho2, none = ctx.normalise_peakgram(d_wide[:, 30:170], window=101, want_peak=False)
    assert none is None and same_floats(d_rho2.cpu().numpy(), want)
    none, d_peak2 = ctx.normalise_peakgram(d_wide[:, 30:170], window=101, want_rho=False)
    assert none is None and np.array_equal(d_peak2.cpu().numpy().view(np.uint32), oracle.peakgram(want))
    # another threshold and another bias
    rho_b, peak_b = run_front(torch, ctx, x, 101, bias=math.log(2.0), rho_th=2.5)
    want_b = oracle.normalise(x, 101, bias=math.log(2.0))
    assert same_floats(rho_b, want_b) and np.array_equal(peak_b, oracle.peakgram(want_b, 2.5))


def test_frontend_rejects_bad_arguments(bsh, torch, ctx):
    d_x = torch.from_numpy(synth.raw_sft_bins(1, 4, 120)).cuda()
    for window in (0, 100, 121, -3):
        with pytest.raises(bsh.BshError):
            ctx.normalise_peakgram(d_x, window=window)
    with pytest.raises(bsh.BshError):
        ctx.normalise_peakgram(d_x, window=101, bias=0.0)
    with pytest.raises(bsh.BshError):
        ctx.normalise_peakgram(d_x, window=101, want_rho=False, want_peak=False)
    with pytest.raises(bsh.BshError):
        ctx.normalise_peakgram(torch.zeros((2, 2049), dtype=torch.complex64, device="cuda"), window=101)


def test_config4_from_raw_bins_recovers_the_injections(bsh, torch, ctx):
    """BASELINE.json configs[3] started where the paper starts: complex SFT bins of a non-stationary,
    coloured detector -> front end -> peakgram -> stage 1 -> stage 2.  The front end's output equals the oracle's bit for
    bit, every injection is the loudest candidate of its patch, and counts and powers equal the oracle's on that input."""
    c4 = synth.config4()
    bins = []
    for inj in c4.injections:
        wl_p = c4.patch_workload(inj.patch, None)
        bins.append(oracle.track(wl_p, inj.pix, inj.ia, inj.ip, inj.it, inj.j, mode=oracle.DIRECT))
    raw = c4.raw_bins(bins, window=101)
    assert raw.shape == (6000, c4.base.n_bins + 100)
    want_rho = oracle.normalise(raw, 101)
    pk = oracle.peakgram(want_rho)
    d_raw = torch.from_numpy(raw).cuda()
    d_rho, d_peak = ctx.normalise_peakgram(d_raw, window=101)
    assert same_floats(d_rho.cpu().numpy(), want_rho)
    assert np.array_equal(d_peak.cpu().numpy().view(np.uint32), pk)
    for inj in c4.injections[:4]:
        wl = c4.patch_workload(inj.patch, want_rho)
        d_top, n_top = ctx.stage1_hough(d_peak, wl, mode=bsh.BSH_UNWEIGHTED, topk=1000)
        top = ctx.records(d_top, n_top)
        want = oracle.encode_index(wl, inj.pix, inj.ia, inj.ip, inj.it, inj.j)
        assert int(top["index"][0]) == want, inj.patch
        n_o, _, _ = oracle.score(wl, top["index"], peak=pk, w=None)
        assert np.array_equal(top["count"], n_o)
        ctx.stage2_power(d_rho, wl, d_top, n_top, d_w=None, sort_by_power=True)
        recs = ctx.records(d_top, n_top)
        assert int(recs["index"][0]) == want
        p_o = oracle.stage2(wl, recs["index"][:50], want_rho, None)
        assert np.allclose(recs["power"][:50], p_o, rtol=1e-5, atol=0)
