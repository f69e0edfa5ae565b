"""Post-processing on the GPU (section V.E, Eq. 44) against the oracle: pair lists, cluster labels
and member counts bit-exact (the distance decisions are FP64 in the same operation order on both sides), centroids and
significances equal to the last bit (same summation order).  Needs a B200: -m gpu."""
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


def dev(torch, c):
    return tuple(torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (c.param, c.res, c.sig))


def check_cluster(torch, ctx, c, window, prune=0.0):
    got = ctx.post_cluster(dev(torch, c), float(window), float(prune))
    want = oracle.cluster(c.param, c.res, c.sig, float(window), float(prune))
    assert np.array_equal(got["label"].cpu().numpy(), want["label"])
    assert np.array_equal(got["root"].cpu().numpy(), want["root"])
    assert np.array_equal(got["n_members"].cpu().numpy(), want["n_members"])
    assert np.array_equal(got["significance"].cpu().numpy(), want["significance"])
    assert np.array_equal(got["centroid"].cpu().numpy(), want["centroid"])
    assert got["best"] == want["best"]
    return want


@pytest.mark.parametrize("seed,n_bg,window,prune", [(1, 300, 3.0, 0.0), (2, 300, math.sqrt(14.0), 0.0), (3, 1000, 3.0, 2.0),
                                                    (4, 31, 1.0, 0.0), (5, 33, 50.0, 3.0), (6, 4900, math.sqrt(14.0), 0.0),
                                                    (7, 4900, math.sqrt(14.0), 3.0)])
def test_clusters_and_centroids(bsh, torch, ctx, seed, n_bg, window, prune):
    c = synth.candidate_list(seed, n_background=n_bg, chain=40 if n_bg > 100 else 5)
    want = check_cluster(torch, ctx, c, window, prune)
    if n_bg >= 300 and window >= 3.0 and prune == 0.0:
        assert want["n_members"].max() >= 20                    # the planted groups and the chain were found


def test_hand_example_empty_and_single(bsh, torch, ctx):
    f = np.array([0, 10, 1, 10, 2, 50, 10, 10], np.float64)
    x = np.array([0, 0, 0, 1, 0, 50, 2, 6], np.float64)
    p = np.zeros((8, 6))
    p[:, 0], p[:, 1] = f, x
    r = np.ones((8, 6))
    r[7] = 3.0
    c = synth.Candidates(param=p, res=r, sig=np.array([1, 4, 2, 1, 3, 9, 5, 2], np.float64), truth=np.zeros(8, int))
    for window, prune in ((1.5, 0.0), (2.5, 0.0), (1.5, 1.5)):
        check_cluster(torch, ctx, c, window, prune)
    got = ctx.post_cluster(dev(torch, c), 1.5)
    assert got["label"].cpu().tolist() == [0, 1, 0, 1, 0, 5, 1, 7] and got["best"] == 1
    empty = synth.Candidates(param=np.zeros((0, 6)), res=np.ones((0, 6)), sig=np.zeros(0), truth=np.zeros(0, int))
    e = ctx.post_cluster(dev(torch, empty), 1.0)
    assert e["label"].numel() == 0 and e["root"].numel() == 0 and e["best"] == -1
    one = synth.Candidates(param=np.zeros((1, 6)), res=np.ones((1, 6)), sig=np.ones(1), truth=np.zeros(1, int))
    check_cluster(torch, ctx, one, 1.0)
    pa, pb, cen, sig = ctx.post_coincidences(dev(torch, c), dev(torch, empty), 3.0)
    assert pa.numel() == 0
    with pytest.raises(bsh.BshError):
        ctx.post_cluster(dev(torch, c), 0.0)


@pytest.mark.parametrize("na,nb,window", [(300, 300, 3.0), (1000, 777, 3.0), (65, 31, 10.0), (4900, 4900, 3.0)])
def test_coincidences(bsh, torch, ctx, na, nb, window):
    a = synth.candidate_list(20 + na, n_background=na)
    b = synth.candidate_list(21 + nb, n_background=nb)
    m = min(a.n, b.n, 60)
    b.param[:m] = a.param[:m] + 0.7 * a.res[:m] * np.random.default_rng(na).standard_normal((m, 6))
    b.res[:m] = synth.resolutions(b.param[:m, 0], b.param[:m, 3], b.param[:m, 4])
    ia, ib, cen, sig = oracle.coincidences(a.param, a.res, a.sig, b.param, b.res, b.sig, window)
    pa, pb, gcen, gsig = ctx.post_coincidences(dev(torch, a), dev(torch, b), window)
    assert ia.size >= 20
    assert np.array_equal(pa.cpu().numpy(), ia) and np.array_equal(pb.cpu().numpy(), ib)
    assert np.array_equal(gcen.cpu().numpy(), cen) and np.array_equal(gsig.cpu().numpy(), sig)
    # a buffer that is too small reports the full count and fills what fits
    pa2, pb2, _, _ = ctx.post_coincidences(dev(torch, a), dev(torch, b), window, max_pairs=5)
    assert pa2.numel() == 5 and np.array_equal(pa2.cpu().numpy(), ia[:5]) and np.array_equal(pb2.cpu().numpy(), ib[:5])
