"""Pins for the post-processing oracle (oracle/bsh_oracle.c: orc_distance2, orc_coincidences, orc_cluster; PAPER.md section
V.E, L385-L407, Eq. 44): a hand-placed example, scipy's connected components and single-linkage clustering, numpy
averages.  CPU only."""
import os

import numpy as np
import pytest
import scipy.cluster.hierarchy as sch
import scipy.sparse as sp
import scipy.sparse.csgraph as csg
import scipy.spatial.distance as ssd

import oracle
import synth

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _golden():
    out = {}
    with open(os.path.join(GOLDEN, "cluster_example.txt")) as fh:
        for line in fh:
            line = line.split("#")[0].strip()
            if "=" in line:
                k, v = line.split("=", 1)
                out[k.strip()] = np.array([float(t) for t in v.split()])
    return out


def _hand():
    g = _golden()
    n = g["f"].size
    p = np.zeros((n, 6))
    p[:, 0], p[:, 1] = g["f"], g["x"]
    r = np.ones((n, 6))
    r[7] = 3.0
    return g, p, r, g["sig"]


def test_hand_placed_clusters():
    g, p, r, s = _hand()
    assert oracle.distance2(p[0], r[0], p[4], r[4]) == 4.0
    assert oracle.distance2(p[6], r[6], p[7], r[7]) == 4.0                # (6 - 2) / ((1 + 3) / 2) = 2 bins
    c = oracle.cluster(p, r, s, 1.5)
    assert np.array_equal(c["label"], g["labels_w1p5"].astype(np.int32))
    assert np.array_equal(c["root"], [0, 1, 5, 7]) and np.array_equal(c["n_members"], [3, 3, 1, 1])
    assert np.allclose(c["significance"], [6, 10, 9, 2], rtol=0, atol=0)
    assert np.allclose(c["centroid"][:, 0], [8 / 6, 10, 50, 10], rtol=1e-15)
    assert np.allclose(c["centroid"][:, 1], [0, 1.1, 50, 6], rtol=1e-15)
    assert c["best"] == 1
    c = oracle.cluster(p, r, s, 2.5)
    assert np.array_equal(c["label"], g["labels_w2p5"].astype(np.int32))
    assert np.isclose(c["centroid"][1, 1], 23 / 12, rtol=1e-15) and c["significance"][1] == 12 and c["best"] == 1
    c = oracle.cluster(p, r, s, 1.5, prune_window=1.5)
    assert np.array_equal(c["label"], g["labels_pruned"].astype(np.int32))
    assert np.array_equal(c["root"], [0, 1, 5, 7]) and np.array_equal(c["n_members"], [2, 2, 1, 1])
    assert np.isclose(c["centroid"][0, 0], 1.6, rtol=1e-15) and np.isclose(c["centroid"][1, 1], 11 / 6, rtol=1e-15)
    assert c["best"] == 2                                                # label 5, s = 9
    # coincidences between the list and itself shifted by 0.5 in f: pairs closer than 1 bin
    q = p.copy()
    q[:, 0] += 0.5
    ia, ib, cen, sig = oracle.coincidences(p, r, s, q, r, s, 1.0)
    # (same index: 0.5 bins, or 0.5 / 3 for candidate 7; (2, 0) and (4, 2): f differs by 0.5; (1, 3), (3, 1): sqrt(1.25) > 1;
    #  (7, 6): (0.5 / 2)^2 + (4 / 2)^2 > 1)
    assert list(zip(ia.tolist(), ib.tolist())) == [(0, 0), (1, 1), (2, 0), (2, 2), (3, 3), (4, 2), (4, 4), (5, 5), (6, 6),
                                                    (7, 7)]
    assert np.isclose(cen[2, 0], (2 * 1.0 + 1 * 0.5) / 3) and sig[2] == 3    # pair (2, 0): s = 2 + 1


def _dist_matrix(p, r):
    res = 0.5 * (r[:, None, :] + r[None, :, :])
    return np.sqrt((((p[:, None, :] - p[None, :, :]) / res) ** 2).sum(-1))


@pytest.mark.parametrize("seed,window", [(1, 3.0), (2, np.sqrt(14.0)), (3, 1.0)])
def test_clusters_equal_scipy_connected_components_and_single_linkage(seed, window):
    """coincidence window 3 bins, clustering window sqrt(14) bins."""
    c = synth.candidate_list(seed, chain=9)
    d = _dist_matrix(c.param, c.res)
    assert np.abs(np.abs(d - window) - 0).min() > 1e-9                    # no pair sits on the threshold
    got = oracle.cluster(c.param, c.res, c.sig, float(window))
    adj = sp.csr_matrix((d < window) & ~np.eye(c.n, dtype=bool))
    n_comp, comp = csg.connected_components(adj, directed=False)
    first = np.full(n_comp, c.n)
    np.minimum.at(first, comp, np.arange(c.n))
    assert np.array_equal(got["label"], first[comp])                       # label = smallest member index
    assert got["root"].size == n_comp
    link = sch.fcluster(sch.linkage(ssd.squareform(d, checks=False), "single"), t=float(window), criterion="distance")
    for lab in np.unique(link):
        assert np.unique(got["label"][link == lab]).size == 1
    assert np.unique(link).size == n_comp
    # centroids and significances: numpy's weighted average over the members
    for k, root in enumerate(got["root"]):
        m = got["label"] == root
        assert got["n_members"][k] == m.sum()
        assert np.isclose(got["significance"][k], c.sig[m].sum(), rtol=1e-13)
        assert np.allclose(got["centroid"][k], np.average(c.param[m], axis=0, weights=c.sig[m]), rtol=1e-12)
    assert got["best"] == int(np.argmax(got["significance"]))
    if window >= 3.0:                                                      # the chain (0.9-bin steps) is one cluster, the planted
        for g in range(4):                                                 # groups are recovered
            assert np.unique(got["label"][c.truth == g]).size == 1


def test_distance_properties_and_coincidences_bruteforce():
    a, b = synth.candidate_list(11), synth.candidate_list(12)
    b.param[:40] = a.param[:40] + 0.7 * a.res[:40] * np.random.default_rng(0).standard_normal((40, 6))
    b.res[:40] = synth.resolutions(b.param[:40, 0], b.param[:40, 3], b.param[:40, 4])
    for i, j in [(0, 0), (5, 17), (39, 2)]:
        d2 = oracle.distance2(a.param[i], a.res[i], b.param[j], b.res[j])
        assert d2 == oracle.distance2(b.param[j], b.res[j], a.param[i], a.res[i])            # symmetric, exactly
        want = (((a.param[i] - b.param[j]) / (0.5 * (a.res[i] + b.res[j]))) ** 2).sum()
        assert np.isclose(d2, want, rtol=1e-14)
        assert np.isclose(oracle.distance2(a.param[i], 2 * a.res[i], b.param[j], 2 * b.res[j]), d2 / 4, rtol=1e-15)
    assert oracle.distance2(a.param[3], a.res[3], a.param[3], a.res[3]) == 0.0
    ia, ib, cen, sig = oracle.coincidences(a.param, a.res, a.sig, b.param, b.res, b.sig, 3.0)
    res = 0.5 * (a.res[:, None, :] + b.res[None, :, :])
    d = np.sqrt((((a.param[:, None, :] - b.param[None, :, :]) / res) ** 2).sum(-1))
    want = np.argwhere(d < 3.0)
    assert want.shape[0] >= 30 and np.array_equal(np.stack([ia, ib], 1), want)
    assert np.allclose(sig, a.sig[ia] + b.sig[ib], rtol=1e-15)
    w = np.stack([a.sig[ia], b.sig[ib]], 1)
    assert np.allclose(cen, (w[:, :1] * a.param[ia] + w[:, 1:] * b.param[ib]) / w.sum(1, keepdims=True), rtol=1e-13)


def test_prune_keeps_members_near_the_top_template():
    c = synth.candidate_list(5, groups=((30, 2.5),), n_background=50)
    full = oracle.cluster(c.param, c.res, c.sig, 3.0)
    cut = oracle.cluster(c.param, c.res, c.sig, 3.0, prune_window=2.0)
    d = _dist_matrix(c.param, c.res)
    for root in full["root"]:
        m = np.flatnonzero(full["label"] == root)
        top = m[np.argmax(c.sig[m])]
        keep = m[(d[m, top] < 2.0) | (m == top)]
        assert np.array_equal(np.flatnonzero(cut["label"] == root), keep)
    assert (cut["label"] == -1).sum() == c.n - sum((cut["label"] == r).sum() for r in full["root"])
    assert (cut["label"] == -1).sum() > 0
    # empty and single-candidate lists
    e = oracle.cluster(np.zeros((0, 6)), np.ones((0, 6)), np.zeros(0), 1.0)
    assert e["label"].size == 0 and e["root"].size == 0 and e["best"] == -1
    one = oracle.cluster(np.zeros((1, 6)), np.ones((1, 6)), np.ones(1), 1.0)
    assert one["label"].tolist() == [0] and one["best"] == 0
