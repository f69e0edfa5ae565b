"""Pins for the CPU oracle (oracle/bsh_oracle.c): each test checks it against something OTHER than itself --
a hand-worked example, a closed form, a library routine, a 50-digit independent evaluation of the paper's
phase model, or an invariant the paper states.  CPU only (-m "not gpu")."""
import dataclasses
import math
import os

import mpmath as mp
import numpy as np
import pytest
import scipy.stats as st

import oracle
import synth

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _read_golden(name):
    out = {}
    with open(os.path.join(GOLDEN, name)) as fh:
        for line in fh:
            line = line.split("#")[0].strip()
            if "=" in line:
                k, v = line.split("=", 1)
                out[k.strip()] = v.strip()
    return out


def _pack_bits(bits):
    """independent packing: numpy packbits, little bit order, padded to 32-bit words"""
    bits = np.asarray(bits, np.uint8)
    n, k = bits.shape
    wpr = (k + 31) // 32
    padded = np.zeros((n, wpr * 32), np.uint8)
    padded[:, :k] = bits
    return np.packbits(padded, axis=1, bitorder="little").view(np.uint32).reshape(n, wpr)


# ------------------------------------------------------------------------------------------------------------
# paper constants
# ------------------------------------------------------------------------------------------------------------
def test_paper_constants():
    g = _read_golden("paper_constants.txt")
    assert float(g["rho_th"]) == oracle.RHO_TH == 1.6
    assert int(g["n_f0_per_0p1Hz_at_900s"]) == synth.config2().n_f0 == 90
    assert abs(oracle.P_PEAK - 0.20189651799465538) < 1e-15


# ------------------------------------------------------------------------------------------------------------
# peakgram: library routine + closed-form fraction
# ------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n,k", [(1, 1), (3, 31), (5, 32), (7, 33), (64, 63), (50, 172), (9, 257)])
def test_peakgram_equals_numpy_packbits(n, k):
    rng = np.random.default_rng(n * 1000 + k)
    rho = rng.standard_exponential((n, k)).astype(np.float32)
    rho[0, 0] = np.float32(1.6)                        # exactly at threshold: strict '>' -> 0   (R-8)
    if k > 2:
        rho[0, 1] = np.nextafter(np.float32(1.6), np.float32(2))   # one ulp above -> 1
        rho[0, 2] = np.nan                                             # NaN -> 0
    got = oracle.peakgram(rho)
    want = _pack_bits(rho > np.float32(1.6))
    assert got.dtype == np.uint32 and got.shape == want.shape
    assert np.array_equal(got, want)
    assert (got[0, 0] & 1) == 0
    if k > 2:
        assert (got[0, 0] >> 1) & 1 == 1 and (got[0, 0] >> 2) & 1 == 0


def test_peakgram_fraction_is_exp_minus_rho_th():
    wl = synth.config2()
    pk = oracle.peakgram(wl.rho)
    ones = int(np.unpackbits(pk.view(np.uint8)).sum())
    n = wl.n_sft * wl.n_bins
    p = math.exp(-1.6)
    assert abs(ones / n - p) < 4 * math.sqrt(p * (1 - p) / n)
    # pad bits are zero
    pad = pk[:, -1] >> np.uint32(wl.n_bins - 32 * (pk.shape[1] - 1)) if wl.n_bins % 32 else np.zeros(1, np.uint32)
    assert not pad.any()


# ------------------------------------------------------------------------------------------------------------
# hand-worked example (tests/golden/hand_track_example.txt): pins the SIGN and size of the binary term
# ------------------------------------------------------------------------------------------------------------
def _hand_workload():
    P = 4000.0
    ap = 0.002 * P / (2 * math.pi)
    return synth.Workload(name="hand", seed=0, t_sft=1.0, t_mid=np.array([0.0, 1000.0, 2000.0]),
                          v_over_c=np.zeros((3, 3)), t_search_mid=0.0, k_slab0=996, n_bins=11, k_band0=1000, n_f0=3,
                          rho=None, w=None, alpha=np.array([0.3]), delta=np.array([-0.2]), ap=np.array([ap]),
                          P=np.array([P]), tasc_frac=np.array([0.0]), topk=3)


@pytest.mark.parametrize("mode", [oracle.DIRECT, oracle.CANONICAL])
def test_hand_worked_example(mode):
    g = _read_golden("hand_track_example.txt")
    rows = np.array([[int(x) for x in g[f"row{i}"].split()] for i in range(3)], np.uint8)
    w = np.array([float(x) for x in g["weights"].split()], np.float32)
    wl = _hand_workload()
    for j in range(3):
        assert list(oracle.track(wl, 0, 0, 0, 0, j, mode=mode)) == [2 + j, 4 + j, 6 + j]
    cnt, wc = oracle.stage1(wl, _pack_bits(rows), w, mode=mode)
    assert list(cnt) == [int(x) for x in g["counts"].split()]
    assert np.allclose(wc, [float(x) for x in g["wcounts"].split()], rtol=0, atol=1e-12)
    # stage 2 on the same tracks: power = sum w_i rho[i][k_i] with rho = 10*row + column index (hand-checkable)
    rho = (10.0 * rows + np.arange(11)[None, :]).astype(np.float32)
    pw = oracle.stage2(wl, np.arange(3, dtype=np.uint64), rho, w, mode=mode)
    want = [0.5 * rho[0, 2 + j] + 1.0 * rho[1, 4 + j] + 1.5 * rho[2, 6 + j] for j in range(3)]
    assert np.allclose(pw, want, rtol=0, atol=1e-12)


# ------------------------------------------------------------------------------------------------------------
# brute force at 50 digits from the PHASE model, Eq. (13) with e = 0: f = (1/2pi) dphi/dt.
# Independent of Eq. (15) as typed in the oracle: the detector POSITION model is differentiated numerically, so a
# wrong sign, a dropped Omega factor, a_p in the wrong units or a swapped sin/cos in the oracle would show.
# ------------------------------------------------------------------------------------------------------------
def _mp_position_over_c(t, lat_deg=30.6, theta0=0.0):
    lam = 2 * mp.pi * t / mp.mpf(synth.YEAR_S)
    eps = mp.mpf(synth.OBLIQUITY)
    r_orb = mp.mpf(synth.V_ORB) * mp.mpf(synth.YEAR_S) / (2 * mp.pi)
    th = mp.mpf(theta0) + 2 * mp.pi * t / mp.mpf(synth.T_SIDEREAL)
    r_rot = mp.mpf(synth.R_EARTH) * mp.cos(mp.radians(mp.mpf(lat_deg)))
    x = r_orb * mp.cos(lam) + r_rot * mp.cos(th)
    y = r_orb * mp.sin(lam) * mp.cos(eps) + r_rot * mp.sin(th)
    z = r_orb * mp.sin(lam) * mp.sin(eps)
    c = mp.mpf(synth.C_LIGHT)
    return x / c, y / c, z / c


def test_track_against_phase_model_derivative_50_digits():
    mp.mp.dps = 50
    wl = synth.config1(pixel="ecliptic")
    nvec = (mp.cos(mp.mpf(wl.delta[0])) * mp.cos(mp.mpf(wl.alpha[0])),
            mp.cos(mp.mpf(wl.delta[0])) * mp.sin(mp.mpf(wl.alpha[0])), mp.sin(mp.mpf(wl.delta[0])))
    T = mp.mpf(wl.t_sft)
    h = mp.mpf(10) ** -12                                # central difference step, seconds: error O(h^2) << 1e-15 bins
    # absolute detector time of SFT i: synth uses t_abs = start + T/2 with t_ref = first start = 0
    checked = near = 0
    for ia in range(len(wl.ap)):
        for ip in range(len(wl.P)):
            for it in range(len(wl.tasc_frac)):
                P = mp.mpf(wl.P[ip])
                Om = 2 * mp.pi / P
                tasc = mp.mpf(wl.t_search_mid) + mp.mpf(wl.tasc_frac[it]) * P
                ap = mp.mpf(wl.ap[ia])
                for j in (0, 17, 44):
                    f0 = mp.mpf(wl.k_band0 + j) / T

                    def phase_over_2pi(t):           # Eq. (13), e = 0, constants dropped
                        rx, ry, rz = _mp_position_over_c(t)
                        return f0 * (t + rx * nvec[0] + ry * nvec[1] + rz * nvec[2] - ap * mp.sin(Om * (t - tasc)))

                    kd, xd = oracle.track(wl, 0, ia, ip, it, j, mode=oracle.DIRECT, with_aux=True)
                    kc = oracle.track(wl, 0, ia, ip, it, j, mode=oracle.CANONICAL)
                    for i in range(0, wl.n_sft, 3):
                        t = mp.mpf(wl.t_mid[i])
                        f = (phase_over_2pi(t + h) - phase_over_2pi(t - h)) / (2 * h)
                        x = (f - mp.mpf(wl.k_slab0) / T) * T
                        assert abs(x - mp.mpf(xd[i])) < mp.mpf("1e-7"), (ia, ip, it, j, i, x, xd[i])
                        frac = x + mp.mpf("0.5")
                        if abs(frac - mp.nint(frac)) < mp.mpf("1e-7"):
                            near += 1
                            continue
                        k = int(mp.floor(frac))
                        assert k == kd[i] == kc[i], (ia, ip, it, j, i)
                        checked += 1
    assert checked > 2000 and near < 5


def test_track_bruteforce_eq15_50_digits_all_of_config1():
    """Every (template, SFT) of config 1 (both pixels): Eq. (15) evaluated in 50-digit arithmetic from the same FP64
    inputs; bins must match both oracle modes except where x + 1/2 is within 1e-9 of an integer."""
    mp.mp.dps = 50
    total = near = 0
    for pixel in ("ecliptic", "pole"):
        wl = synth.config1(pixel=pixel)
        a, d = mp.mpf(wl.alpha[0]), mp.mpf(wl.delta[0])
        nvec = (mp.cos(d) * mp.cos(a), mp.cos(d) * mp.sin(a), mp.sin(d))
        D = [sum(mp.mpf(wl.v_over_c[i, c]) * nvec[c] for c in range(3)) for i in range(wl.n_sft)]
        m = wl.k_band0 - wl.k_slab0
        for ip in range(len(wl.P)):
            P = mp.mpf(wl.P[ip])
            Om = 2 * mp.pi / P
            for it in range(len(wl.tasc_frac)):
                tasc = mp.mpf(wl.t_search_mid) + mp.mpf(wl.tasc_frac[it]) * P
                cphi = [mp.cos(Om * (mp.mpf(wl.t_mid[i]) - tasc)) for i in range(wl.n_sft)]
                for ia in range(len(wl.ap)):
                    g = [D[i] - mp.mpf(wl.ap[ia]) * Om * cphi[i] for i in range(wl.n_sft)]
                    for j in range(wl.n_f0):
                        kd = oracle.track(wl, 0, ia, ip, it, j, mode=oracle.DIRECT)
                        kc = oracle.track(wl, 0, ia, ip, it, j, mode=oracle.CANONICAL)
                        u = mp.mpf(wl.k_band0 + j)
                        for i in range(wl.n_sft):
                            xh = m + j + u * g[i] + mp.mpf("0.5")
                            total += 1
                            if abs(xh - mp.nint(xh)) < mp.mpf("1e-9"):
                                near += 1
                                continue
                            k = int(mp.floor(xh))
                            assert k == kd[i] == kc[i], (pixel, ia, ip, it, j, i)
    assert total == 2 * 1620 * 64 and near <= 2


# ------------------------------------------------------------------------------------------------------------
# a_p = 0 limit (Eq. 15 without its third term is the isolated-star track of SkyHough, L199)
# ------------------------------------------------------------------------------------------------------------
def test_ap_zero_reduces_to_isolated_track_and_to_column_sums():
    wl = synth.noise_workload(seed=11, n_sft=300, n_f0=40, margin=14, f_band_start=100.0, n_pix_side=2,
                              ap=(0.0,), P_days=(15.0, 33.0), n_t=3)
    pk = oracle.peakgram(wl.rho)
    bits = np.unpackbits(pk.view(np.uint8), axis=1, bitorder="little")[:, :wl.n_bins]
    nvec = np.stack([np.cos(wl.delta) * np.cos(wl.alpha), np.cos(wl.delta) * np.sin(wl.alpha), np.sin(wl.delta)], -1)
    D = (wl.v_over_c.astype(np.longdouble) @ nvec.T.astype(np.longdouble)).T            # [pix, N], 80-bit
    u = (wl.k_band0 + np.arange(wl.n_f0)).astype(np.longdouble)
    x = u[None, :, None] * (1 + D[:, None, :]) - np.longdouble(wl.k_slab0)               # [pix, j, N]
    near = np.abs(x + 0.5 - np.rint(x + 0.5)) < 1e-9
    k_iso = np.floor(x + np.longdouble(0.5)).astype(np.int64)
    for mode in (oracle.DIRECT, oracle.CANONICAL):
        cnt, wc = oracle.stage1(wl, pk, wl.w, mode=mode)
        cnt = cnt.reshape(wl.n_pix, 1, len(wl.P), len(wl.tasc_frac), wl.n_f0)
        # every (P, t_asc) gives the same answer when a_p = 0
        assert (cnt == cnt[:, :, :1, :1, :]).all()
        for pix in range(wl.n_pix):
            for j in range(wl.n_f0):
                k = oracle.track(wl, pix, 0, 1, 2, j, mode=mode)
                ok = ~near[pix, j]
                assert np.array_equal(k[ok], k_iso[pix, j][ok])
                if ok.all():
                    inside = (k_iso[pix, j] >= 0) & (k_iso[pix, j] < wl.n_bins)
                    want = bits[np.arange(wl.n_sft)[inside], k_iso[pix, j][inside]].sum()
                    assert cnt[pix, 0, 0, 0, j] == want
    # detector at rest as well: the track is the vertical line k = j + m and the count is a column sum
    wl0 = dataclasses.replace(wl, v_over_c=np.zeros_like(wl.v_over_c))
    m = wl0.margin
    for mode in (oracle.DIRECT, oracle.CANONICAL):
        cnt, wc = oracle.stage1(wl0, pk, wl0.w, mode=mode)
        cnt = cnt.reshape(wl.n_pix, -1, wl.n_f0)
        wc = wc.reshape(wl.n_pix, -1, wl.n_f0)
        assert (cnt == bits[:, m:m + wl.n_f0].sum(0)[None, None, :]).all()
        want_w = wl0.w.astype(np.float64) @ bits[:, m:m + wl.n_f0].astype(np.float64)
        assert np.allclose(wc, want_w[None, None, :], rtol=1e-13, atol=0)
        idx = np.arange(wl0.n_templates, dtype=np.uint64)
        pw = oracle.stage2(wl0, idx, wl0.rho, wl0.w, mode=mode).reshape(wl.n_pix, -1, wl.n_f0)
        want_p = wl0.w.astype(np.float64) @ wl0.rho[:, m:m + wl.n_f0].astype(np.float64)
        assert np.allclose(pw, want_p[None, None, :], rtol=1e-12, atol=0)


# ------------------------------------------------------------------------------------------------------------
# invariants the paper states: t_asc defined modulo P (L303); and a_p -> -a_p  <=>  t_asc -> t_asc + P/2
# ------------------------------------------------------------------------------------------------------------
def test_tasc_periodicity_and_half_period_symmetry():
    wl = synth.config1(pixel="pole")
    pk = oracle.peakgram(wl.rho)
    base, _ = oracle.stage1(wl, pk, None, mode=oracle.DIRECT)
    shifted = dataclasses.replace(wl, tasc_frac=wl.tasc_frac + 1.0)
    got, _ = oracle.stage1(shifted, pk, None, mode=oracle.DIRECT)
    # identical up to near-tie events (expected ~1e-9 * 1e5 accumulations -> none)
    assert np.array_equal(base, got)
    flipped = dataclasses.replace(wl, ap=-wl.ap, tasc_frac=wl.tasc_frac + 0.5)
    got2, _ = oracle.stage1(flipped, pk, None, mode=oracle.DIRECT)
    assert np.array_equal(base, got2)
    # excursion bound |k - (j + m)| <= ceil(u (max|D| + a_p Omega))
    bound = synth.slab_margin(wl.k_band0 + wl.n_f0, wl.v_over_c, wl.ap.max(), wl.P.min())
    for ia, ip, it, j in [(0, 0, 0, 0), (2, 0, 3, 44), (1, 2, 2, 20)]:
        k = oracle.track(wl, 0, ia, ip, it, j)
        assert np.abs(k - (j + wl.margin)).max() <= bound


def test_direct_and_canonical_agree_except_flagged_near_ties():
    wl = synth.noise_workload(seed=5, n_sft=500, n_f0=30, margin=40, f_band_start=150.0, n_pix_side=2,
                              ap=(10.0, 25.0, 40.0), P_days=(15.0, 22.0, 45.0), n_t=5)
    res = oracle.compare_modes(wl, tol=1e-9)
    assert res["compared"] == wl.n_accumulations
    assert res["unflagged"] == 0
    assert res["flagged"] < 40 + 4e-9 * res["compared"] * 5      # ~2e-9 per accumulation expected


def test_canonical_stage1_equals_per_accumulation_canonical_track():
    """orc_stage1's hoisted CANONICAL loop must equal orc_track_canonical call by call."""
    wl = synth.config1(pixel="ecliptic")
    pk = oracle.peakgram(wl.rho)
    bits = np.unpackbits(pk.view(np.uint8), axis=1, bitorder="little")[:, :wl.n_bins]
    cnt, wc = oracle.stage1(wl, pk, wl.w, mode=oracle.CANONICAL)
    left_slab = 0
    rows = np.arange(wl.n_sft)
    for idx in range(0, wl.n_templates, 7):
        pix, ia, ip, it, j = oracle.decode_index(wl, idx)
        assert oracle.encode_index(wl, pix, ia, ip, it, j) == idx
        k = oracle.track(wl, pix, ia, ip, it, j, mode=oracle.CANONICAL)
        inside = (k >= 0) & (k < wl.n_bins)
        left_slab += int((~inside).sum())
        b = np.zeros(wl.n_sft, np.int64)
        b[inside] = bits[rows[inside], k[inside]]
        assert cnt[idx] == b.sum()
        assert abs(wc[idx] - (wl.w.astype(np.float64) * b).sum()) < 1e-12
    assert left_slab > 0, "config1-ecliptic must exercise tracks leaving the slab (R-6)"
    c2, w2, _ = oracle.score(wl, np.arange(0, wl.n_templates, 7), peak=pk, w=wl.w)
    assert np.array_equal(c2, cnt[::7]) and np.allclose(w2, wc[::7], rtol=0, atol=1e-12)


# ------------------------------------------------------------------------------------------------------------
# noise statistics: counts ~ Binomial(N, e^-1.6); power ~ Gamma(N, 1)
# ------------------------------------------------------------------------------------------------------------
def test_noise_counts_are_binomial_and_power_is_gamma():
    p = math.exp(-1.6)
    counts, z_w, z_p, pw_unw = [], [], [], []
    n_sft = 64
    for seed in range(60):
        wl = synth.config1(seed=100 + seed, pixel="pole")
        pk = oracle.peakgram(wl.rho)
        # one (pixel, binary template): its 45 f0 templates read disjoint cells -> independent samples
        sub = wl.subgrid(ia=[seed % 3], ip=[(seed // 3) % 3], it=[seed % 4])
        c, wc = oracle.stage1(sub, pk, wl.w, mode=oracle.CANONICAL)
        counts.append(c)
        w = wl.w.astype(np.float64)
        z_w.append((wc - p * w.sum()) / math.sqrt(p * (1 - p) * (w * w).sum()))
        idx = np.arange(sub.n_templates, dtype=np.uint64)
        z_p.append(oracle.significance_power(oracle.stage2(sub, idx, wl.rho, wl.w), wl.w))
        pw_unw.append(oracle.stage2(sub, idx, wl.rho, None))
    counts = np.concatenate(counts)
    n = counts.size
    assert n == 60 * 45
    assert abs(counts.mean() - n_sft * p) < 4 * math.sqrt(n_sft * p * (1 - p) / n)
    var = counts.var(ddof=1)
    assert abs(var / (n_sft * p * (1 - p)) - 1) < 4 * math.sqrt(2.0 / n) * 1.3
    # chi-square against the binomial pmf, tails pooled
    lo, hi = 6, 21
    obs = np.array([(counts <= lo).sum()] + [(counts == v).sum() for v in range(lo + 1, hi)] + [(counts >= hi).sum()])
    pmf = st.binom.pmf(np.arange(0, n_sft + 1), n_sft, p)
    exp = n * np.array([pmf[:lo + 1].sum()] + [pmf[v] for v in range(lo + 1, hi)] + [pmf[hi:].sum()])
    chi2 = ((obs - exp) ** 2 / exp).sum()
    assert chi2 < st.chi2.ppf(0.9999, len(obs) - 1)
    for z in (np.concatenate(z_w), np.concatenate(z_p)):
        assert abs(z.mean()) < 4 / math.sqrt(n)
        assert abs(z.var(ddof=1) - 1) < 0.2
    pu = np.concatenate(pw_unw)                                    # Gamma(N, 1): mean N, variance N
    assert abs(pu.mean() - n_sft) < 4 * math.sqrt(n_sft / n)
    assert abs(pu.var(ddof=1) / n_sft - 1) < 0.2
    assert st.kstest(pu, st.gamma(a=n_sft).cdf).pvalue > 1e-4


# ------------------------------------------------------------------------------------------------------------
# toplist = full sort by (value desc, index asc)  (L217, L225; R-11) against numpy lexsort
# ------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n,k", [(1, 1), (10, 20), (1620, 10), (5000, 1000)])
def test_toplist_equals_lexsort(n, k):
    rng = np.random.default_rng(n)
    v = rng.integers(0, 12, n).astype(np.float64)                  # many ties
    got = oracle.toplist(v, k)
    want = np.lexsort((np.arange(n), -v))[:k]
    assert np.array_equal(got, want.astype(np.uint64))


# ------------------------------------------------------------------------------------------------------------
# injected signal is recovered as the loudest candidate; its count matches the noncentral chi-square closed form
# ------------------------------------------------------------------------------------------------------------
def _mp_track_bins(wl, alpha, delta, ap, P, tasc, u):
    """Eq. (15) bins at 30 digits, independent of the oracle (used to DEPOSIT the injection)."""
    mp.mp.dps = 30
    a, d = mp.mpf(alpha), mp.mpf(delta)
    nvec = (mp.cos(d) * mp.cos(a), mp.cos(d) * mp.sin(a), mp.sin(d))
    Om = 2 * mp.pi / mp.mpf(P)
    out = np.zeros(wl.n_sft, np.int64)
    for i in range(wl.n_sft):
        D = sum(mp.mpf(wl.v_over_c[i, c]) * nvec[c] for c in range(3))
        f = mp.mpf(u) / mp.mpf(wl.t_sft) * (1 + D - mp.mpf(ap) * Om * mp.cos(Om * (mp.mpf(wl.t_mid[i]) - mp.mpf(tasc))))
        out[i] = int(mp.floor((f - mp.mpf(wl.k_slab0) / mp.mpf(wl.t_sft)) * mp.mpf(wl.t_sft) + mp.mpf("0.5")))
    return out


def test_injected_signal_is_loudest_and_count_matches_marcum_q():
    n_sft, t_sft = 1500, 600.0
    starts = np.arange(n_sft) * (45.0 * synth.DAY / n_sft)
    v = synth.detector_velocity_over_c(starts + 0.5 * t_sft)
    ap, P, tf = np.linspace(10, 40, 4), np.linspace(15, 45, 5) * synth.DAY, synth.tasc_fractions(6)
    margin = synth.slab_margin(int(400.05 * t_sft), v, ap.max(), P.min())
    rng = np.random.Generator(np.random.Philox(key=[44, 0]))
    k_bins = 30 + 2 * margin
    re = rng.standard_normal((n_sft, k_bins)) * math.sqrt(0.5)
    im = rng.standard_normal((n_sft, k_bins)) * math.sqrt(0.5)
    alpha, delta = synth.patch_pixels(1.0, 0.4, synth.pixel_size(t_sft, 400.0, 1.0), 3, 3)
    base = synth._finish("inj", 44, t_sft, starts, v, 400.0, 30 / t_sft, margin, None, np.ones(n_sft, np.float32),
                         alpha, delta, ap, P, tf, topk=20)
    inj = synth.Injection(patch=0, pix=4, ia=2, ip=1, it=3, j=11, phases=rng.uniform(0, 2 * math.pi, n_sft))
    c4 = synth.Config4(base=base, re=re, im=im, patches=[(alpha, delta)], injections=[inj], amp2=0.3)
    tasc = base.t_search_mid + tf[inj.it] * P[inj.ip]
    bins = _mp_track_bins(base, alpha[inj.pix], delta[inj.pix], ap[inj.ia], P[inj.ip], tasc, base.k_band0 + inj.j)
    rho = c4.deposit([bins])
    wl = c4.patch_workload(0, rho)
    pk = oracle.peakgram(rho)
    cnt, _ = oracle.stage1(wl, pk, None, mode=oracle.CANONICAL)
    top = oracle.toplist(cnt.astype(np.float64), 20)
    want = oracle.encode_index(wl, inj.pix, inj.ia, inj.ip, inj.it, inj.j)
    assert int(top[0]) == want
    # P(rho > 1.6 | |A|^2 = 0.3): 2 rho is noncentral chi-square(2 dof, nc = 2 |A|^2)  -> 0.29568
    p_sig = st.ncx2.sf(2 * 1.6, 2, 2 * 0.3)
    assert abs(p_sig - 0.29568) < 1e-4
    assert abs(cnt[want] - n_sft * p_sig) < 4.5 * math.sqrt(n_sft * p_sig * (1 - p_sig))
    # stage 2 is the more sensitive statistic (L229): the injected template also tops the power ranking
    pw = oracle.stage2(wl, top, rho, None)
    assert int(top[np.argmax(pw)]) == want
    assert abs(pw[0] - n_sft * 1.3) < 5 * math.sqrt(n_sft * (1 + 2 * 0.3))     # E[rho] = 1 + |A|^2, var = 1 + 2|A|^2


def test_ties_round_to_even():
    """R-1: the bin is round(y) to the nearest integer, ties to even.  With the tie workload y = q / 2 exactly at j = 0
    (k_band0 = 2^17, v_x / c = q 2^-18, n = (1, 0, 0), no binary term), so the expected bins follow from Python's own
    round() (banker's rounding) -- nothing of the oracle is used to form them."""
    wl = synth.tie_workload()
    q = [1, 3, 5, -1, -3, 2, 0, 7]
    want = np.array([wl.margin + round(v / 2) for v in q])
    assert [round(v / 2) for v in q] == [0, 2, 2, 0, -2, 1, 0, 4]
    assert np.array_equal(oracle.track(wl, 0, 0, 0, 0, 0, mode=oracle.CANONICAL), want)
    # DIRECT evaluates Eq. (15) as printed: its x carries a few ulps of rounding, so at an exact tie it may fall on either
    # side (these are the flagged near-ties of compare_modes); away from ties it must agree
    direct = oracle.track(wl, 0, 0, 0, 0, 0, mode=oracle.DIRECT)
    tie = np.array([v % 2 != 0 for v in q])
    assert np.array_equal(direct[~tie], want[~tie]) and np.all(np.abs(direct[tie] - want[tie]) <= 1)
    # one bin up the lattice (u = 2^17 + 1) y is no longer a tie: ordinary rounding of q/2 (1 + 2^-17)
    want1 = np.array([wl.margin + 1 + math.floor(v / 2 * (1 + 2.0 ** -17) + 0.5) for v in q])
    assert np.array_equal(oracle.track(wl, 0, 0, 0, 0, 1, mode=oracle.CANONICAL), want1)
    # and the counts see the parity of the bins (peaks on even columns only)
    pk = oracle.peakgram(wl.rho)
    cnt, _ = oracle.stage1(wl, pk, None, mode=oracle.CANONICAL)
    assert cnt[0] == int(np.sum(want % 2 == 0))


# ------------------------------------------------------------------------------------------------------------
# Front end: running-median normalisation, Eq. (20)-(21), reading R-22
# ------------------------------------------------------------------------------------------------------------
def test_normalise_hand_worked_example():
    g = _read_golden("running_median_example.txt")
    amp = np.array([float(v) for v in g["amplitudes"].split()])
    want = np.array([float(v) for v in g["rho"].split()])
    x = amp.astype(np.complex64)[None, :]
    got = oracle.normalise(x, window=int(g["window"]))
    assert np.allclose(got[0], want, rtol=3e-7, atol=0)
    assert abs(oracle.median_bias(3) - float(g["bias"])) < 1e-15
    # the same powers carried by the imaginary part, or split between the two, give the same rho (|x|^2 = re^2 + im^2)
    assert np.array_equal(oracle.normalise((1j * amp).astype(np.complex64)[None, :], window=3), got)
    x2 = (amp * (0.6 + 0.8j)).astype(np.complex64)[None, :]
    assert np.allclose(oracle.normalise(x2, window=3), got, rtol=1e-6)
    # peak bits of the example: only column 1 exceeds 1.0; none exceeds the paper's 1.6
    assert oracle.peakgram(got, 1.0)[0, 0] == 0b0010 and oracle.peakgram(got, 1.6)[0, 0] == 0


def test_median_bias_closed_form_and_monte_carlo():
    from fractions import Fraction
    g = _read_golden("running_median_example.txt")
    assert abs(oracle.median_bias(101) - float(g["median_bias_101"])) < 1e-14
    for w in (1, 3, 5, 21, 101):
        exact = sum(Fraction(1, i) for i in range((w + 1) // 2, w + 1))       # E of the middle order statistic of Exp(1)
        assert abs(oracle.median_bias(w) - float(exact)) < 1e-14
    assert oracle.median_bias(1) == 1.0                                      # window of one bin: the mean itself
    assert 0 < oracle.median_bias(100001) - float(g["ln2"]) < 1e-5          # large-window limit ln 2
    rng = np.random.default_rng(7)
    med = np.median(rng.standard_exponential((200000, 101)), axis=1)
    assert abs(med.mean() - oracle.median_bias(101)) < 5 * med.std() / math.sqrt(med.size)


@pytest.mark.parametrize("n,n_raw,window", [(3, 101, 101), (5, 150, 101), (4, 40, 3), (2, 64, 1), (6, 352, 101), (2, 33, 33)])
def test_normalise_equals_numpy_sliding_median(n, n_raw, window):
    """np.median over numpy's sliding_window_view is a library routine, not the oracle's copy-sort-pick loop."""
    x = synth.raw_sft_bins(11, n, n_raw)
    got = oracle.normalise(x, window)
    re, im = x.real.astype(np.float32), x.imag.astype(np.float32)
    p = re * re + im * im
    med = np.median(np.lib.stride_tricks.sliding_window_view(p, window, axis=1), axis=-1).astype(np.float32)
    h = (window - 1) // 2
    want = p[:, h:n_raw - h] / (med / np.float32(oracle.median_bias(window)))
    assert got.shape == (n, n_raw - window + 1)
    assert np.array_equal(got, want)


def test_normalise_statistics_scale_invariance_and_lines():
    n, k, window = 400, 200, 101
    x = synth.raw_sft_bins(5, n, k + window - 1, noise_sigma=3.0)            # per-SFT noise levels spread over e^{+-4.5}
    rho = oracle.normalise(x, window).astype(np.float64)
    # normalised noise power is Exp(1): mean 1, P(rho > 1.6) = e^{-1.6}.  The 101-bin median estimate has a
    # relative scatter of ~1/sqrt(101 ln^2 2 ...) ~ 10 %, which biases <1/median> up by ~1 %: allow 3 %.
    assert abs(rho.mean() - 1.0) < 0.03
    frac = (rho > 1.6).mean()
    assert abs(frac - math.exp(-1.6)) < 0.01
    # every SFT is normalised on its own: per-row means agree although the raw levels differ by orders of magnitude
    raw_level = (np.abs(x) ** 2).mean(axis=1)
    assert raw_level.max() / raw_level.min() > 1e2
    assert np.abs(rho.mean(axis=1) - 1.0).max() < 0.35
    # scaling one SFT by a power of two changes nothing, bit for bit (every operation scales exactly)
    y = x.copy()
    y[3] *= np.complex64(2.0 ** 7)
    y[9] *= np.complex64(2.0 ** -5)
    assert np.array_equal(oracle.normalise(y, window), oracle.normalise(x, window))
    # a narrow spectral line (3 bins, 1000 x the noise power) stands out and barely moves the noise estimate around it:
    z = x.copy()
    z[:, 150:153] *= np.complex64(math.sqrt(1000.0))
    rz = oracle.normalise(z, window).astype(np.float64)
    h = (window - 1) // 2
    assert (rz[:, 150 - h:153 - h] > 20).mean() > 0.96                       # P(1000 Exp(1) > 20) = 0.98
    far = np.r_[0:40]                                                        # columns whose windows do not contain the line
    assert np.array_equal(rz[:, far], rho[:, far])
    near = np.r_[60:99]                                                      # windows containing the 3 line bins: the median
    ratio = rho[:, near] / rz[:, near]                                       # moves up by ~3 order statistics of 101 (~6 %)
    assert 1.0 <= ratio.min() and ratio.mean() < 1.12


def test_normalise_special_values():
    """Constant power -> rho = bias (|x|^2 / (|x|^2 / bias)); zero median -> inf / NaN; NaN bins rank last."""
    b = np.float32(oracle.median_bias(5))
    x = np.full((1, 9), 3.0 + 4.0j, np.complex64)                            # |x|^2 = 25 everywhere
    got = oracle.normalise(x, 5)
    assert np.allclose(got, b, rtol=2e-7)
    x = np.zeros((1, 7), np.complex64)
    x[0, 3] = 2.0
    got = oracle.normalise(x, 5)                                             # medians are 0: 0/0 = NaN, 4/0 = inf
    assert np.isnan(got[0, 0]) and np.isinf(got[0, 1]) and np.isnan(got[0, 2])
    assert oracle.peakgram(got)[0, 0] == 0b010                               # NaN > 1.6 is false, inf > 1.6 is true
    x = (np.arange(1, 8) + 0j).astype(np.complex64)[None, :]
    x[0, 1] = np.nan
    got = oracle.normalise(x, 3)
    # windows of |x|^2: (1, NaN, 9) -> median 9; (NaN, 9, 16) -> 16; (9, 16, 25) -> 16; ...
    b3 = np.float32(oracle.median_bias(3))
    assert np.isnan(got[0, 0])                                               # centre bin is the NaN
    assert np.isclose(got[0, 1], np.float32(9.0) / (np.float32(16.0) / b3))
    assert np.isclose(got[0, 2], np.float32(16.0) / (np.float32(16.0) / b3))


# ------------------------------------------------------------------------------------------------------------
# Eccentric (ELL1) tracks: PAPER.md Eq. (14), derived from the timing model Eq. (11)-(13) L78-L91
# ------------------------------------------------------------------------------------------------------------
def test_eccentric_zero_pair_reproduces_circular_tracks_bit_for_bit():
    wl = synth.config1(pixel="ecliptic")
    we = synth.eccentric(wl)                                 # pair 0 is (0, 0)
    assert we.n_ecc == 7 and we.n_templates == 7 * wl.n_templates and we.ecosw[0] == 0.0 and we.esinw[0] == 0.0
    pk = oracle.peakgram(wl.rho)
    for mode in (oracle.DIRECT, oracle.CANONICAL):
        base_n, base_w = oracle.stage1(wl, pk, wl.w, mode=mode)
        n, w = oracle.stage1(we, pk, wl.w, mode=mode)
        shape = (1, 3, 3, 4, 7, 45)
        assert np.array_equal(n.reshape(shape)[:, :, :, :, 0, :].ravel(), base_n)
        assert np.array_equal(w.reshape(shape)[:, :, :, :, 0, :].ravel(), base_w)
        assert not np.array_equal(n.reshape(shape)[:, :, :, :, 3, :].ravel(), base_n)     # e = 0.05 moves the tracks
        for (ia, ip, it, j) in [(0, 0, 0, 0), (2, 1, 3, 44)]:
            k0, a0 = oracle.track(wl, 0, ia, ip, it, j, mode=mode, with_aux=True)
            k1, a1 = oracle.track(we, 0, ia, ip, it, j, mode=mode, with_aux=True, ie=0)
            assert np.array_equal(k0, k1) and np.array_equal(a0, a1)
    # index helpers with the extra axis
    for idx in (0, 1, 44, 45, 7 * 45 - 1, 7 * 45, we.n_templates - 1, 12345):
        pix, ia, ip, it, ie, j = oracle.decode_index(we, idx)
        assert oracle.encode_index(we, pix, ia, ip, it, j, ie=ie) == idx


def test_eccentric_track_bruteforce_eq14_50_digits():
    """Eq. (14) as printed, in 50-digit arithmetic from the same FP64 inputs, against both oracle modes."""
    mp.mp.dps = 50
    we = synth.eccentric(synth.config1(pixel="pole"))
    a, d = mp.mpf(we.alpha[0]), mp.mpf(we.delta[0])
    nvec = (mp.cos(d) * mp.cos(a), mp.cos(d) * mp.sin(a), mp.sin(d))
    D = [sum(mp.mpf(we.v_over_c[i, c]) * nvec[c] for c in range(3)) for i in range(we.n_sft)]
    m = we.k_band0 - we.k_slab0
    total = near = 0
    for ip in range(len(we.P)):
        P = mp.mpf(we.P[ip])
        Om = 2 * mp.pi / P
        for it in (0, 3):
            tasc = mp.mpf(we.t_search_mid) + mp.mpf(we.tasc_frac[it]) * P
            ph = [Om * (mp.mpf(we.t_mid[i]) - tasc) for i in range(we.n_sft)]
            for ia in (0, 2):
                ap = mp.mpf(we.ap[ia])
                for ie in range(we.n_ecc):
                    ecw, esw = mp.mpf(we.ecosw[ie]), mp.mpf(we.esinw[ie])
                    g = [D[i] - ap * Om * mp.cos(ph[i]) - ap * Om * ecw * mp.cos(2 * ph[i]) + ap * Om * esw * mp.sin(2 * ph[i])
                         for i in range(we.n_sft)]
                    for j in (0, 13, 44):
                        kd = oracle.track(we, 0, ia, ip, it, j, mode=oracle.DIRECT, ie=ie)
                        kc = oracle.track(we, 0, ia, ip, it, j, mode=oracle.CANONICAL, ie=ie)
                        u = mp.mpf(we.k_band0 + j)
                        for i in range(we.n_sft):
                            xh = m + j + u * g[i] + mp.mpf("0.5")
                            total += 1
                            if abs(xh - mp.nint(xh)) < mp.mpf("1e-9"):
                                near += 1
                                continue
                            assert int(mp.floor(xh)) == kd[i] == kc[i], (ip, it, ia, ie, j, i)
    assert total == 3 * 2 * 2 * 7 * 3 * 64 and near <= 2


def test_eccentric_track_against_kepler_orbit_to_first_order_in_e():
    """Independent of Eq. (14) as typed: the projected orbit of Eq. (9) (L68) with the eccentric anomaly from Kepler's
    equation (7) and t_asc = t_p - omega / Omega (Eq. 10), differentiated numerically at 40 digits.  The ELL1 track
    is its expansion to first order in e (L72, L80), so the two bin coordinates differ by at most ~ 2 e^2 a_p Omega u.
    DESIGN.md R-24: expanding Eq. (9)-(10) gives R/c = a_p [sin psi + (e cos w / 2) sin 2 psi - (e sin w / 2) cos 2 psi];
    Eq. (11)-(14) print the last term with the opposite sign.  The oracle follows Eq. (14) as printed, so its pair
    (e cos w, e sin w) corresponds to the Kepler orbit with argument of periapsis -w: the test passes
    esinw = -e sin(w_Kepler).  With esinw = +e sin(w_Kepler) the same comparison is off by O(e), which is asserted too."""
    mp.mp.dps = 40
    base = synth.config1(pixel="pole")
    T = mp.mpf(base.t_sft)
    for e, omega in [(0.01, 0.7), (0.03, 2.9), (0.002, 4.4)]:
        we = dataclasses.replace(base, ecosw=np.array([e * math.cos(omega)]), esinw=np.array([-e * math.sin(omega)]))
        wrong = dataclasses.replace(base, ecosw=np.array([e * math.cos(omega)]), esinw=np.array([e * math.sin(omega)]))
        for (ia, ip, it, j) in [(2, 0, 1, 10), (0, 2, 3, 40)]:
            P = mp.mpf(we.P[ip])
            Om = 2 * mp.pi / P
            ap, ee, om = mp.mpf(we.ap[ia]), mp.mpf(e), mp.mpf(omega)
            tasc = mp.mpf(we.t_search_mid) + mp.mpf(we.tasc_frac[it]) * P
            tp = tasc + om / Om                                                   # Eq. (10)
            u = mp.mpf(we.k_band0 + j)

            def roemer(t):                                                         # R(t)/c, Eq. (9) with Eq. (7)
                M = Om * (t - tp)
                E = mp.findroot(lambda x: x - ee * mp.sin(x) - M, M)
                return ap * (mp.sin(om) * (mp.cos(E) - ee) + mp.cos(om) * mp.sin(E) * mp.sqrt(1 - ee * ee))

            _, xd = oracle.track(we, 0, ia, ip, it, j, mode=oracle.DIRECT, with_aux=True, ie=0)
            _, xw = oracle.track(wrong, 0, ia, ip, it, j, mode=oracle.DIRECT, with_aux=True, ie=0)
            _, x0 = oracle.track(base, 0, ia, ip, it, j, mode=oracle.DIRECT, with_aux=True)
            worst = worst_wrong = 0
            for i in range(0, we.n_sft, 5):
                t = mp.mpf(we.t_mid[i])
                dR = mp.diff(roemer, t)                                            # f = f0 (1 + v.n/c - dR/dt), Eq. (13)
                circ = -ap * Om * mp.cos(Om * (t - tasc))                          # the e = 0 term the circular track has
                want_delta = u * (-dR - circ)                                      # bins the eccentricity moves the track by
                got_delta = mp.mpf(xd[i]) - mp.mpf(x0[i])
                worst = max(worst, abs(want_delta - got_delta))
                worst_wrong = max(worst_wrong, abs(want_delta - (mp.mpf(xw[i]) - mp.mpf(x0[i]))))
                assert abs(want_delta - got_delta) < 2.5 * ee * ee * ap * Om * u + mp.mpf("1e-7"), (e, omega, ia, ip, it, i)
            assert worst_wrong > 0.5 * ee * abs(mp.sin(om)) * ap * Om * u          # the other sign is an O(e) error
            # and the first-order terms are really there (a dropped or mis-signed term is O(e), not O(e^2))
            assert max(abs(xd[i] - x0[i]) for i in range(we.n_sft)) > 0.5 * e * float(ap * Om * u) * 0.5


def test_eccentric_modes_agree_and_symmetry():
    wl = synth.eccentric(synth.noise_workload(seed=5, n_sft=300, n_f0=30, margin=44, f_band_start=150.0, n_pix_side=2,
                                              ap=(10.0, 40.0), P_days=(15.0, 45.0), n_t=3), e_max=0.1)
    res = oracle.compare_modes(wl, tol=1e-9)
    assert res["compared"] == wl.n_accumulations and res["unflagged"] == 0
    assert res["flagged"] < 40 + 4e-9 * res["compared"] * 5
    # (a_p, t_asc, e cos w, e sin w) -> (-a_p, t_asc + P/2, -e cos w, -e sin w) is the same track (Eq. 14: phi -> phi - pi)
    pk = oracle.peakgram(wl.rho)
    base, _ = oracle.stage1(wl, pk, None, mode=oracle.DIRECT)
    flipped = dataclasses.replace(wl, ap=-wl.ap, tasc_frac=wl.tasc_frac + 0.5, ecosw=-wl.ecosw, esinw=-wl.esinw)
    got, _ = oracle.stage1(flipped, pk, None, mode=oracle.DIRECT)
    assert np.array_equal(base, got)
    # hoisted CANONICAL loop == per-accumulation canonical track, eccentric templates included
    bits = np.unpackbits(pk.view(np.uint8), axis=1, bitorder="little")[:, :wl.n_bins]
    cnt, _ = oracle.stage1(wl, pk, None, mode=oracle.CANONICAL)
    rows = np.arange(wl.n_sft)
    for idx in range(3, wl.n_templates, 97):
        pix, ia, ip, it, ie, j = oracle.decode_index(wl, idx)
        k = oracle.track(wl, pix, ia, ip, it, j, mode=oracle.CANONICAL, ie=ie)
        inside = (k >= 0) & (k < wl.n_bins)
        assert cnt[idx] == bits[rows[inside], k[inside]].sum()
