"""Python face of the plain-C oracle (oracle/bsh_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this package.
It never imports paper_1904_04873_b200 (the CUDA path) and the CUDA path never imports it.

Functions take a "workload" object: anything with the plain-data attributes of synth.Workload
(t_sft, t_mid, v_over_c, t_search_mid, k_slab0, n_bins, k_band0, n_f0, alpha, delta, ap, P, tasc_frac).
"""
from __future__ import annotations

import ctypes as C
import math
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "bsh_oracle.c")
_LIB = os.path.join(_HERE, "libbsh_oracle.so")

DIRECT, CANONICAL = 0, 1
RHO_TH = 1.6
P_PEAK = math.exp(-RHO_TH)                       # P(rho > rho_th) in Gaussian noise


def build(force: bool = False) -> str:
    """gcc -O2, no FMA contraction, OpenMP over templates.  (Also builds the tier-2 reference.)"""
    build_tier2(force)
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-shared", "-fPIC", "-std=c11",
               "-Wall", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True, capture_output=True)
    return _LIB


class _Problem(C.Structure):
    _fields_ = [("n_sft", C.c_int32), ("t_sft", C.c_double), ("t_mid", C.c_void_p), ("v_over_c", C.c_void_p),
                ("t_search_mid", C.c_double), ("k_slab0", C.c_int64), ("n_bins", C.c_int32), ("k_band0", C.c_int64),
                ("n_f0", C.c_int32), ("n_pix", C.c_int32), ("alpha", C.c_void_p), ("delta", C.c_void_p),
                ("n_ap", C.c_int32), ("ap", C.c_void_p), ("n_P", C.c_int32), ("P", C.c_void_p),
                ("n_tasc", C.c_int32), ("tasc_frac", C.c_void_p),
                ("n_ecc", C.c_int32), ("ecosw", C.c_void_p), ("esinw", C.c_void_p)]


_SRC2 = os.path.join(_HERE, "bsh_tier2.c")
_LIB2 = os.path.join(_HERE, "libbsh_tier2.so")
_lib2 = None


def build_tier2(force: bool = False) -> str:
    """The tier-2 CPU reference (bsh_tier2.c): gcc -O3 (integer loops vectorise), no FMA contraction, OpenMP."""
    if force or not os.path.exists(_LIB2) or os.path.getmtime(_LIB2) < os.path.getmtime(_SRC2):
        cmd = ["gcc", "-O3", "-march=native", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-shared", "-fPIC",
               "-std=c11", "-Wall", "-o", _LIB2, _SRC2, "-lm"]
        subprocess.run(cmd, check=True, capture_output=True)
    return _LIB2


def tier2_stage1(wl, peak: np.ndarray, w=None, n_threads=0, want_wcount=False):
    """Tier-2 CPU reference (SURVEY 8(c) coverage plan): counts (and FP64 weighted counts) of EVERY template of the grid,
    one track evaluation per (pixel, binary template, SFT).  Must equal stage1(..., mode=CANONICAL) bit for bit."""
    global _lib2
    if _lib2 is None:
        _lib2 = C.CDLL(build_tier2())
    pb = Problem(wl)
    peak = np.ascontiguousarray(peak, np.uint32)
    wv = None if w is None else np.ascontiguousarray(w, np.float32)
    cnt = np.zeros(pb.n_templates, np.int32)
    wc = np.zeros(pb.n_templates, np.float64) if want_wcount else None
    _lib2.t2_stage1(pb.ref, C.c_void_p(peak.ctypes.data), C.c_int32(peak.shape[1]),
                    C.c_void_p(wv.ctypes.data if wv is not None else None), C.c_void_p(cnt.ctypes.data),
                    C.c_void_p(wc.ctypes.data if wc is not None else None), C.c_int(n_threads))
    return (cnt, wc) if want_wcount else cnt


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_track_direct.restype = C.c_int64
        _lib.orc_track_canonical.restype = C.c_int64
        _lib.orc_toplist.restype = C.c_int64
        _lib.orc_max_threads.restype = C.c_int
        _lib.orc_median_bias.restype = C.c_double
        _lib.orc_distance2.restype = C.c_double
        _lib.orc_coincidences.restype = C.c_int64
        _lib.orc_cluster.restype = C.c_int32
    return _lib


def max_threads() -> int:
    return int(lib().orc_max_threads())


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


class Problem:
    """Keeps the numpy arrays alive next to the C struct that points into them."""

    def __init__(self, wl):
        self.arrays = dict(t_mid=_f64(wl.t_mid), v_over_c=_f64(wl.v_over_c), alpha=_f64(wl.alpha),
                           delta=_f64(wl.delta), ap=_f64(wl.ap), P=_f64(wl.P), tasc_frac=_f64(wl.tasc_frac))
        ecw, esw = getattr(wl, "ecosw", None), getattr(wl, "esinw", None)
        n_ecc = 0 if ecw is None else len(ecw)
        if n_ecc:
            self.arrays.update(ecosw=_f64(ecw), esinw=_f64(esw))
            assert self.arrays["ecosw"].shape == self.arrays["esinw"].shape == (n_ecc,)
        a = self.arrays
        self.c = _Problem(n_sft=a["t_mid"].shape[0], t_sft=float(wl.t_sft), t_mid=a["t_mid"].ctypes.data,
                          v_over_c=a["v_over_c"].ctypes.data, t_search_mid=float(wl.t_search_mid),
                          k_slab0=int(wl.k_slab0), n_bins=int(wl.n_bins), k_band0=int(wl.k_band0), n_f0=int(wl.n_f0),
                          n_pix=a["alpha"].shape[0], alpha=a["alpha"].ctypes.data, delta=a["delta"].ctypes.data,
                          n_ap=a["ap"].shape[0], ap=a["ap"].ctypes.data, n_P=a["P"].shape[0], P=a["P"].ctypes.data,
                          n_tasc=a["tasc_frac"].shape[0], tasc_frac=a["tasc_frac"].ctypes.data,
                          n_ecc=n_ecc, ecosw=a["ecosw"].ctypes.data if n_ecc else None,
                          esinw=a["esinw"].ctypes.data if n_ecc else None)
        self.n_sft = self.c.n_sft
        self.n_ecc = n_ecc
        self.shape = (self.c.n_pix, self.c.n_ap, self.c.n_P, self.c.n_tasc, max(1, n_ecc), self.c.n_f0)
        self.n_templates = int(np.prod([int(s) for s in self.shape]))

    @property
    def ref(self):
        return C.byref(self.c)


def words_per_row(n_bins: int) -> int:
    return (n_bins + 31) // 32


def peakgram(rho: np.ndarray, rho_th: float = RHO_TH) -> np.ndarray:
    """PAPER.md L176 -> bit-packed uint32 [N, ceil(K/32)], LSB first."""
    rho = np.ascontiguousarray(rho, np.float32)
    n, k = rho.shape
    wpr = words_per_row(k)
    out = np.zeros((n, wpr), np.uint32)
    lib().orc_peakgram(C.c_void_p(rho.ctypes.data), C.c_int32(n), C.c_int32(k), C.c_float(rho_th),
                       C.c_void_p(out.ctypes.data), C.c_int32(wpr))
    return out


def median_bias(window: int = 101) -> float:
    """E[median of `window` iid Exp(1) draws] = sum_{i=(window+1)/2}^{window} 1/i  (R-22; -> ln 2 for large windows)."""
    return float(lib().orc_median_bias(C.c_int32(window)))


def normalise(sft: np.ndarray, window: int = 101, bias=None) -> np.ndarray:
    """PAPER.md Eq. (20)-(21), L167-L174: complex64 SFT bins [N, n_raw] -> normalised powers f32 [N, n_raw - window + 1]
    (slab column k = raw bin k + (window - 1) / 2), noise estimated by the running median over `window` bins."""
    sft = np.ascontiguousarray(sft, np.complex64)
    n, n_raw = sft.shape
    assert window % 2 == 1 and 1 <= window <= n_raw
    b = np.float32(median_bias(window) if bias is None else bias)
    out = np.zeros((n, n_raw - window + 1), np.float32)
    lib().orc_normalise(C.c_void_p(sft.ctypes.data), C.c_int32(n), C.c_int32(n_raw), C.c_int32(window), C.c_float(b),
                        C.c_void_p(out.ctypes.data))
    return out


def track(wl, pix, ia, ip, it, j, mode=CANONICAL, with_aux=False, ie=0):
    """Slab column per SFT for one template (Eq. 15; Eq. 14 when the workload has eccentricity pairs, `ie` = pair index).
    aux = x (DIRECT) or y (CANONICAL), the unrounded values."""
    pb = Problem(wl)
    k = np.zeros(pb.n_sft, np.int64)
    aux = np.zeros(pb.n_sft, np.float64)
    lib().orc_track(pb.ref, C.c_int(mode), C.c_int(pix), C.c_int(ia), C.c_int(ip), C.c_int(it), C.c_int(ie), C.c_int(j),
                    C.c_void_p(k.ctypes.data), C.c_void_p(aux.ctypes.data))
    return (k, aux) if with_aux else k


def stage1(wl, peak: np.ndarray, w=None, mode=CANONICAL, n_threads=0, want_count=True, want_wcount=True):
    """All templates of the grid: (count int32 [n_templates], wcount f64 [n_templates]) in R-11 order."""
    pb = Problem(wl)
    peak = np.ascontiguousarray(peak, np.uint32)
    wv = None if w is None else np.ascontiguousarray(w, np.float32)
    cnt = np.zeros(pb.n_templates, np.int32) if want_count else None
    wc = np.zeros(pb.n_templates, np.float64) if want_wcount else None
    lib().orc_stage1(pb.ref, C.c_int(mode), C.c_void_p(peak.ctypes.data), C.c_int32(peak.shape[1]),
                     C.c_void_p(wv.ctypes.data if wv is not None else None),
                     C.c_void_p(cnt.ctypes.data if cnt is not None else None),
                     C.c_void_p(wc.ctypes.data if wc is not None else None), C.c_int(n_threads))
    return cnt, wc


def compare_modes(wl, tol=1e-9):
    pb = Problem(wl)
    out = np.zeros(4, np.int64)
    lib().orc_compare_modes(pb.ref, C.c_double(tol), C.c_void_p(out.ctypes.data))
    return dict(compared=int(out[0]), disagree=int(out[1]), unflagged=int(out[2]), flagged=int(out[3]))


def score(wl, idx, peak=None, rho=None, w=None, mode=CANONICAL, n_threads=0):
    """count / wcount / power (Eq. 26) for an explicit list of template indices."""
    pb = Problem(wl)
    idx = np.ascontiguousarray(idx, np.uint64)
    n = idx.shape[0]
    pk = None if peak is None else np.ascontiguousarray(peak, np.uint32)
    rh = None if rho is None else np.ascontiguousarray(rho, np.float32)
    wv = None if w is None else np.ascontiguousarray(w, np.float32)
    cnt = np.zeros(n, np.int32) if pk is not None else None
    wc = np.zeros(n, np.float64) if pk is not None else None
    pw = np.zeros(n, np.float64) if rh is not None else None
    p = lambda a: C.c_void_p(a.ctypes.data if a is not None else None)
    lib().orc_score(pb.ref, C.c_int(mode), p(idx), C.c_int64(n), p(pk), C.c_int32(pk.shape[1] if pk is not None else 0),
                    p(rh), p(wv), p(cnt), p(wc), p(pw), C.c_int(n_threads))
    return cnt, wc, pw


def stage2(wl, idx, rho, w=None, mode=CANONICAL, n_threads=0):
    """Eq. (26): P = sum_i w_i rho[i][k_i] for each candidate index."""
    return score(wl, idx, peak=None, rho=rho, w=w, mode=mode, n_threads=n_threads)[2]


def toplist(values, k: int) -> np.ndarray:
    """Indices of the k best by (value desc, index asc), via a full sort (R-11)."""
    v = np.ascontiguousarray(values, np.float64)
    out = np.zeros(min(k, v.shape[0]), np.uint64)
    kk = lib().orc_toplist(C.c_void_p(v.ctypes.data), C.c_int64(v.shape[0]), C.c_int64(k), C.c_void_p(out.ctypes.data))
    return out[:kk]


def decode_index(wl, idx):
    """(pix, ia, ip, it, j) for a circular grid, (pix, ia, ip, it, ie, j) when the workload has eccentricity pairs."""
    pb = Problem(wl)
    out = np.zeros(6, np.int32)
    lib().orc_decode_index(pb.ref, C.c_uint64(int(idx)), C.c_void_p(out.ctypes.data))
    t = tuple(int(x) for x in out)
    return t if pb.n_ecc else t[:4] + t[5:]


def encode_index(wl, pix, ia, ip, it, j, ie=0) -> int:
    n_ecc = 1 if getattr(wl, "ecosw", None) is None else len(wl.ecosw)
    return (((((pix * len(wl.ap) + ia) * len(wl.P) + ip) * len(wl.tasc_frac) + it) * n_ecc + ie) * wl.n_f0 + j)


# --- significances (R-10): derived from independent Bernoulli(p) / Exp(1) terms; constant within a patch -------
def significance_count(nw, w, p=P_PEAK):
    w = np.asarray(w, np.float64)
    return (np.asarray(nw, np.float64) - p * w.sum()) / math.sqrt(p * (1 - p) * (w * w).sum())


def significance_power(pw, w):
    w = np.asarray(w, np.float64)
    return (np.asarray(pw, np.float64) - w.sum()) / math.sqrt((w * w).sum())


# --- post-processing of the toplists (section V.E, Eq. 44) ---------------------------
NPAR = 6                                         # (f, x, y, a_p, Omega, t_asc), the order of Eq. (44)


def _cand(p, r, s):
    p, r, s = _f64(p), _f64(r), _f64(s)
    assert p.ndim == 2 and p.shape[1] == NPAR and r.shape == p.shape and s.shape == (p.shape[0],)
    return p, r, s


def distance2(pa, ra, pb, rb) -> float:
    """Eq. (44): squared parameter-space distance in bins, mean of the two points' resolutions (L399)."""
    pa, ra, pb, rb = (_f64(x) for x in (pa, ra, pb, rb))
    return float(lib().orc_distance2(C.c_void_p(pa.ctypes.data), C.c_void_p(ra.ctypes.data), C.c_void_p(pb.ctypes.data),
                                     C.c_void_p(rb.ctypes.data)))


def coincidences(pa, ra, sa, pb, rb, sb, window):
    """Step 1 (L387-L393): pairs closer than `window`, (a, b) order.  -> (pair_a, pair_b, centroid [n, 6], significance)."""
    pa, ra, sa = _cand(pa, ra, sa)
    pb, rb, sb = _cand(pb, rb, sb)
    cap = max(1, pa.shape[0] * pb.shape[0])
    ia, ib = np.zeros(cap, np.int32), np.zeros(cap, np.int32)
    cen, sig = np.zeros((cap, NPAR), np.float64), np.zeros(cap, np.float64)
    v = lambda a: C.c_void_p(a.ctypes.data)
    n = lib().orc_coincidences(C.c_int32(pa.shape[0]), v(pa), v(ra), v(sa), C.c_int32(pb.shape[0]), v(pb), v(rb), v(sb),
                               C.c_double(window), C.c_int64(cap), v(ia), v(ib), v(cen), v(sig))
    return ia[:n].copy(), ib[:n].copy(), cen[:n].copy(), sig[:n].copy()


def cluster(p, r, s, window, prune_window=0.0):
    """Steps 2-3 (L401-L405).  -> dict(label [n] (smallest member index, -1 pruned), root, centroid, significance,
    n_members (per cluster, increasing label), best (position of the most significant cluster or -1))."""
    p, r, s = _cand(p, r, s)
    n = p.shape[0]
    label = np.zeros(max(n, 1), np.int32)
    root, members = np.zeros(max(n, 1), np.int32), np.zeros(max(n, 1), np.int32)
    cen, sig = np.zeros((max(n, 1), NPAR), np.float64), np.zeros(max(n, 1), np.float64)
    best = C.c_int32(-1)
    v = lambda a: C.c_void_p(a.ctypes.data)
    nc = lib().orc_cluster(C.c_int32(n), v(p), v(r), v(s), C.c_double(window), C.c_double(prune_window), v(label), v(root),
                           v(cen), v(sig), v(members), C.byref(best))
    return dict(label=label[:n].copy(), root=root[:nc].copy(), centroid=cen[:nc].copy(), significance=sig[:nc].copy(),
                n_members=members[:nc].copy(), best=int(best.value))
