"""Seeded synthetic inputs for the BinarySkyHough hot path (shared by oracle tests, GPU tests and bench.py).

This module holds NONE of the method's arithmetic (no track, no peakgram, no count, no power sum): it only
draws the inputs -- SFT times, detector velocities, normalised powers, weights, sky pixels and the template
grid axes -- with the shapes and distributions of the paper's workloads.  The five configurations are the ones
BASELINE.json lists; every choice the configs leave open is a DESIGN.md reading (R-numbers quoted below).

Stand-in statement: the paper searches LIGO O1 H1+L1 SFTs; that data is not available, so
exponential powers (p(rho) = exp(-rho) in Gaussian noise) and an analytic detector-velocity
model stand in for it.

All randomness comes from numpy's counter-based Philox generator keyed by the config seed.
"""
from __future__ import annotations

import dataclasses
import math
from typing import List, Optional

import numpy as np

C_LIGHT = 299_792_458.0          # m/s
V_ORB = 29.8e3                   # m/s  (BASELINE.json config 1: "circular 1 AU orbit at 29.8 km/s")
YEAR_S = 365.25 * 86400.0
OBLIQUITY = math.radians(23.4393)
R_EARTH = 6_378_137.0            # m
T_SIDEREAL = 23.934 * 3600.0     # s   (config 1: "sidereal rotation 23.934 h")
DAY = 86400.0


@dataclasses.dataclass
class Workload:
    """One (SFT set, sky patch, template grid) problem instance.  Plain data only."""
    name: str
    seed: int
    t_sft: float                 # T, seconds
    t_mid: np.ndarray            # [N] f64, SFT mid-times relative to t_ref = first SFT start (R-2)
    v_over_c: np.ndarray         # [N,3] f64, detector velocity / c, equatorial frame
    t_search_mid: float          # mid-time of the search, same origin as t_mid (Eq. 35)
    k_slab0: int                 # absolute bin index of slab column 0
    n_bins: int                  # K
    k_band0: int                 # absolute bin index of f0 lattice point j = 0
    n_f0: int
    rho: Optional[np.ndarray]    # [N,K] f32 normalised powers (None when supplied separately, config 4/5)
    w: np.ndarray                # [N] f32 weights, sum ~ N
    alpha: np.ndarray            # [n_pix] f64 right ascension, rad
    delta: np.ndarray            # [n_pix] f64 declination, rad
    ap: np.ndarray               # [n_a] f64 projected semi-major axis, light-seconds
    P: np.ndarray                # [n_P] f64 orbital period, seconds
    tasc_frac: np.ndarray        # [n_t] f64 in [-0.5, 0.5): t_asc = t_search_mid + frac * P   (Eq. 35)
    topk: int
    rho_th: float = 1.6
    ecosw: Optional[np.ndarray] = None   # [n_ecc] f64 e cos(omega), Eq. (14); None = circular orbits
    esinw: Optional[np.ndarray] = None   # [n_ecc] f64 e sin(omega)

    @property
    def n_sft(self) -> int:
        return int(self.t_mid.shape[0])

    @property
    def n_pix(self) -> int:
        return int(self.alpha.shape[0])

    @property
    def margin(self) -> int:
        return int(self.k_band0 - self.k_slab0)

    @property
    def n_ecc(self) -> int:
        return 0 if self.ecosw is None else int(len(self.ecosw))

    @property
    def n_binary(self) -> int:
        return len(self.ap) * len(self.P) * len(self.tasc_frac) * max(1, self.n_ecc)

    @property
    def n_templates(self) -> int:
        return self.n_pix * self.n_binary * self.n_f0

    @property
    def n_accumulations(self) -> int:
        return self.n_templates * self.n_sft

    def subgrid(self, ia=None, ip=None, it=None, pix=None, name_suffix="sub") -> "Workload":
        """Same data, a sub-selection of the grid axes (index arrays); used to make oracle-sized cases."""
        sel = lambda a, ix: a if ix is None else np.ascontiguousarray(a[np.asarray(ix)])
        return dataclasses.replace(
            self, name=f"{self.name}-{name_suffix}",
            ap=sel(self.ap, ia), P=sel(self.P, ip), tasc_frac=sel(self.tasc_frac, it),
            alpha=sel(self.alpha, pix), delta=sel(self.delta, pix))


def _rng(seed: int, stream: int = 0) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(key=[seed, stream]))


def detector_velocity_over_c(t_abs: np.ndarray, lat_deg: float = 30.6, theta0: float = 0.0) -> np.ndarray:
    """Analytic v_det/c (R-19): circular 1 AU orbit + sidereal rotation, equatorial frame.  t_abs in seconds."""
    lam = 2.0 * math.pi * t_abs / YEAR_S
    v_orb = V_ORB * np.stack([-np.sin(lam), np.cos(lam) * math.cos(OBLIQUITY), np.cos(lam) * math.sin(OBLIQUITY)], -1)
    th = theta0 + 2.0 * math.pi * t_abs / T_SIDEREAL
    vr = 2.0 * math.pi * R_EARTH * math.cos(math.radians(lat_deg)) / T_SIDEREAL
    v_rot = vr * np.stack([-np.sin(th), np.cos(th), np.zeros_like(th)], -1)
    return np.ascontiguousarray((v_orb + v_rot) / C_LIGHT, dtype=np.float64)


def slab_margin(f_max_bin: int, v_over_c: np.ndarray, ap_max: float, P_min: float) -> int:
    """Harness rule for configs that say only 'plus margin' (R-6): a bound on the track excursion, in bins.
    This is slab sizing (how many columns to load), not a track evaluation."""
    vmax = float(np.sqrt((v_over_c ** 2).sum(-1)).max())
    return int(math.ceil(f_max_bin * (vmax + ap_max * 2.0 * math.pi / P_min))) + 1


def pixel_size(t_sft: float, f: float, pixel_factor: float) -> float:
    """Sky resolution delta-Theta = c / (v T f P_F), Eq. 34 (L289); only used to size synthetic pixels."""
    return C_LIGHT / (V_ORB * t_sft * f * pixel_factor)


def patch_pixels(alpha0: float, delta0: float, dtheta: float, nx: int = 8, ny: int = 8):
    ix, iy = np.meshgrid(np.arange(nx), np.arange(ny), indexing="xy")
    alpha = alpha0 + (ix.ravel() - (nx - 1) / 2.0) * dtheta / max(math.cos(delta0), 0.05)
    delta = delta0 + (iy.ravel() - (ny - 1) / 2.0) * dtheta
    delta = np.clip(delta, -math.pi / 2, math.pi / 2)
    return np.ascontiguousarray(alpha, np.float64), np.ascontiguousarray(delta, np.float64)


def exp_powers(rng: np.random.Generator, n_sft: int, n_bins: int) -> np.ndarray:
    return np.ascontiguousarray(rng.standard_exponential((n_sft, n_bins), dtype=np.float32))


def lognormal_weights(rng: np.random.Generator, n_sft: int, sigma: float = 0.3) -> np.ndarray:
    s_n = np.exp(sigma * rng.standard_normal(n_sft))
    w = 1.0 / s_n
    w *= n_sft / w.sum()
    return np.ascontiguousarray(w, np.float32)


def tasc_fractions(n_t: int) -> np.ndarray:
    """R-13: frac_q = -1/2 + q/n_t, the half-open range of Eq. 35."""
    return -0.5 + np.arange(n_t, dtype=np.float64) / n_t


def _finish(name, seed, t_sft, starts, v_over_c, f_band_start, bandwidth, margin, rho, w, alpha, delta, ap, P,
            tasc_frac, topk) -> Workload:
    t_ref = float(starts.min())
    t_mid = np.ascontiguousarray(starts - t_ref + 0.5 * t_sft, np.float64)
    t_search_mid = 0.5 * ((float(starts.min()) - t_ref) + (float(starts.max()) + t_sft - t_ref))
    k_band0 = int(round(f_band_start * t_sft))
    assert abs(k_band0 - f_band_start * t_sft) < 1e-6, "band edge must sit on the 1/T lattice (R-3)"
    n_f0 = int(round(bandwidth * t_sft))
    return Workload(name=name, seed=seed, t_sft=t_sft, t_mid=t_mid, v_over_c=v_over_c, t_search_mid=t_search_mid,
                    k_slab0=k_band0 - margin, n_bins=n_f0 + 2 * margin, k_band0=k_band0, n_f0=n_f0, rho=rho, w=w,
                    alpha=alpha, delta=delta, ap=np.ascontiguousarray(ap, np.float64),
                    P=np.ascontiguousarray(P, np.float64), tasc_frac=np.ascontiguousarray(tasc_frac, np.float64),
                    topk=topk)


# ----------------------------------------------------------------------------------------------------------------
# Config 1: tiny, one sky pixel
# ----------------------------------------------------------------------------------------------------------------
def config1(seed: int = 0, pixel: str = "ecliptic") -> Workload:
    """BASELINE.json configs[0].  pixel='ecliptic' puts the pixel where Earth's Doppler shift is largest so that
    some tracks leave the 9-bin margin (exercises R-6); pixel='pole' keeps every track inside."""
    n, t_sft = 64, 900.0
    starts = np.arange(n, dtype=np.float64) * (10.0 * DAY / n)
    v = detector_velocity_over_c(starts + 0.5 * t_sft)
    rng = _rng(seed)
    margin = 9                                       # "plus a 0.01 Hz Doppler margin" = 0.01 * 900
    n_f0 = 45
    rho = exp_powers(rng, n, n_f0 + 2 * margin)
    w = rng.uniform(0.5, 1.5, n)
    w *= n / w.sum()
    if pixel == "ecliptic":
        # along -v_orb(t=0)-ish direction in the ecliptic plane: alpha = 90 deg, delta = +23.44 deg
        alpha, delta = np.array([math.pi / 2]), np.array([OBLIQUITY])
    else:
        # north ecliptic pole: alpha = 270 deg, delta = 66.56 deg
        alpha, delta = np.array([1.5 * math.pi]), np.array([math.pi / 2 - OBLIQUITY])
    return _finish(f"config1-{pixel}", seed, t_sft, starts, v, 100.0, 0.05, margin, rho,
                   np.ascontiguousarray(w, np.float32), alpha, delta,
                   ap=[10.0, 12.0, 14.0], P=np.array([15.0, 16.0, 17.0]) * DAY,
                   tasc_frac=np.array([-0.5, -0.25, 0.0, 0.25]), topk=10)


# ----------------------------------------------------------------------------------------------------------------
# Config 2: single sky patch, noise only  (the bench workload)
# ----------------------------------------------------------------------------------------------------------------
def _binary_grid_c2():
    return np.linspace(10.0, 40.0, 20), np.linspace(15.0, 45.0, 30) * DAY, tasc_fractions(40)


def config2(seed: int = 2) -> Workload:
    """BASELINE.json configs[1]."""
    n, t_sft = 2000, 900.0
    starts = np.arange(n, dtype=np.float64) * (60.0 * DAY / n)
    v = detector_velocity_over_c(starts + 0.5 * t_sft)
    ap, P, tf = _binary_grid_c2()
    f0, bw = 150.0, 0.1
    margin = slab_margin(int(round((f0 + bw) * t_sft)), v, ap.max(), P.min())
    rng = _rng(seed)
    n_f0 = int(round(bw * t_sft))
    rho = exp_powers(rng, n, n_f0 + 2 * margin)
    w = lognormal_weights(rng, n)
    a0, d0 = rng.uniform(0, 2 * math.pi), math.asin(rng.uniform(-0.8, 0.8))
    alpha, delta = patch_pixels(a0, d0, pixel_size(t_sft, f0, 1.0))
    return _finish("config2", seed, t_sft, starts, v, f0, bw, margin, rho, w, alpha, delta, ap, P, tf, topk=1000)


# ----------------------------------------------------------------------------------------------------------------
# Config 3: full-size search patch (two detectors x 4000 SFTs with gaps, weighted)
# ----------------------------------------------------------------------------------------------------------------
def _two_detector_times(rng, n_per_det=4000, n_slots=5714, span_days=270.0, t_sft=900.0):
    spacing = span_days * DAY / n_slots
    starts, vel = [], []
    for lat, th0 in ((30.6, 0.0), (46.5, -0.5)):
        keep = np.sort(rng.choice(n_slots, size=n_per_det, replace=False))
        s = keep.astype(np.float64) * spacing
        starts.append(s)
        vel.append(detector_velocity_over_c(s + 0.5 * t_sft, lat, th0))
    return np.concatenate(starts), np.concatenate(vel)


def config3(seed: int = 3) -> Workload:
    """BASELINE.json configs[2]."""
    t_sft = 900.0
    rng = _rng(seed)
    starts, v = _two_detector_times(rng, t_sft=t_sft)
    n = starts.shape[0]
    ap, P, tf = np.linspace(10.0, 40.0, 40), np.linspace(15.0, 45.0, 60) * DAY, tasc_fractions(120)
    f0, bw = 200.0, 0.1
    margin = slab_margin(int(round((f0 + bw) * t_sft)), v, ap.max(), P.min())
    n_f0 = int(round(bw * t_sft))
    rho = exp_powers(rng, n, n_f0 + 2 * margin)
    w = lognormal_weights(rng, n)
    a0, d0 = rng.uniform(0, 2 * math.pi), math.asin(rng.uniform(-0.8, 0.8))
    alpha, delta = patch_pixels(a0, d0, pixel_size(t_sft, f0, 1.0))
    return _finish("config3", seed, t_sft, starts, v, f0, bw, margin, rho, w, alpha, delta, ap, P, tf, topk=1000)


# ----------------------------------------------------------------------------------------------------------------
# Config 4: signal recovery.  The generator draws noise bins and injection PARAMETERS; the bins the injected
# tracks land in are supplied by the caller (tests get them from the oracle) -- no track arithmetic here.
# ----------------------------------------------------------------------------------------------------------------
@dataclasses.dataclass
class Injection:
    patch: int
    pix: int
    ia: int
    ip: int
    it: int
    j: int
    phases: np.ndarray           # [N] seeded uniform phases of the deposited amplitude


@dataclasses.dataclass
class Config4:
    base: Workload               # rho=None, alpha/delta of patch 0
    re: np.ndarray               # [N,K] f64 noise, variance 1/2
    im: np.ndarray
    patches: List[tuple]         # (alpha[64], delta[64]) per patch
    injections: List[Injection]
    amp2: float = 0.3

    def patch_workload(self, ipatch: int, rho: np.ndarray) -> Workload:
        a, d = self.patches[ipatch]
        return dataclasses.replace(self.base, name=f"config4-patch{ipatch}", alpha=a, delta=d, rho=rho)

    def deposit(self, bins_per_injection: List[np.ndarray]) -> np.ndarray:
        """rho = |x|^2 after adding A*exp(i*phi_i) to bin bins[inj][i] of SFT i (R-17); bins < 0 or >= K skip."""
        re, im = self.deposit_bins(bins_per_injection)
        return np.ascontiguousarray(re * re + im * im, np.float32)

    def raw_bins(self, bins_per_injection: List[np.ndarray], window: int = 101, noise_sigma: float = 1.0) -> np.ndarray:
        """Complex SFT bins as the front end takes them (Eq. 19-20): the K slab bins of deposit_bins()
        plus (window - 1) / 2 wing bins of fresh noise on each side, every SFT scaled by a seeded log-normal noise
        amplitude sqrt(S_J) (a non-stationary detector) and by a gentle slope across the band (a coloured spectrum) --
        what the running-median normalisation has to take out again.  complex64 [N, K + window - 1]."""
        re, im = self.deposit_bins(bins_per_injection)
        n, k = re.shape
        h = (window - 1) // 2
        rng = _rng(self.base.seed, 4242)
        wing = rng.standard_normal((n, 2, h, 2)) * math.sqrt(0.5)
        x = np.empty((n, k + 2 * h), np.complex128)
        x[:, h:h + k] = re + 1j * im
        x[:, :h] = wing[:, 0, :, 0] + 1j * wing[:, 0, :, 1]
        x[:, h + k:] = wing[:, 1, :, 0] + 1j * wing[:, 1, :, 1]
        amp = np.exp(0.5 * noise_sigma * rng.standard_normal(n))[:, None]
        slope = 1.0 + 0.2 * (np.arange(k + 2 * h)[None, :] / (k + 2 * h) - 0.5)
        return np.ascontiguousarray(x * amp * np.sqrt(slope), np.complex64)

    def deposit_bins(self, bins_per_injection: List[np.ndarray]):
        """(re, im) [N, K] f64 after adding A*exp(i*phi_i) to bin bins[inj][i] of SFT i (R-17); bins outside the slab skip."""
        re, im = self.re.copy(), self.im.copy()
        amp = math.sqrt(self.amp2)
        n, k = re.shape
        rows = np.arange(n)
        for inj, bins in zip(self.injections, bins_per_injection):
            bins = np.asarray(bins)
            ok = (bins >= 0) & (bins < k)
            re[rows[ok], bins[ok]] += amp * np.cos(inj.phases[ok])
            im[rows[ok], bins[ok]] += amp * np.sin(inj.phases[ok])
        return re, im


def config4(seed: int = 4, n_patches: int = 10) -> Config4:
    """BASELINE.json configs[3]."""
    n, t_sft = 6000, 600.0
    starts = np.arange(n, dtype=np.float64) * (180.0 * DAY / n)
    v = detector_velocity_over_c(starts + 0.5 * t_sft)
    ap, P, tf = _binary_grid_c2()
    f0, bw = 400.0, 0.1
    margin = slab_margin(int(round((f0 + bw) * t_sft)), v, ap.max(), P.min())
    n_f0 = int(round(bw * t_sft))
    k = n_f0 + 2 * margin
    rng = _rng(seed)
    re = rng.standard_normal((n, k)) * math.sqrt(0.5)
    im = rng.standard_normal((n, k)) * math.sqrt(0.5)
    dth = pixel_size(t_sft, f0, 1.0)
    patches, injections = [], []
    for ipatch in range(n_patches):
        a0, d0 = rng.uniform(0, 2 * math.pi), math.asin(rng.uniform(-0.8, 0.8))
        patches.append(patch_pixels(a0, d0, dth))
        injections.append(Injection(patch=ipatch, pix=int(rng.integers(64)), ia=int(rng.integers(len(ap))),
                                    ip=int(rng.integers(len(P))), it=int(rng.integers(len(tf))),
                                    j=int(rng.integers(n_f0)), phases=rng.uniform(0, 2 * math.pi, n)))
    w = np.ones(n, np.float32)
    base = _finish("config4", seed, t_sft, starts, v, f0, bw, margin, None, w, patches[0][0], patches[0][1],
                   ap, P, tf, topk=1000)
    return Config4(base=base, re=re, im=im, patches=patches, injections=injections)


# ----------------------------------------------------------------------------------------------------------------
# Config 5: batched multi-patch sweep, one shared spectrogram, per-patch pixels and weights
# ----------------------------------------------------------------------------------------------------------------
@dataclasses.dataclass
class Config5:
    base: Workload               # rho shared by all patches
    centres: np.ndarray          # [n_patches, 2] (alpha0, delta0)
    dtheta: float

    @property
    def n_patches(self) -> int:
        return int(self.centres.shape[0])

    def patch_workload(self, ipatch: int) -> Workload:
        a0, d0 = self.centres[ipatch]
        alpha, delta = patch_pixels(float(a0), float(d0), self.dtheta)
        w = lognormal_weights(_rng(self.base.seed, 1000 + ipatch), self.base.n_sft)
        return dataclasses.replace(self.base, name=f"config5-patch{ipatch}", alpha=alpha, delta=delta, w=w)


def config5(seed: int = 5, n_side: int = 16) -> Config5:
    """BASELINE.json configs[4]."""
    t_sft = 900.0
    rng = _rng(seed)
    starts, v = _two_detector_times(rng, t_sft=t_sft)
    n = starts.shape[0]
    ap, P, tf = _binary_grid_c2()
    f0, bw = 300.0, 0.1
    margin = slab_margin(int(round((f0 + bw) * t_sft)), v, ap.max(), P.min())
    n_f0 = int(round(bw * t_sft))
    rho = exp_powers(rng, n, n_f0 + 2 * margin)
    ia, idl = np.meshgrid(np.arange(n_side), np.arange(n_side), indexing="ij")
    centres = np.stack([2 * math.pi * (ia.ravel() + 0.5) / n_side, np.arcsin((idl.ravel() + 0.5) / n_side)], -1)
    dth = pixel_size(t_sft, f0, 2.0)
    alpha, delta = patch_pixels(float(centres[0, 0]), float(centres[0, 1]), dth)
    base = _finish("config5", seed, t_sft, starts, v, f0, bw, margin, rho, lognormal_weights(_rng(seed, 1000), n),
                   alpha, delta, ap, P, tf, topk=1000)
    return Config5(base=base, centres=centres, dtheta=dth)


def noise_workload(seed: int, n_sft: int, n_f0: int, margin: int, f_band_start: float, t_sft: float = 900.0,
                   span_days: float = 30.0, n_pix_side: int = 2, ap=(10.0, 20.0), P_days=(15.0, 20.0), n_t: int = 4,
                   topk: int = 16, weights: str = "lognormal") -> Workload:
    """Free-form small noise workload for edge-case tests (ragged sizes, tiny grids)."""
    starts = np.arange(n_sft, dtype=np.float64) * (span_days * DAY / max(n_sft, 1))
    v = detector_velocity_over_c(starts + 0.5 * t_sft)
    rng = _rng(seed)
    rho = exp_powers(rng, n_sft, n_f0 + 2 * margin)
    w = lognormal_weights(rng, n_sft) if weights == "lognormal" else np.ones(n_sft, np.float32)
    a0, d0 = rng.uniform(0, 2 * math.pi), math.asin(rng.uniform(-0.8, 0.8))
    alpha, delta = patch_pixels(a0, d0, pixel_size(t_sft, f_band_start, 1.0), n_pix_side, n_pix_side)
    return _finish(f"noise-{seed}", seed, t_sft, starts, v, f_band_start, n_f0 / t_sft, margin, rho, w, alpha, delta,
                   np.asarray(ap, np.float64), np.asarray(P_days, np.float64) * DAY, tasc_fractions(n_t), topk)


def raw_sft_bins(seed: int, n_sft: int, n_raw: int, noise_sigma: float = 2.0) -> np.ndarray:
    """Noise-only complex SFT bins for the front end (Eq. 19-21): unit complex Gaussian bins times a seeded
    log-normal per-SFT amplitude (orders of magnitude apart) and a slope across the band.  complex64 [N, n_raw]."""
    rng = _rng(seed, 4243)
    x = (rng.standard_normal((n_sft, n_raw)) + 1j * rng.standard_normal((n_sft, n_raw))) * math.sqrt(0.5)
    amp = np.exp(0.5 * noise_sigma * rng.standard_normal(n_sft))[:, None]
    slope = 1.0 + 0.3 * (np.arange(n_raw)[None, :] / max(n_raw, 1) - 0.5)
    return np.ascontiguousarray(x * amp * np.sqrt(slope), np.complex64)


def widened(wl: Workload, extra: int) -> Workload:
    """The same workload on a slab with `extra` more margin columns on each side (fresh Exp(1) powers): room for the larger
    excursion of eccentric tracks (a_p Omega e more bins), so that no track leaves the slab."""
    n_bins = wl.n_bins + 2 * extra
    return dataclasses.replace(wl, name=f"{wl.name}-wide{extra}", k_slab0=wl.k_slab0 - extra, n_bins=n_bins,
                               rho=exp_powers(_rng(wl.seed, 5500 + extra), wl.n_sft, n_bins))


def eccentric(wl: Workload, e_max: float = 0.05, n_e: int = 2, n_omega: int = 3) -> Workload:
    """The same workload with an eccentricity axis (Eq. 14, the ELL1 model for e << 1): pairs
    (e cos omega, e sin omega) on n_e rings e = e_max m / n_e (m = 1..n_e) x n_omega arguments of periapsis, plus the
    circular pair (0, 0) first.  Fig. 2 of the paper: most binary pulsars have e < 0.01; e_max = 0.05 keeps e << 1."""
    ks, hs = [0.0], [0.0]
    for m in range(1, n_e + 1):
        for q in range(n_omega):
            om = 2.0 * math.pi * (q + 0.25 * m) / n_omega
            ks.append(e_max * m / n_e * math.cos(om))
            hs.append(e_max * m / n_e * math.sin(om))
    return dataclasses.replace(wl, name=wl.name + "-ecc", ecosw=np.asarray(ks, np.float64), esinw=np.asarray(hs, np.float64))


def tie_workload() -> Workload:
    """Inputs whose bin coordinate y = u_j g lands EXACTLY on half-integers at j = 0 (R-1 pins the tie rule):
    k_band0 = 2^17, one pixel at alpha = delta = 0 (n = (1, 0, 0) exactly), a_p = 0 (no binary term), and detector
    velocities v_x / c = q 2^-18 for q = 1, 3, 5, -1, -3, 2, 0, 7, so that y = q / 2 at j = 0.  Powers alternate between
    a peak on the even slab columns and none on the odd ones: a bin that is off by one changes the count."""
    q = np.array([1, 3, 5, -1, -3, 2, 0, 7], np.float64)
    n, t_sft, margin, n_f0 = len(q), 900.0, 8, 4
    v = np.zeros((n, 3), np.float64)
    v[:, 0] = q * 2.0 ** -18
    starts = np.arange(n, dtype=np.float64) * 1800.0
    rho = np.where(np.arange(n_f0 + 2 * margin)[None, :] % 2 == 0, 2.0, 0.5).astype(np.float32).repeat(n, axis=0)
    k_band0 = 1 << 17
    t_mid = starts + 0.5 * t_sft
    return Workload(name="ties", seed=0, t_sft=t_sft, t_mid=t_mid, v_over_c=v,
                    t_search_mid=0.5 * (starts[0] + starts[-1] + t_sft), k_slab0=k_band0 - margin,
                    n_bins=n_f0 + 2 * margin, k_band0=k_band0, n_f0=n_f0, rho=np.ascontiguousarray(rho),
                    w=np.ones(n, np.float32), alpha=np.zeros(1), delta=np.zeros(1), ap=np.zeros(1),
                    P=np.array([15.0 * DAY]), tasc_frac=np.zeros(1), topk=4)


def overlapped_stage2_set(wl: Workload, seed: int = 0, lat_deg: float = 30.6, theta0: float = 0.0) -> Workload:
    """Stage-2 SFT set of PAPER.md L233: the stage-1 SFTs plus a second set whose start times are shifted by T_sft / 2
    (N-bar ~ 2 N in Table I).  Same template grid, same time origin and the SAME t_search_mid as `wl` (the templates
    -- their t_asc -- must not move); fresh Exp(1) powers and log-normal weights for the 2 N rows.  Single-detector
    velocity model (the test workloads it is used with are single-detector)."""
    t1 = np.asarray(wl.t_mid, np.float64)
    t2 = np.sort(np.concatenate([t1, t1 + 0.5 * wl.t_sft]))
    rng = _rng(seed, 77)
    n2 = t2.shape[0]
    # t_mid is relative to the first SFT start; the velocity model wants absolute mid-times with the same origin
    v2 = detector_velocity_over_c(t2, lat_deg, theta0)
    return dataclasses.replace(wl, name=wl.name + "-stage2", t_mid=np.ascontiguousarray(t2), v_over_c=v2,
                               rho=exp_powers(rng, n2, wl.n_bins), w=lognormal_weights(rng, n2))


# ----------------------------------------------------------------------------------------------------------------
# Candidate lists for the post-processing (section V.E): toplist entries as points of parameter space with
# the resolutions of Eq. 30-33 at each point.  Inputs only: no distance, no clustering here.
# ----------------------------------------------------------------------------------------------------------------
@dataclasses.dataclass
class Candidates:
    param: np.ndarray            # [n, 6] f64: f [Hz], x, y (ecliptic plane), a_p [s], Omega [rad/s], t_asc [s]
    res: np.ndarray              # [n, 6] f64: delta f, delta theta, delta theta, delta a_p, delta Omega, delta t_asc
    sig: np.ndarray              # [n] f64 significance
    truth: np.ndarray            # [n] int: index of the planted group the candidate was drawn around, -1 = background

    @property
    def n(self) -> int:
        return int(self.param.shape[0])


def resolutions(f, ap, Om, t_sft=900.0, t_obs=60 * DAY, m_a=0.4, m_om=0.4, m_t=0.4, pixel_factor=1.0) -> np.ndarray:
    """Eq. 30-33 (L270-L290) at the given points: [.., 6] = (1/T, dTheta, dTheta, d a_p, d Omega, d t_asc)."""
    f, ap, Om = (np.asarray(v, np.float64) for v in (f, ap, Om))
    dth = C_LIGHT / (V_ORB * t_sft * f * pixel_factor)
    da = math.sqrt(6 * m_a) / (math.pi * t_sft * f * Om)
    dom = math.sqrt(72 * m_om) / (math.pi * t_sft * f * ap * Om * t_obs)
    dt = math.sqrt(6 * m_t) / (math.pi * t_sft * f * ap * Om ** 2)
    return np.stack([np.full_like(f, 1.0 / t_sft), dth, dth, da, dom, dt], -1)


def candidate_list(seed: int, n_background: int = 300, groups=((12, 0.8), (7, 0.8), (20, 1.5)), f_band=(150.0, 150.1),
                   chain: int = 0) -> Candidates:
    """A toplist-like set of points: `n_background` isolated candidates spread over the band / patch / binary ranges of
    config 2, plus planted groups (n_members, spread in bins) scattered around seeded centres (what a signal or a line
    leaves in a toplist), plus optionally a `chain` of points 0.9 bins apart (a cluster held together by single links).
    Significances: exponential background, louder group members."""
    rng = _rng(seed, 909)
    lo = np.array([f_band[0], -0.02, -0.02, 10.0, 2 * math.pi / (45 * DAY), 0.0])
    hi = np.array([f_band[1], 0.02, 0.02, 40.0, 2 * math.pi / (15 * DAY), 15 * DAY])
    pts = [lo + (hi - lo) * rng.random((n_background, 6))]
    truth = [np.full(n_background, -1)]
    sig = [5.0 + rng.standard_exponential(n_background)]
    for g, (members, spread) in enumerate(groups):
        c = lo + (hi - lo) * (0.2 + 0.6 * rng.random(6))
        r = resolutions(c[0], c[3], c[4])
        pts.append(c + spread / math.sqrt(6.0) * r * rng.standard_normal((members, 6)))
        truth.append(np.full(members, g))
        sig.append(8.0 + 4.0 * rng.random(members))
    if chain:
        c = lo + (hi - lo) * 0.5
        r = resolutions(c[0], c[3], c[4])
        step = np.zeros(6)
        step[0] = 0.9 * r[0]
        pts.append(c + np.arange(chain)[:, None] * step)
        truth.append(np.full(chain, len(groups)))
        sig.append(6.0 + rng.random(chain))
    param = np.concatenate(pts)
    order = rng.permutation(param.shape[0])
    param = np.ascontiguousarray(param[order])
    return Candidates(param=param, res=np.ascontiguousarray(resolutions(param[:, 0], param[:, 3], param[:, 4])),
                      sig=np.ascontiguousarray(np.concatenate(sig)[order]), truth=np.concatenate(truth)[order])
