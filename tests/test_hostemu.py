"""GPU-less check of the kernels' per-thread logic: tests/hostemu/hostemu.cpp runs the code of csrc/bsh_core.cuh and
csrc/bsh_host.hpp (the same headers the CUDA kernels compile) with plain loops instead of the grid, and must reproduce
the oracle's CANONICAL counts bit for bit.  This is host-logic coverage; the parity tests proper are the -m gpu ones."""
import ctypes as C
import os
import subprocess

import numpy as np
import pytest

import oracle
import synth

HERE = os.path.join(os.path.dirname(os.path.abspath(__file__)), "hostemu")


@pytest.fixture(scope="module")
def emu():
    src, lib = os.path.join(HERE, "hostemu.cpp"), os.path.join(HERE, "libhostemu.so")
    deps = [src] + [os.path.join(HERE, "..", "..", "paper_1904_04873_b200", "csrc", f) for f in ("bsh_core.cuh", "bsh_host.hpp")]
    if not os.path.exists(lib) or any(os.path.getmtime(d) > os.path.getmtime(lib) for d in deps):
        subprocess.run(["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-shared", "-fPIC", "-Wno-unknown-pragmas",
                        "-o", lib, src], check=True)
    return C.CDLL(lib)


def run_emu(emu, wl, peak, weighted=False, force_clamp=False, nw=0, pix=False):
    f64 = lambda a: np.ascontiguousarray(a, np.float64)
    arrs = [f64(wl.t_mid), f64(wl.v_over_c), f64(wl.alpha), f64(wl.delta), f64(wl.ap), f64(wl.P), f64(wl.tasc_frac)]
    t_mid, v, alpha, delta, ap, P, tf = arrs
    peak = np.ascontiguousarray(peak, np.uint32)
    w = np.ascontiguousarray(wl.w, np.float32)
    counts = np.zeros(wl.n_templates, np.int32)
    wcounts = np.zeros(wl.n_templates, np.float32)
    info = np.zeros(4, np.int32)
    p = lambda a: C.c_void_p(a.ctypes.data)
    rc = emu.emu_stage1(C.c_int(wl.n_sft), p(t_mid), p(v), C.c_double(wl.t_search_mid), C.c_int64(wl.k_slab0),
                        C.c_int(wl.n_bins), C.c_int64(wl.k_band0), C.c_int(wl.n_f0), C.c_int(wl.n_pix), p(alpha), p(delta),
                        C.c_int(len(ap)), p(ap), C.c_int(len(P)), p(P), C.c_int(len(tf)), p(tf), p(peak),
                        C.c_int(peak.shape[1]), p(w), C.c_int(2 if pix else int(weighted)), C.c_int(int(force_clamp)), C.c_int(nw),
                        p(counts), p(wcounts), p(info))
    assert rc == 0
    return counts, wcounts, info


@pytest.mark.parametrize("pixel,force_clamp,nw", [("ecliptic", False, 0), ("pole", False, 0), ("pole", True, 0),
                                                  ("ecliptic", False, 1), ("pole", False, 1), ("ecliptic", False, 3)])
def test_emulated_kernel_logic_matches_oracle_config1(emu, pixel, force_clamp, nw):
    wl = synth.config1(pixel=pixel)
    pk = oracle.peakgram(wl.rho)
    want, want_w = oracle.stage1(wl, pk, wl.w, mode=oracle.CANONICAL)
    got, _, info = run_emu(emu, wl, pk, force_clamp=force_clamp, nw=nw)
    got_pix, _, _ = run_emu(emu, wl, pk, force_clamp=force_clamp, nw=nw, pix=True)
    assert np.array_equal(got_pix, want)
    if pixel == "ecliptic":
        assert info[0] == 1, "tracks leave the slab here: the clamped table must be chosen"
    assert np.array_equal(got, want)
    _, got_w, _ = run_emu(emu, wl, pk, weighted=True, force_clamp=force_clamp, nw=nw)
    assert np.allclose(got_w, want_w, rtol=1e-5, atol=0)


@pytest.mark.parametrize("n_sft,n_f0,margin,f0", [(1, 1, 3, 50.0), (33, 7, 12, 80.0), (64, 90, 30, 120.0),
                                                   (200, 96, 45, 150.0), (130, 97, 45, 150.0), (70, 200, 60, 200.0)])
def test_emulated_kernel_logic_ragged_sizes_and_breaks(emu, n_sft, n_f0, margin, f0):
    wl = synth.noise_workload(seed=n_sft + n_f0, n_sft=n_sft, n_f0=n_f0, margin=margin, f_band_start=f0, n_pix_side=2,
                              ap=(10.0, 40.0), P_days=(15.0, 31.0), n_t=3)
    pk = oracle.peakgram(wl.rho)
    want, want_w = oracle.stage1(wl, pk, wl.w, mode=oracle.CANONICAL)
    for force_clamp in (False, True):
        got, _, info = run_emu(emu, wl, pk, force_clamp=force_clamp)
        assert np.array_equal(got, want), (force_clamp, info)
        got, _, info = run_emu(emu, wl, pk, force_clamp=force_clamp, pix=True)      # position table + lean fix-ups
        assert np.array_equal(got, want), ("pix", force_clamp, info)
        _, got_w, _ = run_emu(emu, wl, pk, weighted=True, force_clamp=force_clamp)
        assert np.allclose(got_w, want_w, rtol=1e-5, atol=1e-6)


def test_emulated_kernel_logic_multiple_breaks_per_band(emu):
    """Unphysically large a_p Omega: the rounded shift changes by more than one bin across the f0 band, which takes the
    per-bin fallback of break_window(); tracks also leave the slab (clamped table)."""
    wl = synth.noise_workload(seed=77, n_sft=96, n_f0=90, margin=40, f_band_start=150.0, n_pix_side=1,
                              ap=(2500.0, 6000.0), P_days=(15.0,), n_t=4)
    pk = oracle.peakgram(wl.rho)
    want, want_w = oracle.stage1(wl, pk, wl.w, mode=oracle.CANONICAL)
    got, _, info = run_emu(emu, wl, pk)
    assert info[0] == 1
    assert np.array_equal(got, want)
    got, _, _ = run_emu(emu, wl, pk, pix=True)
    assert np.array_equal(got, want)
    assert want.max() > 0


def test_emulated_pixel_lane_fixups_with_many_breaks(emu):
    """A wide band (n_f0 = 96) at a high frequency with fast orbits: about 1 % of the 32000 (pixel, template, SFT) triples
    break inside the tile (345, in both directions), so the estimated break bin of exact_window_pos() is exercised all
    over the tile."""
    wl = synth.noise_workload(seed=91, n_sft=400, n_f0=96, margin=250, f_band_start=900.0, n_pix_side=2,
                              ap=(30.0, 40.0), P_days=(15.0, 16.0), n_t=5)
    pk = oracle.peakgram(wl.rho)
    want, _ = oracle.stage1(wl, pk, wl.w, mode=oracle.CANONICAL, want_wcount=False)
    got, _, info = run_emu(emu, wl, pk, pix=True)
    assert info[0] == 0, "unclamped geometry expected"
    assert np.array_equal(got, want)


def test_emulated_kernels_round_ties_to_even(emu):
    """R-1 on the kernel side: exact half-integer bin coordinates (synth.tie_workload) give the oracle's counts."""
    wl = synth.tie_workload()
    pk = oracle.peakgram(wl.rho)
    want, _ = oracle.stage1(wl, pk, None, mode=oracle.CANONICAL)
    for pix in (False, True):
        for force_clamp in (False, True):
            got, _, _ = run_emu(emu, wl, pk, force_clamp=force_clamp, pix=pix)
            assert np.array_equal(got, want), (pix, force_clamp)
