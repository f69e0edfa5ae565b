"""The tier-2 CPU reference (oracle/bsh_tier2.c; SURVEY.md 8(c) coverage plan) equals the plain oracle's CANONICAL mode bit
for bit on every grid the plain oracle can run: config 1 (tracks leaving the slab), ragged noise grids, bands where the
shift changes several times, eccentric grids.  It is then the full-grid comparator of the GPU tests.  CPU only."""
import numpy as np
import pytest

import oracle
import synth


def _check(wl, weighted=True):
    pk = oracle.peakgram(wl.rho)
    n, w = oracle.stage1(wl, pk, wl.w, mode=oracle.CANONICAL)
    n2, w2 = oracle.tier2_stage1(wl, pk, wl.w, want_wcount=True)
    assert np.array_equal(n2, n)
    assert np.array_equal(w2, w)                       # same FP64 additions in the same (SFT) order
    assert np.array_equal(oracle.tier2_stage1(wl, pk), n)
    return n


@pytest.mark.parametrize("pixel", ["ecliptic", "pole"])
def test_tier2_equals_plain_oracle_on_config1(pixel):
    _check(synth.config1(pixel=pixel))
    _check(synth.eccentric(synth.config1(pixel=pixel)))


@pytest.mark.parametrize("n_sft,n_f0,margin,f0,side", [(1, 1, 3, 50.0, 1), (33, 7, 12, 80.0, 2), (64, 90, 30, 120.0, 2),
                                                        (200, 96, 45, 150.0, 3), (130, 97, 5, 150.0, 2), (70, 200, 60, 200.0, 1)])
def test_tier2_equals_plain_oracle_on_ragged_grids(n_sft, n_f0, margin, f0, side):
    wl = synth.noise_workload(seed=n_sft + n_f0, n_sft=n_sft, n_f0=n_f0, margin=margin, f_band_start=f0, n_pix_side=side,
                              ap=(10.0, 40.0), P_days=(15.0, 31.0), n_t=3)
    _check(wl)


def test_tier2_handles_many_breaks_and_tracks_far_outside_the_slab():
    wl = synth.noise_workload(seed=77, n_sft=96, n_f0=90, margin=40, f_band_start=150.0, n_pix_side=1,
                              ap=(2500.0, 6000.0, 60000.0), P_days=(15.0,), n_t=4)      # unphysical a_p: several breaks per band
    n = _check(wl)
    assert n.max() > 0
    wl = synth.tie_workload()                                                          # exact half-integer coordinates
    _check(wl)


def test_tier2_config2_subgrid_equals_plain_oracle():
    wl = synth.config2()
    sub = wl.subgrid(ia=[0, 7, 19], ip=[0, 11, 29], it=[0, 13, 39], pix=[0, 9, 63])
    _check(sub)
