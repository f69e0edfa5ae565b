"""CPU-side checks of the boundary: libbsh.so builds for sm_100a, loads, and exports every symbol include/bsh.h
declares; pure-host entry points behave; and nothing computes without a GPU (no CPU fallback)."""
import ctypes as C
import os
import re
import subprocess

import numpy as np
import pytest

import synth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    import paper_1904_04873_b200 as b
    lib = b.library()
    header = open(os.path.join(ROOT, "include", "bsh.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(bsh_[a-z0-9_]+)\s*\(", header))
    assert {"bsh_build_peakgram", "bsh_stage1_hough", "bsh_stage2_power"} <= declared
    for name in declared:
        assert hasattr(lib, name), name
    assert lib.bsh_version() >= 100
    assert declared == set(b.binding.EXPORTS)


def test_library_is_built_for_sm_100a_with_tma_and_fp64_no_fma():
    import paper_1904_04873_b200 as b
    path = b.build.build_library()
    out = subprocess.run(["cuobjdump", "-lelf", path], capture_output=True, text=True).stdout
    assert "sm_100a" in out
    sass = subprocess.run(["cuobjdump", "-sass", path], capture_output=True, text=True).stdout
    kernels = sass.split("Function : ")
    # every accumulation-kernel family: the ones the bench runs (pixel-lane, weighted pixel-lane), the template-lane
    # position-table kernels and the funnel-shift fallbacks
    families = {"stage1_unweighted_pix_kernel": "LOP3", "stage1_weighted_pix_kernel": "FADD",
                "stage1_unweighted_pos_kernel": "LOP3", "stage1_weighted_pos_kernel": "FADD",
                "stage1_unweighted_kernel": "LOP3", "stage1_weighted_kernel": "FADD"}
    for name, count_op in families.items():
        acc = [k for k in kernels if k.startswith(f"_ZN3bsh{len(name)}{name}")]
        assert acc, name
        for k in acc:
            assert "UBLKCP" in k, f"{name}: accumulation kernels stage their tables with TMA bulk copies"
            assert "DFMA" not in k, f"{name}: track arithmetic must not contract to FMA (DESIGN.md R-5)"
            assert "DMUL" in k and "DADD" in k and count_op in k, name
    pix = [k for k in kernels if k.startswith("_ZN3bsh28stage1_unweighted_pix_kernel")]
    assert all("LDS.64" in k for k in pix), "pixel-lane kernel: 8-byte window reads from the position-major table"
    assert all("DSETP" in k for k in pix if "Lb0ELb" in k.split("\n")[0]), "unclamped pixel-lane kernel: FP64 break predicate"
    assert any("Lb0ELb0EEE" in k.split("\n")[0] for k in pix) and any("Lb0ELb1EEE" in k.split("\n")[0] for k in pix)
    wpix = [k for k in kernels if k.startswith("_ZN3bsh26stage1_weighted_pix_kernel")]
    assert all("R2P" in k for k in wpix), "weighted pixel-lane kernel: predicates of a byte of bins set by one R2P"
    front = [k for k in kernels if k.startswith("_ZN3bsh25normalise_peakgram_kernel")]
    assert front and all("FMUL" in k and "FADD" in k for k in front), "front end: |x|^2 as rounded FP32 products and sum (R-22)"


def test_template_index_roundtrip_and_order():
    import paper_1904_04873_b200 as b
    wl = synth.config2()
    rng = np.random.default_rng(0)
    for _ in range(50):
        pix, ia, ip, it, j = (int(rng.integers(n)) for n in (64, 20, 30, 40, 90))
        idx = b.template_index(wl, pix, ia, ip, it, j)
        assert idx == ((((pix * 20 + ia) * 30 + ip) * 40 + it) * 90 + j)
        assert b.template_decode(wl, idx) == (pix, ia, ip, it, j)
    assert b.CAND_DTYPE.itemsize == 24


def test_no_cpu_fallback():
    import torch
    import paper_1904_04873_b200 as b
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(b.BshError):
        b.Context(0)
    ctx = C.c_void_p()
    assert b.library().bsh_create(C.byref(ctx), 0, None) < 0 and not ctx.value


def test_product_path_does_not_import_the_oracle():
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_1904_04873_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".hpp", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle|bsh_oracle|#include\s+\"[^\"]*oracle|CDLL\([^)]*oracle", text, re.M), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(import|from)\s+paper_1904_04873_b200|#include\s+\"[^\"]*csrc|libbsh\.so", text, re.M), f
