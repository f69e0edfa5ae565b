"""Build libbsh.so (CUDA, sm_100a) in-tree with nvcc.  No GPU is needed to build."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libbsh.so")
SOURCES = [os.path.join(CSRC, "bsh_api.cu")]
DEPS = SOURCES + [os.path.join(CSRC, "bsh_kernels.cuh"), os.path.join(CSRC, "bsh_core.cuh"),
                  os.path.join(CSRC, "bsh_pos.cuh"), os.path.join(CSRC, "bsh_pix.cuh"), os.path.join(CSRC, "bsh_peaks.cuh"), os.path.join(CSRC, "bsh_wpix.cuh"), os.path.join(CSRC, "bsh_frontend.cuh"), os.path.join(CSRC, "bsh_post.cuh"), os.path.join(CSRC, "bsh_sort.cuh"),
                  os.path.join(CSRC, "bsh_host.hpp"),
                  os.path.join(HERE, "..", "include", "bsh.h")]

NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC,-ffp-contract=off,-O2", "-shared", "--fmad=false"]


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(d) > t for d in DEPS)


def build_library(force: bool = False, verbose: bool = False, extra=()) -> str:
    if force or needs_build():
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        cmd = [nvcc, *NVCC_FLAGS, *extra, "-o", LIB, *SOURCES]
        res = subprocess.run(cmd, capture_output=True, text=True)
        if verbose or res.returncode != 0:
            sys.stderr.write(res.stdout + res.stderr)
        if res.returncode != 0:
            raise RuntimeError("nvcc failed building libbsh.so")
    return LIB


if __name__ == "__main__":
    print(build_library(force=True, verbose=True, extra=sys.argv[1:]))
