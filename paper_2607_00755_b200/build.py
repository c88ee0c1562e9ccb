"""Compile csrc/*.cu -> libkx.so for sm_100a with nvcc (cross-compiles without a GPU).

    python -m paper_2607_00755_b200.build [--force]

The library is built in-tree so that it travels with the repository snapshot; it is git-ignored.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libkx.so")
SOURCES = ["kx_api.cu", "kx_build.cu", "kx_contract.cu", "kx_stream_bt1.cu", "kx_stream_bt2.cu", "kx_stream_bt4.cu", "kx_stream_bt8.cu",
           "kx_tiled_build.cu", "kx_tiled.cu", "kx_probe.cu", "kx_static.cu"]
HEADERS = [os.path.join(CSRC, "kx_internal.cuh"), os.path.join(CSRC, "kx_entry.cuh"), os.path.join(CSRC, "kx_device.cuh"), os.path.join(CSRC, "kx_stream.cuh"), os.path.join(HERE, "..", "include", "kx.h")]
# --fmad=false: validity decisions, omega and the Runge-Kutta updates must not depend on implicit FMA
# contraction; the hot loops call fma() explicitly.
NVCC_FLAGS = ["-O3", "-std=c++17", "--threads", "0", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "--fmad=false", "-Xcompiler", "-fPIC", "-shared"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + HEADERS
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or needs_build():
        cmd = [_nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB] + \
              [os.path.join(CSRC, s) for s in SOURCES]
        subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
