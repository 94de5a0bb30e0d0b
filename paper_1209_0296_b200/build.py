"""Build liblsm.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_1209_0296_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU, so this also runs on the CPU-only box.
"""
from __future__ import annotations

import os
import subprocess
import sys

PKG = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(PKG, "csrc")
LIB = os.path.join(PKG, "liblsm.so")
SOURCES = ["lsm_api.cu", "lsm_generic.cu", "lsm_tiled.cu", "lsm_tiled_bulk.cu", "lsm_small.cu", "lsm_slab.cu", "lsm_ne_tile.cu"]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-lineinfo", "-O3", "-std=c++17",
    # the threshold arithmetic of reading D3 must be plain IEEE double on the host
    "-Xcompiler", "-fPIC,-ffp-contract=off",
    "-shared", "--threads", "0",
]


PROBE_LIB = os.path.join(PKG, "libpipe_probe.so")
PROBE_SRC = os.path.join(CSRC, "probe", "pipe_probe.cu")


def build_probe(force: bool = False) -> str:
    """libpipe_probe.so: the integer-pipe microbenchmarks behind `bench.py --pipe-probe` (not part of liblsm.so)."""
    if not force and os.path.exists(PROBE_LIB) and os.path.getmtime(PROBE_LIB) >= os.path.getmtime(PROBE_SRC):
        return PROBE_LIB
    tmp = PROBE_LIB + f".tmp{os.getpid()}"
    r = subprocess.run([os.environ.get("NVCC", "nvcc"), *NVCC_FLAGS, "-o", tmp, PROBE_SRC], capture_output=True, text=True)
    if r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
        raise RuntimeError("nvcc failed building libpipe_probe.so")
    os.replace(tmp, PROBE_LIB)
    return PROBE_LIB


def _inputs():
    out = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cu", ".cuh", ".h"))]   # not csrc/probe/
    out.append(os.path.join(os.path.dirname(PKG), "include", "lsm.h"))
    return out


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(p) > t for p in _inputs())


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not needs_build():
        return LIB
    nvcc = os.environ.get("NVCC", "nvcc")
    tmp = LIB + f".tmp{os.getpid()}"
    cmd = [nvcc, *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []), "-o", tmp,
           *[os.path.join(CSRC, s) for s in SOURCES]]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed building liblsm.so")
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
