"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol that
include/lsm.h declares; host-only entry points behave; the binding knows every symbol."""
import ctypes
import math
import os
import re

import numpy as np
import pytest

from oracle import lsm_oracle as O
from paper_1209_0296_b200 import build as B
from paper_1209_0296_b200 import lsm

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    B.build()
    return lsm.load()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "lsm.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(lsm_[a-z0-9_]+)\s*\(", text)))


def test_every_declared_symbol_is_exported_and_bound(lib):
    names = declared_symbols()
    assert len(names) >= 25
    raw = ctypes.CDLL(lsm.lib_path())
    for n in names:
        assert hasattr(raw, n), f"{n} declared in lsm.h but not exported by liblsm.so"
        assert n in lsm.SIGNATURES, f"{n} missing from the Python binding"
    assert sorted(lsm.SIGNATURES) == names


def test_product_does_not_touch_the_oracle():
    """The CUDA path and the oracle share no code and neither imports the other."""
    pkg = os.path.join(ROOT, "paper_1209_0296_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                src = open(os.path.join(dirpath, f)).read()
                assert "lsm_oracle" not in src and "import oracle" not in src and "from oracle" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_1209_0296_b200" not in src and "from paper_1209_0296_b200" not in src
            assert "csrc" not in src and "#include \"lsm" not in src


def test_workspace_and_argument_errors(lib):
    n = ctypes.c_size_t()
    assert lib.lsm_workspace_bytes(2, 64, 1, lsm.ISING, ctypes.byref(n)) == lsm.OK
    assert n.value >= 64 * 64
    assert lsm.workspace_bytes(3, 512) >= 512 ** 3
    assert lib.lsm_workspace_bytes(2, 63, 1, lsm.ISING, ctypes.byref(n)) == lsm.ERR_ARG
    assert lib.lsm_workspace_bytes(2, 2, 1, lsm.ISING, ctypes.byref(n)) == lsm.ERR_ARG
    assert lib.lsm_workspace_bytes(4, 64, 1, lsm.ISING, ctypes.byref(n)) == lsm.ERR_ARG
    assert lib.lsm_workspace_bytes(2, 64, 3, lsm.ISING, ctypes.byref(n)) == lsm.ERR_UNSUPPORTED
    assert lib.lsm_workspace_bytes(3, 64, 1, lsm.NE_HEATBATH, ctypes.byref(n)) == lsm.ERR_UNSUPPORTED
    assert lib.lsm_workspace_bytes(2, 64, 1, 7, ctypes.byref(n)) == lsm.ERR_ARG
    assert lib.lsm_workspace_bytes(2, 64, 1, lsm.ISING, None) == lsm.ERR_ARG
    h = ctypes.c_void_p()
    # NULL workspace / bad temperature are rejected before any CUDA call
    assert lib.lsm_create(2, 64, 1, 0, 1.0, 0.0, 2.0, 1, None, 0, None, ctypes.byref(h)) == lsm.ERR_ARG
    fake = ctypes.c_void_p(4096)
    assert lib.lsm_create(2, 64, 1, 0, 1.0, 0.0, -1.0, 1, fake, 1 << 20, None, ctypes.byref(h)) == lsm.ERR_ARG
    assert lib.lsm_create(2, 64, 1, 0, 1.0, 0.0, float("nan"), 1, fake, 1 << 20, None, ctypes.byref(h)) == lsm.ERR_ARG
    assert lib.lsm_create(2, 64, 1, 0, 1.0, 0.0, 2.0, 1, fake, 16, None, ctypes.byref(h)) == lsm.ERR_WORKSPACE
    assert lib.lsm_create(2, 64, 1, 0, 1.0, 0.0, 2.0, 1, ctypes.c_void_p(4100), 1 << 20, None, ctypes.byref(h)) == lsm.ERR_WORKSPACE
    assert lib.lsm_create(2, 64, 1, lsm.NE_HEATBATH, 1.0, 0.0, 2.0, 1, fake, 1 << 20, None, ctypes.byref(h)) == lsm.ERR_UNSUPPORTED
    assert not h.value
    assert lib.lsm_sweep(None, 1, None) == lsm.ERR_ARG
    assert lib.lsm_destroy(None) == lsm.ERR_ARG
    # entry points added in round 3: argument errors are found before any CUDA call
    buf = ctypes.c_void_p(8)
    assert lib.lsm_sweep_record_host_noalloc(None, 1, buf, None) == lsm.ERR_ARG
    assert lib.lsm_batch_sweep_random_tile(None, 1, 32, 16, 0, None, None) == lsm.ERR_ARG
    assert b"LSM_NOALLOC_MAX_SWEEPS" in lib.lsm_strerror(lsm.ERR_LIMIT)
    text = open(os.path.join(ROOT, "include", "lsm.h")).read()
    assert f"LSM_NOALLOC_MAX_SWEEPS = {lsm.NOALLOC_MAX_SWEEPS}" in text and "LSM_ERR_LIMIT = -6" in text
    for code in (0, -1, -2, -3, -4, -5, -6, -99):
        assert len(lib.lsm_strerror(code)) > 0


def test_no_cpu_fallback_without_device():
    import torch

    if torch.cuda.is_available():
        pytest.skip("CUDA device present")
    with pytest.raises(RuntimeError):
        lsm.Lattice(2, 16, T=2.0, seed=1)


def test_derived_quantities_match_oracle_side(lib):
    """Binder cumulant, heat capacity, Phi, persistence: library (long double / int128) vs the
    oracle side (exact rationals) within 1e-9 relative (BASELINE.json north_star)."""
    rng = np.random.default_rng(7)
    for N, scale in ((4096, 300), (8192 * 8192, 3_000_000), (512 ** 3, 40_000_000)):
        n = 5000
        M = (rng.normal(0, scale, n)).astype(np.int64)
        Bs = (rng.normal(-1.4 * N, scale * 2, n)).astype(np.int64)
        obs = np.stack([Bs, M], axis=1)
        u_lib, u_orc = lsm.binder_u4(obs), O.binder_u4(M)
        assert abs(u_lib - u_orc) <= 1e-9 * abs(u_orc)
        for J, h, T in ((1.0, 0.0, 2.269), (1.0, 0.01, 3.0)):
            c_lib = lsm.heat_capacity(obs, N, J, h, T)
            c_orc = O.heat_capacity_per_site(obs[:400], N, J, h, T)
            c_lib_400 = lsm.heat_capacity(obs[:400], N, J, h, T)
            assert abs(c_lib_400 - c_orc) <= 1e-9 * abs(c_orc)
            assert c_lib > 0
    for c in (0.1, 0.2, 0.3):
        N = 8192 * 8192
        for ov in (N, int(0.7 * N), int((2 * c - 1) ** 2 * N)):
            a, b = lsm.phi(ov, N, c), O.phi(ov, N, c)
            assert abs(a - b) <= 1e-9 * max(abs(b), 1e-12) or abs(a - b) < 1e-15
        assert lsm.persistence_fraction(12345, N) == O.persistence_fraction(12345, N)
    assert lsm.phi(100, 100, 0.3) == 1.0
    assert lsm.energy(lsm.ISING, 1.0, 0.01, 100, -7) == O.energy_from_int(100, -7, 1.0, 0.01)
    assert lsm.energy(lsm.NE_HEATBATH, 0.0, 0.0, 0, 55) == 55.0
    out = ctypes.c_double()
    assert lib.lsm_binder_u4(None, 5, ctypes.byref(out)) == lsm.ERR_ARG
    assert lib.lsm_phi(1, 0, 0.3, ctypes.byref(out)) == lsm.ERR_ARG


def test_workload_table():
    from paper_1209_0296_b200 import workloads as W

    cfg = W.configs()
    assert cfg["cfg1"].N == 4096 and cfg["cfg3"].N == 512 ** 3 and cfg["cfg4"].two_S == 2
    assert len({w.seed for w in cfg.values()}) == len(cfg)
    for c in (0.1, 0.2, 0.3):
        T = W.ne_temperature(c)
        assert abs(1.0 / (1.0 + math.exp(1.0 / T)) - c) < 1e-12
    assert abs(W.ne_temperature(0.10) - 0.455120) < 1e-6
    assert cfg["cfg2_T2.269"].scaled(256, 100).N == 65536
