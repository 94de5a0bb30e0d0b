"""ctypes view of oracle/lsm_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, bench.py's cpu_baseline / --impl reference leg and
__graft_entry__.smoke() may import this module.  It shares nothing with
paper_1209_0296_b200/ (the CUDA path): it compiles its own C file with gcc and
never imports the package.

The derived floating-point quantities at the bottom follow SURVEY.md 8(c)
readings D11 (Phi), D12 (persistence) and D13 (heat capacity, Binder cumulant)
and are evaluated with exact Python integers before the final division, so
they carry no accumulation error of their own.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from fractions import Fraction

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lsm_oracle.c")
_LIB = os.path.join(_HERE, "liblsm_oracle.so")
# tests/test_oracle_mutants.py points this at a deliberately broken copy of lsm_oracle.c to prove that the pins
# notice; nothing else sets it.
if os.environ.get("LSM_ORACLE_SRC"):
    _SRC = os.path.abspath(os.environ["LSM_ORACLE_SRC"])
    _LIB = _SRC + ".so"

ISING, NE_HEATBATH, NE_METROPOLIS, EA, POTTS = 0, 1, 2, 3, 4


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, no FMA contraction: the threshold
    arithmetic of reading D3 must be plain IEEE double)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(
            ["gcc", "-O2", "-ffp-contract=off", "-std=c11", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"]
        )
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        vp, i32, i64, u64, dbl = ctypes.c_void_p, ctypes.c_int, ctypes.c_int64, ctypes.c_uint64, ctypes.c_double
        L.orc_create.restype = vp
        L.orc_create.argtypes = [i32, i32, i32, i32, dbl, dbl, dbl, u64]
        L.orc_destroy.argtypes = [vp]
        L.orc_sweep.argtypes = [vp, i64]
        L.orc_sweep_ordered.argtypes = [vp, i64, i32]
        L.orc_sweep_record.argtypes = [vp, i64, vp]
        L.orc_measure.argtypes = [vp, vp, vp]
        L.orc_energy.restype = dbl
        L.orc_energy.argtypes = [vp]
        L.orc_persistence.argtypes = [vp, vp, vp]
        L.orc_reset_reference.argtypes = [vp]
        L.orc_get_spins.argtypes = [vp, vp]
        L.orc_set_spins.argtypes = [vp, vp, u64]
        L.orc_set_temperature.restype = i32
        L.orc_set_temperature.argtypes = [vp, dbl]
        L.orc_get_thresholds.restype = i32
        L.orc_get_thresholds.argtypes = [vp, vp]
        L.orc_sweeps_done.restype = u64
        L.orc_sweeps_done.argtypes = [vp]
        L.orc_num_sites.restype = i64
        L.orc_num_sites.argtypes = [vp]
        L.orc_concentration.restype = dbl
        L.orc_concentration.argtypes = [vp]
        L.orc_philox4x32_10.argtypes = [vp, vp, vp]
        L.orc_get_bonds.argtypes = [vp, vp]
        L.orc_set_bonds.restype = i32
        L.orc_set_bonds.argtypes = [vp, vp]
        L.orc_sweep_random_tile.restype = i32
        L.orc_sweep_random_tile.argtypes = [vp, i64, i32, i32, i32]
        L.orc_sweep_random_tile_balanced.restype = i32
        L.orc_sweep_random_tile_balanced.argtypes = [vp, i64, i32, i32, i32]
        L.orc_sweep_random_tile_record.restype = i32
        L.orc_sweep_random_tile_record.argtypes = [vp, i64, i32, i32, vp]
        L.orc_sweep_random_tile_balanced_record.restype = i32
        L.orc_sweep_random_tile_balanced_record.argtypes = [vp, i64, i32, i32, vp]
        _lib = L
    return _lib


def philox4x32_10(ctr, key):
    c = (ctypes.c_uint32 * 4)(*ctr)
    k = (ctypes.c_uint32 * 2)(*key)
    o = (ctypes.c_uint32 * 4)()
    lib().orc_philox4x32_10(c, k, o)
    return tuple(int(v) for v in o)


class Oracle:
    """One lattice; the arguments are those of lsm_create (include/lsm.h)."""

    def __init__(self, dims, L, two_S=1, model=ISING, J=1.0, h=0.0, T=1.0, seed=0):
        self._h = lib().orc_create(dims, L, two_S, model, float(J), float(h), float(T), int(seed))
        if not self._h:
            raise ValueError("orc_create rejected the arguments")
        self.dims, self.L, self.two_S, self.model = dims, L, two_S, model
        self.J, self.h, self.T, self.seed = float(J), float(h), float(T), int(seed)
        self.N = int(lib().orc_num_sites(self._h))

    def close(self):
        if self._h:
            lib().orc_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def sweep(self, n=1, descending=False):
        lib().orc_sweep_ordered(self._h, int(n), 1 if descending else 0)

    def sweep_record(self, n):
        obs = np.zeros((int(n), 2), dtype=np.int64)
        lib().orc_sweep_record(self._h, int(n), obs.ctypes.data)
        return obs

    def sweep_random_tile(self, n=1, b=32, lam=16, tiles_descending=False):
        """The paper's corrected North-East algorithm (readings D17-D21)."""
        if lib().orc_sweep_random_tile(self._h, int(n), int(b), int(lam), 1 if tiles_descending else 0) != 0:
            raise ValueError("random-tile schedule: NE model, b | L and 2*lambda | b*b required")

    def sweep_random_tile_balanced(self, n=1, b=32, lam=16, tiles_descending=False):
        """The balance-preserving variant (readings D22-D24): colour-restricted picks, 4 launches."""
        if lib().orc_sweep_random_tile_balanced(self._h, int(n), int(b), int(lam), 1 if tiles_descending else 0) != 0:
            raise ValueError("balanced random-tile schedule: NE model, even b | L and 8*lambda | b*b required")

    def sweep_random_tile_record(self, n, b=32, lam=16):
        obs = np.zeros((int(n), 2), dtype=np.int64)
        if lib().orc_sweep_random_tile_record(self._h, int(n), int(b), int(lam), obs.ctypes.data) != 0:
            raise ValueError("random-tile schedule: NE model, b | L and 2*lambda | b*b required")
        return obs

    def sweep_random_tile_balanced_record(self, n, b=32, lam=16):
        obs = np.zeros((int(n), 2), dtype=np.int64)
        if lib().orc_sweep_random_tile_balanced_record(self._h, int(n), int(b), int(lam), obs.ctypes.data) != 0:
            raise ValueError("balanced random-tile schedule: NE model, even b | L and 8*lambda | b*b required")
        return obs

    def measure_int(self):
        B, M = ctypes.c_int64(), ctypes.c_int64()
        lib().orc_measure(self._h, ctypes.byref(B), ctypes.byref(M))
        return int(B.value), int(M.value)

    def energy(self):
        return float(lib().orc_energy(self._h))

    def persistence(self):
        a, b = ctypes.c_int64(), ctypes.c_int64()
        lib().orc_persistence(self._h, ctypes.byref(a), ctypes.byref(b))
        return int(a.value), int(b.value)

    def reset_reference(self):
        lib().orc_reset_reference(self._h)

    def get_spins(self):
        out = np.empty(self.N, dtype=np.int8)
        lib().orc_get_spins(self._h, out.ctypes.data)
        return out

    def set_spins(self, spins, sweep_counter):
        a = np.ascontiguousarray(spins, dtype=np.int8).reshape(-1)
        assert a.size == self.N
        lib().orc_set_spins(self._h, a.ctypes.data, int(sweep_counter))

    def get_bonds(self):
        """EA model (reading D25): bond signs [dims, N]; [a, i] joins site i and its neighbour in direction +a."""
        out = np.empty((self.dims, self.N), dtype=np.int8)
        lib().orc_get_bonds(self._h, out.ctypes.data)
        return out

    def set_bonds(self, tau):
        a = np.ascontiguousarray(tau, dtype=np.int8).reshape(-1)
        assert a.size == self.dims * self.N
        if lib().orc_set_bonds(self._h, a.ctypes.data) != 0:
            raise ValueError("bonds belong to the EA model")

    def set_temperature(self, T):
        if lib().orc_set_temperature(self._h, float(T)) != 0:
            raise ValueError("bad temperature")
        self.T = float(T)

    def thresholds(self):
        buf = (ctypes.c_uint64 * 128)()
        n = lib().orc_get_thresholds(self._h, buf)
        return [int(buf[i]) for i in range(n)]

    @property
    def sweeps_done(self):
        return int(lib().orc_sweeps_done(self._h))

    @property
    def concentration(self):
        return float(lib().orc_concentration(self._h))


# ---------------------------------------------------------------------------
# Derived quantities (host doubles from the integer series), readings D11-D13.
# ---------------------------------------------------------------------------
def energy_from_int(B, M, J, h, model=ISING):
    """E = -J*B - h*M (Ising, PAPER.md:86 with the field term of reading D1);
    E = M for the North-East model (H = sum n_i, reading D15)."""
    if model in (ISING, EA):
        return -float(J) * float(B) - float(h) * float(M)
    if model == POTTS:
        return -float(J) * float(B)
    return float(M)


def binder_u4(M_series):
    """U4 = 1 - <M^4> / (3 <M^2>^2) over the given sweeps (reading D13)."""
    m = [int(v) for v in M_series]
    n = len(m)
    s2 = sum(v * v for v in m)
    s4 = sum(v ** 4 for v in m)
    return float(1 - Fraction(s4 * n, 3 * s2 * s2))


def heat_capacity_per_site(obs, N, J, h, T):
    """C/N = (<E^2> - <E>^2) / (N T^2) (reading D13).  Exact for the integer
    J = 1, h = 0 case; general J, h evaluated through exact rationals."""
    Jf, hf = Fraction(J), Fraction(h)
    e = [-Jf * int(b) - hf * int(m) for b, m in obs]
    n = len(e)
    mean = sum(e, Fraction(0)) / n
    var = sum((v * v for v in e), Fraction(0)) / n - mean * mean
    return float(var) / (N * T * T)


def persistence_fraction(never_changed, N):
    """P(t) = never_changed / N (reading D12)."""
    return never_changed / N


def phi(overlap, N, c):
    """Phi(t) = [overlap/N - (2c-1)^2] / [1 - (2c-1)^2] (reading D11)."""
    q = (2.0 * c - 1.0) ** 2
    return (overlap / N - q) / (1.0 - q)
