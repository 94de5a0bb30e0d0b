"""Exact / closed-form references used to pin the oracle.

Everything here is computed from first principles (enumeration of all states,
an elliptic integral, a published series) and shares no code with oracle/ or
with the CUDA path.  tests/golden/exact_values.txt holds the survey's digits
for the same quantities; the tests check both against each other.
"""
from __future__ import annotations

import ctypes
import functools
import math
import os
import subprocess

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))


def golden(path=os.path.join(HERE, "golden", "exact_values.txt")):
    out = {}
    with open(path) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            k, *v = line.split()
            out[k] = [float(x) for x in v]
    return out


# ------------------------------------------------------------------ 4x4 spin-1/2
@functools.lru_cache(maxsize=None)
def ising4x4_states():
    """All 2^16 states of the periodic 4x4 lattice: spins[state, site] in {-1,+1},
    bond sum B (each of the 32 bonds once) and magnetisation M."""
    codes = np.arange(1 << 16, dtype=np.int64)
    spins = (((codes[:, None] >> np.arange(16)[None, :]) & 1) * 2 - 1).astype(np.int64)
    g = spins.reshape(-1, 4, 4)  # [state, y, x]
    B = (g * np.roll(g, -1, axis=2)).sum(axis=(1, 2)) + (g * np.roll(g, -1, axis=1)).sum(axis=(1, 2))
    M = spins.sum(axis=1)
    return spins, B, M


def ising4x4_exact(T, J=1.0, h=0.0):
    """Boltzmann averages per site: <E>/N, <|M|>/N, C/N, U4."""
    _, B, M = ising4x4_states()
    E = -J * B - h * M
    w = np.exp(-(E - E.min()) / T)
    Z = w.sum()
    N = 16
    e1 = (w * E).sum() / Z
    e2 = (w * E * E).sum() / Z
    absm = (w * np.abs(M)).sum() / Z
    m2 = (w * M.astype(float) ** 2).sum() / Z
    m4 = (w * M.astype(float) ** 4).sum() / Z
    return e1 / N, absm / N, (e2 - e1 * e1) / (N * T * T), 1.0 - m4 / (3.0 * m2 * m2)


def ising4x4_density_of_states():
    _, B, _ = ising4x4_states()
    E = -B
    vals, counts = np.unique(E, return_counts=True)
    return dict(zip(vals.tolist(), counts.tolist()))


def ising4x4_flip_probability(thr_table, site):
    """Exact probability thr/2^32 that `site` flips, for every state (vector of 2^16).
    thr_table: the oracle's spin-1/2 2D table, index b*5 + (nn+4)/2."""
    spins, _, _ = ising4x4_states()
    g = spins.reshape(-1, 4, 4)
    nn = (np.roll(g, 1, axis=2) + np.roll(g, -1, axis=2) + np.roll(g, 1, axis=1) + np.roll(g, -1, axis=1)).reshape(-1, 16)
    b = (spins[:, site] + 1) // 2
    idx = b * 5 + (nn[:, site] + 4) // 2
    thr = np.asarray(thr_table, dtype=np.float64)
    return thr[idx] / 2.0 ** 32


def ising4x4_parity_sites(parity):
    return [x + 4 * y for y in range(4) for x in range(4) if (x + y) % 2 == parity]


def ising4x4_evolve_sweep(p, thr_table):
    """Exact evolution of a probability vector over the 2^16 states through one
    checkerboard sweep (parity 0 then parity 1); sites of one parity are updated
    one after the other, which is equivalent because they do not interact."""
    codes = np.arange(1 << 16)
    for parity in (0, 1):
        for site in ising4x4_parity_sites(parity):
            f = ising4x4_flip_probability(thr_table, site)
            flipped = codes ^ (1 << site)
            p = p * (1.0 - f) + p[flipped] * f[flipped]
    return p


# ------------------------------------------------------------------ Onsager
def onsager_u(T, J=1.0):
    from scipy.special import ellipk

    K = J / T
    k = 2.0 * math.sinh(2 * K) / math.cosh(2 * K) ** 2
    K1 = ellipk(k * k)
    return -J / math.tanh(2 * K) * (1.0 + (2.0 / math.pi) * (2.0 * math.tanh(2 * K) ** 2 - 1.0) * K1)


def onsager_m(T, J=1.0):
    K = J / T
    x = math.sinh(2 * K) ** -4
    return (1.0 - x) ** 0.125 if x < 1.0 else 0.0


# ------------------------------------------------------------------ 3D series
def sc_high_T_series_u(T, J=1.0):
    """Simple-cubic high-temperature series: lnZ/N = ln2 + 3 ln cosh K + 3v^4 + 22v^6 + 187.5v^8,
    v = tanh K  =>  u = -J [3v + (12v^3 + 132v^5 + 1500v^7)(1 - v^2)]."""
    v = math.tanh(J / T)
    return -J * (3 * v + (12 * v ** 3 + 132 * v ** 5 + 1500 * v ** 7) * (1 - v * v))


# ------------------------------------------------------------------ 4x4 spin-1
@functools.lru_cache(maxsize=None)
def spin1_4x4_histogram():
    src = os.path.join(HERE, "exact", "enum_spin1.c")
    so = os.path.join(HERE, "exact", "libenum_spin1.so")
    if not os.path.exists(so) or os.path.getmtime(so) < os.path.getmtime(src):
        tmp = so + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-fPIC", "-shared", "-o", tmp, src])
        os.replace(tmp, so)
    lib = ctypes.CDLL(so)
    g = np.zeros((65, 33, 17), dtype=np.int64)
    lib.enum_spin1_4x4(ctypes.c_void_p(g.ctypes.data))
    assert g.sum() == 3 ** 16
    return g


def spin1_4x4_exact(T, J=1.0, h=0.0):
    """<E>/N, C/N, <M>/N, <|M|>/N, <s^2> for H = -J B - h M."""
    g = spin1_4x4_histogram().astype(np.float64)
    B = np.arange(-32, 33)[:, None, None].astype(float)
    M = np.arange(-16, 17)[None, :, None].astype(float)
    Q = np.arange(0, 17)[None, None, :].astype(float)
    E = -J * B - h * M + 0 * Q
    w = g * np.exp(-(E - E[g > 0].min()) / T)
    Z = w.sum()
    N = 16
    e1 = (w * E).sum() / Z
    e2 = (w * E * E).sum() / Z
    return (
        e1 / N,
        (e2 - e1 * e1) / (N * T * T),
        (w * M).sum() / Z / N,
        (w * np.abs(M)).sum() / Z / N,
        (w * Q).sum() / Z / N,
    )


# ------------------------------------------------------------------ statistics
def binned_mean_err(x, nbins=32):
    """Mean and binning estimate of its standard error for a correlated series."""
    x = np.asarray(x, dtype=np.float64)
    n = (len(x) // nbins) * nbins
    b = x[:n].reshape(nbins, -1).mean(axis=1)
    return b.mean(), b.std(ddof=1) / math.sqrt(nbins)


# ------------------------------------------------------------------ 4x4 +/-J bonds (reading D25)
def ea4x4_exact(T, tau, J=1.0, h=0.0):
    """Boltzmann <E>/N and <B>/N of the 4x4 periodic lattice with bond signs tau[a, i] (a = 0: bond to x+1,
    1: bond to y+1) by enumeration of all 2^16 states: H = -J sum tau_ij s_i s_j - h sum s_i."""
    spins, _, M = ising4x4_states()
    g = spins.reshape(-1, 4, 4)
    t = np.asarray(tau, dtype=np.int64).reshape(2, 4, 4)
    B = (t[0][None] * g * np.roll(g, -1, axis=2)).sum(axis=(1, 2)) + (t[1][None] * g * np.roll(g, -1, axis=1)).sum(axis=(1, 2))
    E = -J * B - h * M
    w = np.exp(-(E - E.min()) / T)
    Z = w.sum()
    return (w * E).sum() / Z / 16, (w * B).sum() / Z / 16


# ------------------------------------------------------------------ 4x4 Potts (reading D26)
@functools.lru_cache(maxsize=None)
def potts3_4x4_histogram():
    src = os.path.join(HERE, "exact", "enum_potts3.c")
    so = os.path.join(HERE, "exact", "libenum_potts3.so")
    if not os.path.exists(so) or os.path.getmtime(so) < os.path.getmtime(src):
        tmp = so + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-fPIC", "-shared", "-o", tmp, src])
        os.replace(tmp, so)
    lib = ctypes.CDLL(so)
    g = np.zeros((33, 17), dtype=np.int64)
    lib.enum_potts3_4x4(ctypes.c_void_p(g.ctypes.data))
    assert g.sum() == 3 ** 16
    return g


def potts3_4x4_exact(T, J=1.0):
    """<E>/N, C/N, <N0>/N, <N0^2>/N^2 of the 4x4 3-state Potts lattice, H = -J * (equal bonds)."""
    g = potts3_4x4_histogram().astype(np.float64)
    B = np.arange(0, 33)[:, None].astype(float)
    N0 = np.arange(0, 17)[None, :].astype(float)
    E = -J * B + 0 * N0
    w = g * np.exp(-(E - E[g > 0].min()) / T)
    Z = w.sum()
    e1 = (w * E).sum() / Z
    e2 = (w * E * E).sum() / Z
    return e1 / 16, (e2 - e1 * e1) / (16 * T * T), (w * N0).sum() / Z / 16, (w * N0 * N0).sum() / Z / 256


def potts2_4x4_exact(T, J=1.0):
    """q = 2: delta(s, s') = (1 + s s')/2, so H = -(J/2) sum s s' - 16 J: the Ising enumeration at coupling J/2."""
    _, B, _ = ising4x4_states()
    E = -J * (B + 32) / 2.0
    w = np.exp(-(E - E.min()) / T)
    return (w * E).sum() / w.sum() / 16
