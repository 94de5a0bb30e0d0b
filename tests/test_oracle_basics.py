"""Deterministic pins of the CPU oracle: P1 (Philox), P2 (thresholds), P4 (exact
reversibility), P9 (order independence), P10 (geometry) of SURVEY.md 8(c)."""
import math
import os

import numpy as np
import pytest

from oracle import lsm_oracle as O
from tests import exact_ref as X

GOLD = X.golden()


def test_p1_philox_known_answers():
    path = os.path.join(os.path.dirname(__file__), "golden", "philox4x32_10_kat.txt")
    n = 0
    for line in open(path):
        if line.startswith("#") or not line.strip():
            continue
        v = [int(t, 16) for t in line.split()]
        assert O.philox4x32_10(v[0:4], v[4:6]) == tuple(v[6:10])
        n += 1
    assert n == 3


def test_p1_philox_round_structure():
    """Independent re-statement of one Philox round applied ten times (python ints):
    catches a swapped multiplier or key word that the three vectors could share."""
    rng = np.random.default_rng(5)
    for _ in range(50):
        c = [int(v) for v in rng.integers(0, 2 ** 32, 4)]
        k = [int(v) for v in rng.integers(0, 2 ** 32, 2)]
        c0, c1, c2, c3 = c
        k0, k1 = k
        for _r in range(10):
            p0 = 0xD2511F53 * c0
            p1 = 0xCD9E8D57 * c2
            c0, c1, c2, c3 = (p1 >> 32) ^ c1 ^ k0, p1 & 0xFFFFFFFF, (p0 >> 32) ^ c3 ^ k1, p0 & 0xFFFFFFFF
            k0 = (k0 + 0x9E3779B9) & 0xFFFFFFFF
            k1 = (k1 + 0xBB67AE85) & 0xFFFFFFFF
        assert O.philox4x32_10(c, k) == (c0, c1, c2, c3)


@pytest.mark.parametrize("T", [2.0, 2.269, 2.6])
def test_p2_thresholds_2d(T):
    o = O.Oracle(2, 8, T=T, seed=1)
    thr = o.thresholds()
    assert len(thr) == 10
    # index b*5 + j, nn = 2j-4; dE = 2 s nn (J=1,h=0): s=-1 -> dE = -2nn ; s=+1 -> dE = 2nn
    for b in (0, 1):
        for j in range(5):
            s, nn = 2 * b - 1, 2 * j - 4
            dE = 2 * s * nn
            want = 2 ** 32 if dE <= 0 else int(math.floor(math.exp(-dE / T) * 2.0 ** 32))
            assert thr[b * 5 + j] == want
    assert thr[1 * 5 + 3] == int(GOLD[f"thr_T{T}_dE4"][0])
    assert thr[1 * 5 + 4] == int(GOLD[f"thr_T{T}_dE8"][0])
    assert thr[0 * 5 + 1] == int(GOLD[f"thr_T{T}_dE4"][0])
    assert thr[0 * 5 + 0] == int(GOLD[f"thr_T{T}_dE8"][0])


def test_p2_thresholds_3d():
    o = O.Oracle(3, 4, T=4.5115, seed=1)
    thr = o.thresholds()
    assert len(thr) == 14
    assert thr[7 + 4] == int(GOLD["thr_T4.5115_dE4"][0])
    assert thr[7 + 5] == int(GOLD["thr_T4.5115_dE8"][0])
    assert thr[7 + 6] == int(GOLD["thr_T4.5115_dE12"][0])
    assert thr[0] == int(GOLD["thr_T4.5115_dE12"][0])
    assert all(t == 2 ** 32 for t in thr[3:11])


def test_p2_thresholds_field_and_extremes():
    # field sign: h > 0 favours s=+1, so flipping +1 -> -1 with nn=0 costs dE = 2h > 0
    o = O.Oracle(2, 4, J=1.0, h=0.5, T=1.0, seed=0)
    thr = o.thresholds()
    assert thr[1 * 5 + 2] == int(math.floor(math.exp(-1.0) * 2.0 ** 32))  # s=+1, nn=0, dE=2h=1
    assert thr[0 * 5 + 2] == 2 ** 32  # s=-1, nn=0, dE=-1
    # underflow: p < 2^-32 -> threshold 0 = never; dE <= 0 -> 2^32 = always
    o = O.Oracle(2, 4, T=0.05, seed=0)
    thr = o.thresholds()
    assert thr[1 * 5 + 4] == 0 and thr[1 * 5 + 3] == 0
    assert thr[1 * 5 + 2] == 2 ** 32  # dE = 0 accepted with certainty (min[1, e^0])


def test_p2_thresholds_spin1_layout():
    J, h, T = 1.0, 0.01, 3.0
    o = O.Oracle(3, 4, two_S=2, J=J, h=h, T=T, seed=0)
    thr = o.thresholds()
    assert len(thr) == 78
    v = (-1, 0, 1)
    for a in range(3):
        for kk in range(2):
            sp = v[(a + 1 + kk) % 3]
            assert sp != v[a]
            for j in range(13):
                nn = j - 6
                dE = -(sp - v[a]) * (J * nn + h)
                want = 2 ** 32 if dE <= 0 else int(math.floor(math.exp(-dE / T) * 2.0 ** 32))
                assert thr[(a * 2 + kk) * 13 + j] == want
    # both other values are proposed, once each
    for a in range(3):
        assert sorted(v[(a + 1 + kk) % 3] for kk in range(2)) == sorted(set(v) - {v[a]})


def test_p2_ne_thresholds():
    for c in (0.10, 0.20, 0.30):
        T = 1.0 / math.log((1 - c) / c)
        o = O.Oracle(2, 8, model=O.NE_HEATBATH, J=0.0, T=T, seed=0)
        assert abs(o.concentration - c) < 1e-12
        thr = o.thresholds()
        assert thr[0] == int(math.floor(o.concentration * 2.0 ** 32))
        assert thr[1] == int(math.floor(math.exp(-1.0 / T) * 2.0 ** 32))
        assert thr[2] == 2 ** 32


@pytest.mark.parametrize("T", [2.269, 1.0])
def test_p4_exact_reversibility_4x4(T):
    """Each half-sweep is reversible w.r.t. the Boltzmann weight: for all states a and all 2^8
    outcomes b on the active colour, pi(a) P(a->b) = pi(b) P(b->a) (up to the 2^-32 floor)."""
    thr = O.Oracle(2, 4, T=T, seed=0).thresholds()
    _, B, _ = X.ising4x4_states()
    logpi = B / T  # E = -B
    codes = np.arange(1 << 16)
    for parity in (0, 1):
        sites = X.ising4x4_parity_sites(parity)
        f = np.stack([X.ising4x4_flip_probability(thr, s) for s in sites])  # [8, 65536]
        worst = 0.0
        for pattern in range(1, 256):
            mask = 0
            pab = np.ones(1 << 16)
            for j, s in enumerate(sites):
                if (pattern >> j) & 1:
                    mask |= 1 << s
                    pab = pab * f[j]
                else:
                    pab = pab * (1.0 - f[j])
            b = codes ^ mask
            pba = np.ones(1 << 16)
            for j, s in enumerate(sites):
                pba = pba * (f[j][b] if (pattern >> j) & 1 else (1.0 - f[j][b]))
            lhs = pab
            rhs = np.exp(logpi[b] - logpi) * pba
            ok = (lhs > 1e-300) | (rhs > 1e-300)
            rel = np.abs(lhs[ok] - rhs[ok]) / np.maximum(lhs[ok], rhs[ok])
            # floor() perturbs each non-trivial factor by < 2^-32 / p; smallest p here is e^{-8/T}
            worst = max(worst, rel.max())
        assert worst < (1e-6 if T > 2 else 1e-4)


@pytest.mark.parametrize(
    "kw",
    [
        dict(dims=2, L=12, T=2.269),
        dict(dims=3, L=6, T=4.5115),
        dict(dims=3, L=6, two_S=2, h=0.01, T=3.0),
        dict(dims=2, L=12, model=O.NE_HEATBATH, J=0.0, T=1.180223),
        dict(dims=2, L=12, model=O.NE_METROPOLIS, J=0.0, T=1.180223),
    ],
)
def test_p9_order_independence(kw):
    a, b = O.Oracle(seed=77, **kw), O.Oracle(seed=77, **kw)
    a.sweep(25, descending=False)
    b.sweep(25, descending=True)
    assert np.array_equal(a.get_spins(), b.get_spins())
    assert a.persistence() == b.persistence()
    # and the result does depend on the seed / the sweep index
    c = O.Oracle(seed=78, **kw)
    c.sweep(25)
    assert not np.array_equal(a.get_spins(), c.get_spins())


@pytest.mark.parametrize("dims,L", [(2, 8), (2, 6), (3, 4), (3, 6)])
def test_p10_geometry(dims, L):
    N = L ** dims
    o = O.Oracle(dims, L, T=1.0, seed=3)
    up = np.ones(N, dtype=np.int8)
    o.set_spins(up, 0)
    assert o.measure_int() == (dims * N, N)
    # checkerboard +/-: every bond is unsatisfied
    idx = np.arange(N)
    x, y, z = idx % L, (idx // L) % L, idx // (L * L)
    cb = np.where((x + y + z) % 2 == 0, 1, -1).astype(np.int8)
    o.set_spins(cb, 0)
    assert o.measure_int() == (-dims * N, 0)
    # a single flipped spin in the all-up state breaks 2d bonds: B = dN - 4d
    for site in (0, N - 1, N // 2 + 1):
        s = up.copy()
        s[site] = -1
        o.set_spins(s, 0)
        assert o.measure_int() == (dims * N - 4 * dims, N - 2)
    # two flipped neighbours along each axis share one bond: B = dN - 2*(4d) + 4
    for step in (1, L, L * L)[:dims]:
        s = up.copy()
        s[0] = -1
        s[step] = -1
        o.set_spins(s, 0)
        assert o.measure_int() == (dims * N - 8 * dims + 4, N - 4)
    # periodic wrap: flipped pair (0, L-1) along x are neighbours
    s = up.copy()
    s[0] = -1
    s[L - 1] = -1
    o.set_spins(s, 0)
    assert o.measure_int() == (dims * N - 8 * dims + 4, N - 4)


def test_p10_zero_temperature_limit_and_invariants():
    o = O.Oracle(2, 8, T=0.02, seed=9)
    o.set_spins(np.ones(64, dtype=np.int8), 0)
    o.reset_reference()
    o.sweep(50)
    assert np.all(o.get_spins() == 1)  # dE = 8 > 0 is never accepted
    assert o.persistence() == (64, 64)
    o = O.Oracle(2, 16, T=2.269, seed=10)
    N = 256
    for _ in range(30):
        o.sweep(1)
        B, M = o.measure_int()
        assert abs(M) <= N and abs(B) <= 2 * N
        assert (M - N) % 2 == 0
        assert (B - 2 * N) % 4 == 0
        assert o.energy() == -1.0 * B


def test_set_get_spins_and_counter():
    a = O.Oracle(2, 8, T=2.0, seed=4)
    a.sweep(7)
    snap = a.get_spins()
    b = O.Oracle(2, 8, T=2.0, seed=4)
    b.set_spins(snap, 7)
    a.sweep(5)
    b.sweep(5)
    assert np.array_equal(a.get_spins(), b.get_spins())
    assert a.sweeps_done == b.sweeps_done == 12


def test_init_distribution():
    """Reading D4: +/-1 uniform; {-1,0,1} uniform; Bernoulli(c)."""
    o = O.Oracle(2, 256, T=2.0, seed=123)
    s = o.get_spins()
    assert set(np.unique(s)) == {-1, 1}
    assert abs(s.mean()) < 4 / math.sqrt(s.size)
    o = O.Oracle(3, 32, two_S=2, T=2.0, seed=123)
    s = o.get_spins()
    assert set(np.unique(s)) == {-1, 0, 1}
    for v in (-1, 0, 1):
        assert abs((s == v).mean() - 1 / 3) < 4 * math.sqrt(2 / 9 / s.size)
    for c in (0.1, 0.3):
        o = O.Oracle(2, 256, model=O.NE_HEATBATH, J=0.0, T=1.0 / math.log((1 - c) / c), seed=5)
        s = o.get_spins()
        assert set(np.unique(s)) == {0, 1}
        assert abs(s.mean() - c) < 4 * math.sqrt(c * (1 - c) / s.size)


def test_create_rejects_bad_arguments():
    for kw in [
        dict(dims=1, L=8), dict(dims=2, L=7), dict(dims=2, L=2), dict(dims=2, L=8, T=0.0),
        dict(dims=2, L=8, T=float("nan")), dict(dims=2, L=8, two_S=3),
        dict(dims=3, L=8, model=O.NE_HEATBATH, J=0.0), dict(dims=2, L=8, model=O.NE_HEATBATH, J=1.0),
    ]:
        base = dict(T=1.0, seed=0)
        base.update(kw)
        with pytest.raises(ValueError):
            O.Oracle(**base)
