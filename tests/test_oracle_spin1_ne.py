"""Pins of the oracle's spin-1 path (P7, P8) and North-East path (P11-P13, constraint direction)."""
import math

import numpy as np
import pytest

from oracle import lsm_oracle as O
from tests import exact_ref as X

GOLD = X.golden()


# ------------------------------------------------------------------------ spin-1
@pytest.mark.parametrize("dims,L", [(2, 24), (3, 8)])
def test_p7_free_spin_one(dims, L):
    """J = 0: <s> = 2 sinh(bh)/(1+2cosh bh), <s^2> = 2cosh(bh)/(1+2cosh bh)  (proposal + table)."""
    h, T = 0.6, 1.1
    o = O.Oracle(dims, L, two_S=2, J=0.0, h=h, T=T, seed=4242)
    o.sweep(30)
    N = L ** dims
    ms, qs = [], []
    for _ in range(500):
        o.sweep(1)
        s = o.get_spins().astype(np.int64)
        ms.append(s.sum() / N)
        qs.append((s * s).sum() / N)
    bh = h / T
    m_ex = 2 * math.sinh(bh) / (1 + 2 * math.cosh(bh))
    q_ex = 2 * math.cosh(bh) / (1 + 2 * math.cosh(bh))
    m, sm = X.binned_mean_err(ms, 20)
    q, sq = X.binned_mean_err(qs, 20)
    assert abs(m - m_ex) < 4 * sm, (m, m_ex, sm)
    assert abs(q - q_ex) < 4 * sq, (q, q_ex, sq)
    assert sm < 3e-3 and sq < 3e-3


def test_p8_exact_spin1_references_match_survey_digits():
    for T in (3.0, 1.5):
        got = X.spin1_4x4_exact(T, h=0.01)
        assert np.allclose(got, GOLD[f"spin1_4x4_T{T}_h0.01"], rtol=0, atol=2e-9), got


@pytest.mark.slow
@pytest.mark.parametrize("T,nsweeps", [(3.0, 900_000), (1.5, 900_000)])
def test_p8_spin1_4x4_chain_matches_brute_force(T, nsweeps):
    """2D spin-1, 4x4, h = 0.01 (no dE = 0 moves, so no deterministic traps): one long chain
    reproduces the exact averages over all 3^16 states."""
    h = 0.01
    o = O.Oracle(2, 4, two_S=2, J=1.0, h=h, T=T, seed=8675309)
    o.set_spins(np.ones(16, dtype=np.int8), 0)
    o.sweep(5_000)
    E, M, Q = [], [], []
    # <s^2> needs the configuration; sample it every sweep in chunks through get_spins
    obs = np.concatenate([o.sweep_record(100_000) for _ in range(nsweeps // 100_000)])
    E = (-obs[:, 0] - h * obs[:, 1]) / 16.0
    M = obs[:, 1] / 16.0
    e_ex, c_ex, m_ex, absm_ex, q_ex = X.spin1_4x4_exact(T, h=h)
    e, se = X.binned_mean_err(E)
    m, sm = X.binned_mean_err(M)
    am, sam = X.binned_mean_err(np.abs(M))
    assert abs(e - e_ex) < 3.5 * se, (e, e_ex, se)
    assert abs(m - m_ex) < 3.5 * sm, (m, m_ex, sm)
    assert abs(am - absm_ex) < 3.5 * sam, (am, absm_ex, sam)
    assert se < 3e-3 and sam < 2e-3
    c = (E * 16).var() / (16 * T * T)
    assert abs(c - c_ex) < 0.03 * c_ex + 0.01
    for _ in range(4000):
        o.sweep(5)
        s = o.get_spins().astype(np.int64)
        Q.append((s * s).mean())
    q, sq = X.binned_mean_err(Q, 20)
    assert abs(q - q_ex) < 4 * sq, (q, q_ex, sq)


def test_spin1_values_and_moves():
    o = O.Oracle(3, 8, two_S=2, h=0.01, T=3.0, seed=11)
    prev = o.get_spins()
    for _ in range(5):
        o.sweep(1)
        cur = o.get_spins()
        assert set(np.unique(cur)) <= {-1, 0, 1}
        prev = cur
    B, M = o.measure_int()
    assert abs(M) <= 512 and abs(B) <= 3 * 512
    assert abs(o.energy() - (-B - 0.01 * M)) < 1e-12


# ------------------------------------------------------------------ North-East
def T_of_c(c):
    return 1.0 / math.log((1.0 - c) / c)


@pytest.mark.parametrize("model", [O.NE_HEATBATH, O.NE_METROPOLIS])
@pytest.mark.parametrize("c", [0.10, 0.20, 0.30])
def test_p11_product_measure_and_monotone_persistence(model, c):
    L = 192
    N = L * L
    o = O.Oracle(2, L, model=model, J=0.0, T=T_of_c(c), seed=2718 + int(100 * c))
    assert o.persistence() == (N, N)  # P(0) = 1, overlap = N -> Phi(0) = 1
    assert O.phi(N, N, c) == 1.0 and O.persistence_fraction(N, N) == 1.0
    sigma = math.sqrt(c * (1 - c) / N)
    last_nc = N
    for t in range(60):
        o.sweep(1)
        B, M = o.measure_int()
        assert B == 0
        assert abs(M / N - c) < 4 * sigma, (t, M / N, c, sigma)
        nc, ov = o.persistence()
        assert nc <= last_nc
        last_nc = nc
        assert o.energy() == float(M)


@pytest.mark.parametrize("model,formula", [
    (O.NE_HEATBATH, lambda c: 1 - 2 * c ** 3 * (1 - c)),
    (O.NE_METROPOLIS, lambda c: 1 - 2 * c ** 3),
])
@pytest.mark.parametrize("c", [0.10, 0.20, 0.30])
def test_p12_first_sweep_persistence_closed_form(model, formula, c):
    L = 256
    N = L * L
    o = O.Oracle(2, L, model=model, J=0.0, T=T_of_c(c), seed=161803 + int(1000 * c))
    o.sweep(1)
    nc, _ = o.persistence()
    P = formula(c)
    sigma = math.sqrt(P * (1 - P) / N)
    assert abs(nc / N - P) < 5 * sigma, (nc / N, P, sigma)


@pytest.mark.parametrize("model", [O.NE_HEATBATH, O.NE_METROPOLIS])
def test_constraint_direction_north_and_east(model):
    """Reading D8: a site may change only if (x, y+1) and (x+1, y) are both up at the time of its
    half-sweep.  Parity-0 sites see the initial state; parity-1 sites see the final parity-0 values."""
    L = 48
    c = 0.35
    o = O.Oracle(2, L, model=model, J=0.0, T=T_of_c(c), seed=55)
    for _ in range(12):
        before = o.get_spins().reshape(L, L).copy()  # [y, x]
        o.sweep(1)
        after = o.get_spins().reshape(L, L)
        y, x = np.mgrid[0:L, 0:L]
        par = (x + y) % 2
        changed = before != after
        for p, ref in ((0, before), (1, after)):
            north = np.roll(ref, -1, axis=0)  # value at (x, y+1)
            east = np.roll(ref, -1, axis=1)   # value at (x+1, y)
            fac = (north == 1) & (east == 1)
            assert not np.any(changed & (par == p) & ~fac)
            # and facilitated sites do move at the expected rate (direction is not vacuous)
            assert np.any(changed & (par == p))
        # south / west must NOT be what matters: some changed site has south or west down
        south = np.roll(before, 1, axis=0)
        west = np.roll(before, 1, axis=1)
        assert np.any(changed & (par == 0) & ((south == 0) | (west == 0)))


def test_metropolis_rule_details():
    """NE Metropolis: a facilitated up site always goes down (dE = -1 < 0)."""
    L = 32
    o = O.Oracle(2, L, model=O.NE_METROPOLIS, J=0.0, T=T_of_c(0.3), seed=8)
    before = o.get_spins().reshape(L, L).copy()
    o.sweep(1)
    after = o.get_spins().reshape(L, L)
    y, x = np.mgrid[0:L, 0:L]
    par0 = (x + y) % 2 == 0
    fac = (np.roll(before, -1, 0) == 1) & (np.roll(before, -1, 1) == 1)
    sel = par0 & fac & (before == 1)
    assert sel.sum() > 5 and np.all(after[sel] == 0)


@pytest.mark.parametrize("c", [0.10, 0.20])
def test_p13_frozen_set_bound(c):
    L = 48
    N = L * L
    o = O.Oracle(2, L, model=O.NE_HEATBATH, J=0.0, T=T_of_c(c), seed=1234)
    n0 = o.get_spins().reshape(L, L).astype(bool)  # [y, x]
    Z = ~n0
    while True:
        keep = Z & (np.roll(Z, -1, axis=0) | np.roll(Z, -1, axis=1))  # north in Z or east in Z
        if np.array_equal(keep, Z):
            break
        Z = keep
    blocked = np.roll(Z, -1, axis=0) | np.roll(Z, -1, axis=1)
    assert np.all(blocked[Z])
    bound = int(blocked.sum())
    assert bound > 0
    for t in range(40):
        o.sweep(5)
        nc, _ = o.persistence()
        assert nc >= bound
        s = o.get_spins().reshape(L, L)
        assert np.all(s[Z] == 0)
        assert np.array_equal(s[blocked].astype(bool), n0[blocked])


def test_derived_quantities():
    assert abs(O.binder_u4([1, -1, 1, -1]) - (1 - 1 / 3)) < 1e-15
    assert abs(O.binder_u4([2, 0, -2, 0]) - (1 - (8.0) / (3 * 4.0))) < 1e-15
    obs = np.array([[10, 2], [14, 4], [6, 0]])
    # E = -B: mean -10, var = (0+16+16)/3
    assert abs(O.heat_capacity_per_site(obs, N=16, J=1, h=0, T=2.0) - (32 / 3) / (16 * 4)) < 1e-15
    assert O.phi(50, 100, 0.5) == 0.5
    assert abs(O.phi(100 * (0.6 ** 2), 100, 0.2)) < 1e-15
    assert O.energy_from_int(7, 3, 1.0, 0.5) == -8.5
    assert O.energy_from_int(0, 9, 0.0, 0.0, model=O.NE_HEATBATH) == 9.0
