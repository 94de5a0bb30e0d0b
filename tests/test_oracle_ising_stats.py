"""Statistical pins of the oracle's Ising path against exact results:
P3 (4x4 brute force), P15 (exact transient), P5 (Onsager), P6 (3D series), P7 (free spins).
All chains are seeded, so each test is deterministic; tolerances are k*sigma with sigma from binning."""
import math

import numpy as np
import pytest

from oracle import lsm_oracle as O
from tests import exact_ref as X

GOLD = X.golden()


def test_exact_references_match_survey_digits():
    """The recomputed exact values agree with the digits printed in SURVEY.md 8(c)."""
    dos = X.ising4x4_density_of_states()
    assert dos == {-32: 2, -24: 32, -20: 64, -16: 424, -12: 1728, -8: 6688, -4: 13568, 0: 20524,
                   4: 13568, 8: 6688, 12: 1728, 16: 424, 20: 64, 24: 32, 32: 2}
    for T in (2.269, 2.0, 3.0):
        assert np.allclose(X.ising4x4_exact(T), GOLD[f"ising4x4_T{T}"], rtol=0, atol=2e-9)
    for T in (2.0, 2.6, 1.5, 3.0):
        u, m = GOLD[f"onsager_T{T}"]
        assert abs(X.onsager_u(T) - u) < 2e-8 and abs(X.onsager_m(T) - m) < 2e-8
    assert abs(X.sc_high_T_series_u(20.0) - GOLD["sc_series_T20"][0]) < 1e-6
    assert abs(X.sc_high_T_series_u(10.0) - GOLD["sc_series_T10"][0]) < 1e-6
    # Onsager's Tc = 2/log(1+sqrt 2) is where m vanishes
    Tc = 2.0 / math.log(1.0 + math.sqrt(2.0))
    assert X.onsager_m(Tc - 1e-6) > 0 and X.onsager_m(Tc + 1e-6) == 0.0


@pytest.mark.slow
@pytest.mark.parametrize("T,nsweeps", [(2.269, 2_400_000), (2.0, 1_200_000), (3.0, 1_200_000)])
def test_p3_4x4_chain_matches_brute_force(T, nsweeps):
    """One long chain from the all-up start (reading D16) reproduces the exact 4x4 Boltzmann
    averages: validates table, neighbour code, sweep order and the balance claim."""
    o = O.Oracle(2, 4, T=T, seed=20120903)
    o.set_spins(np.ones(16, dtype=np.int8), 0)
    o.sweep(10_000)
    chunks = []
    left = nsweeps
    while left > 0:
        n = min(left, 200_000)
        chunks.append(o.sweep_record(n))
        left -= n
    obs = np.concatenate(chunks)
    E = -obs[:, 0] / 16.0
    M = obs[:, 1] / 16.0
    e_ex, absm_ex, c_ex, u4_ex = X.ising4x4_exact(T)
    e, se = X.binned_mean_err(E)
    am, sam = X.binned_mean_err(np.abs(M))
    assert abs(e - e_ex) < 3.5 * se, (e, e_ex, se)
    assert abs(am - absm_ex) < 3.5 * sam, (am, absm_ex, sam)
    assert se < 2e-3 and sam < 1e-3  # the test has teeth
    # heat capacity and Binder cumulant from binned moments (jackknife over 32 bins)
    nb = 32
    n = (len(E) // nb) * nb
    Eb = (E[:n] * 16).reshape(nb, -1)
    Mb = (M[:n] * 16).reshape(nb, -1)
    def jack(f):
        full = f(Eb.ravel(), Mb.ravel())
        loo = np.array([f(np.delete(Eb, i, 0).ravel(), np.delete(Mb, i, 0).ravel()) for i in range(nb)])
        return full, math.sqrt((nb - 1) / nb * ((loo - loo.mean()) ** 2).sum())
    c, sc = jack(lambda e_, m_: e_.var() / (16 * T * T))
    u4, su4 = jack(lambda e_, m_: 1 - (m_ ** 4).mean() / (3 * (m_ ** 2).mean() ** 2))
    assert abs(c - c_ex) < 4 * sc, (c, c_ex, sc)
    assert abs(u4 - u4_ex) < 4 * su4, (u4, u4_ex, su4)


def test_p15_exact_transient_4x4():
    """Dynamics pin: evolve the exact probability vector through checkerboard sweeps from the
    uniform distribution and compare <E>/N after 1, 2, 5, 10 sweeps with an ensemble of oracle
    runs (fresh seed = fresh random start)."""
    T = 2.269
    thr = O.Oracle(2, 4, T=T, seed=0).thresholds()
    _, B, _ = X.ising4x4_states()
    p = np.full(1 << 16, 1.0 / (1 << 16))
    exact = {}
    for t in range(1, 11):
        p = X.ising4x4_evolve_sweep(p, thr)
        exact[t] = float((p * (-B)).sum() / 16.0)
    assert abs(p.sum() - 1.0) < 1e-12
    want = GOLD["transient4x4_T2.269"]
    for t, w in zip((1, 2, 5, 10), want[:4]):
        assert abs(exact[t] - w) < 2e-9
    nseeds = 60_000
    acc = {t: [] for t in (1, 2, 5, 10)}
    for seed in range(nseeds):
        o = O.Oracle(2, 4, T=T, seed=1_000_003 * seed + 17)
        obs = o.sweep_record(10)
        for t in acc:
            acc[t].append(-obs[t - 1, 0] / 16.0)
        o.close()
    for t in acc:
        a = np.asarray(acc[t])
        se = a.std(ddof=1) / math.sqrt(nseeds)
        assert abs(a.mean() - exact[t]) < 3.5 * se, (t, a.mean(), exact[t], se)
        assert se < 4e-3


def test_p15_trapped_states_are_exactly_the_36_zero_energy_cycles():
    """Reading D16: with dE = 0 accepted with certainty the chain has closed period-2 states in
    which every spin has two like and two unlike neighbours; on 4x4 there are exactly 36."""
    spins, B, _ = X.ising4x4_states()
    g = spins.reshape(-1, 4, 4)
    nn = np.roll(g, 1, 2) + np.roll(g, -1, 2) + np.roll(g, 1, 1) + np.roll(g, -1, 1)
    trapped = np.where(np.all(nn == 0, axis=(1, 2)))[0]
    assert len(trapped) == 36 and np.all(B[trapped] == 0)
    o = O.Oracle(2, 4, T=2.269, seed=5)
    for code in trapped[:8]:
        s0 = spins[code].astype(np.int8)
        o.set_spins(s0, 0)
        o.sweep(1)
        s1 = o.get_spins()
        assert o.measure_int()[0] == 0 and not np.array_equal(s1, s0)
        o.sweep(1)
        assert np.array_equal(o.get_spins(), s0)


@pytest.mark.slow
def test_p5_onsager_below_tc():
    """L=128, T=2.0, all-up start: infinite-lattice u and m (finite-size corrections ~ e^{-L/xi})."""
    T, L = 2.0, 128
    o = O.Oracle(2, L, T=T, seed=31415)
    o.set_spins(np.ones(L * L, dtype=np.int8), 0)
    o.sweep(300)
    obs = o.sweep_record(900)
    u, su = X.binned_mean_err(-obs[:, 0] / (L * L), 18)
    m, sm = X.binned_mean_err(np.abs(obs[:, 1]) / (L * L), 18)
    assert abs(u - X.onsager_u(T)) < 4 * su + 2e-4, (u, X.onsager_u(T), su)
    assert abs(m - X.onsager_m(T)) < 4 * sm + 2e-4, (m, X.onsager_m(T), sm)
    assert su < 1.5e-3


@pytest.mark.slow
def test_p5_onsager_above_tc():
    T, L = 2.6, 128
    o = O.Oracle(2, L, T=T, seed=27182)
    o.sweep(400)
    obs = o.sweep_record(1400)
    u, su = X.binned_mean_err(-obs[:, 0] / (L * L), 14)
    assert abs(u - X.onsager_u(T)) < 4 * su + 3e-4, (u, X.onsager_u(T), su)
    assert su < 2e-3
    m = obs[:, 1] / (L * L)
    assert abs(m.mean()) < 0.05  # no spontaneous magnetisation above Tc


@pytest.mark.slow
@pytest.mark.parametrize("T,nsweeps", [(20.0, 2500), (10.0, 3500)])
def test_p6_3d_high_temperature_series(T, nsweeps):
    L = 16
    o = O.Oracle(3, L, T=T, seed=1618)
    o.sweep(50)
    obs = o.sweep_record(nsweeps)
    u, su = X.binned_mean_err(-obs[:, 0] / L ** 3, 25)
    assert abs(u - X.sc_high_T_series_u(T)) < 4 * su + 5e-5, (u, X.sc_high_T_series_u(T), su)
    assert su < 8e-4  # resolves the 3v leading term (0.15 / 0.30) to 0.5 %, and the v^3 term


@pytest.mark.parametrize("dims,L", [(2, 32), (3, 10)])
def test_p7_free_spin_half(dims, L):
    """J = 0: independent spins in a field, <s> = tanh(h/T) (field sign, table rows)."""
    h, T = 0.7, 1.3
    o = O.Oracle(dims, L, J=0.0, h=h, T=T, seed=99)
    o.sweep(20)
    obs = o.sweep_record(600)
    N = L ** dims
    m, sm = X.binned_mean_err(obs[:, 1] / N, 20)
    assert abs(m - math.tanh(h / T)) < 4 * sm, (m, math.tanh(h / T), sm)
    assert sm < 2e-3
    assert np.all(obs[:, 0] * 0 == 0) and o.energy() == -h * obs[-1, 1]
