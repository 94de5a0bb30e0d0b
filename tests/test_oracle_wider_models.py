"""CPU pins of the oracle's NEXT-4 models: Edwards-Anderson +/-J bonds (reading D25)
and the q-state Potts model (reading D26).  No GPU."""
import math

import numpy as np
import pytest

from oracle import lsm_oracle as O
from tests import exact_ref as X
from tests.test_oracle_restatement import ALWAYS, M32, philox_py, thr_metropolis, thr_of, words


# ============================================================================ Edwards-Anderson +/-J
def test_ea_all_ferromagnetic_bonds_is_the_ising_rule():
    """tau = +1 on every bond: configuration, (B, M) and persistence of every sweep equal the Ising oracle's."""
    for dims, L, h, T in ((2, 16, 0.0, 2.2), (2, 12, 0.3, 1.9), (3, 8, -0.1, 4.2)):
        e = O.Oracle(dims, L, model=O.EA, h=h, T=T, seed=41)
        i = O.Oracle(dims, L, model=O.ISING, h=h, T=T, seed=41)
        e.set_bonds(np.ones((dims, e.N), dtype=np.int8))
        assert np.array_equal(e.get_spins(), i.get_spins()) and e.thresholds() == i.thresholds()
        assert e.measure_int() == i.measure_int()
        for _ in range(6):
            e.sweep(1)
            i.sweep(1)
            assert np.array_equal(e.get_spins(), i.get_spins())
            assert e.measure_int() == i.measure_int() and e.persistence() == i.persistence()
            assert abs(e.energy() - i.energy()) < 1e-12


@pytest.mark.parametrize("dims,L,T", [(2, 16, 2.269), (2, 10, 1.5), (3, 8, 4.5115), (3, 6, 3.0)])
def test_ea_mattis_gauge_reproduces_the_ferromagnet(dims, L, T):
    """Gauge pin: bonds tau_ij = g_i g_j with the state gauge-transformed (s_i -> g_i s_i) are the ferromagnet in
    disguise (h = 0): nn_eff = g_i nn and the Metropolis threshold depends on s * nn only, so under the same seed the
    EA run must reproduce the ferromagnet's B series bit for bit and its configuration up to the gauge."""
    rng = np.random.default_rng(1234 + L)
    N = L ** dims
    g = rng.choice(np.array([-1, 1], dtype=np.int8), size=N)
    shape = (L,) * dims                                            # [z][y][x]
    gg = g.reshape(shape)
    tau = np.stack([gg * np.roll(gg, -1, axis=dims - 1 - a) for a in range(dims)]).reshape(dims, N).astype(np.int8)
    f = O.Oracle(dims, L, model=O.ISING, T=T, seed=99)
    e = O.Oracle(dims, L, model=O.EA, T=T, seed=99)
    e.set_bonds(tau)
    e.set_spins(f.get_spins() * g, 0)
    e.reset_reference()
    assert e.measure_int()[0] == f.measure_int()[0]
    for _ in range(8):
        f.sweep(1)
        e.sweep(1)
        assert np.array_equal(e.get_spins(), f.get_spins() * g)
        assert e.measure_int()[0] == f.measure_int()[0]
        assert e.measure_int()[1] == int((f.get_spins().astype(np.int64) * g).sum())
        assert e.persistence() == f.persistence()                 # changes and s(0) s(t) are gauge invariant


def test_ea_bonds_from_seed_and_geometry():
    """D25: bond id b = a*N + i, group b>>2, word b&3, stream tag 3, tau = +1 iff the top bit is set.  One antiferro
    bond in the all-up state costs 2 in B; which two sites feel it fixes the (a, i) convention."""
    dims, L, seed = 3, 6, (7 << 33) + 5
    o = O.Oracle(dims, L, model=O.EA, T=2.0, seed=seed)
    N = o.N
    tau = o.get_bonds()
    want = np.array([[1 if words(seed, (a * N + i) >> 2, 0, 3)[(a * N + i) & 3] >> 31 else -1 for i in range(N)]
                     for a in range(dims)], dtype=np.int8)
    assert np.array_equal(tau, want)
    big = O.Oracle(2, 128, model=O.EA, T=2.0, seed=3).get_bonds()
    assert abs(big.mean()) < 5 / math.sqrt(big.size)               # +/-J with p = 1/2
    for a in range(dims):
        o.set_bonds(np.ones((dims, N), dtype=np.int8))
        o.set_spins(np.ones(N, dtype=np.int8), 0)
        assert o.measure_int() == (dims * N, N)
        t = np.ones((dims, N), dtype=np.int8)
        x, y, z = 2, 3, 4
        i = x + L * (y + L * z)
        t[a, i] = -1
        o.set_bonds(t)
        assert o.measure_int() == (dims * N - 2, N)
        # T -> 0+, h = 0: only sites with nn_eff <= 0 can flip; with one bad bond every site still has nn_eff >= 2d - 2 > 0
        cold = O.Oracle(dims, L, model=O.EA, T=1e-3, seed=1)
        cold.set_bonds(t)
        cold.set_spins(np.ones(N, dtype=np.int8), 0)
        cold.sweep(2)
        assert cold.measure_int() == (dims * N - 2, N)
        # the two ends of that bond, and nobody else, see a reduced field: flip them by a strong negative field on a
        # lattice where J is small -- instead check the local fields directly through one hot sweep's thresholds:
        # a site's flip probability at nn_eff = 2d - 2 differs from the bulk's at 2d.  Count flips over many seeds.
        j = [i + 1, i + L, i + L * L][a] if [x, y, z][a] + 1 < L else None
        assert j is not None
        flips = np.zeros(N)
        for sd in range(300):
            hot = O.Oracle(dims, L, model=O.EA, T=6.0, seed=1000 + sd)
            hot.set_bonds(t)
            hot.set_spins(np.ones(N, dtype=np.int8), 0)
            hot.sweep(1)
            flips += hot.get_spins() == -1
        par0 = [k for k in range(N) if ((k % L) + (k // L) % L + k // (L * L)) % 2 == 0]
        # compare within the colour updated first (their neighbours are still all up when they are visited)
        first = i if i in par0 else j
        rate_bulk = np.mean([flips[k] for k in par0 if k != first]) / 300
        p_bulk, p_end = math.exp(-2 * 2 * dims / 6.0), math.exp(-2 * (2 * dims - 2) / 6.0)
        assert abs(rate_bulk - p_bulk) < 0.01
        assert abs(flips[first] / 300 - p_end) < 5 * math.sqrt(p_end * (1 - p_end) / 300)


def ea_reference_sweep(s, tau, dims, L, J, h, T, seed, t):
    """Reading D25 on dicts: s[(x, y, z)], tau[(a, x, y, z)] = sign of the bond from (x, y, z) in direction +a."""
    def at(x, y, z):
        return s[(x % L, y % L, z % L if dims == 3 else 0)]

    def bond(a, x, y, z):
        return tau[(a, x % L, y % L, z % L if dims == 3 else 0)]

    sites = sorted(s.keys(), key=lambda p: (p[2], p[1], p[0]))
    for half in (0, 1):
        new = {}
        for (x, y, z) in sites:
            if (x + y + z) & 1 != half:
                continue
            nn = (bond(0, x, y, z) * at(x + 1, y, z) + bond(0, x - 1, y, z) * at(x - 1, y, z)
                  + bond(1, x, y, z) * at(x, y + 1, z) + bond(1, x, y - 1, z) * at(x, y - 1, z))
            if dims == 3:
                nn += bond(2, x, y, z) * at(x, y, z + 1) + bond(2, x, y, z - 1) * at(x, y, z - 1)
            k = (x + L * (y + L * z)) >> 1
            w = words(seed, k >> 2, t, half)[k & 3]
            v = s[(x, y, z)]
            new[(x, y, z)] = -v if w < thr_metropolis(J, h, T, v, -v, nn) else v
        s.update(new)


@pytest.mark.parametrize("dims,L,J,h,T", [(2, 4, 1.0, 0.0, 1.8), (2, 6, 1.0, 0.2, 1.2), (3, 4, 1.0, 0.0, 2.5), (3, 6, -0.7, 0.1, 2.0)])
def test_ea_sweep_matches_the_dict_restatement(dims, L, J, h, T):
    seed = (0xEA << 36) + 13 * L + dims
    o = O.Oracle(dims, L, model=O.EA, J=J, h=h, T=T, seed=seed)
    Lz = L if dims == 3 else 1
    sites = [(x, y, z) for z in range(Lz) for y in range(L) for x in range(L)]
    sp, tb = o.get_spins(), o.get_bonds()
    s = {p: int(sp[p[0] + L * (p[1] + L * p[2])]) for p in sites}
    tau = {(a, *p): int(tb[a, p[0] + L * (p[1] + L * p[2])]) for a in range(dims) for p in sites}
    t0 = (3 << 32) + 1
    o.set_spins(sp, t0)
    for k in range(4):
        ea_reference_sweep(s, tau, dims, L, J, h, T, seed, t0 + k)
        o.sweep(1)
        want = np.array([s[p] for p in sites], dtype=np.int8)
        assert np.array_equal(o.get_spins(), want), k
        B = sum(s[p] * sum(tau[(a, *p)] * s[tuple((p[i] + (1 if i == a else 0)) % (L if (i < 2 or dims == 3) else 1) for i in range(3))]
                           for a in range(dims)) for p in sites)
        assert o.measure_int() == (B, int(want.sum()))


@pytest.mark.slow
def test_ea_4x4_fixed_bonds_against_enumeration():
    """4x4 with a fixed random +/-J bond set: Boltzmann <E>/N by enumeration of the 2^16 states; one long chain."""
    T = 2.0
    o = O.Oracle(2, 4, model=O.EA, T=T, seed=20240229)
    tau = o.get_bonds()
    assert 8 <= int((tau == -1).sum()) <= 24                       # a genuinely mixed bond set
    e_ex, b_ex = X.ea4x4_exact(T, tau)
    o.sweep(2000)
    E = []
    for _ in range(60000):
        o.sweep(3)
        E.append(o.energy() / 16)
    e, se = X.binned_mean_err(E)
    assert abs(e - e_ex) < 3.5 * se and se < 4e-3, (e, e_ex, se)


# ============================================================================ Potts
def potts_thr(J, T, d):
    out = []
    for dn in range(-2 * d, 2 * d + 1):
        dE = -(J * float(dn))
        out.append(ALWAYS if dE <= 0.0 else thr_of(math.exp(-dE / T)))
    return out


def test_potts_table_and_q2_is_ising_at_half_coupling():
    for d, J, T in ((2, 1.0, 1.1), (3, 1.0, 1.8), (2, -0.5, 0.7)):
        p = O.Oracle(d, 8, two_S=2, model=O.POTTS, J=J, T=T, seed=1)
        assert p.thresholds() == potts_thr(J, T, d)
        # q = 2: flipping s with aligned-minus-antialigned neighbours s*nn = -(n_new - n_old) costs 2 (J/2) s nn
        p2 = O.Oracle(d, 8, two_S=1, model=O.POTTS, J=J, T=T, seed=1).thresholds()
        i = O.Oracle(d, 8, two_S=1, model=O.ISING, J=J / 2, T=T, seed=1).thresholds()     # idx b*(2d+1) + (nn+2d)/2
        for dn in range(-2 * d, 2 * d + 1, 2):
            snn = -dn
            assert p2[dn + 2 * d] == i[1 * (2 * d + 1) + (snn + 2 * d) // 2] == i[0 * (2 * d + 1) + (-snn + 2 * d) // 2]


def potts_reference(dims, L, q, J, T, seed, nsweeps, t0=0):
    """Reading D26 on a dict; returns the configuration after every sweep and the set of sites that ever changed."""
    Lz = L if dims == 3 else 1
    sites = [(x, y, z) for z in range(Lz) for y in range(L) for x in range(L)]
    s = {}
    for (x, y, z) in sites:
        i = x + L * (y + L * z)
        s[(x, y, z)] = (words(seed, i >> 2, 0, 2)[i & 3] * q) >> 32
    thr = potts_thr(J, T, dims)
    out, changed = [np.array([s[p] for p in sites], dtype=np.int8)], set()
    nbrs = [(-1, 0, 0), (1, 0, 0), (0, -1, 0), (0, 1, 0)] + ([(0, 0, -1), (0, 0, 1)] if dims == 3 else [])
    for k in range(nsweeps):
        for half in (0, 1):
            new = {}
            for (x, y, z) in sites:
                if (x + y + z) & 1 != half:
                    continue
                kk = (x + L * (y + L * z)) >> 1
                w4 = words(seed, kk >> 1, t0 + k, half)
                w0, w1 = w4[2 * (kk & 1)], w4[2 * (kk & 1) + 1]
                old = s[(x, y, z)]
                prop = (old + 1 + ((w0 * (q - 1)) >> 32)) % q
                nb = [s[((x + a) % L, (y + b) % L, (z + c) % L if dims == 3 else 0)] for a, b, c in nbrs]
                dn = nb.count(prop) - nb.count(old)
                new[(x, y, z)] = prop if w1 < thr[dn + 2 * dims] else old
            for p, v in new.items():
                if v != s[p]:
                    changed.add(p)
                s[p] = v
        out.append(np.array([s[p] for p in sites], dtype=np.int8))
    return out, changed, s, sites


@pytest.mark.parametrize("dims,L,q,J,T", [(2, 4, 3, 1.0, 1.0), (2, 6, 5, 1.0, 0.8), (2, 8, 2, 1.0, 1.2), (3, 4, 3, 1.0, 1.8),
                                          (3, 6, 4, -1.0, 1.5), (2, 6, 16, 1.0, 0.6)])
def test_potts_matches_the_dict_restatement(dims, L, q, J, T):
    seed = (0x9077 << 32) + 31 * L + q
    t0 = (1 << 32) - 2
    states, changed, s, sites = potts_reference(dims, L, q, J, T, seed, 4, t0)
    o = O.Oracle(dims, L, two_S=q - 1, model=O.POTTS, J=J, T=T, seed=seed)
    assert np.array_equal(o.get_spins(), states[0])
    o.set_spins(o.get_spins(), t0)
    for k in range(4):
        o.sweep(1)
        assert np.array_equal(o.get_spins(), states[k + 1]), k
    assert 0 < len(changed)
    nc, ov = o.persistence()
    assert nc == o.N - len(changed) and ov == int((states[0] == states[-1]).sum())
    a = states[-1].astype(np.int64).reshape((L,) * dims)
    B = sum(int((a == np.roll(a, -1, axis=ax)).sum()) for ax in range(dims))
    assert o.measure_int() == (B, int((a == 0).sum()))
    assert abs(o.energy() + J * B) < 1e-12


def test_potts_closed_forms():
    """(i) J = 0: every proposal costs nothing and is a different state: every site changes in every sweep, the state
    histogram stays uniform.  (ii) T -> 0+, J > 0, all sites equal: nothing can move (dn = -2d).  (iii) T -> 0+ from a
    random start: the number of equal bonds never decreases."""
    q, L = 4, 64
    o = O.Oracle(2, L, two_S=q - 1, model=O.POTTS, J=0.0, T=1.0, seed=5)
    before = o.get_spins().copy()
    o.sweep(1)
    after = o.get_spins()
    assert o.persistence()[0] == 0 and not np.any(before == after)
    counts = np.bincount(after, minlength=q) / o.N
    assert np.all(np.abs(counts - 1 / q) < 5 * math.sqrt((1 / q) * (1 - 1 / q) / o.N))
    assert set(np.unique(after)) == set(range(q))
    o = O.Oracle(3, 8, two_S=2, model=O.POTTS, J=1.0, T=1e-3, seed=6)
    o.set_spins(np.full(o.N, 2, dtype=np.int8), 0)
    o.sweep(3)
    assert o.measure_int() == (3 * o.N, 0) and o.persistence()[0] == o.N
    o = O.Oracle(2, 32, two_S=2, model=O.POTTS, J=1.0, T=1e-3, seed=7)
    last = o.measure_int()[0]
    for _ in range(10):
        o.sweep(1)
        b = o.measure_int()[0]
        assert b >= last
        last = b
    assert last > 1.3 * o.N                                        # coarsened well beyond the random-start 2N/3


@pytest.mark.slow
@pytest.mark.parametrize("q,T", [(3, 1.2), (2, 1.3)])
def test_potts_4x4_against_enumeration(q, T):
    """4x4 brute force (3^16 states for q = 3; the Ising enumeration at J/2 for q = 2): <E>/N (and <N0>/N = 1/q)."""
    o = O.Oracle(2, 4, two_S=q - 1, model=O.POTTS, J=1.0, T=T, seed=4321 + q)
    if q == 3:
        e_ex, c_ex, n0_ex, _ = X.potts3_4x4_exact(T)
        assert abs(n0_ex - 1 / 3) < 1e-12
    else:
        e_ex = X.potts2_4x4_exact(T)
    o.sweep(2000)
    E, N0 = [], []
    for _ in range(60000):
        o.sweep(3)
        B, M = o.measure_int()
        E.append(-B / 16)
        N0.append(M / 16)
    e, se = X.binned_mean_err(E)
    n0, sn = X.binned_mean_err(N0)
    assert abs(e - e_ex) < 3.5 * se and se < 4e-3, (e, e_ex, se)
    assert abs(n0 - 1 / q) < 3.5 * sn, (n0, sn)


def test_wider_models_reject_bad_arguments():
    with pytest.raises(ValueError):
        O.Oracle(2, 8, two_S=2, model=O.EA, T=1.0)                # EA is spin-1/2
    with pytest.raises(ValueError):
        O.Oracle(2, 8, two_S=0, model=O.POTTS, T=1.0)             # q >= 2
    with pytest.raises(ValueError):
        O.Oracle(2, 8, two_S=16, model=O.POTTS, T=1.0)            # q <= 16
    with pytest.raises(ValueError):
        O.Oracle(2, 8, two_S=2, model=O.POTTS, h=0.1, T=1.0)      # no field term in reading D26
    with pytest.raises(ValueError):
        O.Oracle(2, 8, T=1.0).set_bonds(np.ones((2, 64), dtype=np.int8))
