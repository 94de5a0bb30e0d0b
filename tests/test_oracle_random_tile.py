"""CPU pins of the oracle's random-tile schedule for the North-East model -- the paper's "corrected algorithm"
(steps 3-10; readings D17-D21 in DESIGN.md).  No GPU."""
import math

import numpy as np
import pytest

from oracle import lsm_oracle as O


def T_of_c(c):
    return 1.0 / math.log((1.0 - c) / c)


def philox_py(ctr, key):
    """Ten Philox4x32 rounds in python integers (independent of the C oracle; the oracle's own routine is
    pinned to the known-answer vectors in test_oracle_basics.py)."""
    c0, c1, c2, c3 = ctr
    k0, k1 = key
    for _ in range(10):
        p0, p1 = 0xD2511F53 * c0, 0xCD9E8D57 * c2
        c0, c1, c2, c3 = (p1 >> 32) ^ c1 ^ k0, p1 & 0xFFFFFFFF, (p0 >> 32) ^ c3 ^ k1, p0 & 0xFFFFFFFF
        k0, k1 = (k0 + 0x9E3779B9) & 0xFFFFFFFF, (k1 + 0xBB67AE85) & 0xFFFFFFFF
    return c0, c1, c2, c3


def reference_sweep(n, L, b, lam, seed, t, thr, metropolis):
    """The algorithm of PAPER.md:128-140 restated on a dict keyed by (x, y): per launch, per tile, q sub-steps of
    lam simultaneous random picks; boundary cells come from the lattice at launch start."""
    key = (seed & 0xFFFFFFFF, seed >> 32)
    P, nt = b * b, L // b
    q, calls = P // (2 * lam), (lam + 1) // 2
    changed = set()
    for launch in (0, 1):
        at_start = dict(n)
        for T in range(nt * nt):
            tx, ty = T % nt, T // nt
            inside = lambda x, y: tx * b <= x < (tx + 1) * b and ty * b <= y < (ty + 1) * b   # noqa: E731
            for k in range(q):
                writes = {}
                for j in range(lam):
                    w = philox_py((T, k * calls + (j >> 1), t & 0xFFFFFFFF, (4 + launch) | (((t >> 32) << 4) & 0xFFFFFFFF)), key)
                    w_pos, w_acc = w[2 * (j & 1)], w[2 * (j & 1) + 1]
                    r = (w_pos * P) >> 32
                    x, y = tx * b + r % b, ty * b + r // b
                    nb = []
                    for (xx, yy) in ((x, y + 1), (x + 1, y)):                  # north, east
                        nb.append(n[(xx, yy)] if inside(xx, yy) else at_start[(xx % L, yy % L)])
                    new = n[(x, y)]
                    if nb == [1, 1]:
                        if metropolis:
                            if new == 1 or w_acc < thr[1]:
                                new = 1 - new
                        else:
                            new = 1 if w_acc < thr[0] else 0
                    writes[(x, y)] = new                                       # a later thread overrides an earlier one
                for site, v in writes.items():
                    if n[site] != v:
                        changed.add(site)
                    n[site] = v
    return changed


@pytest.mark.parametrize("model", [O.NE_HEATBATH, O.NE_METROPOLIS])
@pytest.mark.parametrize("L,b,lam", [(8, 2, 2), (8, 4, 4), (12, 4, 1), (16, 8, 16), (8, 8, 1), (12, 6, 3)])
def test_matches_the_dict_restatement(model, L, b, lam):
    """Small lattices where collisions between the lam picks of a sub-step are frequent (b = 2, lam = 2: P = 4)."""
    c = 0.45
    o = O.Oracle(2, L, model=model, J=0.0, T=T_of_c(c), seed=(77 << 32) + 5 * L + b)
    thr = o.thresholds()
    s = o.get_spins().reshape(L, L)
    n = {(x, y): int(s[y, x]) for y in range(L) for x in range(L)}
    ever = set()
    for t in range(6):
        ever |= reference_sweep(n, L, b, lam, o.seed, t, thr, model == O.NE_METROPOLIS)
        o.sweep_random_tile(1, b, lam)
        got = o.get_spins().reshape(L, L)
        want = np.array([[n[(x, y)] for x in range(L)] for y in range(L)], dtype=np.int8)
        assert np.array_equal(got, want), (t, np.argwhere(got != want)[:4])
        assert o.persistence()[0] == L * L - len(ever)
    assert len(ever) > 0
    assert o.sweeps_done == 6


@pytest.mark.parametrize("b,lam", [(32, 16), (16, 4), (64, 1)])
def test_tile_order_is_immaterial(b, lam):
    """Reading D18 (boundaries frozen at launch start): each tile is handled once per launch (PAPER.md step 5), so
    which block takes which tile cannot matter -- ascending and descending tile order give the same lattice."""
    kw = dict(dims=2, L=64, model=O.NE_HEATBATH, J=0.0, T=T_of_c(0.35), seed=99)
    a, d = O.Oracle(**kw), O.Oracle(**kw)
    a.sweep_random_tile(5, b, lam, tiles_descending=False)
    d.sweep_random_tile(5, b, lam, tiles_descending=True)
    assert np.array_equal(a.get_spins(), d.get_spins())
    assert a.persistence() == d.persistence()


@pytest.mark.parametrize("model", [O.NE_HEATBATH, O.NE_METROPOLIS])
@pytest.mark.parametrize("c", [0.20, 0.42])
def test_product_measure_is_stationary(model, c):
    """Up-density stays at c (c is "also the equilibrium density"): a pick never reads the site it
    redraws, so the Bernoulli(c) product measure survives simultaneous and stale-boundary updates."""
    L = 192
    N = L * L
    o = O.Oracle(2, L, model=model, J=0.0, T=T_of_c(c), seed=4242 + int(100 * c))
    sigma = math.sqrt(c * (1 - c) / N)
    last = N
    obs = o.sweep_random_tile_record(40, 32, 16)
    assert np.all(obs[:, 0] == 0)
    assert np.all(np.abs(obs[:, 1] / N - c) < 4 * sigma), (obs[:, 1] / N, c, sigma)
    assert obs[-1, 1] == o.measure_int()[1]
    for _ in range(5):
        o.sweep_random_tile(1, 32, 16)
        nc, _ = o.persistence()
        assert nc <= last
        last = nc


@pytest.mark.parametrize("c", [0.20, 0.30, 0.42])
def test_first_sweep_persistence_closed_form(c):
    """One sweep = P random picks per tile of P sites, so a site is picked K ~ Binomial(P, 1/P) times.  Whether it is
    facilitated (probability c^2 at an i.i.d. start) hardly changes within one sweep -- its neighbours change at a
    rate of order c^3 -- so it is the same for all K picks; a facilitated site of value v survives a pick with
    probability 1 - p_v (p_1 = 1-c, p_0 = c: the heat-bath redraw differs):
    E[P(1)] = 1 - c^2 { 1 - [ c (1 - (1-c)/P)^P + (1-c) (1 - c/P)^P ] }."""
    L, b, lam = 512, 32, 16
    N, P = L * L, b * b
    o = O.Oracle(2, L, model=O.NE_HEATBATH, J=0.0, T=T_of_c(c), seed=31337 + int(1000 * c))
    o.sweep_random_tile(1, b, lam)
    nc, _ = o.persistence()
    want = 1 - c * c * (1 - (c * (1 - (1 - c) / P) ** P + (1 - c) * (1 - c / P) ** P))
    sigma = math.sqrt(want * (1 - want) / N)
    # lost writes of same-site collisions (< lam / 2P of the picks) and neighbours that change within the sweep
    # (order c^3 of them): second order
    assert abs(nc / N - want) < 5 * sigma, (nc / N, want, sigma)
    # and it must differ from the checkerboard sweep's 1 - 2c^3(1-c) where the two are far enough apart
    cb = 1 - 2 * c ** 3 * (1 - c)
    if abs(cb - want) > 12 * sigma:
        assert abs(nc / N - cb) > 5 * sigma


def test_frozen_set_bound_and_constraint_direction():
    """P13 under the random-tile schedule: initially-down sites whose north or east is in the frozen set never
    change, whatever the order of the picks (fixes north = y+1, east = x+1, both required)."""
    L, c = 64, 0.15
    o = O.Oracle(2, L, model=O.NE_HEATBATH, J=0.0, T=T_of_c(c), seed=1234)
    n0 = o.get_spins().reshape(L, L).astype(bool)
    Z = ~n0
    while True:
        keep = Z & (np.roll(Z, -1, axis=0) | np.roll(Z, -1, axis=1))
        if np.array_equal(keep, Z):
            break
        Z = keep
    blocked = np.roll(Z, -1, axis=0) | np.roll(Z, -1, axis=1)
    bound = int(blocked.sum())
    assert bound > 0
    for _ in range(20):
        o.sweep_random_tile(5, 32, 16)
        assert o.persistence()[0] >= bound
        s = o.get_spins().reshape(L, L)
        assert np.all(s[Z] == 0)
        assert np.array_equal(s[blocked].astype(bool), n0[blocked])


def test_serial_limit_relaxes_like_random_sequential_dynamics():
    """Q = lambda = 1 "is in fact serial": one tile = the whole lattice, one pick per sub-step, i.e.
    random-sequential dynamics with N picks per sweep.  Same closed form as above with P = N."""
    L, c = 128, 0.42
    N = L * L
    o = O.Oracle(2, L, model=O.NE_HEATBATH, J=0.0, T=T_of_c(c), seed=2024)
    o.sweep_random_tile(1, L, 1)
    nc = o.persistence()[0] / N
    want = 1 - c * c * (1 - (c * (1 - (1 - c) / N) ** N + (1 - c) * (1 - c / N) ** N))
    sigma = math.sqrt(want * (1 - want) / N)
    assert abs(nc - want) < 5 * sigma


def test_rejects_bad_schedules():
    o = O.Oracle(2, 64, model=O.NE_HEATBATH, J=0.0, T=1.0, seed=1)
    with pytest.raises(ValueError):
        o.sweep_random_tile(1, 24, 16)      # b does not divide L
    with pytest.raises(ValueError):
        o.sweep_random_tile(1, 32, 3)       # 2*lambda does not divide P
    i = O.Oracle(2, 64, T=2.0, seed=1)
    with pytest.raises(ValueError):
        i.sweep_random_tile(1, 32, 16)      # Ising: the schedule belongs to the North-East model


# ------------------------------------------------------------------ NEXT-2: the balance-preserving variant
def reference_sweep_balanced(n, L, b, lam, seed, t, thr, metropolis):
    """PAPER.md:148-158 on a dict keyed by (x, y): 4 launches; a sub-step = lam picks among the tile's red sites
    ((x+y) even), then lam picks among its white sites; one Philox call per thread and sub-step (D22-D24)."""
    key = (seed & 0xFFFFFFFF, seed >> 32)
    P, nt = b * b, L // b
    q = P // (8 * lam)
    changed = set()
    for launch in range(4):
        at_start = dict(n)
        for T in range(nt * nt):
            tx, ty = T % nt, T // nt
            sites = {col: [(tx * b + px, ty * b + py) for py in range(b) for px in range(b) if (px + py) % 2 == col]
                     for col in (0, 1)}                                # row-major list of each colour's sites
            for k in range(q):
                for col in (0, 1):
                    writes = {}
                    for j in range(lam):
                        w = philox_py((T, k * lam + j, t & 0xFFFFFFFF, (8 + launch) | (((t >> 32) << 4) & 0xFFFFFFFF)), key)
                        w_pos, w_acc = w[2 * col], w[2 * col + 1]
                        x, y = sites[col][(w_pos * (P // 2)) >> 32]
                        nb = []
                        for (xx, yy) in ((x, y + 1), (x + 1, y)):
                            ins = tx * b <= xx < (tx + 1) * b and ty * b <= yy < (ty + 1) * b
                            nb.append(n[(xx, yy)] if ins else at_start[(xx % L, yy % L)])
                        new = n[(x, y)]
                        if nb == [1, 1]:
                            if metropolis:
                                if new == 1 or w_acc < thr[1]:
                                    new = 1 - new
                            else:
                                new = 1 if w_acc < thr[0] else 0
                        writes[(x, y)] = new
                    for site, v in writes.items():
                        if n[site] != v:
                            changed.add(site)
                        n[site] = v
    return changed


@pytest.mark.parametrize("model", [O.NE_HEATBATH, O.NE_METROPOLIS])
@pytest.mark.parametrize("L,b,lam", [(8, 4, 2), (16, 8, 8), (12, 4, 1), (16, 16, 4), (24, 12, 2)])
def test_balanced_matches_the_dict_restatement(model, L, b, lam):
    c = 0.45
    o = O.Oracle(2, L, model=model, J=0.0, T=T_of_c(c), seed=(78 << 32) + 5 * L + b)
    thr = o.thresholds()
    s = o.get_spins().reshape(L, L)
    n = {(x, y): int(s[y, x]) for y in range(L) for x in range(L)}
    ever = set()
    for t in range(6):
        ever |= reference_sweep_balanced(n, L, b, lam, o.seed, t, thr, model == O.NE_METROPOLIS)
        o.sweep_random_tile_balanced(1, b, lam)
        got = o.get_spins().reshape(L, L)
        want = np.array([[n[(x, y)] for x in range(L)] for y in range(L)], dtype=np.int8)
        assert np.array_equal(got, want), (t, np.argwhere(got != want)[:4])
        assert o.persistence()[0] == L * L - len(ever)
    assert len(ever) > 0 and o.sweeps_done == 6


def test_balanced_tile_order_measure_and_persistence():
    """Tile order immaterial (D18); product measure stationary; one MC step attempts P updates per tile (D23), so the
    first-step persistence follows the closed form of the base algorithm with Binomial(P/2, 2/P) picks per site (the
    step draws P/2 picks for each colour, each uniform over that colour's P/2 sites)."""
    c, L, b, lam = 0.30, 256, 32, 16
    N, P = L * L, b * b
    kw = dict(dims=2, L=L, model=O.NE_HEATBATH, J=0.0, T=T_of_c(c), seed=5150)
    a, d = O.Oracle(**kw), O.Oracle(**kw)
    a.sweep_random_tile_balanced(1, b, lam)
    d.sweep_random_tile_balanced(1, b, lam, tiles_descending=True)
    assert np.array_equal(a.get_spins(), d.get_spins()) and a.persistence() == d.persistence()
    K = P // 2                                                         # picks that can hit a given site, each w.p. 2/P
    want = 1 - c * c * (1 - (c * (1 - (1 - c) * 2 / P) ** K + (1 - c) * (1 - c * 2 / P) ** K))
    sigma = math.sqrt(want * (1 - want) / N)
    assert abs(a.persistence()[0] / N - want) < 5 * sigma
    s = math.sqrt(c * (1 - c) / N)
    for _ in range(20):
        a.sweep_random_tile_balanced(1, b, lam)
        assert abs(a.measure_int()[1] / N - c) < 4 * s


def test_balanced_rejects_bad_schedules():
    o = O.Oracle(2, 64, model=O.NE_HEATBATH, J=0.0, T=1.0, seed=1)
    with pytest.raises(ValueError):
        o.sweep_random_tile_balanced(1, 32, 3)     # 8*lambda does not divide P
    with pytest.raises(ValueError):
        o.sweep_random_tile_balanced(1, 24, 2)     # b does not divide L
