"""CPU pins of the oracle's checkerboard sweep, initial state and overlap against a SECOND statement of the same
readings, written from the text of SURVEY.md 8(c) ("D2 detail", D3-D9, D11, D12) on a dict keyed by coordinates, with
Python integers and its own Philox.  What this fixes that statistics cannot see: the site -> (group, word, sweep-high-
bits, stream tag) map of D2, the value maps of D4, which word proposes and which accepts (D5), and the overlap of Eq. 4
 at t > 0.  tests/test_oracle_mutants.py breaks each of these in a copy of the oracle and checks that
this file notices.  No GPU."""
import itertools
import math

import numpy as np
import pytest

from oracle import lsm_oracle as O

M32 = 0xFFFFFFFF
ALWAYS = 1 << 32


def philox_py(ctr, key):
    """Philox4x32-10 from the round definition of D2 (independent of the C oracle)."""
    c0, c1, c2, c3 = ctr
    k0, k1 = key
    for _ in range(10):
        p0, p1 = 0xD2511F53 * c0, 0xCD9E8D57 * c2
        c0, c1, c2, c3 = (p1 >> 32) ^ c1 ^ k0, p1 & M32, (p0 >> 32) ^ c3 ^ k1, p0 & M32
        k0, k1 = (k0 + 0x9E3779B9) & M32, (k1 + 0xBB67AE85) & M32
    return c0, c1, c2, c3


def test_python_philox_known_answers():
    """P1: the restatement's own Philox against the published vectors (tests/golden/philox4x32_10_kat.txt)."""
    assert philox_py((0, 0, 0, 0), (0, 0)) == (0x6627E8D5, 0xE169C58D, 0xBC57AC4C, 0x9B00DBD8)
    assert philox_py((M32,) * 4, (M32, M32)) == (0x408F276D, 0x41C83B0E, 0xA20BC7C6, 0x6D5451FD)
    assert philox_py((0x243F6A88, 0x85A308D3, 0x13198A2E, 0x03707344), (0xA4093822, 0x299F31D0)) == (
        0xD16CFE09, 0x94FDCCEB, 0x5001E420, 0x24126EA1)


def words(seed, group, t, tag):
    """D2 detail: key = seed; counter (lo32 g, hi32 g, lo32 t, tag | hi32(t) << 4)."""
    return philox_py((group & M32, group >> 32, t & M32, (tag | ((t >> 32) << 4)) & M32), (seed & M32, seed >> 32))


def thr_of(p):
    return ALWAYS if p >= 1.0 else int(math.floor(math.ldexp(p, 32)))


def thr_metropolis(J, h, T, s_old, s_new, nn):
    """D3, keyed by what the move IS (old value, new value, neighbour sum) rather than by a table index."""
    dE = -float(s_new - s_old) * (J * float(nn) + h)
    return ALWAYS if dE <= 0.0 else thr_of(math.exp(-dE / T))


class Restated:
    """The algorithm box of SURVEY.md 8(c) on a dict {(x, y, z): value}."""

    def __init__(self, dims, L, two_S, model, J, h, T, seed):
        self.d, self.L, self.two_S, self.model, self.J, self.h, self.T, self.seed = dims, L, two_S, model, J, h, T, seed
        self.c = 1.0 / (1.0 + math.exp(1.0 / T))                       # D6
        Lz = L if dims == 3 else 1
        self.sites = [(x, y, z) for z in range(Lz) for y in range(L) for x in range(L)]
        self.s = {}
        for (x, y, z) in self.sites:                                    # D4: stream 2, t = 0, canonical id
            i = x + L * (y + L * z)
            w = words(seed, i >> 2, 0, 2)[i & 3]
            if model != O.ISING:
                self.s[(x, y, z)] = 1 if w < thr_of(self.c) else 0
            elif two_S == 1:
                self.s[(x, y, z)] = 1 if (w >> 31) else -1
            else:
                self.s[(x, y, z)] = ((w * 3) >> 32) - 1
        self.s0 = dict(self.s)
        self.changed = set()
        self.t = 0

    def at(self, x, y, z):
        L = self.L
        return self.s[(x % L, y % L, z % L if self.d == 3 else 0)]

    def sweep(self):
        L = self.L
        for half in (0, 1):                                             # D9: the parity of the origin first
            new = {}
            for (x, y, z) in self.sites:
                if (x + y + z) & 1 != half:
                    continue
                i = x + L * (y + L * z)
                k = i >> 1                                              # compact index = byte offset in its colour
                s = self.s[(x, y, z)]
                if self.model == O.ISING:
                    nn = self.at(x - 1, y, z) + self.at(x + 1, y, z) + self.at(x, y - 1, z) + self.at(x, y + 1, z)
                    if self.d == 3:
                        nn += self.at(x, y, z - 1) + self.at(x, y, z + 1)
                    if self.two_S == 1:                                 # one word per site: group k>>2, word k&3
                        w = words(self.seed, k >> 2, self.t, half)[k & 3]
                        if w < thr_metropolis(self.J, self.h, self.T, s, -s, nn):
                            s = -s
                    else:                                               # D5: two words per site, group k>>1
                        w4 = words(self.seed, k >> 1, self.t, half)
                        w0, w1 = w4[2 * (k & 1)], w4[2 * (k & 1) + 1]
                        kk = w0 >> 31
                        prop = (-1, 0, 1)[(s + 1 + 1 + kk) % 3]
                        if w1 < thr_metropolis(self.J, self.h, self.T, s, prop, nn):
                            s = prop
                else:                                                   # D7, D8
                    if self.at(x, y + 1, z) == 1 and self.at(x + 1, y, z) == 1:
                        w = words(self.seed, k >> 2, self.t, half)[k & 3]
                        if self.model == O.NE_HEATBATH:
                            s = 1 if w < thr_of(self.c) else 0
                        elif s == 1 or w < thr_of(math.exp(-1.0 / self.T)):
                            s = 1 - s
                new[(x, y, z)] = s
            for site, v in new.items():
                if v != self.s[site]:
                    self.changed.add(site)                              # D12
                self.s[site] = v
        self.t += 1

    def array(self):
        return np.array([self.s[p] for p in self.sites], dtype=np.int8)

    def overlap(self):
        f = (lambda v: v) if self.model == O.ISING else (lambda v: 2 * v - 1)   # D11
        return sum(f(self.s0[p]) * f(self.s[p]) for p in self.sites)

    def bond_sum_and_M(self):
        B = 0
        for (x, y, z) in self.sites:
            f = self.at(x + 1, y, z) + self.at(x, y + 1, z) + (self.at(x, y, z + 1) if self.d == 3 else 0)
            B += self.s[(x, y, z)] * f
        return (B if self.model == O.ISING else 0), sum(self.s.values())


CASES = [
    # dims, L, two_S, model, J, h, T
    (2, 4, 1, O.ISING, 1.0, 0.0, 2.269),
    (2, 6, 1, O.ISING, 1.0, 0.3, 1.7),
    (2, 8, 1, O.ISING, -1.0, 0.1, 2.5),
    (3, 4, 1, O.ISING, 1.0, 0.0, 4.5115),
    (3, 6, 1, O.ISING, 1.0, -0.2, 3.0),
    (3, 8, 1, O.ISING, 1.0, 0.0, 4.0),
    (2, 4, 2, O.ISING, 1.0, 0.01, 3.0),
    (2, 6, 2, O.ISING, 1.0, 0.4, 1.5),
    (2, 8, 2, O.ISING, 0.7, 0.0, 2.0),
    (3, 4, 2, O.ISING, 1.0, 0.01, 3.0),
    (3, 6, 2, O.ISING, 1.0, 0.2, 2.2),
    (3, 8, 2, O.ISING, 1.0, 0.01, 3.0),
    (2, 4, 1, O.NE_HEATBATH, 0.0, 0.0, 1.0 / math.log(0.58 / 0.42)),
    (2, 6, 1, O.NE_HEATBATH, 0.0, 0.0, 1.180223),
    (2, 8, 1, O.NE_HEATBATH, 0.0, 0.0, 5.0),
    (2, 4, 1, O.NE_METROPOLIS, 0.0, 0.0, 1.0 / math.log(0.58 / 0.42)),
    (2, 6, 1, O.NE_METROPOLIS, 0.0, 0.0, 1.180223),
    (2, 8, 1, O.NE_METROPOLIS, 0.0, 0.0, 5.0),
]


@pytest.mark.parametrize("dims,L,two_S,model,J,h,T", CASES)
def test_init_matches_the_restatement(dims, L, two_S, model, J, h, T):
    """D4: canonical id, group i>>2, word i&3, stream tag 2; value maps of the three models."""
    seed = (0x1209 << 40) + 977 * L + 31 * dims + two_S + 5 * model
    o = O.Oracle(dims, L, two_S, model, J, h, T, seed)
    r = Restated(dims, L, two_S, model, J, h, T, seed)
    assert np.array_equal(o.get_spins(), r.array())
    assert o.measure_int() == r.bond_sum_and_M()
    assert o.persistence() == (o.N, r.overlap())         # overlap(0) = sum sigma^2 (= N unless spin-1 has zeros)


@pytest.mark.parametrize("t0", [0, (1 << 32) - 2, (7 << 32) + 3])
@pytest.mark.parametrize("dims,L,two_S,model,J,h,T", CASES)
def test_checkerboard_sweep_matches_the_restatement(dims, L, two_S, model, J, h, T, t0):
    """Four sweeps, compared after each: configuration, (B, M), never-changed count and overlap.  t0 moves the sweep
    counter across 2^32 (the high bits enter c3 above the stream tag, D2)."""
    seed = (0x0296 << 44) + 1013 * L + 17 * dims + two_S + 3 * model
    o = O.Oracle(dims, L, two_S, model, J, h, T, seed)
    r = Restated(dims, L, two_S, model, J, h, T, seed)
    o.set_spins(o.get_spins(), t0)
    r.t = t0
    moved = False
    for _ in range(4):
        o.sweep(1)
        r.sweep()
        assert np.array_equal(o.get_spins(), r.array()), (r.t, np.flatnonzero(o.get_spins() != r.array())[:8])
        assert o.measure_int() == r.bond_sum_and_M()
        assert o.persistence() == (o.N - len(r.changed), r.overlap())
        moved |= len(r.changed) > 0
    assert moved and o.sweeps_done == t0 + 4


def test_counter_fields_never_alias():
    """the stream tag owns the low four bits of c3, so the (c2, c3) pairs of all tags in use
    (0, 1 half-sweeps; 2 init; 4, 5 random tiles; 8..11 balanced variant) are pairwise distinct for every t, and the
    words of sweep t and t + 2^32 differ for each of them."""
    tags = [0, 1, 2, 4, 5, 8, 9, 10, 11]
    seen = {}
    for hi, lo, tag in itertools.product([0, 1, 2, 5, (1 << 28) - 1], [0, 7], tags):
        t = (hi << 32) + lo
        c23 = (t & M32, (tag | ((t >> 32) << 4)) & M32)
        assert c23 not in seen, (t, tag, seen[c23])
        seen[c23] = (t, tag)
    # the oracle draws different lattices at t and t + 2^32 under every schedule
    for kind in ("checkerboard", "tile", "balanced"):
        out = []
        for t0 in (3, 3 + (1 << 32), 3 + (2 << 32), 3 + (4 << 32)):
            o = O.Oracle(2, 16, model=O.NE_HEATBATH, J=0.0, T=5.0, seed=99)
            o.set_spins(o.get_spins(), t0)
            {"checkerboard": lambda: o.sweep(1), "tile": lambda: o.sweep_random_tile(1, 8, 4),
             "balanced": lambda: o.sweep_random_tile_balanced(1, 8, 4)}[kind]()
            out.append(o.get_spins().tobytes())
        assert len(set(out)) == len(out), kind
    # and the three schedules do not replay one another's words at shifted high bits
    a = O.Oracle(2, 16, model=O.NE_HEATBATH, J=0.0, T=5.0, seed=99)
    a.sweep_random_tile(1, 8, 4)
    for hi in (1, 2):
        b = O.Oracle(2, 16, model=O.NE_HEATBATH, J=0.0, T=5.0, seed=99)
        b.set_spins(b.get_spins(), hi << 32)
        b.sweep_random_tile_balanced(1, 8, 4)
        assert a.get_spins().tobytes() != b.get_spins().tobytes()


# ------------------------------------------------------------------------- overlap, Eq. 4, at t > 0
@pytest.mark.parametrize("kind", ["ising", "spin1", "ne_checkerboard", "ne_tile", "ne_balanced"])
def test_overlap_from_two_snapshots(kind):
    """overlap(t) = sum_i sigma_i(ref) sigma_i(t) recomputed in numpy from get_spins() snapshots; reference moved by
    reset_reference() in mid-run; never_changed bounded by the sites that differ between the snapshots."""
    if kind == "ising":
        o = O.Oracle(2, 32, T=2.5, seed=11)
    elif kind == "spin1":
        o = O.Oracle(3, 8, two_S=2, T=3.0, h=0.01, seed=12)
    else:
        o = O.Oracle(2, 32, model=O.NE_HEATBATH, J=0.0, T=1.0 / math.log(0.58 / 0.42), seed=13)
    step = {"ne_tile": lambda n: o.sweep_random_tile(n, 8, 4),
            "ne_balanced": lambda n: o.sweep_random_tile_balanced(n, 8, 4)}.get(kind, lambda n: o.sweep(n))
    sig = (lambda a: a.astype(np.int64)) if kind in ("ising", "spin1") else (lambda a: 2 * a.astype(np.int64) - 1)
    ref = sig(o.get_spins())
    seen_below = False
    for n in (1, 2, 5):
        step(n)
        now = sig(o.get_spins())
        nc, ov = o.persistence()
        assert ov == int((ref * now).sum())
        assert nc <= int((ref == now).sum())
        seen_below |= ov < int((ref * ref).sum())
    assert seen_below                                      # the configuration did move away from the reference
    o.reset_reference()
    ref = sig(o.get_spins())
    assert o.persistence() == (o.N, int((ref * ref).sum()))
    step(3)
    assert o.persistence()[1] == int((ref * sig(o.get_spins())).sum())


def test_overlap_closed_forms():
    """(i) T -> infinity, h = 0: every proposed flip has exp(-dE/T) = 1 - O(1e-12), threshold 2^32 - 1 or 2^32, so
    every spin flips in every sweep (unless w = 2^32 - 1): overlap(1) = -N, overlap(2) = +N, never_changed(1) = 0.
    (ii) strong field, low T, J = 0: after one sweep every spin is +1 (flip up certain, flip down exp(-2h/T) = 0):
    overlap(t >= 1) = M(0), never_changed = number of sites that started up.
    (iii) North-East at c = 0.47 >> c*: after decorrelation overlap/N -> (2c-1)^2 (product measure)."""
    o = O.Oracle(2, 32, T=1e12, seed=5)
    N = o.N
    o.sweep(1)
    assert o.persistence() == (0, -N)
    o.sweep(1)
    assert o.persistence() == (0, N)
    o = O.Oracle(3, 8, J=0.0, h=50.0, T=0.05, seed=6)
    M0 = o.measure_int()[1]
    for _ in range(3):
        o.sweep(1)
        assert o.measure_int()[1] == o.N
        assert o.persistence() == ((o.N + M0) // 2, M0)
    c, L = 0.47, 64                                        # far above c* ~ 0.3: decorrelates within ~1e4 sweeps
    o = O.Oracle(2, L, model=O.NE_HEATBATH, J=0.0, T=1.0 / math.log((1 - c) / c), seed=7)
    o.sweep(12000)
    assert o.persistence()[0] == 0
    ov = o.persistence()[1] / o.N
    q = (2 * c - 1) ** 2
    # sigma_i(0) sigma_i(t) for independent Bernoulli(c) values: mean q, variance 1 - q^2
    assert abs(ov - q) < 5 * math.sqrt((1 - q * q) / o.N), (ov, q)
    assert abs(O.phi(o.persistence()[1], o.N, c)) < 5 * math.sqrt((1 - q * q) / o.N) / (1 - q)


def test_balanced_record_is_the_sweep_plus_measure():
    kw = dict(dims=2, L=32, model=O.NE_METROPOLIS, J=0.0, T=1.2, seed=21)
    a, b = O.Oracle(**kw), O.Oracle(**kw)
    obs = a.sweep_random_tile_balanced_record(5, 8, 2)
    for k in range(5):
        b.sweep_random_tile_balanced(1, 8, 2)
        assert tuple(obs[k]) == b.measure_int()
    assert np.array_equal(a.get_spins(), b.get_spins())
