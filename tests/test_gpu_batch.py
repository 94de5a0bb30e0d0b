"""GPU parity of the batch calls (many small lattices in one launch):
every replica of a batch must end exactly as a single lattice with its temperature and seed does under the oracle."""
import numpy as np
import pytest

from oracle import lsm_oracle as O
from paper_1209_0296_b200 import build as B
from paper_1209_0296_b200 import lsm
from paper_1209_0296_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _built():
    B.build()
    lsm.load()


def oracles(kw, T, seeds):
    return [O.Oracle(T=t, seed=s, **kw) for t, s in zip(T, seeds)]


def check_all(batch, orcs, persistence=True):
    bm = batch.measure_int()
    for r, o in enumerate(orcs):
        v = batch.replica(r)
        assert np.array_equal(v.get_spins().cpu().numpy(), o.get_spins()), f"replica {r}"
        assert bm[r] == o.measure_int(), f"replica {r}"
        assert v.measure_int() == (*o.measure_int(), o.sweeps_done)
        assert v.measure_full() == o.measure_int()
        if persistence:
            assert v.persistence() == o.persistence(), f"replica {r}"


CASES = [
    # kwargs of the shape, R, sweeps
    (dict(dims=2, L=128), 32, 12),                                           # the verdict's case: 32 x 128^2
    (dict(dims=2, L=16), 5, 30),
    (dict(dims=2, L=64, h=0.05, J=0.8), 7, 20),
    (dict(dims=3, L=16), 6, 10),
    (dict(dims=3, L=32, two_S=2, h=0.01), 3, 6),
    (dict(dims=2, L=32, two_S=2, h=0.2), 9, 15),
    (dict(dims=2, L=64, model=lsm.NE_HEATBATH, J=0.0), 8, 25),
    (dict(dims=2, L=32, model=lsm.NE_METROPOLIS, J=0.0), 4, 25),
]


@pytest.mark.parametrize("kw,R,n", CASES)
def test_batch_matches_independent_oracles(kw, R, n):
    """Different seeds AND temperatures per replica; record, no-record and tracking-off sweeps; set_temperatures."""
    ne = kw.get("model", lsm.ISING) != lsm.ISING
    T = [W.ne_temperature(0.15 + 0.3 * r / R) for r in range(R)] if ne else [1.8 + 1.7 * r / R for r in range(R)]
    seeds = [W.seed_of(9, 3) + 17 * r + R for r in range(R)]
    batch = lsm.Batch(T=T, seeds=seeds, **kw)
    orcs = oracles(kw, T, seeds)
    check_all(batch, orcs)                                                    # the initial states
    got = batch.sweep_record(n).cpu().numpy()
    for r, o in enumerate(orcs):
        want = o.sweep_record(n)
        assert np.array_equal(got[r], want), (r, np.flatnonzero((got[r] != want).any(axis=1))[:4])
    check_all(batch, orcs)
    batch.sweep(3)                                                            # last sweep measured only
    batch.sweep(1)
    for o in orcs:
        o.sweep(4)
    check_all(batch, orcs)
    T2 = list(reversed(T))
    batch.set_temperatures(T2)
    for o, t in zip(orcs, T2):
        o.set_temperature(t)
    assert batch.replica(1).thresholds() == orcs[1].thresholds()
    batch.set_tracking(False)
    got = batch.sweep_record(5).cpu().numpy()
    for r, o in enumerate(orcs):
        assert np.array_equal(got[r], o.sweep_record(5))
    check_all(batch, orcs, persistence=False)
    batch.close()


def test_batch_is_one_launch_and_cluster_sizes_agree():
    kw = dict(dims=2, L=128)
    R = 12
    T = [2.0 + 0.05 * r for r in range(R)]
    seeds = [1000 + r for r in range(R)]
    ref = None
    for c in (0, 1, 2, 4, 8, 16):
        batch = lsm.Batch(T=T, seeds=seeds, **kw)
        batch.set_cluster(c)
        n0 = batch.launch_count
        got = batch.sweep_record(20).cpu().numpy()
        assert batch.launch_count - n0 == 1            # ONE launch for R lattices x 20 sweeps
        n0 = batch.launch_count
        batch.sweep(7)
        assert batch.launch_count - n0 == 2            # 6 unmeasured sweeps + the measured last one
        state = [batch.replica(r).get_spins().cpu().numpy().copy() for r in range(R)]
        if ref is None:
            ref = (got, state)
        else:
            assert np.array_equal(got, ref[0])
            assert all(np.array_equal(a, b) for a, b in zip(state, ref[1]))
        batch.close()
    o = O.Oracle(T=T[5], seed=seeds[5], **kw)
    assert np.array_equal(ref[0][5], o.sweep_record(20))


def test_batch_more_replicas_than_one_launch_holds():
    """300 replicas of 16^2: two launches (256 + 44); spot-check replicas on both sides of the cut."""
    R = 300
    T = [2.269] * R
    seeds = [77 + r for r in range(R)]
    batch = lsm.Batch(dims=2, L=16, T=T, seeds=seeds)
    n0 = batch.launch_count
    got = batch.sweep_record(10).cpu().numpy()
    assert batch.launch_count - n0 == 2
    for r in (0, 1, 255, 256, 299):
        o = O.Oracle(2, 16, T=T[r], seed=seeds[r])
        assert np.array_equal(got[r], o.sweep_record(10)), r
        assert np.array_equal(batch.replica(r).get_spins().cpu().numpy(), o.get_spins())
    batch.close()


@pytest.mark.parametrize("kw", [dict(dims=2, L=34), dict(dims=2, L=96), dict(dims=2, L=64, Tlow=True)])
def test_batch_falls_back_to_one_replica_after_the_other(kw):
    """Lattices the one-launch kernel does not cover (L not a power of two; a table with a 'never' entry) still work."""
    kw = dict(kw)
    low = kw.pop("Tlow", False)
    R = 3
    T = [0.05, 2.0, 0.07] if low else [2.0, 2.3, 2.6]
    seeds = [5, 6, 7]
    batch = lsm.Batch(T=T, seeds=seeds, **kw)
    orcs = oracles(kw, T, seeds)
    got = batch.sweep_record(8).cpu().numpy()
    for r, o in enumerate(orcs):
        assert np.array_equal(got[r], o.sweep_record(8))
    check_all(batch, orcs)
    batch.close()


def test_batch_lockstep_and_argument_errors():
    batch = lsm.Batch(dims=2, L=32, T=[2.0, 2.5], seeds=[1, 2])
    batch.replica(0).sweep(1)                          # one replica runs ahead on its own
    with pytest.raises(lsm.LsmError) as e:
        batch.sweep(1)
    assert e.value.code == lsm.ERR_STATE
    batch.replica(1).sweep(1)
    batch.sweep(1)                                     # back in lockstep
    with pytest.raises(lsm.LsmError):
        batch.set_cluster(3)
    with pytest.raises(lsm.LsmError):
        batch.set_temperatures([1.0, -1.0])
    batch.close()
    with pytest.raises(lsm.LsmError):
        lsm.Batch(dims=2, L=33, T=[2.0], seeds=[1])


@pytest.mark.parametrize("model", [lsm.NE_HEATBATH, lsm.NE_METROPOLIS])
@pytest.mark.parametrize("L,R,b,lam,balanced", [
    (128, 30, 32, 16, False),          # the paper's case: 30 realisations of 128^2, 32 x 32 tiles, lambda = 16
    (128, 30, 32, 16, True),
    (64, 7, 8, 32, False),             # collisions in almost every sub-step; R * tiles is odd per warp pair
    (64, 5, 16, 4, True),
    (96, 3, 32, 1, False),             # lambda = 1: one lane per tile, 9 tiles per lattice (groups of a warp in different lattices)
    (512, 4, 32, 16, False),
    (256, 3, 128, 4, False),           # tiles too large for every group of a warp to hold one
])
def test_batch_random_tile_matches_independent_oracles(model, L, R, b, lam, balanced):
    """lsm_batch_sweep_random_tile (SURVEY.md 8(f) NEXT-1 x NEXT-3): every replica must end exactly as the
    oracle's random-tile schedule leaves a single lattice with its temperature and seed -- recorded series, unrecorded
    sweeps, mixed with checkerboard batch sweeps, persistence included."""
    kw = dict(dims=2, L=L, model=model, J=0.0)
    T = [W.ne_temperature(0.2 + 0.25 * r / R) for r in range(R)]
    seeds = [W.seed_of(12, 1) + 13 * r for r in range(R)]
    batch = lsm.Batch(T=T, seeds=seeds, **kw)
    orcs = oracles(kw, T, seeds)
    rec = (lambda o, n: o.sweep_random_tile_balanced_record(n, b, lam)) if balanced else (lambda o, n: o.sweep_random_tile_record(n, b, lam))
    n = 4
    l0 = batch.launch_count
    got = batch.sweep_random_tile(n, b, lam, record=True, balanced=balanced).cpu().numpy()
    assert batch.launch_count - l0 == n * (4 if balanced else 2)            # launches do not grow with R
    for r, o in enumerate(orcs):
        assert np.array_equal(got[r], rec(o, n)), r
    check_all(batch, orcs)
    batch.sweep_random_tile(3, b, lam, balanced=balanced)                   # only the last sweep is measured
    batch.sweep(2)                                                          # checkerboard sweeps of the same batch in between
    got = batch.sweep_random_tile(1, b, lam, record=True, balanced=balanced).cpu().numpy()
    for r, o in enumerate(orcs):
        rec(o, 3)
        o.sweep(2)
        assert np.array_equal(got[r], rec(o, 1)), r
    check_all(batch, orcs)
    # a replica swept on its own puts the batch out of lockstep
    batch.replica(1).sweep_random_tile(1, b, lam, balanced=balanced)
    with pytest.raises(lsm.LsmError) as e:
        batch.sweep_random_tile(1, b, lam, balanced=balanced)
    assert e.value.code == lsm.ERR_STATE
    batch.close()


def test_batch_random_tile_argument_checks():
    batch = lsm.Batch(T=[2.0, 2.1], seeds=[1, 2], dims=2, L=64)
    with pytest.raises(lsm.LsmError) as e:
        batch.sweep_random_tile(1, 32, 16)                                  # Ising batch
    assert e.value.code == lsm.ERR_UNSUPPORTED
    batch.close()
    batch = lsm.Batch(T=[1.0, 1.1], seeds=[1, 2], dims=2, L=64, model=lsm.NE_HEATBATH, J=0.0)
    with pytest.raises(lsm.LsmError) as e:
        batch.sweep_random_tile(1, 24, 16)                                  # tile edge not a power of two
    assert e.value.code == lsm.ERR_UNSUPPORTED
    assert batch.sweep_random_tile(0, 32, 16) is None
    batch.close()
