"""One small case per kernel family and synchronisation scheme, each held to the oracle: a quick GPU test on its own, and
the file to point `compute-sanitizer` at ("Race detection / sanitizers") where that tool may run -- on this
GPU pool it is closed, so these oracle comparisons are the stand-in.  Shapes are the smallest each family
accepts so that memcheck / racecheck / synccheck would finish in minutes: generic (one thread per site), tiled (cp.async ring), bulk (cp.async.bulk + mbarrier ring), small (cluster
barriers + distributed shared memory, also 16 blocks per lattice through the batch call), slab (L2 mailboxes, temporal
depths 1-4), the random-tile kernel (claim bytes, collisions), Edwards-Anderson
and Potts."""
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


def check(kw, family, n=3, depth=None):
    lat, orc = lsm.Lattice(**kw), O.Oracle(**kw)
    try:
        lat.set_kernel(family)
    except lsm.LsmError as e:
        assert e.code == lsm.ERR_UNSUPPORTED
        pytest.skip("family does not run this lattice")
    if depth is not None:
        lat.set_temporal_depth(depth)
    assert np.array_equal(lat.sweep_record(n).cpu().numpy(), orc.sweep_record(n))
    lat.sweep(2)
    orc.sweep(2)
    assert np.array_equal(lat.get_spins().cpu().numpy(), orc.get_spins())
    assert lat.measure_int() == (*orc.measure_int(), n + 2) and lat.measure_full() == orc.measure_int()
    assert lat.persistence() == orc.persistence()
    lat.close()


NE = dict(model=lsm.NE_HEATBATH, J=0.0, T=W.ne_temperature(0.25))


@pytest.mark.parametrize("kw", [dict(dims=2, L=6, T=2.0, seed=1), dict(dims=3, L=4, two_S=2, T=3.0, h=0.1, seed=2),
                                dict(dims=2, L=10, seed=3, **NE)])
def test_generic(kw):
    check(kw, lsm.KERNEL_GENERIC)


@pytest.mark.parametrize("kw", [dict(dims=2, L=64, T=2.269, seed=4), dict(dims=3, L=32, two_S=2, T=3.0, h=0.01, seed=5),
                                dict(dims=2, L=64, seed=6, **NE), dict(dims=3, L=32, model=lsm.EA, T=1.1, seed=7),
                                dict(dims=2, L=64, two_S=2, model=lsm.POTTS, T=0.995, seed=8),
                                dict(dims=2, L=64, T=0.2, seed=9)])                  # "never" thresholds
def test_tiled(kw):
    check(kw, lsm.KERNEL_TILED)


@pytest.mark.parametrize("kw", [dict(dims=2, L=64, T=2.269, seed=10), dict(dims=3, L=16, T=4.5, seed=11),
                                dict(dims=2, L=32, two_S=2, T=1.7, seed=12), dict(dims=2, L=256, seed=13, **NE)])
def test_small_cluster(kw):
    check(kw, lsm.KERNEL_SMALL)


@pytest.mark.parametrize("depth", [1, 2, 3, 4])
def test_slab_depths(depth):
    check(dict(dims=2, L=512, T=2.269, seed=14), lsm.KERNEL_SLAB, n=3, depth=depth)


@pytest.mark.parametrize("kw", [dict(dims=2, L=128, model=lsm.EA, T=0.9, seed=15), dict(dims=3, L=32, two_S=3, model=lsm.POTTS, T=1.5, seed=16),
                                dict(dims=3, L=64, T=4.5115, seed=17), dict(dims=2, L=512, seed=18, **NE)])
def test_slab_models(kw):
    check(kw, lsm.KERNEL_SLAB)


def test_resident_family_is_gone():
    lat = lsm.Lattice(dims=2, L=1024, T=2.269, seed=19)
    with pytest.raises(lsm.LsmError) as e:
        lat.set_kernel(lsm.KERNEL_RESIDENT)            # removed in round 3: the value is reserved, the call refuses it
    assert e.value.code == lsm.ERR_UNSUPPORTED and lat.kernel == lsm.KERNEL_SLAB


def test_bulk_against_tiled():
    """8192^2 is the smallest lattice of the bulk-copy family; its oracle parity at that size is in test_gpu_parity.py.
    Here: two sweeps against the tiled family, and one oracle sweep from the resulting state."""
    kw = dict(dims=2, L=8192, T=2.269, seed=20)
    a, b = lsm.Lattice(**kw), lsm.Lattice(**kw)
    a.set_kernel(lsm.KERNEL_BULK)
    b.set_kernel(lsm.KERNEL_TILED)
    assert np.array_equal(a.sweep_record(2).cpu().numpy(), b.sweep_record(2).cpu().numpy())
    assert np.array_equal(a.get_spins_host(), b.get_spins_host())


@pytest.mark.parametrize("balanced", [False, True])
def test_random_tile_with_collisions(balanced):
    """8 x 8 tiles with 32 (unbalanced) or 8 (balanced) picks per sub-step out of 64 (32) sites: same-site collisions in
    almost every sub-step (reading D20: the highest thread wins)."""
    kw = dict(dims=2, L=64, seed=21, **NE)
    lam = 8 if balanced else 32
    lat, orc = lsm.Lattice(**kw), O.Oracle(**kw)
    got = lat.sweep_random_tile(4, 8, lam, record=True, balanced=balanced).cpu().numpy()
    want = orc.sweep_random_tile_balanced_record(4, 8, lam) if balanced else orc.sweep_random_tile_record(4, 8, lam)
    assert np.array_equal(got, want)
    assert np.array_equal(lat.get_spins().cpu().numpy(), orc.get_spins()) and lat.persistence() == orc.persistence()


@pytest.mark.parametrize("cluster", [0, 16])
def test_batch(cluster):
    kw, R = dict(dims=2, L=256), 3
    T, seeds = [2.0, 2.269, 2.6], [31, 32, 33]
    batch = lsm.Batch(T=T, seeds=seeds, **kw)
    batch.set_cluster(cluster)
    got = batch.sweep_record(3).cpu().numpy()
    for r in range(R):
        o = O.Oracle(T=T[r], seed=seeds[r], **kw)
        assert np.array_equal(got[r], o.sweep_record(3))
        assert np.array_equal(batch.replica(r).get_spins().cpu().numpy(), o.get_spins())
        assert batch.measure_int()[r] == o.measure_int()
    batch.close()


def test_host_series_without_device_scratch():
    kw = dict(dims=2, L=64, T=2.269, seed=41)
    lat, orc = lsm.Lattice(**kw), O.Oracle(**kw)
    assert np.array_equal(lat.sweep_record_host_noalloc(5), orc.sweep_record(5))
