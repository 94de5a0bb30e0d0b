"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element.

Integer results (configuration, bond sum B, magnetisation M, never-changed count, overlap) must be
bit-exact after every sweep; derived doubles within 1e-9 relative (BASELINE.json north_star)."""
import ctypes
import math

import numpy as np
import pytest
import torch

from oracle import lsm_oracle as O
from paper_1209_0296_b200 import build as B
from paper_1209_0296_b200 import lsm
from paper_1209_0296_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _built():
    B.build()
    lsm.load()


def make_pair(family=lsm.KERNEL_AUTO, **kw):
    lat = lsm.Lattice(**kw)
    if family != lsm.KERNEL_AUTO:
        lat.set_kernel(family)
    return lat, O.Oracle(**kw)


def assert_same_state(lat, orc, check_persistence=True):
    g = lat.get_spins().cpu().numpy()
    o = orc.get_spins()
    bad = np.flatnonzero(g != o)
    assert bad.size == 0, f"{bad.size} sites differ, first at {bad[:5]}"
    Bg, Mg, tg = lat.measure_int()
    assert (Bg, Mg) == orc.measure_int()
    assert tg == orc.sweeps_done
    assert lat.measure_full() == (Bg, Mg)      # P14: fused running sums == full reduction
    if check_persistence:
        assert lat.persistence() == orc.persistence()


SHAPES = [
    # (kwargs, sweeps) -- sizes span several tiles and ragged tails; L not a multiple of 32 included
    (dict(dims=2, L=4, T=2.269), 40),
    (dict(dims=2, L=6, T=2.0), 40),
    (dict(dims=2, L=8, T=2.269), 40),                # one 32-bit lane per compact row (small family)
    (dict(dims=2, L=16, T=2.0, h=0.1), 40),
    (dict(dims=2, L=34, T=2.269), 30),
    (dict(dims=2, L=64, T=2.269), 60),
    (dict(dims=2, L=96, T=2.6, h=0.05), 30),
    (dict(dims=2, L=160, T=1.5, J=0.7, h=-0.3), 25),
    (dict(dims=2, L=256, T=2.269), 25),
    (dict(dims=2, L=64, T=0.05), 20),               # thresholds 0 ("never") and 2^32 ("always")
    (dict(dims=2, L=64, T=1e6), 10),                # p ~ 1 - 1e-5: thresholds just below 2^32
    (dict(dims=2, L=32, T=2.0, J=0.0, h=0.4), 20),  # free spins
    (dict(dims=2, L=32, T=2.0, J=-1.0), 20),        # antiferromagnet
    (dict(dims=3, L=4, T=4.5115), 30),
    (dict(dims=3, L=6, T=4.0, h=0.1), 20),
    (dict(dims=3, L=8, T=4.5115), 30),
    (dict(dims=3, L=16, T=4.0, h=-0.05), 20),
    (dict(dims=3, L=32, T=4.5115), 20),
    (dict(dims=3, L=64, T=4.5115), 8),
    (dict(dims=3, L=34, T=3.0), 8),
    (dict(dims=2, L=4, two_S=2, T=3.0, h=0.01), 40),
    (dict(dims=2, L=8, two_S=2, T=2.0, h=0.3), 30),       # small family with a single warp: 64-entry table, 32 threads
    (dict(dims=2, L=16, two_S=2, T=3.9, h=-0.4), 30),
    (dict(dims=2, L=64, two_S=2, T=1.5, h=0.01), 30),
    (dict(dims=3, L=6, two_S=2, T=3.0, h=0.01), 20),
    (dict(dims=3, L=16, two_S=2, T=3.0, h=0.01), 20),
    (dict(dims=3, L=32, two_S=2, T=3.0, h=0.01), 12),
    (dict(dims=3, L=64, two_S=2, T=3.0, h=0.01), 6),
    (dict(dims=2, L=4, model=lsm.NE_HEATBATH, J=0.0, T=W.ne_temperature(0.3)), 40),
    (dict(dims=2, L=16, model=lsm.NE_HEATBATH, J=0.0, T=W.ne_temperature(0.3)), 40),
    (dict(dims=2, L=34, model=lsm.NE_HEATBATH, J=0.0, T=W.ne_temperature(0.2)), 40),
    (dict(dims=2, L=64, model=lsm.NE_HEATBATH, J=0.0, T=W.ne_temperature(0.1)), 60),
    (dict(dims=2, L=256, model=lsm.NE_HEATBATH, J=0.0, T=W.ne_temperature(0.3)), 40),
    (dict(dims=2, L=64, model=lsm.NE_METROPOLIS, J=0.0, T=W.ne_temperature(0.3)), 60),
    (dict(dims=2, L=160, model=lsm.NE_METROPOLIS, J=0.0, T=W.ne_temperature(0.2)), 30),
    # larger lattices: several march segments per word column (tiled), many rows per slab
    (dict(dims=2, L=1024, T=2.269), 12),
    (dict(dims=2, L=2048, T=2.0, h=0.02), 7),
    (dict(dims=3, L=128, T=4.5115), 5),
    (dict(dims=2, L=1024, two_S=2, T=1.5, h=0.01), 8),
    (dict(dims=3, L=96, two_S=2, T=3.0, h=0.01), 6),
    (dict(dims=2, L=1024, model=lsm.NE_HEATBATH, J=0.0, T=W.ne_temperature(0.3)), 16),
    (dict(dims=2, L=3072, model=lsm.NE_METROPOLIS, J=0.0, T=W.ne_temperature(0.2)), 6),
]
FAMILIES = [lsm.KERNEL_GENERIC, lsm.KERNEL_TILED, lsm.KERNEL_SMALL, lsm.KERNEL_SLAB]   # + BULK: below


def test_device_philox_known_answers_and_random():
    rows = []
    want = []
    for line in open(__file__.replace("test_gpu_parity.py", "golden/philox4x32_10_kat.txt")):
        if line.startswith("#") or not line.strip():
            continue
        v = [int(t, 16) for t in line.split()]
        rows.append(v[:6])
        want.append(v[6:])
    rng = np.random.default_rng(3)
    extra = rng.integers(0, 2 ** 32, size=(500, 6), dtype=np.uint64)
    rows += extra.tolist()
    want += [list(O.philox4x32_10(r[:4], r[4:])) for r in extra.tolist()]
    got = lsm.philox_device(np.array(rows, dtype=np.uint64).astype(np.uint32))
    assert np.array_equal(got, np.array(want, dtype=np.uint64).astype(np.uint32))


@pytest.mark.parametrize("kw", [
    dict(dims=2, L=8, T=2.269), dict(dims=2, L=8, T=2.0, J=0.5, h=0.25), dict(dims=3, L=8, T=4.5115),
    dict(dims=3, L=8, T=0.3, h=-0.2), dict(dims=2, L=8, two_S=2, T=3.0, h=0.01),
    dict(dims=3, L=8, two_S=2, T=3.0, h=0.01), dict(dims=3, L=8, two_S=2, T=0.4, J=2.0, h=0.0),
    dict(dims=2, L=8, model=lsm.NE_HEATBATH, J=0.0, T=W.ne_temperature(0.1)),
    dict(dims=2, L=8, model=lsm.NE_METROPOLIS, J=0.0, T=W.ne_temperature(0.3)),
])
def test_threshold_tables_identical(kw):
    lat, orc = make_pair(seed=1, **kw)
    assert lat.thresholds() == orc.thresholds()
    for T in (0.02, 1.0, 2.269, 37.5):
        lat.set_temperature(T)
        orc.set_temperature(T)
        assert lat.thresholds() == orc.thresholds()


@pytest.mark.parametrize("family", FAMILIES)
@pytest.mark.parametrize("kw,nsweeps", SHAPES)
def test_sweep_parity(kw, nsweeps, family):
    """Initial state, every per-sweep (B, M), final configuration, persistence and overlap."""
    try:
        lat, orc = make_pair(family, seed=W.seed_of(9, nsweeps), **kw)
    except lsm.LsmError as e:
        if e.code == lsm.ERR_UNSUPPORTED and family != lsm.KERNEL_GENERIC:
            pytest.skip("this family does not cover this lattice (generic covers it)")
        raise
    assert lat.kernel == family
    assert_same_state(lat, orc)                      # a1: initial state from the seed
    half = nsweeps // 2
    got = lat.sweep_record(half).cpu().numpy()
    want = orc.sweep_record(half)
    assert np.array_equal(got, want), np.flatnonzero((got != want).any(axis=1))[:5]
    assert_same_state(lat, orc)
    lat.sweep(nsweeps - half)                        # no per-sweep record: observables of the last sweep only
    orc.sweep(nsweeps - half)
    assert_same_state(lat, orc)
    E, M = lat.measure()
    assert E == orc.energy() and M == orc.measure_int()[1]


SLAB_DEPTH_CASES = [
    # (kwargs, depths): temporal blocking of the slab family -- every depth the shape allows, incl. a "never" table
    (dict(dims=2, L=512, T=2.269), (1, 2, 3, 4)),
    (dict(dims=2, L=1024, T=0.3, h=0.1), (2, 4)),
    (dict(dims=2, L=1024, two_S=2, T=1.5, h=0.01), (1, 3)),
    (dict(dims=2, L=512, model=lsm.NE_HEATBATH, J=0.0, T=W.ne_temperature(0.3)), (2, 3, 4)),
    (dict(dims=2, L=1024, model=lsm.NE_METROPOLIS, J=0.0, T=W.ne_temperature(0.2)), (4,)),
    (dict(dims=2, L=2048, T=2.269, h=-0.02), (1, 2)),
    (dict(dims=2, L=4096, T=2.6), (1,)),
    (dict(dims=3, L=64, T=4.5115), (1,)),
    (dict(dims=3, L=128, two_S=2, T=3.0, h=0.01), (1,)),
    (dict(dims=2, L=512, model=lsm.EA, T=1.1, h=0.05), (1, 2, 3)),      # +/-J bonds resident beside the spins
    (dict(dims=2, L=2048, model=lsm.EA, T=0.2), (2,)),                  # "never" thresholds
    (dict(dims=3, L=64, model=lsm.EA, T=1.2), (1,)),
    (dict(dims=2, L=1024, two_S=2, model=lsm.POTTS, T=0.995), (1, 2, 4)),   # 3-state Potts
    (dict(dims=3, L=64, two_S=7, model=lsm.POTTS, T=0.9), (1,)),           # q = 8
    (dict(dims=2, L=128, model=lsm.EA, T=0.9), (1, 2, 3, 4)),              # small lattices of the models without a small family
    (dict(dims=3, L=32, two_S=3, model=lsm.POTTS, T=1.5), (1,)),
    # L not a power of two: the index arithmetic divides by multiplication
    (dict(dims=2, L=1536, T=2.269), (1, 2)),
    (dict(dims=2, L=1056, two_S=2, T=1.5, h=0.01), (2,)),
    (dict(dims=2, L=736, T=2.0), (3, 4)),
    (dict(dims=2, L=3072, model=lsm.NE_HEATBATH, J=0.0, T=W.ne_temperature(0.2)), (1,)),
    (dict(dims=3, L=96, T=4.5115, h=0.05), (1,)),
    (dict(dims=2, L=160, model=lsm.EA, T=1.0), (1, 2)),
    (dict(dims=2, L=320, T=2.269), (1, 3)),
    (dict(dims=2, L=224, model=lsm.NE_METROPOLIS, J=0.0, T=W.ne_temperature(0.3)), (4,)),
]


@pytest.mark.parametrize("kw,depths", SLAB_DEPTH_CASES)
def test_slab_temporal_blocking_parity(kw, depths):
    """SURVEY 8(f) NEXT-4, temporal blocking: `depth` half-sweeps between two boundary exchanges with redundant halo
    updates must give the oracle's configuration and per-sweep (B, M) for every depth, across calls whose lengths leave
    partial epochs (odd numbers of sweeps, one-sweep calls, calls with and without the record)."""
    calls = ((5, True), (3, False), (1, True), (4, True))
    orc = O.Oracle(seed=W.seed_of(11, 1), **kw)
    want, states = [], []
    for n, rec in calls:
        want.append(orc.sweep_record(n) if rec else orc.sweep(n))
        states.append((orc.get_spins().copy(), orc.measure_int(), orc.persistence()))
    for depth in depths:
        lat = lsm.Lattice(seed=W.seed_of(11, 1), **kw)
        lat.set_kernel(lsm.KERNEL_SLAB)
        lat.set_temporal_depth(depth)
        assert lat.kernel == lsm.KERNEL_SLAB and lat.temporal_depth == depth
        for (n, rec), w, (spins, bm, pers) in zip(calls, want, states):
            if rec:
                got = lat.sweep_record(n).cpu().numpy()
                assert np.array_equal(got, w), (depth, n)
            else:
                lat.sweep(n)
            assert np.array_equal(lat.get_spins().cpu().numpy(), spins), (depth, n)
            assert lat.measure_int()[:2] == bm and lat.measure_full() == bm
            assert lat.persistence() == pers
        lat.close()
    lat = lsm.Lattice(seed=1, **kw)
    lat.set_kernel(lsm.KERNEL_SLAB)
    with pytest.raises(lsm.LsmError):
        lat.set_temporal_depth(5)
    lat.close()


@pytest.mark.parametrize("kw,depth,n", [
    (dict(dims=2, L=512, T=2.269), 3, 60000),
    (dict(dims=2, L=1024, T=2.0, h=0.1), 2, 40000),
    (dict(dims=3, L=128, T=4.5115), 1, 10000),
    (dict(dims=2, L=1536, model=lsm.NE_HEATBATH, J=0.0, T=W.ne_temperature(0.3)), 2, 20000),
    # depth 1 with at least 768 words per step: the "early" exchange, which polls the neighbours' mailbox words before
    # the CTA barrier (slab_plan: 2048^2, 3072^2, 4096^2 at depth 1)
    (dict(dims=2, L=2048, T=2.269), 1, 12000),
    (dict(dims=2, L=4096, T=2.269), 1, 10000),
])
def test_slab_long_run_against_the_tiled_family(kw, depth, n):
    """The mailbox protocol of the slab family over 10^4 ... 10^5 sweeps (2 x 10^4 ... 10^5 exchanges per CTA pair): the
    configuration, the running sums and the persistence counts must equal those of the tiled family, which the other
    tests hold to the oracle sweep by sweep; at the end the oracle itself checks one more slab sweep from the late state
    (the random words are a pure function of (seed, sweep, half, site))."""
    a, b = lsm.Lattice(seed=77, **kw), lsm.Lattice(seed=77, **kw)
    a.set_kernel(lsm.KERNEL_SLAB)
    a.set_temporal_depth(depth)
    b.set_kernel(lsm.KERNEL_TILED)
    for _ in range(2):
        a.sweep(n // 2)
        b.sweep(n // 2)
        assert a.measure_int() == b.measure_int()
    assert torch.equal(a.get_spins(), b.get_spins())
    assert a.persistence() == b.persistence() and a.measure_full() == a.measure_int()[:2]
    # late one-step spot check against the oracle: its state := the slab family's at sweep n, one sweep on either side
    orc = O.Oracle(seed=77, **kw)
    orc.set_spins(a.get_spins_host(), n)
    assert orc.measure_int() == a.measure_int()[:2]
    series = a.sweep_record(1).cpu().numpy()
    orc.sweep(1)
    assert np.array_equal(a.get_spins_host(), orc.get_spins())
    assert tuple(series[0]) == orc.measure_int() and a.measure_int()[2] == n + 1
    a.close()
    b.close()


def test_auto_mixes_short_and_long_calls_on_the_largest_slab_lattice():
    """4096^2 under AUTO: calls of fewer than 8 sweeps run as launches per half-sweep, longer ones as one slab launch
    (the slab launch reads and writes the whole lattice once); the results must not show the seam."""
    kw = dict(dims=2, L=4096, T=2.269, h=0.02)
    seed = W.seed_of(13, 0)
    lat, orc = lsm.Lattice(seed=seed, **kw), O.Oracle(seed=seed, **kw)
    assert lat.kernel == lsm.KERNEL_SLAB
    for n, rec in ((3, True), (9, True), (2, False), (1, True)):
        if rec:
            assert np.array_equal(lat.sweep_record(n).cpu().numpy(), orc.sweep_record(n)), n
        else:
            lat.sweep(n)
            orc.sweep(n)
        assert_same_state(lat, orc)
    lat.close()


BULK_CASES = [
    dict(dims=2, L=8192, T=2.269, h=0.05),
    dict(dims=2, L=8192, T=0.3),                                   # "never" thresholds: the two-compare kernels
    dict(dims=2, L=8192, model=lsm.NE_HEATBATH, J=0.0, T=W.ne_temperature(0.3)),
    dict(dims=2, L=16384, model=lsm.NE_METROPOLIS, J=0.0, T=W.ne_temperature(0.1)),   # two 256-word chunks per row
]


@pytest.mark.parametrize("kw", BULK_CASES)
def test_bulk_copy_family_parity(kw):
    """LSM_KERNEL_BULK: the tiled half-sweep fed by bulk asynchronous copies (cp.async.bulk + mbarrier, one producer
    thread per CTA).  Against the oracle for the first sweeps (every (B, M), configuration, persistence), then against
    the tiled family for a longer run with tracking switched: bit-identical."""
    seed = W.seed_of(12, kw["L"] // 8192)
    lat = lsm.Lattice(seed=seed, **kw)
    lat.set_kernel(lsm.KERNEL_BULK)
    assert lat.kernel == lsm.KERNEL_BULK
    n = 3 if kw["L"] == 8192 else 1
    orc = O.Oracle(seed=seed, **kw)
    assert np.array_equal(lat.sweep_record(n).cpu().numpy(), orc.sweep_record(n))
    assert_same_state(lat, orc)
    ref = lsm.Lattice(seed=seed, **kw)
    ref.set_kernel(lsm.KERNEL_TILED)
    ref.sweep(n)
    for track in (False, True):
        lat.set_tracking(track)
        ref.set_tracking(track)
        assert torch.equal(lat.sweep_record(7), ref.sweep_record(7))
        lat.sweep(2)
        ref.sweep(2)
        assert torch.equal(lat.get_spins(), ref.get_spins())
        assert lat.measure_int() == ref.measure_int() and lat.measure_full() == lat.measure_int()[:2]
    assert lat.persistence() == ref.persistence()
    small = lsm.Lattice(dims=2, L=4096, T=2.0, seed=1)
    with pytest.raises(lsm.LsmError) as e:
        small.set_kernel(lsm.KERNEL_BULK)
    assert e.value.code == lsm.ERR_UNSUPPORTED
    for x in (lat, ref, small):
        x.close()


@pytest.mark.parametrize("family", FAMILIES)
def test_cfg1_full_length(family):
    """BASELINE.json config 1 at full length: 64x64, T=2.269, 1000 sweeps, (E, M) after every sweep."""
    w = W.configs()["cfg1"]
    try:
        lat, orc = make_pair(family, **w.create_args())
    except lsm.LsmError as e:
        if e.code == lsm.ERR_UNSUPPORTED and family == lsm.KERNEL_SLAB:
            pytest.skip("64 x 64 is below the slab family's sizes")
        raise
    got = lat.sweep_record(w.sweeps).cpu().numpy()
    want = orc.sweep_record(w.sweeps)
    assert np.array_equal(got, want)
    assert_same_state(lat, orc)
    # derived doubles within 1e-9 relative
    u_g, u_o = lsm.binder_u4(got[500:]), O.binder_u4(want[500:, 1])
    assert abs(u_g - u_o) <= 1e-9 * abs(u_o)
    c_g, c_o = lsm.heat_capacity(got[500:], w.N, w.J, w.h, w.T), O.heat_capacity_per_site(want[500:], w.N, w.J, w.h, w.T)
    assert abs(c_g - c_o) <= 1e-9 * abs(c_o)


@pytest.mark.parametrize("name,L,nsweeps", [
    ("cfg2_T2.0", 256, 300), ("cfg2_T2.269", 256, 1000), ("cfg2_T2.6", 512, 100),
    ("cfg3", 64, 150), ("cfg4", 64, 60), ("cfg5_c0.10", 256, 1000), ("cfg5_c0.30", 256, 400),
])
def test_reduced_shapes_of_configs_2_to_5(name, L, nsweeps):
    """Same physics and seeds as BASELINE.json configs 2-5 on lattices the oracle finishes in seconds."""
    w = W.configs()[name].scaled(L, nsweeps)
    lat, orc = make_pair(**w.create_args())
    is_ne = w.model != lsm.ISING
    chunk = 100 if is_ne else nsweeps
    done = 0
    while done < nsweeps:
        n = min(chunk, nsweeps - done)
        got = lat.sweep_record(n).cpu().numpy()
        want = orc.sweep_record(n)
        assert np.array_equal(got, want)
        done += n
        if is_ne:   # cfg5: persistence (and Phi) every 100 sweeps
            nc_g, ov_g = lat.persistence()
            nc_o, ov_o = orc.persistence()
            assert (nc_g, ov_g) == (nc_o, ov_o)
            c = orc.concentration
            assert lsm.persistence_fraction(nc_g, w.N) == O.persistence_fraction(nc_o, w.N)
            a, b = lsm.phi(ov_g, w.N, c), O.phi(ov_o, w.N, c)
            assert abs(a - b) <= 1e-9 * max(abs(b), 1e-300)
    assert_same_state(lat, orc)


def test_checkpoint_resume_and_host_buffers():
    kw = dict(dims=2, L=64, T=2.269, seed=5)
    lat, orc = make_pair(**kw)
    lat.sweep(7)
    orc.sweep(7)
    snap = lat.get_spins_host()
    assert np.array_equal(snap, orc.get_spins())
    lat2 = lsm.Lattice(**kw)
    lat2.set_spins_host(snap, 7)
    assert lat2.measure_int() == lat.measure_int()
    h1 = lat.sweep_record_host(9)
    h2 = lat2.sweep_record_host(9)
    want = orc.sweep_record(9)
    assert np.array_equal(np.asarray(h1), want) and np.array_equal(np.asarray(h2), want)
    assert_same_state(lat, orc, check_persistence=True)
    # set_spins leaves the reference snapshot and flags alone: lat2 was re-referenced at create (t=0 draw)
    import torch

    up = torch.ones(64 * 64, dtype=torch.int8, device="cuda")
    lat.set_spins(up, 100)
    orc.set_spins(np.ones(64 * 64, dtype=np.int8), 100)
    assert lat.measure_int() == (2 * 4096, 4096, 100)
    lat.reset_reference()
    orc.reset_reference()
    lat.sweep(5)
    orc.sweep(5)
    assert_same_state(lat, orc)


def test_tracking_off_and_on():
    kw = dict(dims=2, L=64, T=2.269, seed=6)
    lat, orc = make_pair(**kw)
    lat.set_tracking(False)
    with pytest.raises(lsm.LsmError) as ei:
        lat.persistence()
    assert ei.value.code == lsm.ERR_STATE
    lat.sweep(6)
    orc.sweep(6)
    assert_same_state(lat, orc, check_persistence=False)
    lat.reset_reference()
    orc.reset_reference()
    lat.sweep(6)
    orc.sweep(6)
    assert_same_state(lat, orc)


def test_zero_sweeps_and_temperature_change():
    kw = dict(dims=3, L=8, T=4.5115, seed=8)
    lat, orc = make_pair(**kw)
    lat.sweep(0)
    assert lat.sweep_record(0).shape == (0, 2)
    assert_same_state(lat, orc)
    for T in (1.0, 6.0, 0.1):
        lat.set_temperature(T)
        orc.set_temperature(T)
        got = lat.sweep_record(5).cpu().numpy()
        assert np.array_equal(got, orc.sweep_record(5))
    assert_same_state(lat, orc)
    assert lat.launch_count > 0


@pytest.mark.parametrize("family", FAMILIES)
@pytest.mark.parametrize("kw", [dict(dims=2, L=32, T=2.269), dict(dims=2, L=1024, T=2.269),
                                dict(dims=3, L=32, two_S=2, T=3.0, h=0.01),
                                dict(dims=2, L=64, model=lsm.NE_HEATBATH, J=0.0, T=W.ne_temperature(0.3))])
def test_sweep_counter_above_32_bits(kw, family):
    """The 64-bit sweep counter reaches the Philox counter's c3 field (reading D2), also when the counter's low word
    wraps in the middle of a call (kernels that run several sweeps per launch compute it on the device)."""
    lat, orc = make_pair(seed=11, **kw)
    try:
        lat.set_kernel(family)
    except lsm.LsmError as e:
        assert e.code == lsm.ERR_UNSUPPORTED
        pytest.skip("this family does not cover this lattice")
    t0 = (5 << 32) + 0xFFFFFFFE
    s = orc.get_spins()
    lat.set_spins_host(s, t0)
    orc.set_spins(s, t0)
    got = lat.sweep_record(4).cpu().numpy()
    assert np.array_equal(got, orc.sweep_record(4))
    assert_same_state(lat, orc, check_persistence=False)
    if kw.get("model", lsm.ISING) != lsm.ISING:
        lat.set_spins_host(s, t0)
        orc.set_spins(s, t0)
        for bal in (False, True):
            lat.sweep_random_tile(3, 32, 16, balanced=bal)
            (orc.sweep_random_tile_balanced if bal else orc.sweep_random_tile)(3, 32, 16)
        assert_same_state(lat, orc, check_persistence=False)


FULL = [
    # (config, sweeps checked from t=0, late time for the one-step spot check)
    ("cfg2_T2.0", 1, 11),
    ("cfg2_T2.269", 2, 37),
    ("cfg2_T2.6", 1, 1003),      # a spot check beyond 10^3 sweeps
    ("cfg3", 1, 21),
    ("cfg4", 2, 15),
    ("cfg5_c0.10", 2, 1101),     # the per-lane facilitation branch (ne_all4 = 0), late
    ("cfg5_c0.20", 2, 203),
    ("cfg5_c0.30", 1, 57),
]


@pytest.mark.parametrize("family", [lsm.KERNEL_AUTO, lsm.KERNEL_TILED])
@pytest.mark.parametrize("name,k_first,t_late", FULL)
def test_full_size_prefix_and_late_spot_check(name, k_first, t_late, family):
    """BASELINE.json's full sizes in the launch configuration bench.py times (AUTO kernel family,
    tracking as bench.py sets it): the first sweeps element by element, then a one-step spot check at
    a late time -- download the GPU state at sweep t, hand it to the oracle with the same counter,
    one oracle sweep, compare with the GPU at t+1.  Valid because the random words are a pure
    function of (seed, sweep, half, site)."""
    w = W.configs()[name]
    lat, orc = make_pair(family, **w.create_args())
    if w.model == lsm.ISING:
        lat.set_tracking(False)      # as bench.py runs cfg1-4
    if family != lsm.KERNEL_AUTO:
        assert lat.kernel == family
    g0 = lat.get_spins_host()
    assert np.array_equal(g0, orc.get_spins())
    got = lat.sweep_record(k_first).cpu().numpy()
    want = orc.sweep_record(k_first)
    assert np.array_equal(got, want)
    assert np.array_equal(lat.get_spins_host(), orc.get_spins())
    lat.sweep(t_late - k_first)
    state = lat.get_spins_host()
    orc.set_spins(state, t_late)
    series = lat.sweep_record(1).cpu().numpy()
    orc.sweep(1)
    after = lat.get_spins_host()
    ref = orc.get_spins()
    assert np.array_equal(after, ref)
    assert tuple(series[0]) == orc.measure_int()
    # properties that hold at any size
    N = w.N
    Bv, Mv, t = lat.measure_int()
    assert t == t_late + 1 and abs(Mv) <= N and abs(Bv) <= w.dims * N
    assert lat.measure_full() == (Bv, Mv)
    if w.model != lsm.ISING:
        # a9 at full size (BASELINE.json config 5: lsm_persistence every 100 sweeps).  The oracle saw sweeps
        # 0..k_first-1 and t_late only, so: both take a new reference now, one more sweep, counts must agree exactly;
        # and the GPU's count since t = 0 is bounded by what the oracle can derive from the two states.
        nc_run, ov_run = lat.persistence()
        sig0, sig1 = 2 * g0.astype(np.int64) - 1, 2 * after.astype(np.int64) - 1
        assert ov_run == int((sig0 * sig1).sum())                 # Eq. 4 numerator against the t = 0 configuration
        assert nc_run <= int((g0 == after).sum())                 # a site that differs has certainly changed
        lat.reset_reference()
        orc.reset_reference()
        lat.sweep(1)
        orc.sweep(1)
        assert lat.persistence() == orc.persistence()
        assert np.array_equal(lat.get_spins_host(), orc.get_spins())


# ------------------------------------------------------------------ NEXT-1: the paper's corrected North-East algorithm
@pytest.mark.parametrize("model", [lsm.NE_HEATBATH, lsm.NE_METROPOLIS])
@pytest.mark.parametrize("L,b,lam,c,nsweeps", [
    (64, 32, 16, 0.42, 30),      # the paper's best configuration (32 x 32 tiles, lambda = 16)
    (64, 8, 4, 0.45, 20),        # small tiles: same-site collisions in most sub-steps
    (64, 8, 32, 0.45, 20),       # lambda = P/2: a single sub-step per launch
    (128, 16, 1, 0.30, 12),      # lambda = 1: serial inside a tile
    (64, 64, 1, 0.42, 6),        # Q = lambda = 1: the serial limit
    (256, 64, 8, 0.20, 10),
    (384, 128, 32, 0.30, 5),     # tiles of 16 KiB, L not a power of two
    (1024, 32, 16, 0.42, 4),     # several waves of CTAs, tail groups
])
def test_random_tile_schedule_parity(model, L, b, lam, c, nsweeps):
    """Configuration, per-sweep M, persistence and overlap after every stage; mixes with checkerboard sweeps."""
    kw = dict(dims=2, L=L, model=model, J=0.0, T=W.ne_temperature(c), seed=W.seed_of(5, 7) + L + lam)
    lat, orc = make_pair(**kw)
    half = nsweeps // 2
    got = lat.sweep_random_tile(half, b, lam, record=True).cpu().numpy()
    want = orc.sweep_random_tile_record(half, b, lam)
    assert np.array_equal(got, want), np.flatnonzero((got != want).any(axis=1))[:5]
    assert_same_state(lat, orc)
    lat.sweep_random_tile(nsweeps - half, b, lam)            # no record: running M of the last sweep only
    orc.sweep_random_tile(nsweeps - half, b, lam)
    assert_same_state(lat, orc)
    lat.sweep(3)                                             # the checkerboard sweep shares state and sweep counter
    orc.sweep(3)
    lat.sweep_random_tile(2, b, lam)
    orc.sweep_random_tile(2, b, lam)
    assert_same_state(lat, orc)
    lat.set_tracking(False)
    lat.sweep_random_tile(2, b, lam)
    orc.sweep_random_tile(2, b, lam)
    assert np.array_equal(lat.get_spins().cpu().numpy(), orc.get_spins())
    assert lat.measure_int()[:2] == orc.measure_int()


@pytest.mark.parametrize("model", [lsm.NE_HEATBATH, lsm.NE_METROPOLIS])
@pytest.mark.parametrize("L,b,lam", [(128, 128, 1), (128, 128, 4), (64, 64, 1), (256, 128, 2)])
def test_random_tile_large_tiles_small_lambda(model, L, b, lam):
    """Tiles too large for every lane group of a warp to hold one (128 x 128 with lambda <= 4), down to the serial
    limit Q = lambda = 1 of PAPER.md:142 on a 128^2 lattice."""
    kw = dict(dims=2, L=L, model=model, J=0.0, T=W.ne_temperature(0.42), seed=W.seed_of(5, 11) + L + lam)
    lat, orc = make_pair(**kw)
    got = lat.sweep_random_tile(3, b, lam, record=True).cpu().numpy()
    assert np.array_equal(got, orc.sweep_random_tile_record(3, b, lam))
    assert_same_state(lat, orc)


@pytest.mark.slow
def test_lambda_convergence_to_the_serial_limit():
    """PAPER.md:142,155 (Fig. 5): Phi(t) of the corrected algorithm with 32 x 32 tiles follows the serial limit
    Q = lambda = 1 for lambda up to 16 (about 1.5 % of the tile).  Statistical: 6 realisations of a 128^2 lattice at
    c = 0.42; tolerance = 4 standard errors of the difference + 0.02."""
    from paper_1209_0296_b200 import lambda_scan

    times = [10, 30, 100, 300]
    res = lambda_scan.phi_curves(128, 0.42, [(128, 1), (32, 1), (32, 4), (32, 16), (8, 32)], times, 6)
    ref = res[(128, 1)]
    assert all(0.0 < p < 1.0 for p in ref["phi"]) and ref["phi"] == sorted(ref["phi"], reverse=True)   # a decaying curve
    for key in ((32, 1), (32, 4), (32, 16)):
        for p, se, q, sq in zip(res[key]["phi"], res[key]["se"], ref["phi"], ref["se"]):
            assert abs(p - q) < 4 * math.hypot(se, sq) + 0.02, (key, res[key], ref)


def test_random_tile_schedule_rejections():
    lat = lsm.Lattice(dims=2, L=64, model=lsm.NE_HEATBATH, J=0.0, T=1.0, seed=3)
    for b, lam in ((24, 16), (32, 3), (4, 2), (32, 64), (256, 16)):
        with pytest.raises(lsm.LsmError) as e:
            lat.sweep_random_tile(1, b, lam)
        assert e.value.code == lsm.ERR_UNSUPPORTED
    ising = lsm.Lattice(dims=2, L=64, T=2.0, seed=3)
    with pytest.raises(lsm.LsmError) as e:
        ising.sweep_random_tile(1, 32, 16)
    assert e.value.code == lsm.ERR_UNSUPPORTED


def test_random_tile_schedule_full_size_prefix():
    """BASELINE.json config 5 lattice (8192^2, c = 0.30) under the paper's corrected algorithm in its best configuration
    (32 x 32 tiles, lambda = 16: 65 536 tiles, many waves of CTAs): first sweep, element by element."""
    w = W.configs()["cfg5_c0.30"]
    lat, orc = make_pair(**w.create_args())
    got = lat.sweep_random_tile(1, 32, 16, record=True).cpu().numpy()
    want = orc.sweep_random_tile_record(1, 32, 16)
    assert np.array_equal(got, want)
    assert_same_state(lat, orc)


# ------------------------------------------------------------------ NEXT-2: the balance-preserving variant
@pytest.mark.parametrize("model", [lsm.NE_HEATBATH, lsm.NE_METROPOLIS])
@pytest.mark.parametrize("L,b,lam,c,nsweeps", [
    (64, 32, 16, 0.42, 20),
    (64, 8, 8, 0.45, 20),        # P/2 = 32 sites per colour and 8 picks: collisions in most phases
    (128, 16, 1, 0.30, 8),
    (64, 64, 1, 0.42, 4),
    (384, 128, 32, 0.30, 4),
    (1024, 32, 16, 0.42, 3),
])
def test_random_tile_balanced_parity(model, L, b, lam, c, nsweeps):
    kw = dict(dims=2, L=L, model=model, J=0.0, T=W.ne_temperature(c), seed=W.seed_of(5, 9) + L + lam)
    lat, orc = make_pair(**kw)
    got = lat.sweep_random_tile(nsweeps, b, lam, record=True, balanced=True).cpu().numpy()
    want = orc.sweep_random_tile_balanced_record(nsweeps, b, lam)
    assert np.array_equal(got, want), np.flatnonzero((got != want).any(axis=1))[:5]    # the whole per-step series
    assert_same_state(lat, orc)
    lat.sweep_random_tile(1, b, lam)                         # the three schedules share state and sweep counter
    orc.sweep_random_tile(1, b, lam)
    lat.sweep(1)
    orc.sweep(1)
    lat.sweep_random_tile(2, b, lam, balanced=True)
    orc.sweep_random_tile_balanced(2, b, lam)
    assert_same_state(lat, orc)
    with pytest.raises(lsm.LsmError):
        lat.sweep_random_tile(1, 8, 16, balanced=True)       # 8 * lambda does not divide P = 64


# ------------------------------------------------------------------ NEXT-3: the temperature ramp of the paper's Fig. 6
def test_temperature_ramp_matches_the_oracle():
    """start at T = 2.4, lower T in steps, measure M, E and the heat capacity at each T -- one lattice
    carried through; integer series identical to the oracle's, derived doubles within 1e-9."""
    from paper_1209_0296_b200 import ramp

    temps = ramp.temperatures(2.4, 2.1, 0.1)
    assert temps == [2.4, 2.3, 2.2, 2.1]
    kw = dict(dims=2, L=128, T=temps[0], seed=W.seed_of(6, 1))
    lat, orc = make_pair(**kw)
    assert lat.kernel == lsm.KERNEL_SMALL                       # one launch per block of sweeps on the paper's own size
    rows = ramp.temperature_ramp(lat, temps, n_equil=30, n_meas=60, keep_series=True)
    for r in rows:
        orc.set_temperature(r["T"])
        orc.sweep(30)
        want = orc.sweep_record(60)
        assert np.array_equal(r["series"], want)
        c_o = O.heat_capacity_per_site(want, lat.N, 1.0, 0.0, r["T"])
        assert abs(r["c"] - c_o) <= 1e-9 * abs(c_o)
        u_o = O.binder_u4(want[:, 1])
        assert abs(r["u4"] - u_o) <= 1e-9 * abs(u_o)
        e_o = sum(O.energy_from_int(int(b), int(m), 1.0, 0.0) for b, m in want) / (len(want) * lat.N)
        assert abs(r["e"] - e_o) <= 1e-9 * abs(e_o)
    assert_same_state(lat, orc, check_persistence=False)


def test_temperature_ramp_finds_the_transition():
    """Equilibrium check of the whole chain on the paper's protocol (shortened): the heat capacity of a 64^2 lattice
    peaks within 0.06 of Tc = 2/ln(1+sqrt 2), and |m| follows Onsager's 0.911 at T = 2.0 within 1 %."""
    from paper_1209_0296_b200 import ramp

    temps = ramp.temperatures(2.5, 2.0, 0.02)
    lat = lsm.Lattice(dims=2, L=64, T=temps[0], seed=W.seed_of(6, 2))
    lat.set_tracking(False)
    rows = ramp.temperature_ramp(lat, temps, n_equil=3000, n_meas=20000)
    peak = max(rows, key=lambda r: r["c"])
    assert abs(peak["T"] - ramp.TC_2D) < 0.06, peak
    assert abs(rows[-1]["abs_m"] - 0.91131938) < 0.01, rows[-1]
    assert abs(rows[-1]["e"] - (-1.74556458)) < 0.01, rows[-1]


# ------------------------------------------------------------------ seeded random parameters across all families
def _fuzz_cases():
    rng = np.random.default_rng(20121209)
    cases = []
    for i in range(24):
        kind = i % 4
        if kind == 0:
            kw = dict(dims=2, L=int(rng.choice([32, 64, 96, 128, 224])), T=float(rng.uniform(0.3, 6.0)),
                      J=float(rng.choice([-1.0, 0.5, 1.0, 2.0])), h=float(rng.choice([0.0, 0.0, -0.7, 0.13, 3.0])))
        elif kind == 1:
            kw = dict(dims=3, L=int(rng.choice([8, 16, 32, 64])), T=float(rng.uniform(0.5, 9.0)),
                      J=float(rng.choice([-1.0, 1.0, 0.3])), h=float(rng.choice([0.0, 0.25, -2.0])))
        elif kind == 2:
            kw = dict(dims=int(rng.choice([2, 3])), L=int(rng.choice([16, 32, 64])), two_S=2, T=float(rng.uniform(0.4, 5.0)),
                      J=float(rng.choice([-1.0, 1.0, 0.6])), h=float(rng.choice([0.01, -0.4, 1.5])))
        else:
            kw = dict(dims=2, L=int(rng.choice([16, 64, 96, 256])), model=int(rng.choice([lsm.NE_HEATBATH, lsm.NE_METROPOLIS])),
                      J=0.0, T=W.ne_temperature(float(rng.uniform(0.03, 0.49))))
        kw["seed"] = int(rng.integers(1, 2 ** 62))
        cases.append(kw)
    return cases


@pytest.mark.parametrize("kw", _fuzz_cases())
def test_seeded_random_parameters_all_families(kw):
    """Couplings of either sign, fields that make some moves certain or impossible, temperatures from frozen to hot,
    concentrations on both sides of the per-word / per-lane switch of the North-East rule: every family that accepts
    the lattice must reproduce the oracle (families whose tables cannot express a "never" threshold refuse)."""
    ran = 0
    for family in FAMILIES:
        lat = lsm.Lattice(**kw)
        try:
            lat.set_kernel(family)
        except lsm.LsmError as e:
            assert e.code == lsm.ERR_UNSUPPORTED
            continue
        if lat.kernel != family:                      # the library fell back (e.g. a "never" entry): covered by that family
            continue
        orc = O.Oracle(**kw)
        got = lat.sweep_record(6).cpu().numpy()
        assert np.array_equal(got, orc.sweep_record(6)), (family, kw)
        assert_same_state(lat, orc)
        ran += 1
        lat.close()
    assert ran >= 1


def _tile_fuzz_cases():
    rng = np.random.default_rng(1209029601)
    cases = []
    while len(cases) < 16:
        b = int(rng.choice([8, 16, 32, 64]))
        lam = int(rng.choice([1, 2, 4, 8, 16, 32]))
        bal = bool(rng.integers(0, 2))
        if (b * b) % ((8 if bal else 2) * lam) != 0:
            continue
        if lam == 1 and b > 32:
            continue                                  # one thread walking P/2 sub-steps of a big tile: slow, covered above
        L = b * int(rng.choice([1, 2, 3, 5, 8]))
        cases.append((L, b, lam, bal, float(rng.uniform(0.05, 0.49)), int(rng.choice([lsm.NE_HEATBATH, lsm.NE_METROPOLIS])),
                      int(rng.integers(1, 2 ** 62))))
    return cases


@pytest.mark.parametrize("L,b,lam,bal,c,model,seed", _tile_fuzz_cases())
def test_seeded_random_tile_schedules(L, b, lam, bal, c, model, seed):
    kw = dict(dims=2, L=L, model=model, J=0.0, T=W.ne_temperature(c), seed=seed)
    lat, orc = make_pair(**kw)
    got = lat.sweep_random_tile(4, b, lam, record=True, balanced=bal).cpu().numpy()
    if bal:
        orc.sweep_random_tile_balanced(4, b, lam)
        assert got[-1, 1] == orc.measure_int()[1]
    else:
        assert np.array_equal(got, orc.sweep_random_tile_record(4, b, lam))
    assert_same_state(lat, orc)


def test_checkpoint_roundtrip_random_states():
    """get_spins / set_spins (word-granular and scalar conversion kernels) on arbitrary configurations: what goes in comes
    out, flags and snapshot survive, and the run continues bit-exactly from the restored state and sweep counter."""
    rng = np.random.default_rng(7)
    for kw, values in ((dict(dims=2, L=96, T=2.3), (-1, 1)), (dict(dims=2, L=34, T=2.3), (-1, 1)),
                       (dict(dims=3, L=32, two_S=2, T=3.0, h=0.01), (-1, 0, 1)), (dict(dims=3, L=6, two_S=2, T=3.0), (-1, 0, 1)),
                       (dict(dims=2, L=64, model=lsm.NE_HEATBATH, J=0.0, T=1.0), (0, 1))):
        lat, orc = make_pair(seed=11, **kw)
        lat.sweep(3)
        orc.sweep(3)
        state = rng.choice(np.array(values, dtype=np.int8), size=lat.N)
        import torch
        lat.set_spins(torch.from_numpy(state).cuda(), 1000)
        orc.set_spins(state, 1000)
        assert np.array_equal(lat.get_spins().cpu().numpy(), state)
        assert_same_state(lat, orc)                   # persistence / overlap against the untouched snapshot and flags
        got = lat.sweep_record(4).cpu().numpy()
        assert np.array_equal(got, orc.sweep_record(4))
        assert_same_state(lat, orc)


@pytest.mark.parametrize("case", range(8))
def test_seeded_random_operation_sequences(case):
    """A handle driven through a random sequence of calls -- sweeps with and without record, kernel-family switches,
    temperature changes, tracking off/on, reference resets, random-tile sweeps -- stays identical to the oracle driven
    through the same sequence."""
    rng = np.random.default_rng(4000 + case)
    ne = case % 2 == 1
    if ne:
        kw = dict(dims=2, L=int(rng.choice([64, 128])), model=int(rng.choice([lsm.NE_HEATBATH, lsm.NE_METROPOLIS])), J=0.0,
                  T=W.ne_temperature(float(rng.uniform(0.1, 0.45))))
    else:
        kw = dict(dims=int(rng.choice([2, 3])), L=32, two_S=int(rng.choice([1, 2])), T=float(rng.uniform(1.5, 5.0)),
                  h=float(rng.choice([0.0, 0.05])))
    kw["seed"] = int(rng.integers(1, 2 ** 62))
    lat, orc = make_pair(**kw)
    tracking = True
    for step in range(14):
        op = int(rng.integers(0, 7))
        n = int(rng.integers(1, 5))
        if op == 0:
            lat.sweep(n)
            orc.sweep(n)
        elif op == 1:
            assert np.array_equal(lat.sweep_record(n).cpu().numpy(), orc.sweep_record(n)), (case, step)
        elif op == 2:
            try:
                lat.set_kernel(int(rng.choice(FAMILIES + [lsm.KERNEL_AUTO])))
            except lsm.LsmError as e:
                assert e.code == lsm.ERR_UNSUPPORTED
        elif op == 3:
            T = W.ne_temperature(float(rng.uniform(0.1, 0.45))) if ne else float(rng.uniform(1.0, 6.0))
            lat.set_temperature(T)
            orc.set_temperature(T)
        elif op == 4:
            tracking = not tracking
            lat.set_tracking(tracking)
            if tracking:
                orc.reset_reference()                 # switching tracking on is a reference reset (include/lsm.h)
        elif op == 5 and tracking:
            lat.reset_reference()
            orc.reset_reference()
        elif op == 6 and ne:
            bal = bool(rng.integers(0, 2))
            lat.sweep_random_tile(n, 32, 16, balanced=bal)
            (orc.sweep_random_tile_balanced if bal else orc.sweep_random_tile)(n, 32, 16)
        assert_same_state(lat, orc, check_persistence=tracking)
