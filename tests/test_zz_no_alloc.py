"""lsm_sweep_record_host_noalloc against lsm_sweep_record_host (collected last: the file name sorts after the others).

Who needs the entry point: users who drive liblsm from a place where device memory cannot be allocated -- a plug-in
living under a host program's memory pool that owns the whole GPU, a loop that cannot tolerate cudaMalloc's
device-wide synchronisation, a job whose memory quota went into the lattice.  lsm_sweep_record_host asks them for
16*n bytes of device scratch they cannot produce; the _noalloc form stages the (B, M) series in a 64 KiB array
built into liblsm.so instead (at most lsm.NOALLOC_MAX_SWEEPS sweeps per call).

What is checked: the series and the final state of the new call equal those of the existing call on a twin lattice,
bit for bit (the tolerance every integer result of this suite is held to), on two calls in a row -- the second one
shorter and on another lattice shape, so anything left in the shared array by the first call would show -- and
both are held to the CPU oracle as well; sizes beyond the limit are refused without touching the lattice.
The test builds its own lattices and relies on nothing other tests left behind: it passes alone in a fresh process
(where its first call is the one that looks the array's address up) and at the end of the whole suite."""
import ctypes

import numpy as np
import pytest

from oracle import lsm_oracle as O
from paper_1209_0296_b200 import build as B
from paper_1209_0296_b200 import lsm

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _built():
    B.build()
    lsm.load()


def _twin_calls(kw, n, family=lsm.KERNEL_AUTO):
    """n recorded sweeps through the existing path (caller's device scratch) and through the no-allocation path on
    two lattices created alike; returns after asserting that series, configuration and running sums agree."""
    old, new, orc = lsm.Lattice(**kw), lsm.Lattice(**kw), O.Oracle(**kw)
    for lat in (old, new):
        if family != lsm.KERNEL_AUTO:
            lat.set_kernel(family)
    for k in (n, max(n // 3, 1)):               # two calls in a row on the same handles; the second is shorter
        want = np.asarray(old.sweep_record_host(k))
        got = new.sweep_record_host_noalloc(k)
        assert got.shape == (k, 2) and got.dtype == np.int64
        assert np.array_equal(got, want), f"series differ at sweeps {np.flatnonzero((got != want).any(axis=1))[:5]}"
        assert np.array_equal(got, orc.sweep_record(k))
        assert np.array_equal(new.get_spins().cpu().numpy(), old.get_spins().cpu().numpy())
        assert new.measure_int() == old.measure_int()
        assert new.measure_full() == old.measure_full() == orc.measure_int()
    assert np.array_equal(new.get_spins().cpu().numpy(), orc.get_spins())
    return new


def test_noalloc_series_equals_the_scratch_buffer_path_on_consecutive_calls():
    # first call of the process on this GPU when the file runs alone: includes the address look-up
    _twin_calls(dict(dims=2, L=64, T=2.269, seed=11), 40)                       # small family (one launch per call)
    _twin_calls(dict(dims=3, L=32, T=4.5, seed=12), 12, lsm.KERNEL_TILED)       # a launch per half-sweep adds into the array
    _twin_calls(dict(dims=2, L=96, T=2.0, h=0.1, seed=13), 9, lsm.KERNEL_GENERIC)
    ne = _twin_calls(dict(dims=2, L=64, model=lsm.NE_HEATBATH, J=0.0, T=1.2, seed=14), 15)
    ne.close()


def test_noalloc_host_buffer_forms_and_stale_contents():
    kw = dict(dims=2, L=128, T=2.269, seed=21)
    a, b = lsm.Lattice(**kw), lsm.Lattice(**kw)
    long_run = a.sweep_record_host_noalloc(200)          # fills 200 pairs of the array with large sums
    other = lsm.Lattice(dims=2, L=16, T=1.0, seed=3)     # |B|, |M| <= 512: leftovers of `a` would swamp them
    small = other.sweep_record_host_noalloc(200)
    twin = lsm.Lattice(dims=2, L=16, T=1.0, seed=3)
    assert np.array_equal(small, np.asarray(twin.sweep_record_host(200)))
    assert np.array_equal(long_run, np.asarray(b.sweep_record_host(200)))
    # caller-supplied host memory: a numpy array and a pinned tensor
    import torch

    buf = np.full((7, 2), -1, dtype=np.int64)
    pin = torch.full((7, 2), -1, dtype=torch.int64).pin_memory()
    want1 = np.asarray(b.sweep_record_host(7))
    assert a.sweep_record_host_noalloc(7, buf) is buf and np.array_equal(buf, want1)
    want2 = np.asarray(b.sweep_record_host(7))
    a.sweep_record_host_noalloc(7, pin)
    assert np.array_equal(pin.numpy(), want2)
    # n = 0 is a no-op that still succeeds
    assert a.sweep_record_host_noalloc(0).shape == (0, 2)
    assert a.measure_int() == b.measure_int()


def test_noalloc_limit_is_enforced_and_reachable():
    kw = dict(dims=2, L=32, T=2.269, seed=31)
    lat, twin = lsm.Lattice(**kw), lsm.Lattice(**kw)
    before = lat.measure_int()
    with pytest.raises(lsm.LsmError) as e:
        lat.sweep_record_host_noalloc(lsm.NOALLOC_MAX_SWEEPS + 1)
    assert e.value.code == lsm.ERR_LIMIT and "LSM_NOALLOC_MAX_SWEEPS" in str(e.value)
    assert lat.measure_int() == before                   # refused calls sweep nothing (counter included)
    # raw ABI: NULL host buffer, negative n
    L = lsm.load()
    assert L.lsm_sweep_record_host_noalloc(lat._h, 3, None, None) == lsm.ERR_ARG
    assert L.lsm_sweep_record_host_noalloc(lat._h, -1, ctypes.c_void_p(8), None) == lsm.ERR_ARG
    assert L.lsm_sweep_record_host_noalloc(None, 1, ctypes.c_void_p(8), None) == lsm.ERR_ARG
    assert lat.measure_int() == before
    # the full capacity in one call, then the remainder of a longer run in a second call: same series as one long call
    n = lsm.NOALLOC_MAX_SWEEPS
    got = np.concatenate([lat.sweep_record_host_noalloc(n), lat.sweep_record_host_noalloc(100)])
    assert np.array_equal(got, np.asarray(twin.sweep_record_host(n + 100)))
