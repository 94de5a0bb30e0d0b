"""The end-to-end host-buffer pipeline (the sequence bench.py times as `e2e`) held to the CPU oracle.

paper_1209_0296_b200.pipeline.HostPipeline drives lsm_stage_spins_host (copy stream, two alternating staging buffers),
event-ordered lsm_set_spins and lsm_sweep_record_host_async (two pinned series buffers) exactly as bench.py does.  Every
step gets a DIFFERENT configuration with its own sweep counter, so a missing event wait, a staging buffer overwritten
too early or a series downloaded from the wrong buffer changes a number: every downloaded (B, M) series and the final
configuration must equal, bit for bit, what the oracle computes when driven through the same steps
("a test calls through the C-ABI"; BASELINE.json north_star: bit-exact on every config)."""
import numpy as np
import pytest
import torch

from oracle import lsm_oracle as O
from paper_1209_0296_b200 import build as B
from paper_1209_0296_b200 import lsm
from paper_1209_0296_b200 import workloads as W
from paper_1209_0296_b200.pipeline import HostPipeline

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _built():
    B.build()
    lsm.load()


def oracle_steps(kw, counters, S):
    """Configurations of one oracle trajectory at the given sweep counters (ascending), and for each of them the
    series of S further sweeps started from it (computed by a second oracle handle through set_spins)."""
    traj, runner = O.Oracle(**kw), O.Oracle(**kw)
    inputs, want, final = [], [], None
    for t in counters:
        traj.sweep(t - traj.sweeps_done)
        cfg = traj.get_spins().copy()
        runner.set_spins(cfg, t)
        want.append(runner.sweep_record(S))
        final = runner.get_spins().copy()
        inputs.append((cfg, t))
    return inputs, want, final


def run_pipeline(lat, inputs, S):
    pinned = [(torch.from_numpy(cfg).pin_memory(), t) for cfg, t in inputs]
    got = {}
    pipe = HostPipeline(lat, S)
    pipe.run(pinned, consume=lambda k, series: got.__setitem__(k, series.numpy().copy()))
    return pipe, [got[k] for k in range(len(inputs))]


CASES = [
    # (create kwargs, sweep counters of the uploaded configurations, sweeps per step)
    (dict(dims=2, L=256, T=2.269, seed=41), (0, 3, 7, 12, 13, 20), 5),                       # small family
    (dict(dims=2, L=512, T=2.0, h=0.05, seed=42), (0, 3, 7, 12), 9),                         # slab family
    (dict(dims=3, L=32, two_S=2, h=0.01, T=3.0, seed=43), (0, 2, 5, 9, 14), 4),              # spin-1
    (dict(dims=2, L=128, model=lsm.NE_HEATBATH, J=0.0, T=W.ne_temperature(0.2), seed=44), (0, 3, 7, 12), 6),
    (dict(dims=3, L=64, model=lsm.EA, T=1.1, seed=45), (0, 1, 4), 3),
    (dict(dims=2, L=128, two_S=2, model=lsm.POTTS, T=0.995, seed=46), (0, 3, 7), 5),
]


@pytest.mark.parametrize("kw,counters,S", CASES)
@pytest.mark.parametrize("family", [lsm.KERNEL_AUTO, lsm.KERNEL_TILED])
def test_pipeline_series_and_final_state_equal_the_oracle(kw, counters, S, family):
    inputs, want, final = oracle_steps(kw, counters, S)
    lat = lsm.Lattice(**kw)
    try:
        lat.set_kernel(family)
    except lsm.LsmError as e:
        assert e.code == lsm.ERR_UNSUPPORTED
        pytest.skip("family does not run this lattice")
    pipe, got = run_pipeline(lat, inputs, S)
    assert (pipe.h2d_bytes_per_step, pipe.d2h_bytes_per_step) == (lat.N, 16 * S)
    for k, (g, w) in enumerate(zip(got, want)):
        assert np.array_equal(g, w), f"step {k} (counter {counters[k]}): series differs from the oracle"
    assert np.array_equal(lat.get_spins().cpu().numpy(), final)
    Bv, Mv, t = lat.measure_int()
    assert (Bv, Mv) == tuple(want[-1][-1]) and t == counters[-1] + S
    assert lat.measure_full() == (Bv, Mv)
    # a second run on the same pipeline object (events and buffers reused), inputs in reverse order
    rev = list(reversed(range(len(inputs))))
    pinned = [(torch.from_numpy(inputs[i][0]).pin_memory(), inputs[i][1]) for i in rev]
    got2 = {}
    pipe.run(pinned, consume=lambda k, series: got2.__setitem__(k, series.numpy().copy()))
    for k, i in enumerate(rev):
        assert np.array_equal(got2[k], want[i]), f"second run, step {k} (input {i})"


def test_pipeline_with_uploads_that_outlast_the_sweeps():
    """8192^2 (config 2): a 64 MiB upload takes over a millisecond, one sweep about 60 us, so the upload of step k+1 is
    still in flight when the sweeps of step k have finished -- the compute stream has to wait for it, and the copy
    stream has to wait before overwriting a staging buffer.  Three different inputs, one sweep each."""
    w = W.by_name("cfg2_T2.269")
    kw = w.create_args()
    orc = O.Oracle(**kw)
    c0 = orc.get_spins().copy()
    s0 = orc.sweep_record(1)
    c1 = orc.get_spins().copy()
    s1 = orc.sweep_record(1)
    up = np.ones(w.N, dtype=np.int8)
    up[::3] = -1                                       # a configuration unrelated to the trajectory, counter 50
    orc.set_spins(up, 50)
    s2 = orc.sweep_record(1)
    final = orc.get_spins()
    lat = lsm.Lattice(**kw)
    lat.set_tracking(False)
    _, got = run_pipeline(lat, [(c0, 0), (c1, 1), (up, 50)], 1)
    for k, (g, want) in enumerate(zip(got, (s0, s1, s2))):
        assert np.array_equal(g, want), f"step {k}"
    assert np.array_equal(lat.get_spins().cpu().numpy(), final)
    assert lat.measure_int() == (int(s2[0, 0]), int(s2[0, 1]), 51)
