"""GPU parity of the NEXT-4 models: Edwards-Anderson +/-J bonds (reading D25) and q-state Potts
(reading D26), every kernel family that covers them, element by element against the oracle."""
import numpy as np
import pytest
import torch

from oracle import lsm_oracle as O
from paper_1209_0296_b200 import build as B
from paper_1209_0296_b200 import lsm

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _built():
    B.build()
    lsm.load()


def same_state(lat, orc, persistence=True):
    g, o = lat.get_spins().cpu().numpy(), orc.get_spins()
    bad = np.flatnonzero(g != o)
    assert bad.size == 0, f"{bad.size} sites differ, first at {bad[:5]}"
    Bg, Mg, tg = lat.measure_int()
    assert (Bg, Mg) == orc.measure_int() and tg == orc.sweeps_done
    assert lat.measure_full() == (Bg, Mg)
    if persistence:
        assert lat.persistence() == orc.persistence()
    e = lat.measure()[0]
    assert abs(e - orc.energy()) <= 1e-9 * max(1.0, abs(orc.energy()))


EA_SHAPES = [
    (dict(dims=2, L=4, T=1.5), 30),
    (dict(dims=2, L=6, T=1.0, h=0.2), 30),
    (dict(dims=2, L=34, T=1.2), 20),
    (dict(dims=2, L=64, T=0.9, J=0.8, h=-0.1), 25),
    (dict(dims=2, L=96, T=2.0), 12),
    (dict(dims=2, L=256, T=1.1), 12),
    (dict(dims=2, L=64, T=0.05), 10),                # "never" and "always" thresholds
    (dict(dims=3, L=4, T=2.0), 20),
    (dict(dims=3, L=6, T=1.5, h=0.1), 12),
    (dict(dims=3, L=32, T=1.8), 8),
    (dict(dims=3, L=64, T=1.1), 4),
    (dict(dims=3, L=34, T=2.5, J=-1.0), 4),
]


@pytest.mark.parametrize("family", [lsm.KERNEL_AUTO, lsm.KERNEL_GENERIC, lsm.KERNEL_TILED])
@pytest.mark.parametrize("kw,n", EA_SHAPES)
def test_ea_parity(kw, n, family):
    kw = dict(kw, model=lsm.EA, seed=(0xEA << 32) + 7 * kw["L"] + kw["dims"])
    lat, orc = lsm.Lattice(**kw), O.Oracle(**kw)
    try:
        lat.set_kernel(family)
    except lsm.LsmError as e:
        assert e.code == lsm.ERR_UNSUPPORTED
        pytest.skip("this family does not cover this lattice")
    assert np.array_equal(lat.get_bonds().cpu().numpy(), orc.get_bonds())       # the bond stream (tag 3)
    assert lat.thresholds() == orc.thresholds()
    same_state(lat, orc)
    half = n // 2
    got = lat.sweep_record(half).cpu().numpy()
    want = orc.sweep_record(half)
    assert np.array_equal(got, want), np.flatnonzero((got != want).any(axis=1))[:5]
    same_state(lat, orc)
    lat.sweep(n - half)
    orc.sweep(n - half)
    same_state(lat, orc)
    lat.set_tracking(False)
    got = lat.sweep_record(3).cpu().numpy()
    assert np.array_equal(got, orc.sweep_record(3))
    same_state(lat, orc, persistence=False)
    lat.close()


def test_ea_set_bonds_gauge_and_checkpoint():
    """lsm_set_bonds: Mattis bonds tau_i tau_j with a gauge-transformed state follow the ferromagnet (h = 0);
    all-ferromagnetic bonds are the Ising model; a (bonds, spins, counter) checkpoint resumes exactly."""
    for dims, L, T in ((2, 64, 2.269), (3, 32, 4.5115)):
        N = L ** dims
        rng = np.random.default_rng(5 + L)
        g = rng.choice(np.array([-1, 1], dtype=np.int8), size=N)
        gg = g.reshape((L,) * dims)
        tau = np.stack([gg * np.roll(gg, -1, axis=dims - 1 - a) for a in range(dims)]).reshape(dims, N).astype(np.int8)
        f = lsm.Lattice(dims=dims, L=L, T=T, seed=99)
        e = lsm.Lattice(dims=dims, L=L, T=T, seed=99, model=lsm.EA)
        e.set_bonds(torch.as_tensor(tau).cuda())
        assert np.array_equal(e.get_bonds().cpu().numpy(), tau)
        e.set_spins((f.get_spins().cpu() * torch.as_tensor(g)).to(torch.int8).cuda(), 0)
        a = f.sweep_record(12).cpu().numpy()
        b = e.sweep_record(12).cpu().numpy()
        assert np.array_equal(a[:, 0], b[:, 0])                                  # the bond energy series, bit for bit
        assert np.array_equal(e.get_spins().cpu().numpy(), f.get_spins().cpu().numpy() * g)
        e.set_bonds(torch.ones((dims, N), dtype=torch.int8, device="cuda"))
        e.set_spins(f.get_spins(), 12)
        assert np.array_equal(f.sweep_record(5).cpu().numpy(), e.sweep_record(5).cpu().numpy())
        f.close()
        e.close()
    kw = dict(dims=2, L=96, T=1.3, model=lsm.EA, seed=31)
    a = lsm.Lattice(**kw)
    a.sweep(7)
    c = lsm.Lattice(**dict(kw, T=2.9))               # another handle: same seed (= same random words), its own state
    c.set_temperature(1.3)
    c.sweep(3)
    c.set_bonds(a.get_bonds())
    c.set_spins(a.get_spins(), 7)
    a.sweep(5)
    c.sweep(5)
    assert np.array_equal(a.get_spins().cpu().numpy(), c.get_spins().cpu().numpy())
    assert a.measure_int() == c.measure_int()
    with pytest.raises(lsm.LsmError) as err:
        lsm.Lattice(dims=2, L=32, T=1.0).get_bonds()
    assert err.value.code == lsm.ERR_UNSUPPORTED


POTTS_SHAPES = [
    (dict(dims=2, L=4, two_S=2, T=1.0), 30),
    (dict(dims=2, L=6, two_S=4, T=0.8), 30),
    (dict(dims=2, L=34, two_S=1, T=1.2), 20),
    (dict(dims=2, L=64, two_S=2, T=0.995), 25),      # near Tc = 1/ln(1 + sqrt 3)
    (dict(dims=2, L=128, two_S=7, T=0.7), 12),       # q = 8
    (dict(dims=2, L=64, two_S=3, T=0.02), 10),       # "never" thresholds
    (dict(dims=2, L=32, two_S=2, T=1.0, J=-1.0), 15),  # antiferromagnetic Potts
    (dict(dims=3, L=4, two_S=2, T=1.8), 20),
    (dict(dims=3, L=6, two_S=3, T=1.5), 12),
    (dict(dims=3, L=32, two_S=2, T=1.82), 6),
    (dict(dims=3, L=34, two_S=5, T=1.2), 4),
    # whole 16-byte words per row: the vectorised rule of the tiled family (byte-parallel equal-neighbour counts)
    (dict(dims=2, L=256, two_S=2, T=0.995), 12),
    (dict(dims=2, L=96, two_S=1, T=1.1), 12),         # q = 2
    (dict(dims=2, L=160, two_S=6, T=0.75, J=1.3), 10),  # q = 7
    (dict(dims=2, L=1024, two_S=3, T=0.91), 5),
    (dict(dims=3, L=64, two_S=7, T=1.0), 4),          # q = 8 in 3D
    (dict(dims=3, L=96, two_S=2, T=0.05), 3),         # 3D, "never" thresholds
    (dict(dims=3, L=32, two_S=4, T=1.4, J=-0.7), 6),
    (dict(dims=2, L=2048, two_S=2, T=0.995), 4),      # many CTAs, several march segments per word column
    (dict(dims=3, L=128, two_S=2, T=1.82), 3),
]


@pytest.mark.parametrize("family", [lsm.KERNEL_AUTO, lsm.KERNEL_GENERIC, lsm.KERNEL_TILED])
@pytest.mark.parametrize("kw,n", POTTS_SHAPES)
def test_potts_parity(kw, n, family):
    kw = dict(kw, model=lsm.POTTS, seed=(0x9077 << 32) + 11 * kw["L"] + kw["two_S"])
    lat, orc = lsm.Lattice(**kw), O.Oracle(**kw)
    try:
        lat.set_kernel(family)
    except lsm.LsmError as e:
        assert e.code == lsm.ERR_UNSUPPORTED
        pytest.skip("this family does not cover this lattice")
    if family == lsm.KERNEL_AUTO and kw["L"] % 32 == 0:
        assert lat.kernel in (lsm.KERNEL_TILED, lsm.KERNEL_SLAB)       # slab: 512^2 ... 4096^2, 64^3, 128^3
    assert lat.thresholds() == orc.thresholds()
    same_state(lat, orc)
    half = n // 2
    got = lat.sweep_record(half).cpu().numpy()
    want = orc.sweep_record(half)
    assert np.array_equal(got, want), np.flatnonzero((got != want).any(axis=1))[:5]
    same_state(lat, orc)
    s = orc.get_spins()
    t0 = (9 << 32) + 5
    lat.set_spins_host(s, t0)                        # checkpoint round trip with a sweep counter above 2^32
    orc.set_spins(s, t0)
    lat.sweep(n - half)
    orc.sweep(n - half)
    same_state(lat, orc)
    lat.set_tracking(False)
    got = lat.sweep_record(3).cpu().numpy()
    assert np.array_equal(got, orc.sweep_record(3))
    same_state(lat, orc, persistence=False)
    lat.close()


def test_wider_models_argument_checks():
    with pytest.raises(lsm.LsmError) as e:
        lsm.Lattice(dims=2, L=32, two_S=2, model=lsm.EA, T=1.0)
    assert e.value.code == lsm.ERR_UNSUPPORTED
    with pytest.raises(lsm.LsmError) as e:
        lsm.Lattice(dims=2, L=32, two_S=8, model=lsm.POTTS, T=1.0)               # q = 9 > 8
    assert e.value.code == lsm.ERR_UNSUPPORTED
    with pytest.raises(lsm.LsmError) as e:
        lsm.Lattice(dims=2, L=32, two_S=2, model=lsm.POTTS, h=0.1, T=1.0)
    assert e.value.code == lsm.ERR_UNSUPPORTED
    with pytest.raises(lsm.LsmError) as e:
        lsm.Lattice(dims=2, L=32, two_S=2, model=lsm.POTTS, T=1.0).sweep_random_tile(1, 32, 16)
    assert e.value.code == lsm.ERR_UNSUPPORTED
