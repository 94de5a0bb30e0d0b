"""Seeded synthetic workloads shaped like the paper's (shared by tests/ and bench.py).

This module holds configuration data only -- lattice shapes, couplings, temperatures, seeds and run
lengths of BASELINE.json's five configs -- and none of the method's arithmetic.
The lattices themselves are drawn on the device (and, independently, by the oracle) from the seed.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, replace

ISING, NE_HEATBATH, NE_METROPOLIS, EA, POTTS = 0, 1, 2, 3, 4


def seed_of(cfg: int, variant: int = 0) -> int:
    """seed = 12090296 * 2^32 + cfg * 256 + variant (variant = temperature / concentration index)."""
    return (12090296 << 32) + cfg * 256 + variant


def ne_temperature(c: float) -> float:
    """T with c = 1/(1+exp(1/T)) (reading D6): what the harness passes for a target concentration."""
    return 1.0 / math.log((1.0 - c) / c)


@dataclass(frozen=True)
class Workload:
    name: str
    cfg: int
    dims: int
    L: int
    two_S: int = 1
    model: int = ISING
    J: float = 1.0
    h: float = 0.0
    T: float = 1.0
    seed: int = 0
    sweeps: int = 1
    note: str = ""

    @property
    def N(self) -> int:
        return self.L ** self.dims

    def create_args(self):
        return dict(dims=self.dims, L=self.L, two_S=self.two_S, model=self.model, J=self.J, h=self.h,
                    T=self.T, seed=self.seed)

    def scaled(self, L: int, sweeps: int | None = None) -> "Workload":
        """Same physics on a smaller lattice (the reduced shapes of the parity tests)."""
        return replace(self, L=L, sweeps=self.sweeps if sweeps is None else sweeps,
                       name=f"{self.name}@L{L}")


def configs() -> dict[str, Workload]:
    out = {}
    out["cfg1"] = Workload("cfg1", 1, 2, 64, T=2.269, seed=seed_of(1), sweeps=1000,
                           note="2D Ising spin-1/2 64^2 near Tc, (E, M) after every sweep")
    for v, T in enumerate((2.0, 2.269, 2.6)):
        out[f"cfg2_T{T}"] = Workload(f"cfg2_T{T}", 2, 2, 8192, T=T, seed=seed_of(2, v), sweeps=10_000,
                                     note="2D Ising spin-1/2 8192^2, per-sweep E, M, U4 over the last 5000 sweeps")
    out["cfg3"] = Workload("cfg3", 3, 3, 512, T=4.5115, seed=seed_of(3), sweeps=2000,
                           note="3D Ising spin-1/2 512^3 near the 3D Tc")
    out["cfg4"] = Workload("cfg4", 4, 3, 256, two_S=2, h=0.01, T=3.0, seed=seed_of(4), sweeps=2000,
                           note="3D spin-1 Ising 256^3")
    for v, c in enumerate((0.10, 0.20, 0.30)):
        out[f"cfg5_c{c:.2f}"] = Workload(f"cfg5_c{c:.2f}", 5, 2, 8192, model=NE_HEATBATH, J=0.0,
                                         T=ne_temperature(c), seed=seed_of(5, v), sweeps=100_000,
                                         note="2D North-East heat-bath 8192^2, persistence every 100 sweeps")
    return out


def extras() -> dict[str, Workload]:
    """Workloads beyond BASELINE.json's five, used by bench.py for the rooflines: a lattice far larger than the
    126 MB L2 (the HBM-streaming case SURVEY.md 8(d) asks for -- config 3's 128 MiB is borderline), and a cold
    2D lattice whose table has "never" entries (exp(-8/T) < 2^-32 below T ~ 0.36)."""
    out = {}
    out["hbm3d_1024"] = Workload("hbm3d_1024", 6, 3, 1024, T=4.5115, seed=seed_of(6), sweeps=100,
                                 note="3D Ising spin-1/2 1024^3 (1 GiB of spins): the HBM-streaming case")
    out["hbm2d_32768"] = Workload("hbm2d_32768", 6, 2, 32768, T=2.269, seed=seed_of(6, 1), sweeps=100,
                                  note="2D Ising spin-1/2 32768^2 (1 GiB of spins)")
    out["cold2d_T0.30"] = Workload("cold2d_T0.30", 7, 2, 8192, T=0.30, seed=seed_of(7), sweeps=100,
                                   note="2D Ising spin-1/2 8192^2 at T = 0.30: thresholds with never-accepted entries")
    # mid-size lattices (between the paper's own 32^2 ... 512^2, and BASELINE.json's 8192^2): a
    # half-sweep is shorter than a kernel launch, the regime of the slab family (lattice resident in shared memory)
    for L, n in ((512, 2000), (1024, 1000), (2048, 400), (4096, 100)):
        out[f"mid2d_{L}"] = Workload(f"mid2d_{L}", 8, 2, L, T=2.269, seed=seed_of(8, L // 512), sweeps=n,
                                     note=f"2D Ising spin-1/2 {L}^2 near Tc, (E, M) after every sweep")
    # SURVEY.md 8(f) NEXT-4 models (readings D25, D26): the +/-J Edwards-Anderson glass and the q-state Potts model
    out["ea2d_8192"] = Workload("ea2d_8192", 9, 2, 8192, model=EA, T=1.0, seed=seed_of(9, 0), sweeps=100,
                                note="2D Edwards-Anderson +/-J spin glass 8192^2, bonds from the seed")
    out["ea3d_512"] = Workload("ea3d_512", 9, 3, 512, model=EA, T=1.1, seed=seed_of(9, 1), sweeps=40,
                               note="3D Edwards-Anderson +/-J spin glass 512^3 near its glass temperature")
    out["potts2d_q3_4096"] = Workload("potts2d_q3_4096", 9, 2, 4096, two_S=2, model=POTTS, T=0.995, seed=seed_of(9, 2),
                                      sweeps=20, note="2D 3-state Potts 4096^2 at its transition T = 1/ln(1+sqrt 3)")
    out["mid3d_128"] = Workload("mid3d_128", 8, 3, 128, T=4.5115, seed=seed_of(8, 9), sweeps=400,
                                note="3D Ising spin-1/2 128^3 near the 3D Tc")
    return out


def parse_shape(name: str) -> Workload:
    """Any lattice of the models by name, so that every table row under profiles/ has a command
    (`python bench.py --workload ea2d_1024 --kernel tiled --no-extras`):
      ising2d_<L> ising3d_<L> spin1_2d_<L> spin1_3d_<L> ea2d_<L> ea3d_<L> ne2d_c<conc>_<L> potts2d_q<q>_<L> potts3d_q<q>_<L>
    at the temperatures of the named workloads of the same model (2D Ising 2.269, 3D 4.5115, spin-1 3.0 with h = 0.01,
    EA 1.0 / 1.1, Potts at its 2D transition 1/ln(1+sqrt q), 3D q = 3: 1.8164)."""
    import re

    m = re.fullmatch(r"(ising|spin1_|ea|potts|ne)([23])d(?:_q(\d+))?(?:_c([0-9.]+))?_(\d+)", name)
    if not m:
        raise KeyError(name)
    kind, dims, q, c, L = m.group(1), int(m.group(2)), m.group(3), m.group(4), int(m.group(5))
    seed = seed_of(10 + dims, L % 256)
    if kind == "ising":
        return Workload(name, 10, dims, L, T=2.269 if dims == 2 else 4.5115, seed=seed, note=f"Ising spin-1/2 {L}^{dims}")
    if kind == "spin1_":
        return Workload(name, 10, dims, L, two_S=2, h=0.01, T=3.0 if dims == 3 else 1.69, seed=seed, note=f"spin-1 Ising {L}^{dims}")
    if kind == "ea":
        return Workload(name, 10, dims, L, model=EA, T=1.0 if dims == 2 else 1.1, seed=seed, note=f"Edwards-Anderson {L}^{dims}")
    if kind == "ne":
        if dims != 2 or c is None:
            raise KeyError(name)
        return Workload(name, 10, 2, L, model=NE_HEATBATH, J=0.0, T=ne_temperature(float(c)), seed=seed, note=f"North-East {L}^2 c = {c}")
    if q is None:
        raise KeyError(name)
    qq = int(q)
    T = 1.0 / math.log(1.0 + math.sqrt(qq)) if dims == 2 else 1.8164
    return Workload(name, 10, dims, L, two_S=qq - 1, model=POTTS, T=T, seed=seed, note=f"{qq}-state Potts {L}^{dims}")


def by_name(name: str) -> Workload:
    both = {**configs(), **extras()}
    return both[name] if name in both else parse_shape(name)
