"""Temperature-ramp driver: the protocol of the paper's Fig. 6 on the C-ABI library.

    python -m paper_1209_0296_b200.ramp [--L 128] [--T-start 2.4] [--T-stop 2.1] [--T-step 0.01]
                                        [--equil 2000] [--sweeps 10000] [--seed 1]

"The lattice was initialized and allowed to equilibrate at T = 2.4 ... T was decreased by 0.01 down to T = 2.1 ...
at each T, 10^4 measurements were taken" of magnetisation, energy and heat capacity (the paper uses 2*10^7 sweeps
per temperature; the run lengths are arguments here).  One lattice is carried from temperature to temperature;
lsm_set_temperature rebuilds the integer thresholds on the host (reading D3), lsm_sweep_record returns (B, M) after
every sweep, and the averages are host doubles from the integer series (reading D13).  On a 128^2 lattice the small
kernel family runs each block of sweeps in one launch.  Marshalling and bookkeeping only: every update runs in the
CUDA kernels.
"""
from __future__ import annotations

import argparse
import json
import math

import numpy as np

from . import lsm

TC_2D = 2.0 / math.log(1.0 + math.sqrt(2.0))


def temperatures(T_start: float, T_stop: float, T_step: float) -> list[float]:
    """T_start, T_start - step, ... down to T_stop (inclusive), as decimal literals rounded to 1e-9."""
    n = int(round((T_start - T_stop) / T_step))
    return [round(T_start - k * T_step, 9) for k in range(n + 1)]


def summarise(obs: np.ndarray, N: int, J: float, h: float, T: float) -> dict:
    """Per-site averages over a measured (B, M) series: every number comes from the library (lsm_series_means,
    lsm_heat_capacity, lsm_binder_u4: exact integer accumulation, one rounding at the end)."""
    e, abs_m = lsm.series_means(obs, N, J, h)
    return {
        "T": T,
        "e": e,
        "abs_m": abs_m,
        "c": lsm.heat_capacity(obs, N, J, h, T),
        "u4": lsm.binder_u4(obs),
    }


def temperature_ramp(lat: "lsm.Lattice", temps, n_equil: int, n_meas: int, keep_series: bool = False):
    """Carry `lat` through `temps`: at each T, n_equil unrecorded sweeps, then n_meas recorded ones."""
    import torch

    out = []
    buf = torch.empty((max(n_meas, 1), 2), dtype=torch.int64, device=lat.device)
    for T in temps:
        lat.set_temperature(T)
        lat.sweep(n_equil)
        obs = lat.sweep_record(n_meas, out=buf).cpu().numpy()[:n_meas].copy()
        row = summarise(obs, lat.N, lat.J, lat.h, T)
        if keep_series:
            row["series"] = obs
        out.append(row)
    return out


def main(argv=None) -> int:
    ap = argparse.ArgumentParser()
    ap.add_argument("--L", type=int, default=128)
    ap.add_argument("--T-start", type=float, default=2.4)
    ap.add_argument("--T-stop", type=float, default=2.1)
    ap.add_argument("--T-step", type=float, default=0.01)
    ap.add_argument("--equil", type=int, default=2000)
    ap.add_argument("--sweeps", type=int, default=10000)
    ap.add_argument("--seed", type=int, default=1)
    a = ap.parse_args(argv)
    import torch

    temps = temperatures(a.T_start, a.T_stop, a.T_step)
    lat = lsm.Lattice(dims=2, L=a.L, T=temps[0], seed=a.seed)
    lat.set_tracking(False)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    rows = temperature_ramp(lat, temps, a.equil, a.sweeps)
    e1.record()
    torch.cuda.synchronize()
    for r in rows:
        print(json.dumps(r))
    peak = max(rows, key=lambda r: r["c"])
    print(json.dumps({"lattice": f"{a.L}^2", "temperatures": len(temps), "sweeps_per_T": a.equil + a.sweeps,
                      "seconds": e0.elapsed_time(e1) * 1e-3, "heat_capacity_peak_at_T": peak["T"], "Tc_exact": TC_2D,
                      "kernel_family": lat.kernel}))
    return 0


if __name__ == "__main__":
    raise SystemExit(main())
