"""lambda-convergence check of the paper's corrected North-East algorithm (Fig. 5).

    python -m paper_1209_0296_b200.lambda_scan [--L 128] [--c 0.42] [--realisations 8] [--times 10 30 100 300 1000]

"The limit of Q = 1 and lambda = 1 is in fact serial ... The value of lambda is then calibrated to reproduce the
results of the single thread, single block results"; Fig. 5 shows the spin-spin autocorrelation Phi(t)
(Eq. 4) for several lambda at c = 0.42 with 32 x 32 tiles, lambda = 16 being the largest value that
still follows the serial curve.  This driver runs that experiment on the library: for every schedule
(tile edge b, lambda) and realisation it sweeps with lsm_sweep_random_tile and evaluates Phi(t) from lsm_persistence's
overlap with lsm_phi; the reference is b = L, lambda = 1 (one tile, one pick at a time).  Bookkeeping only: every
update and every reduction runs in the CUDA kernels, Phi is formed in the library."""
from __future__ import annotations

import argparse
import json
import math

from . import lsm, workloads as W


def phi_curves(L, c, schedules, times, realisations, seed0=1209, model=lsm.NE_METROPOLIS, device="cuda:0"):
    """{(b, lam): {"phi": [mean Phi(t) for t in times], "se": [standard error of that mean]}}."""
    T = W.ne_temperature(c)
    c_lib = 1.0 / (1.0 + math.exp(1.0 / T))              # the concentration the library derives from T (reading D6)
    out = {}
    for (b, lam) in schedules:
        acc = [[] for _ in times]
        # all realisations of a schedule as one batch: every launch of the schedule covers the tiles of all of them
        # (lsm_batch_sweep_random_tile; replica r is bit-identical to a single lattice with seed seed0 + r)
        batch = lsm.Batch(T=[T] * realisations, seeds=[seed0 + r for r in range(realisations)], dims=2, L=L, model=model,
                          J=0.0, device=device)
        t_now = 0
        for k, t in enumerate(times):
            batch.sweep_random_tile(t - t_now, b, lam)
            t_now = t
            for r in range(realisations):
                _, ov = batch.replica(r).persistence()
                acc[k].append(lsm.phi(ov, batch.N, c_lib))
        batch.close()
        mean = [sum(a) / len(a) for a in acc]
        se = [math.sqrt(sum((x - m) ** 2 for x in a) / max(len(a) - 1, 1) / len(a)) for a, m in zip(acc, mean)]
        out[(b, lam)] = {"phi": mean, "se": se}
    return out


def main(argv=None) -> int:
    ap = argparse.ArgumentParser()
    ap.add_argument("--L", type=int, default=128)
    ap.add_argument("--c", type=float, default=0.42)
    ap.add_argument("--realisations", type=int, default=8)
    ap.add_argument("--times", type=int, nargs="+", default=[10, 30, 100, 300, 1000])
    a = ap.parse_args(argv)
    sched = [(a.L, 1), (32, 1), (32, 4), (32, 16), (32, 32), (16, 32), (8, 32)]
    import time

    t0 = time.perf_counter()
    res = phi_curves(a.L, a.c, sched, a.times, a.realisations)
    wall = time.perf_counter() - t0
    ref = res[(a.L, 1)]
    for (b, lam), v in res.items():
        dev = max(abs(x - y) for x, y in zip(v["phi"], ref["phi"]))
        print(json.dumps({"tile_edge": b, "lambda": lam, "lambda_over_P": lam / (b * b), "times": a.times,
                          "phi": [round(x, 4) for x in v["phi"]], "se": [round(x, 4) for x in v["se"]],
                          "max_abs_dev_from_serial": round(dev, 4)}))
    print(json.dumps({"wall_s": round(wall, 2), "L": a.L, "realisations": a.realisations, "schedules": len(sched),
                      "sweeps_per_realisation_and_schedule": max(a.times)}))
    return 0


if __name__ == "__main__":
    raise SystemExit(main())
