"""Integer-pipe probe: how the ALU pipe and the FMA-heavy pipe share issue on this GPU.

    python -m paper_1209_0296_b200.pipe_probe

Prints cycles per loop iteration and warp for a set of register-only instruction streams; the
sweep kernels are designed around the law these numbers show (an IMAD.WIDE costs 4 FMA-pipe cycles
and one 2-cycle ALU-pipe slot)."""
from __future__ import annotations

import sys

MODES = [
    (0, "16 LOP3", 0, 0, 16),
    (1, "8 IMAD", 0, 8, 0),
    (2, "8 IMAD.WIDE (+8 adds)", 8, 0, 8),
    (3, "8 IMAD + 16 LOP3", 0, 8, 16),
    (4, "4 Philox calls (80 WIDE + 80 LOP3)", 80, 0, 80),
    (5, "4 Philox calls + 80 LOP3", 80, 0, 160),
    (6, "4 Philox calls + 160 LOP3", 80, 0, 240),
    (7, "4 Philox calls + 240 LOP3", 80, 0, 320),
    (8, "4 Philox calls + 80 IMAD", 80, 80, 80),
    (9, "4 Philox calls + 80 IMAD + 80 LOP3", 80, 80, 160),
    (10, "4 Philox calls + 80 IMAD + 160 LOP3", 80, 80, 240),
]


def run(blocks_per_sm=8, iters=1024):
    import torch

    from . import build, lsm

    build.build()
    props = torch.cuda.get_device_properties(0)
    sms = props.multi_processor_count
    try:
        import pynvml

        pynvml.nvmlInit()
        mhz = pynvml.nvmlDeviceGetMaxClockInfo(pynvml.nvmlDeviceGetHandleByIndex(0), pynvml.NVML_CLOCK_SM)
    except Exception:
        mhz = 1965
    out = []
    warps_per_smsp = blocks_per_sm * 8 / 4.0
    for mode, name, W, I, A in MODES:
        lsm.pipe_probe(mode, sms * blocks_per_sm, 32)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        lsm.pipe_probe(mode, sms * blocks_per_sm, iters)
        e1.record()
        torch.cuda.synchronize()
        cyc = e0.elapsed_time(e1) * 1e-3 * mhz * 1e6 / iters / warps_per_smsp
        model = max(4 * W + 2 * I, 2 * (A + W))
        out.append(dict(mode=mode, stream=name, cycles_per_iter_per_warp=cyc, wide=W, imad=I, alu=A,
                        law_max_4W_2I__2A_2W=model, overlap_only_max_4W_2I__2A=max(4 * W + 2 * I, 2 * A)))
    return dict(gpu=props.name, sm_mhz=mhz, warps_per_smsp=warps_per_smsp, rows=out)


def main():
    r = run()
    print(f"# {r['gpu']}  clocks.max.sm {r['sm_mhz']} MHz  {r['warps_per_smsp']:.0f} warps/SMSP")
    print("| stream | measured cycles/iter/warp | law max(4W+2I, 2(A+W)) | if WIDE took no ALU slot |")
    print("|---|---|---|---|")
    for x in r["rows"]:
        print(f"| {x['stream']} | {x['cycles_per_iter_per_warp']:.1f} | {x['law_max_4W_2I__2A_2W']} | {x['overlap_only_max_4W_2I__2A']} |")
    return 0


if __name__ == "__main__":
    sys.exit(main())
