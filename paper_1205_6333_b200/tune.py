"""Dispatch sweep: times every kernel variant of libsd_b200 over N and prints the crossovers.

    python -m paper_1205_6333_b200.tune [f64] [box]

For each N it forces, through sd_set_dispatch, the one-launch warp-per-particle kernel ("small")
and the tiled packed kernels with 2 / 4 / 8 particles per thread (fp64: 1 / 2 / 4), and times
sd_mobility_apply and one Euler step of sd_step (CUDA events, warm caches, mean of many launches).
The defaults compiled into the library (kSmallApplyMax, kIpt4Min, kIpt8Min, kIpt4Min64) are the
crossovers this prints on a B200 (profiles/r01e_sweep.md).  Needs a GPU; argument marshalling and
timing only.
"""
from __future__ import annotations

import sys

import numpy as np

NS = [512, 1024, 1500, 2048, 3000, 4000, 6000, 8192, 12000, 16384, 24576, 32768, 49152, 65536,
      98304, 131072, 196608, 262144]
MODES = {"small": (1 << 30, 0), "i2": (0, 2), "i4": (0, 4), "i8": (0, 8), "auto": (-1, 0)}


def _time(torch, fn, reps):
    for _ in range(3):
        fn()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(reps):
        fn()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) * 1e-3 / reps


def main(argv):
    import torch
    from . import sd, workloads as wl
    sd.load_library()
    torch.cuda.set_device(0)
    f64, box = "f64" in argv, "box" in argv
    prec, npdt = (sd.PREC_F64, np.float64) if f64 else (sd.PREC_F32_KAHAN, np.float32)
    print(f"| N | apply us: small | i2 | i4 | i8 | auto | step us: small | i2 | i4 | i8 | auto | auto kernel "
          f"| pairs/s (auto) |")
    print("|---|---|---|---|---|---|---|---|---|---|---|---|---|")
    for n in NS:
        pos, force = wl.sweep(n)
        dp = torch.from_numpy(wl.to_xyzw(pos, npdt)).cuda()
        df = torch.from_numpy(wl.to_xyzw(force, npdt)).cuda()
        dv = torch.empty_like(dp)
        row = {}
        for mode, (smax, ipt) in MODES.items():
            if (mode == "small" and n > 20000) or (mode == "i8" and n < 8000):
                continue
            ctx = sd.Context(n, wl.A, wl.ETA)
            ctx.set_precision(prec)
            ctx.set_dispatch(smax, ipt)
            if box:
                ctx.set_box(wl.cube_side(n, 0.01))
            reps = max(3, min(200, int(2e11 / n / n)))
            t = _time(torch, lambda: ctx.mobility_apply(dp, df, dv), reps)
            dq = dp.clone()
            ts = _time(torch, lambda: ctx.step(dq, 1e-3, 10, sd.INT_EULER, gravity=(0.0, 0.0, -1.0)),
                       max(2, reps // 10)) / 10
            row[mode] = (t * 1e6, ts * 1e6, ctx.kernel_name)
            ctx.close()

        def cell(mode, k):
            return f"{row[mode][k]:.1f}" if mode in row else "-"
        print(f"| {n} | " + " | ".join(cell(m, 0) for m in MODES) + " | "
              + " | ".join(cell(m, 1) for m in MODES)
              + f" | {row['auto'][2]} | {n * n / row['auto'][0] * 1e6:.3e} |", flush=True)


if __name__ == "__main__":
    main(sys.argv[1:])
