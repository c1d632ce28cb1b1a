"""Dispatch sweep: times every kernel variant of libsd_b200 over N and prints the crossovers.

    python -m paper_1205_6333_b200.tune [f64] [box]
    python -m paper_1205_6333_b200.tune cfg5        (the reporting sweep)
    python -m paper_1205_6333_b200.tune one N IPT   (4 products at one size, for ncu)

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


CFG5_NS = [1024, 4096, 16384, 65536, 262144, 1048576]
PEAK_F32, PEAK_F64 = 148 * 128 * 2 * 1.965e9, 148 * 64 * 2 * 1.965e9
FLOPS = {"rpy": 34, "oseen": 29}


def _times(torch, fn, warm, reps):
    for _ in range(warm):
        fn()
    torch.cuda.synchronize()
    out = []
    for _ in range(reps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        fn()
        e1.record()
        torch.cuda.synchronize()
        out.append(e0.elapsed_time(e1) * 1e-3)
    return np.array(out)


def cfg5(torch, sd, wl):
    """SURVEY.md 8(d), configuration 5: sd_mobility_apply, {fp32-Kahan, fp64} x {RPY, Oseen},
    3 warm-up + 10 timed launches each; best and median pair rate and roofline fraction.  Then
    sd_step steps/s on configurations 1, 3 and 4."""
    print("| N | precision | tensor | kernel | best pairs/s | median pairs/s | best frac of FMA peak | median frac |")
    print("|---|---|---|---|---|---|---|---|")
    for n in CFG5_NS:
        pos, force = wl.sweep(n)
        for pname, prec, npdt, peak in (("fp32-Kahan", sd.PREC_F32_KAHAN, np.float32, PEAK_F32),
                                        ("fp64", sd.PREC_F64, np.float64, PEAK_F64)):
            dp = torch.from_numpy(wl.to_xyzw(pos, npdt)).cuda()
            df = torch.from_numpy(wl.to_xyzw(force, npdt)).cuda()
            dv = torch.empty_like(dp)
            for tname, tensor in (("rpy", sd.TENSOR_RPY), ("oseen", sd.TENSOR_OSEEN)):
                ctx = sd.Context(n, wl.A, wl.ETA)
                ctx.set_tensor(tensor)
                ctx.set_precision(prec)
                t = _times(torch, lambda: ctx.mobility_apply(dp, df, dv), 3, 10)
                best, med = n * n / t.min(), n * n / np.median(t)
                print(f"| {n} | {pname} | {tname} | {ctx.kernel_name} | {best:.3e} | {med:.3e} | "
                      f"{best * FLOPS[tname] / peak:.3f} | {med * FLOPS[tname] / peak:.3f} |", flush=True)
                ctx.close()
    print()
    print("| configuration | N | integrator | precision | steps per call | steps/s (median of 5 calls) |")
    print("|---|---|---|---|---|---|")
    p1, _ = wl.four_sphere(wl.SEED_BASE + 1)
    p3, _ = wl.config3()
    p4, _ = wl.config4()
    for name, pos, integ, iname, dt, steps in (("1", p1, sd.INT_MIDPOINT, "midpoint", 0.01, 10000),
                                               ("3", p3, sd.INT_EULER, "Euler", 0.01, 20),
                                               ("4", p4, sd.INT_MIDPOINT, "midpoint", 0.05, 10)):
        n = pos.shape[0]
        for pname, prec, npdt in (("fp32-Kahan", sd.PREC_F32_KAHAN, np.float32), ("fp64", sd.PREC_F64, np.float64)):
            ctx = sd.Context(n, wl.A, wl.ETA)
            ctx.set_precision(prec)
            dq = torch.from_numpy(wl.to_xyzw(pos, npdt)).cuda()
            t = _times(torch, lambda: ctx.step(dq, dt, steps, integ, gravity=(0.0, 0.0, -1.0)), 1, 5)
            print(f"| {name} | {n} | {iname} | {pname} | {steps} | {steps / np.median(t):.4g} |", flush=True)
            ctx.close()


def main(argv):
    import torch
    from . import sd, workloads as wl
    sd.load_library()
    torch.cuda.set_device(0)
    if "cfg5" in argv:
        return cfg5(torch, sd, wl)
    if argv and argv[0] == "one":
        n, ipt = int(argv[1]), int(argv[2])
        pos, force = wl.sweep(n)
        dp = torch.from_numpy(wl.to_xyzw(pos, np.float32)).cuda()
        df = torch.from_numpy(wl.to_xyzw(force, np.float32)).cuda()
        dv = torch.empty_like(dp)
        ctx = sd.Context(n, wl.A, wl.ETA)
        ctx.set_dispatch(-1 if ipt == 0 else 0, ipt)
        print(n, ctx.kernel_name, _time(torch, lambda: ctx.mobility_apply(dp, df, dv), 1) * 1e6, "us")
        ctx.close()
        return None
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
