"""Long-run numerical-stability experiment of PAPER.md:249-267 (Fig. 4, Fig. 5) on the GPU path.

    python -m paper_1205_6333_b200.stability [--dt 0.01] [--steps 50000000] [--stride 100]

Four equal spheres on a stretched tetrahedron (reading A1) sediment periodically with
T ~ 517 tau_s.  The paper integrates with Euler for ~1000 cycles and compares single against
double-single precision for (a) the accumulation of the hydrodynamic interactions and (b) the
positions.  Here (a) is sd_set_precision (F32_PLAIN / F32_KAHAN), (b) is
sd_set_position_compensation, and an all-fp64 run is added.  Everything runs in the library's
one-launch stepper kernel; this module only drives it, samples x_1, y_1 every `stride` steps
(device-side copies, one download at the end), and reduces the samples the way the paper does:
maxima and minima of x_1(t) by parabolic fits -> cycle duration and amplitude, averaged over
windows of 1e4 tau_s; max |y_1| per window (particle 1 must stay in the xz-plane).

The cluster falls ~1.25 a per tau_s, so every 512 samples all z are shifted up by a multiple of
64 a (exact in fp32, low words stay valid): coordinates stay below 2^11 a, as in a periodic box.
Argument marshalling and post-processing only; needs a GPU.
"""
from __future__ import annotations

import argparse
import sys

import numpy as np

MODES = [  # name, precision attr, position compensation
    ("HI double-single (Kahan), positions double-single", "PREC_F32_KAHAN", True),
    ("HI double-single (Kahan), positions single", "PREC_F32_KAHAN", False),
    ("HI single, positions double-single", "PREC_F32_PLAIN", True),
    ("HI single, positions single", "PREC_F32_PLAIN", False),
    ("all fp64", "PREC_F64", True),
]


def run_mode(torch, sd, wl, prec_name, pos_comp, dt, steps, stride, perturb=0.0):
    prec = getattr(sd, prec_name)
    npdt = np.float64 if prec == sd.PREC_F64 else np.float32
    pos, _ = (wl.four_sphere(jitter_seed=wl.SEED_BASE + 70, jitter=perturb) if perturb > 0.0
              else wl.four_sphere())
    ctx = sd.Context(4, wl.A, wl.ETA)
    ctx.set_precision(prec)
    ctx.set_position_compensation(pos_comp)
    dp = torch.from_numpy(wl.to_xyzw(pos, npdt)).cuda()
    nsamp = steps // stride
    traj = torch.empty((nsamp, 4, 4), dtype=dp.dtype, device=dp.device)
    zshift = np.zeros(nsamp)
    shift = 0.0
    for k in range(nsamp):
        ctx.step(dp, dt, stride, sd.INT_EULER, gravity=(0.0, 0.0, -1.0))
        traj[k].copy_(dp)
        zshift[k] = shift
        if (k & 511) == 511:
            zc = float(dp[:, 2].mean())
            if not np.isfinite(zc):
                break
            s = 64.0 * np.floor(-zc / 64.0)
            if s > 0.0:
                dp[:, 2] += s
                shift += s
    torch.cuda.synchronize()
    out = traj.cpu().numpy().astype(np.float64)
    out[:, :, 2] -= zshift[:, None]
    ctx.close()
    return out


def extrema(t, x):
    """Parabolic fits through the three samples around each local maximum / minimum."""
    res = {}
    for sign, key in ((1.0, "max"), (-1.0, "min")):
        y = sign * x
        idx = np.nonzero((y[1:-1] > y[:-2]) & (y[1:-1] >= y[2:]))[0] + 1
        a, b, c = y[idx - 1], y[idx], y[idx + 1]
        den = a - 2.0 * b + c
        off = np.where(den != 0.0, 0.5 * (a - c) / np.where(den != 0.0, den, 1.0), 0.0)
        h = t[1] - t[0]
        res[key] = (t[idx] + off * h, sign * (b - 0.25 * (a - c) * off))
    return res


def analyse(traj, dt, stride, window=1.0e4):
    t = (np.arange(traj.shape[0]) + 1) * dt * stride
    x1, y1 = traj[:, 0, 0], traj[:, 0, 1]
    ok = np.isfinite(x1)
    ex = extrema(t[ok], x1[ok])
    tmax, xmax = ex["max"]
    tmin, xmin = ex["min"]
    rows = []
    nwin = int(np.ceil(t[-1] / window))
    for w in range(nwin):
        lo, hi = w * window, (w + 1) * window
        sel = (tmax[1:] >= lo) & (tmax[1:] < hi)
        dur = np.diff(tmax)[sel]
        amps = []
        for tm, xm in zip(tmax[(tmax >= lo) & (tmax < hi)], xmax[(tmax >= lo) & (tmax < hi)]):
            j = np.searchsorted(tmin, tm)
            if j < len(tmin):
                amps.append(0.5 * (xm - xmin[j]))
        ysel = (t >= lo) & (t < hi)
        rows.append((lo, hi, len(dur), float(np.mean(dur)) if len(dur) else float("nan"),
                     float(np.std(dur)) if len(dur) else float("nan"),
                     float(np.mean(amps)) if amps else float("nan"),
                     float(np.nanmax(np.abs(y1[ysel]))) if ysel.any() else float("nan")))
    return rows, len(tmax)


def report(name, rows, ncycles, out):
    out.write(f"\n### {name}\n\n{ncycles} maxima of x_1 found.\n\n")
    out.write("| window [tau_s] | cycles | mean cycle duration | std | mean amplitude of x_1 | max abs y_1 |\n")
    out.write("|---|---|---|---|---|---|\n")
    for lo, hi, n, d, sdv, a, y in rows:
        out.write(f"| {lo:.0f} - {hi:.0f} | {n} | {d:.4f} | {sdv:.2e} | {a:.5f} | {y:.3e} |\n")
    out.flush()


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--dt", type=float, default=0.01)
    ap.add_argument("--steps", type=int, default=50_000_000)
    ap.add_argument("--stride", type=int, default=100)
    ap.add_argument("--window", type=float, default=1.0e4)
    ap.add_argument("--every", type=int, default=1, help="print every n-th window")
    ap.add_argument("--perturb", type=float, default=0.0,
                    help="seeded offsets of that size (units of a) on the initial positions: breaks "
                         "the exact mirror symmetry that otherwise keeps y_1 = 0 bit for bit")
    args = ap.parse_args(argv)
    import torch
    from . import sd, workloads as wl
    sd.load_library()
    torch.cuda.set_device(0)
    out = sys.stdout
    out.write(f"## Euler, dt = {args.dt} tau_s, {args.steps} steps = {args.steps * args.dt:.0f} tau_s, "
              f"sampled every {args.stride} steps, initial perturbation {args.perturb:g} a\n")
    for name, prec_name, comp in MODES:
        traj = run_mode(torch, sd, wl, prec_name, comp, args.dt, args.steps, args.stride,
                        args.perturb)
        rows, ncyc = analyse(traj, args.dt, args.stride, args.window)
        report(name, rows[::args.every], ncyc, out)


if __name__ == "__main__":
    main()
