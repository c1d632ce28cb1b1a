#!/usr/bin/env python
"""bench.py -- throughput of the mobility product v = M(r) F on B200 (BASELINE.json metric).

A "step" is one pass of the whole hot path (pack -> all-pairs kernel -> reduce + self term) over
one batch of synthetic particles: sd_mobility_apply at N = 1,048,576 (uniform cube, volume
fraction 0.01, N(0,1) forces, Rotne-Prager-Yamakawa, fp32 terms + Kahan accumulation), the
configuration the north_star target is quoted on.  Prints ONE JSON line.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

N > 1 (torchrun): independent replicas, one per GPU ("replicas only"); the value is
the summed pair rate over the max-over-ranks time.  --impl reference times the CPU oracle on
the host cores on a bounded row sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

FLOPS_PER_PAIR = {"rpy": 34, "oseen": 29}       # algorithmic flops
FLOPS_NEAREST_IMAGE = 15                        # + 3 x (fma, add, fma) per pair in a periodic box
FP32_LANES_PER_SM, FP64_LANES_PER_SM = 128, 64  # CUDA-core FMA lanes per SM (measured: ubench)
# DRAM bytes (read + write) per pair-kernel launch.  NOT measured by this script (ncu cannot run
# inside a timed bench): copied from the committed `ncu --set full` capture of the kernel this
# commit ships, named beside it; a configuration without such a capture reports null.
NCU_TRAFFIC = {
    (1048576, "f32", "rpy", False): (42.7e6, "profiles/r02_pairs_ncu_full.md (dram__bytes_read.sum + "
                                             "dram__bytes_write.sum of pairs_f32_kernel<4,RPY,Kahan,TJ=256>, 34.4 + 8.3 MB)"),
    (1048576, "f32", "rpy", True): (44.2e6, "profiles/r02_pairs_ncu_full.md (pairs_f32_kernel<4,RPY,Kahan,PBC,TJ=256>, 34.4 + 9.7 MB)"),
    (1048576, "f64", "rpy", False): (3.60e9, "profiles/r02_pairs_ncu_full.md (pairs_f64_kernel<4,RPY,TJ=128>, 3.54 GB + 68 MB: "
                                             "L2 misses of the 67-MB record stream)"),
}
CFG5_NS = [1024, 4096, 16384, 65536, 262144, 1048576]   # BASELINE.json configs[4]


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--n", type=int, default=1048576)
    ap.add_argument("--precision", choices=["f32", "f64"], default="f32")
    ap.add_argument("--tensor", choices=["rpy", "oseen"], default="rpy")
    ap.add_argument("--box", action="store_true",
                    help="periodic cube of the cloud's own side, nearest image only (PAPER.md:115)")
    ap.add_argument("--fcc-cells", type=int, default=0,
                    help="instead of the product: the paper's benchmark run (PAPER.md:231), fcc "
                         "lattice of 4 cells^3 spheres at n = 0.1 a^-3 in its periodic box, 100 "
                         "Euler steps of 0.001 tau_s per timed step; reports simulation steps/s")
    ap.add_argument("--staging", choices=["bulk", "naive", "sync"], default="bulk",
                    help="memory-access ablation (PAPER.md Appendix A): how j records reach the threads")
    ap.add_argument("--full-loop", action="store_true",
                    help="with --fcc-cells: run the paper's whole step (PAPER.md:96-109), i.e. switch the "
                         "lubrication correction of the forces on (sd_set_lubrication)")
    ap.add_argument("--lub", action="store_true",
                    help="instead of the product: the lubrication correction of the forces (Eq. 8, "
                         "PAPER.md:80-104) on N uniform points at phi = 0.05; reports particles/s")
    ap.add_argument("--jsplit", choices=["auto", "classic", "warp"], default="auto",
                    help="fp32 mapping of the j sum (sd_set_jsplit): classic tiled kernels (pack + pairs + "
                         "finalize) or the warp-split one-launch kernel; auto = by N")
    ap.add_argument("--launches-per-step", type=int, default=1,
                    help="products enqueued back to back inside one timed step (small N: one launch is "
                         "shorter than the event pair around it); value and ms_per_step are per product")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extra", action="store_true",
                    help="skip the `extra` object (fp64 / Oseen at N = 1M, the configuration-5 sweep, "
                         "sd_step steps/s on configurations 1, 3, 4)")
    ap.add_argument("--extra-only", action="store_true",
                    help="print only the `extra` object (one JSON line)")
    return ap.parse_args()


def workload(n):
    from paper_1205_6333_b200 import workloads as wl
    pos, force = wl.sweep(n)
    return pos, force, wl


def workload_name(args):
    return (f"sd_mobility_apply N={args.n} uniform cube phi=0.01, N(0,1) forces, "
            f"{args.tensor.upper()}, {'fp32-Kahan' if args.precision == 'f32' else 'fp64'}"
            + (", periodic box (nearest image)" if args.box else "")
            + (f", staging={args.staging}" if args.staging != "bulk" else ""))


def box_side(args, wl):
    return wl.cube_side(args.n, 0.01) if args.box else 0.0


def time_oracle(pos64, force64, wl, tensor, target_seconds, box=0.0, image=0):
    """Oracle pair rate on a bounded seeded row sample sized for about target_seconds."""
    from oracle import sd_oracle as orc
    otensor = orc.TENSOR_RPY if tensor == "rpy" else orc.TENSOR_OSEEN
    n = pos64.shape[0]
    cores = orc.num_threads()
    probe_rows = wl.row_subset(n, min(n, 8 * cores), wl.SEED_BASE + 9)
    t0 = time.perf_counter()
    orc.apply_rows(pos64, force64, probe_rows, wl.A, wl.ETA, otensor, box=box, image=image)
    t_probe = max(time.perf_counter() - t0, 1e-6)
    rows = int(min(n, max(len(probe_rows), len(probe_rows) * target_seconds / t_probe)))
    sample = wl.row_subset(n, rows, wl.SEED_BASE + 10)
    t0 = time.perf_counter()
    orc.apply_rows(pos64, force64, sample, wl.A, wl.ETA, otensor, box=box, image=image)
    t = time.perf_counter() - t0
    return len(sample) * n / t, cores, len(sample), t


def cpu_model():
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def run_reference(args, rank):
    """--impl reference: the oracle as it stands, on the host cores."""
    if rank != 0:
        return
    pos, force, wl = workload(args.n)
    p64 = wl.to_xyzw(pos, np.float32)[:, :3].astype(np.float64)
    f64 = wl.to_xyzw(force, np.float32)[:, :3].astype(np.float64)
    from oracle import sd_oracle as orc
    otensor = orc.TENSOR_RPY if args.tensor == "rpy" else orc.TENSOR_OSEEN
    cores = orc.num_threads()
    # size one step for ~2 s so that W + K steps stay within a few minutes
    box = float(np.float32(box_side(args, wl)))
    rate0, _, _, _ = time_oracle(p64, f64, wl, args.tensor, 1.0, box=box)
    rows = int(max(8 * cores, min(args.n, 2.0 * rate0 / args.n)))
    sample = wl.row_subset(args.n, rows, wl.SEED_BASE + 11)
    for _ in range(args.warmup):
        orc.apply_rows(p64, f64, sample, wl.A, wl.ETA, otensor, box=box)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        orc.apply_rows(p64, f64, sample, wl.A, wl.ETA, otensor, box=box)
    t = time.perf_counter() - t0
    value = args.steps * len(sample) * args.n / t
    sample_desc = f"{len(sample)} seeded rows x all {args.n} columns per step"
    line = {
        "impl": "reference", "metric": "pair interactions/s (mobility matvec)", "value": value,
        "unit": "pairs/s", "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": 1e3 * t / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(args), "reference": "CPU oracle (oracle/sd_oracle.c), "
                   "fp64 + long-double rows, OpenMP", "step": sample_desc},
        "cpu_baseline": {"value": value, "unit": "pairs/s", "cores": cores, "kind": "oracle",
                         "sample": sample_desc},
        "e2e": {"value": value, "unit": "pairs/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def run_fcc_steps(args, rank):
    """The paper's own benchmark run: fcc lattice at n = 0.1 a^-3 in its periodic
    box, uniform gravity, Euler steps of 0.001 tau_s, 100 steps per timed "step" of this script.
    Reports simulation steps/s and the pair rate; --impl reference runs the oracle instead (a
    bounded number of simulation steps).  Single GPU (rank 0 only)."""
    if rank != 0:
        return
    from paper_1205_6333_b200 import workloads as wl
    cells = args.fcc_cells
    pos = wl.fcc_lattice(cells, 0.1, jitter_seed=wl.SEED_BASE + 31 + cells)
    L = wl.fcc_box(cells, 0.1)
    n = pos.shape[0]
    sim_steps, dt = 100, 0.001
    f64mode = args.precision == "f64"
    npdt = np.float64 if f64mode else np.float32
    name = (f"sd_step N={n} fcc lattice n=0.1/a^3 (+1e-2 a seeded jitter) in its periodic box "
            f"L={L:.3f} a, nearest image, gravity, Euler dt=0.001, {sim_steps} steps per timed step, "
            f"{args.tensor.upper()}, {'fp64' if f64mode else 'fp32-Kahan'}"
            + (", lubrication correction on (Eq. 8, previous-step velocities)" if args.full_loop else ""))
    base = {"metric": "simulation steps/s at N (Euler step = one mobility product + update)",
            "unit": "steps/s", "n_gpus": 1, "steps": args.steps, "warmup": args.warmup,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "data": "synthetic",
            "paper_context": "5.7 ms per step at N = 4150 on a Tesla C2050 (PAPER.md:281), "
                             "another machine and the whole HAL step: context only"}
    if args.impl == "reference":
        from oracle import sd_oracle as orc
        otensor = orc.TENSOR_RPY if args.tensor == "rpy" else orc.TENSOR_OSEEN
        p64 = wl.to_xyzw(pos, npdt)[:, :3].astype(np.float64)
        F = wl.gravity_forces(n)
        def ostep(k):
            if args.full_loop:
                return orc.step_lub(p64, np.zeros_like(p64), F, wl.A, wl.ETA, dt, k, orc.INT_EULER, otensor, box=L)
            return orc.step(p64, F, wl.A, wl.ETA, dt, k, orc.INT_EULER, otensor, box=L)
        t0 = time.perf_counter()
        ostep(1)
        per = max(time.perf_counter() - t0, 1e-6)
        k = int(max(1, min(sim_steps, 2.0 / per)))  # ~2 s per timed step
        for _ in range(args.warmup):
            ostep(k)
        t0 = time.perf_counter()
        for _ in range(args.steps):
            ostep(k)
        t = time.perf_counter() - t0
        value = args.steps * k / t
        desc = f"{k} Euler steps of all {n} rows per timed step"
        line = dict(base, impl="reference", value=value, ms_per_step=1e3 * t / args.steps,
                    dtype="f64", config={"workload": name, "step": desc},
                    cpu_baseline={"value": value, "unit": "steps/s", "cores": orc.num_threads(),
                                  "kind": "oracle", "sample": desc},
                    e2e={"value": value, "unit": "steps/s", "h2d_bytes_per_step": 0,
                         "d2h_bytes_per_step": 0}, gpu_launches=0)
        print(json.dumps(line), flush=True)
        return

    import torch
    from paper_1205_6333_b200 import benchutil, sd
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU fallback")
    torch.cuda.set_device(0)
    sd.load_library()
    h_pos = torch.from_numpy(wl.to_xyzw(pos, npdt)).pin_memory()
    h_out = torch.empty_like(h_pos).pin_memory()
    d_pos0 = h_pos.cuda()
    d_pos = d_pos0.clone()
    ctx = sd.Context(n, wl.A, wl.ETA)
    ctx.set_precision(sd.PREC_F64 if f64mode else sd.PREC_F32_KAHAN)
    ctx.set_tensor(sd.TENSOR_RPY if args.tensor == "rpy" else sd.TENSOR_OSEEN)
    ctx.set_box(L)
    ctx.set_lubrication(args.full_loop)
    g = (0.0, 0.0, -1.0)

    def one_run():
        d_pos.copy_(d_pos0)
        ctx.reset_compensation()
        ctx.set_velocity(None)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        ctx.step(d_pos, dt, sim_steps, sd.INT_EULER, gravity=g)
        e1.record()
        return e0, e1

    for _ in range(args.warmup):
        one_run()
    torch.cuda.synchronize()
    launches0 = ctx.launch_count
    sampler = benchutil.ClockSampler(0)
    sampler.start()
    evs = [one_run() for _ in range(args.steps)]
    torch.cuda.synchronize()
    clocks = sampler.stop()
    secs = sum(a.elapsed_time(b) for a, b in evs) * 1e-3
    gpu_launches = ctx.launch_count - launches0
    # end to end: positions from pinned host memory, final positions back to the host
    t0 = time.perf_counter()
    for _ in range(args.steps):
        d_pos.copy_(h_pos, non_blocking=True)
        ctx.reset_compensation()
        ctx.step(d_pos, dt, sim_steps, sd.INT_EULER, gravity=g)
        h_out.copy_(d_pos, non_blocking=True)
        torch.cuda.synchronize()
    e2e = time.perf_counter() - t0
    rec_bytes = n * 4 * (8 if f64mode else 4)
    value = args.steps * sim_steps / secs
    line = dict(base, value=value, ms_per_step=1e3 * secs / args.steps,
                dtype="f64" if f64mode else "f32",
                config={"workload": name, "kernel": ctx.kernel_name, "parallelism": "1 GPU",
                        "l2": "whole problem is L2-resident by nature (N x 32 B); no flush: the "
                              "100 steps of one run reuse the same buffers as the paper's run does"},
                clocks=clocks, gpu_launches=gpu_launches,
                ms_per_simulation_step=1e3 * secs / (args.steps * sim_steps),
                pairs_per_s=value * n * n,
                e2e={"value": args.steps * sim_steps / e2e, "unit": "steps/s",
                     "h2d_bytes_per_step": rec_bytes, "d2h_bytes_per_step": rec_bytes})
    ctx.close()
    print(json.dumps(line), flush=True)


def run_lub(args, rank):
    """Lubrication correction (sd_lubrication_apply): an O(N) neighbour-list step, memory bound.
    value = particles/s; roofline against the measured HBM copy bandwidth with 64 B (fp32) / 128 B
    (fp64) algorithmic bytes per particle (pos, vel, F_ext in, force out, each once)."""
    if rank != 0:
        return
    from paper_1205_6333_b200 import workloads as wl
    n, phi = args.n, 0.05
    f64mode = args.precision == "f64"
    npdt = np.float64 if f64mode else np.float32
    pos = wl.uniform_cube(n, phi, wl.SEED_BASE + 300 + n)
    vel = wl.normal_forces(n, wl.SEED_BASE + 302 + n)
    fext = wl.normal_forces(n, wl.SEED_BASE + 303 + n)
    name = (f"sd_lubrication_apply N={n} uniform cube phi={phi} (overlaps allowed, ~1.35 neighbours "
            f"inside 3a per sphere), N(0,1) velocities and forces, {'fp64' if f64mode else 'fp32'}"
            + (", periodic box" if args.box else ""))
    base = {"metric": "particles/s (lubrication correction of the forces, Eq. 8)", "unit": "particles/s",
            "n_gpus": 1, "steps": args.steps, "warmup": args.warmup, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "data": "synthetic"}
    box = wl.cube_side(n, phi) if args.box else 0.0
    if args.impl == "reference":
        from oracle import sd_oracle as orc
        m = min(n, 30000)  # the oracle is O(N^2): a bounded sub-cloud of the same density
        p64 = wl.to_xyzw(wl.uniform_cube(m, phi, wl.SEED_BASE + 300 + n), npdt)[:, :3].astype(np.float64)
        v64 = vel[:m]
        for _ in range(args.warmup):
            orc.lubrication(p64, v64, wl.A, wl.ETA, box=wl.cube_side(m, phi) if args.box else 0.0)
        t0 = time.perf_counter()
        for _ in range(args.steps):
            orc.lubrication(p64, v64, wl.A, wl.ETA, box=wl.cube_side(m, phi) if args.box else 0.0)
        t = time.perf_counter() - t0
        value = args.steps * m / t
        desc = f"all-pairs oracle on a {m}-particle cloud of the same density per step"
        print(json.dumps(dict(base, impl="reference", value=value, ms_per_step=1e3 * t / args.steps,
                              dtype="f64", config={"workload": name, "step": desc},
                              cpu_baseline={"value": value, "unit": "particles/s",
                                            "cores": orc.num_threads(), "kind": "oracle", "sample": desc},
                              e2e={"value": value, "unit": "particles/s", "h2d_bytes_per_step": 0,
                                   "d2h_bytes_per_step": 0}, gpu_launches=0)), flush=True)
        return
    import torch
    from paper_1205_6333_b200 import benchutil, sd
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU fallback")
    torch.cuda.set_device(0)
    sd.load_library()
    hp, hv, hf = (torch.from_numpy(wl.to_xyzw(x, npdt)).pin_memory() for x in (pos, vel, fext))
    hout = torch.empty_like(hp).pin_memory()
    dp, dv, df = hp.cuda(), hv.cuda(), hf.cuda()
    dout = torch.empty_like(dp)
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")
    ctx = sd.Context(n, wl.A, wl.ETA)
    ctx.set_precision(sd.PREC_F64 if f64mode else sd.PREC_F32_KAHAN)
    ctx.set_box(box)
    for _ in range(args.warmup):
        ctx.lubrication_apply(dp, dv, dout, f_ext=df)
    torch.cuda.synchronize()
    launches0 = ctx.launch_count
    sampler = benchutil.ClockSampler(0)
    sampler.start()
    evs = []
    for _ in range(args.steps):
        flush.zero_()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        ctx.lubrication_apply(dp, dv, dout, f_ext=df)
        e1.record()
        evs.append((e0, e1))
    torch.cuda.synchronize()
    clocks = sampler.stop()
    secs = sum(a.elapsed_time(b) for a, b in evs) * 1e-3
    gpu_launches = ctx.launch_count - launches0
    t0 = time.perf_counter()
    for _ in range(args.steps):
        dp.copy_(hp, non_blocking=True)
        dv.copy_(hv, non_blocking=True)
        df.copy_(hf, non_blocking=True)
        ctx.lubrication_apply(dp, dv, dout, f_ext=df)
        hout.copy_(dout, non_blocking=True)
        torch.cuda.synchronize()
    e2e = time.perf_counter() - t0
    rec = n * 4 * (8 if f64mode else 4)
    peaks_path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    hbm, src = 6550.0, "fallback 6550 GB/s (B200_PROFILING.md)"
    if os.path.exists(peaks_path):
        with open(peaks_path) as f:
            hbm = float(json.load(f).get("hbm_gbs", hbm))
            src = "MEASURED_PEAKS.json hbm_gbs (burst copy)"
    achieved = 4.0 * rec * args.steps / secs / 1e9
    line = dict(base, value=args.steps * n / secs, ms_per_step=1e3 * secs / args.steps,
                dtype="f64" if f64mode else "f32",
                config={"workload": name,
                        "kernel": ("lub_small (all pairs)" if n <= 1024 else "lub_one_launch (grid in shared memory)"
                                   if n <= 4096 else "lub_count + lub_scan_totals + lub_scan_apply + lub_scatter + "
                                   "lub_gather + lub_force"),
                        "parallelism": "1 GPU", "l2": "L2 flushed with a 256 MiB write between timed iterations"},
                clocks=clocks, gpu_launches=gpu_launches,
                e2e={"value": args.steps * n / e2e, "unit": "particles/s", "h2d_bytes_per_step": 3 * rec,
                     "d2h_bytes_per_step": rec},
                roofline={"bound": "hbm", "kernel": f"whole lubrication step ({gpu_launches // max(args.steps, 1)} launches)",
                          "achieved": achieved,
                          "peak": hbm, "unit": "GB/s", "frac": achieved / hbm, "traffic": None,
                          "peak_source": src, "bytes_per_particle": 4 * rec // n})
    if not args.no_cpu_baseline:
        from oracle import sd_oracle as orc
        m = min(n, 30000)
        p64 = wl.to_xyzw(wl.uniform_cube(m, phi, wl.SEED_BASE + 300 + n), npdt)[:, :3].astype(np.float64)
        t0 = time.perf_counter()
        orc.lubrication(p64, vel[:m], wl.A, wl.ETA)
        t = time.perf_counter() - t0
        line["cpu_baseline"] = {"value": m / t, "unit": "particles/s", "cores": orc.num_threads(),
                                "kind": "oracle", "sample": f"all-pairs oracle on a {m}-particle cloud of "
                                                            f"the same density, {t:.1f} s"}
    ctx.close()
    print(json.dumps(line), flush=True)


def fma_peaks(sm_count):
    """Derived FMA peaks (TFLOP/s) at sm_max_mhz of MEASURED_PEAKS.json."""
    sm_max_mhz = 1965.0
    peaks_path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(peaks_path):
        with open(peaks_path) as f:
            sm_max_mhz = float(json.load(f).get("sm_max_mhz", sm_max_mhz))
    return {"f32": sm_count * FP32_LANES_PER_SM * 2 * sm_max_mhz * 1e6 / 1e12,
            "f64": sm_count * FP64_LANES_PER_SM * 2 * sm_max_mhz * 1e6 / 1e12}, sm_max_mhz


def graph_of(torch, fn, count):
    """`count` calls of fn captured into one CUDA graph (below N ~ 10^4 a product is shorter than the
    13 us a Python / ctypes call costs on the host: a loop of calls measures the interpreter).
    Returns a callable that replays the graph on the current stream."""
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        fn()
    torch.cuda.current_stream().wait_stream(side)
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=side):
        for _ in range(count):
            fn()
    return g.replay


def _sample_times(torch, fn, warm, samples, per_sample):
    """`samples` timings of `per_sample` back-to-back calls of fn between one pair of CUDA events on
    the current (launching) stream, after `warm` untimed calls; seconds per call.  per_sample > 1:
    the calls are replayed from one CUDA graph (graph_of)."""
    for _ in range(warm):
        fn()
    torch.cuda.synchronize()
    run = graph_of(torch, fn, per_sample) if per_sample > 1 else fn
    out = []
    for _ in range(samples):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        run()
        e1.record()
        torch.cuda.synchronize()
        out.append(e0.elapsed_time(e1) * 1e-3 / per_sample)
    return np.array(out)


def extra_measurements(torch, sd, wl, sm_count, probes):
    """The rest of BASELINE.json's metric, measured in this process:
    configuration 5 (sd_mobility_apply at six sizes x {fp32-Kahan, fp64} x {RPY, Oseen}; best and
    median of 10 samples after 3 warm-ups, warm L2 -- the inputs are at most 67 MB) and sd_step
    steps/s on configurations 1, 3 and 4.  Small products are launch-bound when timed one by one
    (an event pair, and the Python call itself, cost more than the kernel), so a sample is
    `launches_per_sample` back-to-back launches replayed from one CUDA graph, as sd_step issues its
    step loops."""
    peaks, _ = fma_peaks(sm_count)
    sweep = []
    for n in CFG5_NS:
        pos, force = wl.sweep(n)
        per = int(max(1, min(50, 4e9 // (n * n))))
        for pname, prec, npdt in (("f32", sd.PREC_F32_KAHAN, np.float32), ("f64", sd.PREC_F64, np.float64)):
            dp = torch.from_numpy(wl.to_xyzw(pos, npdt)).cuda()
            df = torch.from_numpy(wl.to_xyzw(force, npdt)).cuda()
            dv = torch.empty_like(dp)
            for tname, tensor in (("rpy", sd.TENSOR_RPY), ("oseen", sd.TENSOR_OSEEN)):
                ctx = sd.Context(n, wl.A, wl.ETA)
                ctx.set_tensor(tensor)
                ctx.set_precision(prec)
                t = _sample_times(torch, lambda: ctx.mobility_apply(dp, df, dv), 3, 10, per)
                best, med = n * n / t.min(), n * n / float(np.median(t))
                fl = FLOPS_PER_PAIR[tname] / 1e12
                sweep.append({"n": n, "precision": pname, "tensor": tname, "kernel": ctx.kernel_name,
                              "launches_per_sample": per, "us_per_product_median": 1e6 * float(np.median(t)),
                              "pairs_per_s_best": best, "pairs_per_s_median": med,
                              "frac_of_derived_peak_best": best * fl / peaks[pname],
                              "frac_of_derived_peak_median": med * fl / peaks[pname],
                              "frac_of_probe_median": med * fl / probes[pname]})
                ctx.close()
            del dp, df, dv
    steps = []
    p1, _ = wl.four_sphere(wl.SEED_BASE + 1)
    p3, _ = wl.config3()
    p4, _ = wl.config4()
    for cfg, pos, integ, iname, dt, nsteps in ((1, p1, sd.INT_MIDPOINT, "midpoint", 0.01, 10000),
                                               (3, p3, sd.INT_EULER, "euler", 0.01, 20),
                                               (4, p4, sd.INT_MIDPOINT, "midpoint", 0.05, 10)):
        n = pos.shape[0]
        for pname, prec, npdt in (("f32", sd.PREC_F32_KAHAN, np.float32), ("f64", sd.PREC_F64, np.float64)):
            if cfg == 4 and pname == "f64":
                continue   # BASELINE.json configs[3] is fp32-Kahan only
            ctx = sd.Context(n, wl.A, wl.ETA)
            ctx.set_precision(prec)
            dq = torch.from_numpy(wl.to_xyzw(pos, npdt)).cuda()
            t = _sample_times(torch, lambda: ctx.step(dq, dt, nsteps, integ, gravity=(0.0, 0.0, -1.0)),
                              1, 5, 1)
            steps.append({"config": cfg, "n": n, "integrator": iname, "precision": pname,
                          "steps_per_call": nsteps, "steps_per_s_median": nsteps / float(np.median(t)),
                          "pairs_per_s_median": (2 if iname == "midpoint" else 1) * n * n * nsteps
                          / float(np.median(t))})
            ctx.close()
    # ---- periodic box at the headline size, the paper's own benchmark shape, lubrication
    n = 1048576
    pos, force = wl.sweep(n)
    dp = torch.from_numpy(wl.to_xyzw(pos, np.float32)).cuda()
    df = torch.from_numpy(wl.to_xyzw(force, np.float32)).cuda()
    dv = torch.empty_like(dp)
    ctx = sd.Context(n, wl.A, wl.ETA)
    ctx.set_box(wl.cube_side(n, 0.01))
    t = _sample_times(torch, lambda: ctx.mobility_apply(dp, df, dv), 1, 3, 1)
    flb = (FLOPS_PER_PAIR["rpy"] + FLOPS_NEAREST_IMAGE) / 1e12
    box = {"workload": "sd_mobility_apply N=1048576 uniform cube phi=0.01 in its periodic box (nearest image), RPY, "
                       "fp32-Kahan", "kernel": ctx.kernel_name, "pairs_per_s_median": n * n / float(np.median(t)),
           "flops_per_pair": FLOPS_PER_PAIR["rpy"] + FLOPS_NEAREST_IMAGE,
           "frac_of_derived_peak_median": n * n / float(np.median(t)) * flb / peaks["f32"]}
    ctx.close()
    del dp, df, dv
    fcc = []
    cells = 10
    lat = wl.fcc_lattice(cells, 0.1, jitter_seed=wl.SEED_BASE + 31 + cells)
    d0 = torch.from_numpy(wl.to_xyzw(lat, np.float32)).cuda()
    for full in (False, True):
        ctx = sd.Context(lat.shape[0], wl.A, wl.ETA)
        ctx.set_box(wl.fcc_box(cells, 0.1))
        ctx.set_lubrication(full)
        dq = d0.clone()

        def run():
            dq.copy_(d0)
            ctx.reset_compensation()
            ctx.set_velocity(None)
            ctx.step(dq, 0.001, 100, sd.INT_EULER, gravity=(0.0, 0.0, -1.0))
        t = _sample_times(torch, run, 2, 5, 1)
        fcc.append({"workload": f"sd_step N={lat.shape[0]} fcc lattice n=0.1/a^3 in its periodic box, gravity, Euler "
                                "dt=0.001, 100 steps per call" + (", lubrication correction on" if full else ""),
                    "kernel": ctx.kernel_name, "steps_per_s_median": 100 / float(np.median(t)),
                    "us_per_step_median": 1e4 * float(np.median(t))})
        ctx.close()
    return {"what": "BASELINE.json metric beyond the headline point, same process, CUDA events on the "
                    "launching stream; fractions = pairs/s x (34 RPY | 29 Oseen) flops / FMA peak",
            "fma_probe_tflops": probes, "derived_peak_tflops": peaks,
            "config5_sweep": sweep, "sd_step": steps, "periodic_box": box, "paper_benchmark_shape": fcc,
            "issue_model": issue_model()}


def issue_model():
    """Static issue-cycle model of the hot loops of the library this process runs (paper_1205_6333_b200/
    sassmodel.py: register-bank rule + operand-reuse cache over the SASS; host-side text processing of
    `cuobjdump -sass`): says where the distance to the FMA roofline goes.  null when cuobjdump is missing."""
    try:
        from paper_1205_6333_b200 import sassmodel as sm
        funcs = sm.disassemble()
        out = []
        for label, frag, flops, fp64 in sm.KERNELS:
            names = [n for n in funcs if frag in n]
            if not names:
                continue
            r = sm.analyse(funcs[names[0]], flops, fp64)
            out.append({"kernel": " ".join(label.split()), "instructions_per_iteration": r["instructions"],
                        "fma_class_instructions": r["wide"], "register_bank_conflicts": r["conflicts"],
                        "model_cycles": r["cycles"], "fma_class_cycles": r["ideal_cycles"],
                        "frac_model": r["frac_model"], "frac_without_conflicts": r["frac_no_conflicts"],
                        "frac_fma_class_alone": r["frac_wide_only"]})
        return {"what": "python -m paper_1205_6333_b200.sassmodel (profiles/r02_issue_model.md)", "kernels": out}
    except Exception as e:  # diagnostics only: never fail the bench line
        return {"unavailable": str(e)}


def main():
    args = parse_args()
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.fcc_cells > 0:
        run_fcc_steps(args, rank)
        return
    if args.lub:
        run_lub(args, rank)
        return
    if args.impl == "reference":
        run_reference(args, rank)
        return

    import torch
    import torch.distributed as dist
    from paper_1205_6333_b200 import benchutil, sd

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    sd.load_library()

    n = args.n
    pos, force, wl = workload(n)
    f64mode = args.precision == "f64"
    npdt = np.float64 if f64mode else np.float32
    prec = sd.PREC_F64 if f64mode else sd.PREC_F32_KAHAN
    tensor = sd.TENSOR_RPY if args.tensor == "rpy" else sd.TENSOR_OSEEN
    h_pos = torch.from_numpy(wl.to_xyzw(pos, npdt)).pin_memory()
    h_force = torch.from_numpy(wl.to_xyzw(force, npdt)).pin_memory()
    h_vel = torch.empty_like(h_pos).pin_memory()
    d_pos, d_force = h_pos.to(dev), h_force.to(dev)
    d_vel = torch.empty_like(d_pos)
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=dev)  # > 126 MB L2

    ctx = sd.Context(n, wl.A, wl.ETA)
    ctx.set_precision(prec)
    ctx.set_tensor(tensor)
    ctx.set_box(box_side(args, wl))
    ctx.set_staging({"bulk": 0, "naive": 1, "sync": 2}[args.staging])
    ctx.set_jsplit({"auto": 0, "classic": 1, "warp": 2}[args.jsplit])
    lps = max(1, args.launches_per_step)
    peak_probe = ctx.fma_peak_probe(prec)
    probe64 = peak_probe if f64mode else ctx.fma_peak_probe(sd.PREC_F64)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing ------------------------------------------------------------
    for _ in range(args.warmup):
        ctx.mobility_apply(d_pos, d_force, d_vel)
    barrier()
    # several products per timed step: replayed from one CUDA graph (no per-kernel events then: the
    # roofline below is computed from the whole step)
    c0 = ctx.launch_count
    step_fn = graph_of(torch, lambda: ctx.mobility_apply(d_pos, d_force, d_vel), lps) if lps > 1 else None
    launches_per_product = (ctx.launch_count - c0) // (lps + 1)  # graph_of: one warm call + lps captured ones
    ctx.profile_enable(lps == 1)
    ctx.profile_read()
    launches0 = ctx.launch_count
    sampler = benchutil.ClockSampler(local_rank)
    sampler.start()
    evs = []
    barrier()
    for _ in range(args.steps):
        flush.zero_()  # L2 flush between timed iterations (outside the event pair)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        if step_fn is not None:
            step_fn()
        else:
            ctx.mobility_apply(d_pos, d_force, d_vel)
        e1.record()
        evs.append((e0, e1))
    barrier()
    clocks = sampler.stop()
    local_s = sum(a.elapsed_time(b) for a, b in evs) * 1e-3
    gpu_launches = ctx.launch_count - launches0
    pair_ms, pair_launches = ctx.profile_read()
    if step_fn is not None:  # no per-kernel events inside a graph: whole products stand in
        gpu_launches = launches_per_product * lps * args.steps
        pair_ms, pair_launches = local_s * 1e3, args.steps * lps
    ctx.profile_enable(False)
    units, t_max = benchutil.aggregate_over_ranks(local_s, float(args.steps) * lps * n * n)
    value = units / t_max

    # ---- end to end through the host-buffer entry point ------------------------------------
    ctx.mobility_apply_host(h_pos, h_force, h_vel)
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        ctx.mobility_apply_host(h_pos, h_force, h_vel)  # returns after vel landed on the host
    torch.cuda.synchronize()
    e2e_local = time.perf_counter() - t0
    barrier()
    e2e_units, e2e_t = benchutil.aggregate_over_ranks(e2e_local, float(args.steps) * n * n)
    rec_bytes = n * 4 * (8 if f64mode else 4)

    # ---- roofline of the dominant kernel (compute bound on the CUDA-core FMA pipes) --------
    sm_count = torch.cuda.get_device_properties(dev).multi_processor_count
    peaks, sm_max_mhz = fma_peaks(sm_count)
    pkey = "f64" if f64mode else "f32"
    lanes = FP64_LANES_PER_SM if f64mode else FP32_LANES_PER_SM
    peak_tflops = peaks[pkey]
    flops = FLOPS_PER_PAIR[args.tensor] + (FLOPS_NEAREST_IMAGE if args.box else 0)
    achieved = flops * float(n) * n * pair_launches / (pair_ms * 1e-3) / 1e12 if pair_ms > 0 else None
    traffic, traffic_src = NCU_TRAFFIC.get((n, args.precision, args.tensor, args.box), (None, None))
    if args.staging != "bulk":
        traffic, traffic_src = None, None
    roofline = {
        "bound": "alu", "kernel": ctx.kernel_name, "achieved": achieved, "peak": peak_tflops,
        "unit": "TFLOP/s", "frac": (achieved / peak_tflops) if achieved else None,
        "frac_is": "of the DERIVED peak (no CUDA-core FMA figure in MEASURED_PEAKS.json)",
        "frac_of_probe": (achieved / peak_probe) if achieved and peak_probe else None,
        "traffic": traffic, "traffic_source": traffic_src,
        "peak_source": f"derived: {sm_count} SMs x {lanes} FMA lanes x 2 flop x {sm_max_mhz:.0f} MHz "
                       "(sm_max_mhz of MEASURED_PEAKS.json; DESIGN.md)",
        "fma_probe_tflops": peak_probe,
        "fma_probe_is": "dependent-FMA-chain kernel of this library (sd_fma_peak_probe) timed in this run",
        "flops_per_pair": flops, "kernel_ms": pair_ms / max(pair_launches, 1),
        "kernel_share_of_step": pair_ms * 1e-3 / local_s if local_s > 0 else None,
    }
    if clocks.get("sm_mhz") and abs(clocks["sm_mhz"] - sm_max_mhz) > 1.0 and achieved:
        roofline["frac_at_measured_clock"] = achieved / (peak_tflops * clocks["sm_mhz"] / sm_max_mhz)

    in_mb = 2 * n * 4 * (8 if f64mode else 4) / 1e6
    line = {
        "metric": "pair interactions/s (mobility matvec)", "value": value, "unit": "pairs/s",
        "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": 1e3 * t_max / (args.steps * lps), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64" if f64mode else "f32", "data": "synthetic",
        "config": {"workload": workload_name(args), "kernel": ctx.kernel_name,
                   "jsplit": args.jsplit, "launches_per_step": lps,
                   "parallelism": "replicas only (no sharding, no collective)" if world > 1 else "1 GPU",
                   "l2": f"inputs ({in_mb:.1f} MB) fit in L2; L2 flushed with a 256 MiB write between timed iterations"},
        "clocks": clocks, "gpu_launches": gpu_launches,
        "e2e": {"value": e2e_units / e2e_t, "unit": "pairs/s", "h2d_bytes_per_step": 2 * rec_bytes,
                "d2h_bytes_per_step": rec_bytes},
        "roofline": roofline,
    }

    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        p64 = h_pos.numpy()[:, :3].astype(np.float64)
        f64 = h_force.numpy()[:, :3].astype(np.float64)
        rate, cores, rows, secs = time_oracle(p64, f64, wl, args.tensor, 15.0,
                                              box=float(np.float32(box_side(args, wl))))
        from oracle import sd_oracle as _orc
        _orc.set_num_threads(1)   # also the one-thread figure, on a 3 s sample
        rate1, _, rows1, secs1 = time_oracle(p64, f64, wl, args.tensor, 3.0,
                                             box=float(np.float32(box_side(args, wl))))
        _orc.set_num_threads(cores)
        line["cpu_baseline"] = {"value": rate, "unit": "pairs/s", "cores": cores, "kind": "oracle",
                                "sample": f"{rows} seeded rows x all {n} columns of the same "
                                          f"workload, {secs:.1f} s",
                                "cpu_model": cpu_model(), "one_thread_value": rate1,
                                "one_thread_sample": f"{rows1} rows, {secs1:.1f} s"}
    ctx.close()
    default_point = (n == 1048576 and not f64mode and args.tensor == "rpy" and not args.box
                     and args.staging == "bulk")
    if rank == 0 and world == 1 and default_point and not args.no_extra:
        del d_pos, d_force, d_vel
        probes = {"f32": peak_probe, "f64": probe64}
        line["extra"] = extra_measurements(torch, sd, wl, sm_count, probes)
    if rank == 0:
        print(json.dumps({"extra": line["extra"]} if args.extra_only and "extra" in line else line),
              flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
