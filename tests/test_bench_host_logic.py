"""Host-side bench logic on CPU: multi-rank aggregation over gloo (world_size 2), clock-sample
parsing, and the reference arm's JSON line on a tiny workload."""
import json
import os
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1205_6333_b200 import benchutil

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    units, secs = benchutil.aggregate_over_ranks(1.0 + rank, 100.0 * (rank + 1))
    out[rank] = (units, secs)
    dist.barrier()
    dist.destroy_process_group()


def test_aggregate_over_two_ranks_gloo():
    """value = units of all ranks / max-over-ranks time (replicas only: no data-path collective)."""
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(2, 29531, out), nprocs=2, join=True)
    assert out[0] == out[1] == (300.0, 2.0)


def test_aggregate_single_process_is_identity():
    assert benchutil.aggregate_over_ranks(0.5, 7.0) == (7.0, 0.5)


def test_clock_sample_parsing():
    text = ("1965, 1965, 400.1, Not Active, Not Active, Not Active, Not Active\n"
            "1905, 1965, 950.0, Not Active, Not Active, Not Active, Active\n"
            "1920, 1965, 900.0, Not Active, Not Active, Not Active, Not Active\n")
    c = benchutil.parse_clock_samples(text)
    assert c["sm_mhz"] == 1920 and c["sm_max_mhz"] == 1965
    assert c["reasons"] == ["sw_power_cap"] and c["samples"] == 3
    assert benchutil.parse_clock_samples("")["samples"] == 0


def test_reference_arm_prints_contract_line():
    env = dict(os.environ, OMP_NUM_THREADS="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference",
                        "--n", "3000", "--steps", "2", "--warmup", "1"],
                       capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0, r.stderr
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "pairs/s" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["d2h_bytes_per_step"] == 0
    assert line["steps"] == 2 and line["warmup"] == 1


def test_stability_postprocessing_recovers_period_and_amplitude():
    """paper_1205_6333_b200/stability.py, host side: parabolic fits to the extrema of a sampled
    x_1(t) give cycle duration and amplitude of a known signal."""
    import numpy as np
    from paper_1205_6333_b200 import stability
    dt, stride, T, A = 0.01, 100, 517.04, 4.2617
    t = (np.arange(60000) + 1) * dt * stride
    traj = np.zeros((t.size, 4, 4))
    traj[:, 0, 0] = 6.57 + A * np.cos(2 * np.pi * t / T)
    traj[:, 0, 1] = 1e-7 * np.sin(t)
    rows, ncyc = stability.analyse(traj, dt, stride, window=1.0e4)
    assert ncyc == int(t[-1] // T)
    for lo, hi, n, dur, sd_, amp, ymax in rows[:-1]:
        assert n >= 18 and abs(dur - T) < 1e-3 and abs(amp - A) < 1e-4 and ymax <= 1e-7
