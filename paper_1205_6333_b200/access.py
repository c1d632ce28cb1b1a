"""Appendix A of the paper on this GPU: kernel time per pair for the O(N^2) access kernels.

    python -m paper_1205_6333_b200.access [N ...]          (default N = 16384 65536)

Prints, for float and float4 arrays, the three access patterns (linear, strided p = 131,
unordered) and the staging schemes (naive, small-tiling, tiling, bulk-copy ring), the kernel time
divided by N^2 in picoseconds (Fig. 7 plots the same quantity) and the ratio to the
naive kernel.  Timing and argument marshalling only; the kernels live in csrc/sd_access.cuh.
"""
from __future__ import annotations

import sys

import numpy as np

PATTERNS = ["linear", "strided", "unordered"]
SCHEMES = ["naive", "small-tiling", "tiling", "bulk"]


def main(argv):
    import torch
    from . import sd
    sd.load_library()
    torch.cuda.set_device(0)
    sizes = [int(a) for a in argv] or [16384, 65536]
    rng = np.random.Generator(np.random.PCG64(20120533))
    for n in sizes:
        print(f"\nN = {n}: kernel time / N^2 in ps (ratio to naive)\n")
        print("| element | pattern | " + " | ".join(SCHEMES) + " |")
        print("|---|---|" + "---|" * len(SCHEMES))
        for elem in (1, 4):
            shape = (n,) if elem == 1 else (n, 4)
            d = torch.from_numpy(rng.integers(0, 4, size=shape).astype(np.float32)).cuda()
            out = torch.empty((n,), device="cuda")
            for p, pname in enumerate(PATTERNS):
                cells, base = [], None
                for s, _ in enumerate(SCHEMES):
                    if s == 3 and p != 0:
                        cells.append("-")
                        continue
                    ms = sd.access_bench(d, out, p, s, reps=max(3, min(50, int(3e10 / n / n))))
                    ps = ms * 1e9 / n / n
                    base = ps if s == 0 else base
                    cells.append(f"{ps:.3f} ({ps / base:.2f})")
                print(f"| {'float' if elem == 1 else 'float4'} | {pname} | " + " | ".join(cells) + " |", flush=True)


if __name__ == "__main__":
    main(sys.argv[1:])
