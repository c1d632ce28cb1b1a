"""Issue-cycle model of the hot loops of the shipped pair kernels, read off the SASS of the built library.

    python -m paper_1205_6333_b200.sassmodel            (needs cuobjdump from the CUDA toolkit; no GPU)

For every all-pairs kernel that a large-N product runs (fp32 Rotne-Prager / Oseen / periodic box, fp64) it
finds the innermost loop with the most packed-FP32 (resp. FP64) instructions, prints its instruction mix and
applies a three-line cycle model per warp on its scheduler:

  * an FFMA2 / FMUL2 / FADD2 (two FMAs per lane on a 32-lane pipe) or a DFMA / DMUL / DADD (16 lanes)
    occupies the issue port for max(2, e, o) cycles, where e / o are the numbers of DISTINCT source
    registers it reads from the even / the odd register bank -- a 64-bit operand is one register of each,
    the broadcast scalar of the packed forms one register -- not counting an operand that the previous
    instruction left in the operand-reuse cache of the same slot (`.reuse`);
  * a MUFU counts half a cycle, every other instruction one cycle;
  * the two warps of a scheduler hide each other's latencies (ncu: `wait` + `math_pipe_throttle`, no long
    scoreboard stalls), so the loop takes the sum.

The bank rule is the one /opt/skills/guides/B300_MICROARCH.md states for Blackwell ("rt = max(rt_pipe,
#even_distinct, #odd_distinct)"); the half cycle of a MUFU is fitted to the fp32 kernel.  With
it the model reproduces the ncu cycle counts of profiles/r02_pairs_ncu_full.md to 3 % (fp32 822 against
821 cycles per 4-j iteration, fp64 981 against 998, periodic box 1168 against 1139), which makes it usable
for the one question it is here to answer: WHERE the distance between the kernels and their FMA roofline
goes.  Answer: an instruction with three distinct register operands always has three of them in one bank
(two pairs + a scalar, or three pairs) and costs a third cycle unless the reuse cache serves one; 9 of the
20 packed instructions of a step are of that kind and ptxas finds a reuse partner for a third of them.
profiles/r02_issue_model.md holds the output and the experiments (source order, ptxas flags, immediates,
unroll factors, -O1) that tried to move that share.

Host-side text processing only: nothing here touches the GPU or the method's arithmetic.
"""
from __future__ import annotations

import os
import re
import subprocess
import sys

LIB = os.path.join(os.path.dirname(os.path.abspath(__file__)), "libsd_b200.so")

WIDE = ("FFMA2", "FMUL2", "FADD2", "DFMA", "DMUL", "DADD")
XU = ("MUFU",)

# kernels of a large-N product: (label, mangled-name fragment, flops per pair, fp64?)
KERNELS = [
    ("fp32 Rotne-Prager  pairs_f32_kernel<4,RPY,Kahan,REPAIR=0>", "pairs_f32_kernelILi4ELi0ELi0ELb0ELi0ELi256ELi0E", 34, False),
    ("fp32 Oseen         pairs_f32_kernel<4,Oseen,Kahan,REPAIR=0>", "pairs_f32_kernelILi4ELi1ELi0ELb0ELi0ELi256ELi0E", 29, False),
    ("fp32 periodic box  pairs_f32_kernel<4,RPY,Kahan,PBC,REPAIR=0>", "pairs_f32_kernelILi4ELi0ELi0ELb1ELi0ELi256ELi0E", 49, False),
    ("fp64 Rotne-Prager  pairs_f64_kernel<4,RPY>", "pairs_f64_kernelILi4ELi0ELb0ELi128E", 34, True),
    ("fp64 Oseen         pairs_f64_kernel<4,Oseen>", "pairs_f64_kernelILi4ELi1ELb0ELi128E", 29, True),
]

_INSTR = re.compile(r"\s*/\*([0-9a-f]+)\*/\s+(@!?U?P\d\s+)?(\S+)\s*(.*?);")


def disassemble(lib: str = LIB) -> dict[str, list[tuple[int, str, str]]]:
    """{mangled function name: [(address, opcode, operand text), ...]} from `cuobjdump -sass`."""
    out = subprocess.run(["cuobjdump", "-sass", lib], capture_output=True, text=True, check=True).stdout
    funcs: dict[str, list[tuple[int, str, str]]] = {}
    cur = None
    for line in out.split("\n"):
        if "Function :" in line:
            cur = funcs.setdefault(line.split("Function :")[1].strip(), [])
            continue
        m = _INSTR.match(line)
        if m and cur is not None:
            cur.append((int(m.group(1), 16), m.group(3), m.group(4)))
    return funcs


def innermost_loops(code):
    """(first, last) instruction indices of the loops that hold no other backward branch."""
    index = {a: i for i, (a, _, _) in enumerate(code)}
    loops = []
    for i, (a, op, args) in enumerate(code):
        if not op.startswith("BRA"):
            continue
        m = re.search(r"0x([0-9a-f]+)\s*$", args)
        if m and int(m.group(1), 16) <= a and int(m.group(1), 16) in index:
            loops.append((index[int(m.group(1), 16)], i))
    return [(j, i) for (j, i) in loops if not any(j <= j2 and i2 < i for (j2, i2) in loops if (j2, i2) != (j, i))]


def hot_loop(code):
    """The innermost loop with the most packed-FP32 / FP64 instructions."""
    best = max(innermost_loops(code), key=lambda ji: sum(code[q][1].split(".")[0] in WIDE for q in range(ji[0], ji[1] + 1)))
    return code[best[0]:best[1] + 1]


def cycle_model(body):
    """Issue cycles of one loop iteration per the module docstring; returns a dict of totals."""
    total = 0.0
    mix: dict[str, int] = {}
    conflicts = 0
    three_op = 0
    reuse = {}
    for _, op, args in body:
        base = op.split(".")[0]
        mix[base] = mix.get(base, 0) + 1
        wide = base in WIDE
        srcs = [s.strip() for s in args.split(",")][1:]
        even, odd, keep, regs_named = set(), set(), {}, set()
        for slot, s in enumerate(srcs):
            m = re.match(r"-?\|?R(\d+)", s)
            if not m:
                continue
            r = int(m.group(1))
            pair = wide and (base[0] == "D" or "F32x2" in s)
            regs_named.add((r, pair))
            if reuse.get(slot) != r:
                for q in ((r, r + 1) if pair else (r,)):
                    (odd if q & 1 else even).add(q)
            if "reuse" in s:
                keep[slot] = r
        reuse = keep
        if wide:
            rt = max(2, len(even), len(odd))
            three_op += len(regs_named) >= 3
            conflicts += rt > 2
        elif base in XU:
            rt = 0.5
        else:
            rt = max(1, len(even), len(odd))
        total += rt
    n_wide = sum(v for k, v in mix.items() if k in WIDE)
    return {"cycles": total, "mix": mix, "wide": n_wide, "three_operand": three_op, "conflicts": conflicts}


def analyse(code, flops_per_pair: int, fp64: bool):
    body = hot_loop(code)
    r = cycle_model(body)
    rsq = sum(1 for _, op, _ in body if op.startswith("MUFU.RSQ"))
    r["instructions"] = len(body)
    r["pairs_per_lane"] = rsq  # one reciprocal square root per pair
    lane_flops_per_cycle = 32 if fp64 else 64  # per scheduler: 16 DFMA or 32 x 2 packed FMA lanes, 2 flop each
    r["ideal_cycles"] = 2 * r["wide"]
    r["frac_model"] = flops_per_pair * rsq * 32 / (r["cycles"] * lane_flops_per_cycle)
    r["frac_no_conflicts"] = flops_per_pair * rsq * 32 / ((r["cycles"] - r["conflicts"]) * lane_flops_per_cycle)
    r["frac_wide_only"] = flops_per_pair * rsq * 32 / (r["ideal_cycles"] * lane_flops_per_cycle)
    return r


def main(argv):
    lib = argv[0] if argv else LIB
    funcs = disassemble(lib)
    print("| kernel | instructions per iteration | pairs per lane | packed / fp64 instructions (three distinct register operands) "
          "| bank conflicts | model cycles (FMA-class alone) | roofline fraction: model | without conflicts | FMA-class alone |")
    print("|---|---|---|---|---|---|---|---|---|")
    for label, frag, flops, fp64 in KERNELS:
        names = [n for n in funcs if frag in n]
        if not names:
            print(f"| {label} | not in the library | | | | | | | |")
            continue
        r = analyse(funcs[names[0]], flops, fp64)
        print(f"| {label} | {r['instructions']} | {r['pairs_per_lane']} | {r['wide']} ({r['three_operand']}) | {r['conflicts']} "
              f"| {r['cycles']:.0f} ({r['ideal_cycles']}) | {r['frac_model']:.3f} | {r['frac_no_conflicts']:.3f} | {r['frac_wide_only']:.3f} |")
        mix = ", ".join(f"{v} {k}" for k, v in sorted(r["mix"].items(), key=lambda kv: -kv[1]))
        print(f"|  | {mix} | | | | | | | |")


if __name__ == "__main__":
    main(sys.argv[1:])
