"""FP32-pipe instructions per interaction of the force kernel, counted in its SASS.

    python -m paper_2110_11658_b200.sasscount [--kernel _Z7k_forceILb0ELb0EEv10force_args]

Disassembles libp3t.so (cuobjdump -sass), finds the innermost loops of the kernel that hold MUFU.RSQ (one per
interaction: the particle-cell loop and the far pass of the particle-particle loop) and counts, per MUFU.RSQ,
the FP32-pipe lane-operations FADD / FMUL / FFMA (1 each) and FADD2 / FMUL2 / FFMA2 (2 each: two lanes of work).
These are the "SASS counts" of SURVEY.md 8(d) behind bench.py's `roofline.frac_sass_counts`.  (ncu's
smsp__sass_thread_inst_executed_op_f*_pred_on metrics do not count the packed f32x2 instructions, so the count is
static; the loops are straight-line code, so static = executed.)"""
from __future__ import annotations

import re
import subprocess
import sys
from collections import Counter
from pathlib import Path

LIB = Path(__file__).resolve().parent / "libp3t.so"
FP32 = {"FADD": 1, "FMUL": 1, "FFMA": 1, "FADD2": 2, "FMUL2": 2, "FFMA2": 2}


def loops_with_rsqrt(kernel: str):
    out = subprocess.run(["cuobjdump", "-sass", "-fun", kernel, str(LIB)], capture_output=True, text=True).stdout
    ins = []
    for line in out.splitlines():
        m = re.match(r"\s+/\*([0-9a-f]{4,})\*/\s+(.*?);", line)
        if m:
            ins.append((int(m.group(1), 16), m.group(2)))
    at = {a: i for i, (a, _) in enumerate(ins)}
    loops = []
    for i, (a, t) in enumerate(ins):
        m = re.search(r"\bBRA\b.*?(0x[0-9a-f]+)", t)
        if m and int(m.group(1), 16) < a and int(m.group(1), 16) in at:
            loops.append((at[int(m.group(1), 16)], i))
    res = []
    for lo, hi in loops:
        if any(lo2 >= lo and hi2 <= hi and (lo2, hi2) != (lo, hi) for lo2, hi2 in loops):
            continue                                             # not innermost
        c = Counter()
        for _, t in ins[lo:hi + 1]:
            t = re.sub(r"^@!?U?P\d+\s+", "", t)
            c[t.split()[0].split(".")[0]] += 1
        if c["MUFU"]:
            res.append(dict(begin=hex(ins[lo][0]), end=hex(ins[hi][0]), instructions=hi - lo + 1, rsqrt=c["MUFU"],
                            fp32_lane_ops=sum(FP32[k] * c[k] for k in FP32), mix=dict(c)))
    return res


def main():
    kernel = sys.argv[sys.argv.index("--kernel") + 1] if "--kernel" in sys.argv else "_Z7k_forceILb0ELb0EEv10force_args"
    for r in loops_with_rsqrt(kernel):
        print(f"loop {r['begin']}..{r['end']}: {r['instructions']} instructions, {r['rsqrt']} MUFU.RSQ, "
              f"{r['fp32_lane_ops']} FP32 lane-ops = {r['fp32_lane_ops'] / r['rsqrt']:.2f} per interaction; "
              f"issue slots per interaction {r['instructions'] / r['rsqrt']:.2f}; mix {r['mix']}")


if __name__ == "__main__":
    main()
