"""SASS evidence for libls.so: an opcode histogram of EVERY kernel and the full listing of one kernel per family.

    python -m paper_1612_04040_b200.sass_listing --out profiles/r2_sass

Writes  <out>_histogram.txt   per __global__ function (all template instances, fp64 included): registers are in the
                              ptxas log, here: instruction count and the counts of the opcodes that prove the
                              Blackwell-native paths (UTMALDG / UBLKCP = TMA, LDGSTS = cp.async, SYNCS = mbarrier,
                              FFMA2 / FMUL2 / FADD2 = packed fp32, MUFU, REDUX, ATOMS / ATOMG / RED)
        <out>_kernels.txt     `cuobjdump -sass` of one instance per kernel family, encodings stripped
Runs on the CPU box (cuobjdump is in the CUDA image).
"""
from __future__ import annotations

import argparse
import re
import shutil
import subprocess
from collections import Counter
from pathlib import Path

from . import build as ls_build

WATCH = ["UTMALDG", "UBLKCP", "LDGSTS", "SYNCS", "FFMA2", "FMUL2", "FADD2", "FFMA", "MUFU", "DFMA", "DMUL", "DADD",
         "REDUX", "ATOMS", "ATOMG", "RED", "LDS", "STS", "LDG", "STG", "BAR", "SHFL", "VOTE", "NANOSLEEP"]
# one instance per family gets its full listing: (label, regex on the mangled name)
FAMILIES = [
    ("reinit sweep fp32 (k_band_tile<float, ADV=0, K=1, plain>)", r"k_band_tileIfLb0ELi1ELb0ELb0ELb0E"),
    ("last reinit sweep fp32, clamp + T emission (k_band_tile<float, 0, 1, CLAMP, 0, EMIT_T>)", r"k_band_tileIfLb0ELi1ELb1ELb0ELb1E"),
    ("Advance fp32 (k_band_tile<float, ADV=1, K=1>)", r"k_band_tileIfLb1ELi1E"),
    ("two fused reinit sweeps fp32 (k_band_tile<float, 0, K=2, plain>)", r"k_band_tileIfLb0ELi2ELb0ELb0ELb0E"),
    ("reinit sweep fp64 (k_band_tile<double, 0, 1, plain>)", r"k_band_tileIdLb0ELi1ELb0ELb0ELb0E"),
    ("reinit sweep fp64 with residual (k_band_tile<double, 0, 1, 0, RESIDUAL, 0>)", r"k_band_tileIdLb0ELi1ELb0ELb1ELb0E"),
    ("band builder: dilation + item lists + load maps, incremental (k_dilate_items<1>)", r"k_dilate_itemsILb1E"),
    ("band builder: ordered compaction (k_compact)", r"k_compact"),
    ("whole-grid classification fp32 (k_classify<float, VEC>)", r"k_classifyIfLb1E"),
    ("dense full-domain Advance fp32 (k_advance_dense2)", r"k_advance_dense2"),
    ("whole-grid clamp fp32 (k_clamp_all_v4)", r"k_clamp_all_v4"),
    ("scalar fallback reinit fp32 (k_band_scalar<float, kReinit, plain>)", r"k_band_scalarIfLi1ELb0ELb0ELb0E"),
]


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", required=True)
    args = ap.parse_args(argv)
    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    so = ls_build.build()
    sass = subprocess.run([cuobjdump, "-sass", str(so)], capture_output=True, text=True, check=True).stdout
    funcs, cur = {}, None
    for line in sass.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            cur = m.group(1)
            funcs[cur] = []
            continue
        if cur is None or re.match(r"\s*/\* 0x[0-9a-f]+ \*/\s*$", line):
            continue
        m = re.match(r"\s*/\*([0-9a-f]{4,})\*/\s+(.*?);\s*(/\*.*\*/)?\s*$", line)
        if m:
            funcs[cur].append((m.group(1), m.group(2).strip()))
    demangle = shutil.which("c++filt")

    def pretty(name):
        if not demangle:
            return name
        return subprocess.run([demangle, name], capture_output=True, text=True).stdout.strip() or name

    head = f"# libls.so, csrc {ls_build.source_sha()}; written by python -m paper_1612_04040_b200.sass_listing\n"
    with open(args.out + "_histogram.txt", "w") as f:
        f.write(head + "# instructions | " + " ".join(WATCH) + " | kernel\n")
        for name, ins in sorted(funcs.items(), key=lambda kv: pretty(kv[0])):
            ops = Counter()
            for _, text in ins:
                op = re.sub(r"^@!?U?P\d+\s+", "", text).split()[0].split(".")[0]
                ops[op] += 1
            f.write(f"{len(ins):6d} | " + " ".join(f"{w}={ops[w]}" for w in WATCH if ops[w]) + f" | {pretty(name)}\n")
    with open(args.out + "_kernels.txt", "w") as f:
        f.write(head)
        for label, rx in FAMILIES:
            hits = [n for n in funcs if re.search(rx, n)]
            if not hits:
                f.write(f"\n==== {label}: no such kernel in this build\n")
                continue
            name = sorted(hits)[0]
            f.write(f"\n==== {label}\n==== {pretty(name)}\n")
            for addr, text in funcs[name]:
                f.write(f"  /*{addr}*/  {text}\n")
    print(f"{len(funcs)} kernels -> {args.out}_histogram.txt, {args.out}_kernels.txt")


if __name__ == "__main__":
    main()
