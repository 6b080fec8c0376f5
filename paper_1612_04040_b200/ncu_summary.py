"""Summarise an `ncu --set full` report of bench.py into the tracked files bench.py and the reader use.

    python -m paper_1612_04040_b200.ncu_summary REPORT.ncu-rep --workload cfg4 --out profiles/r2_ncu [--append]

Writes  <out>_kernels.csv   one row per kernel class (key): per-launch averages of the counters bench.py needs
                            (duration, DRAM bytes read / written, warp instructions), tagged with the hash of the
                            kernel sources (build.source_sha) so that a stale capture is never mistaken for this code
        <out>_summary.txt   the metrics a reader checks (throughputs, hit rates, occupancy, stall shares) per launch
The report is read with `ncu -i REPORT --page raw --csv` (ncu is in the CUDA image; no GPU needed).
"""
from __future__ import annotations

import argparse
import csv
import io
import subprocess
import sys
from pathlib import Path

from . import build as ls_build

# kernel class <- substring tests on the demangled kernel name
KEYS = [
    ("reinit_last", lambda n: "k_band_tile<" in n and _targs(n)[1:3] == ["0", "1"] and _targs(n)[5] == "1"),
    ("reinit", lambda n: "k_band_tile<" in n and _targs(n)[1:3] == ["0", "1"]),
    ("reinit2", lambda n: "k_band_tile<" in n and _targs(n)[1:3] == ["0", "2"]),
    ("advance", lambda n: "k_band_tile<" in n and _targs(n)[1] == "1"),
    ("dilate", lambda n: "k_dilate_items" in n),
    ("compact", lambda n: "k_compact" in n),
    ("classify", lambda n: "k_classify" in n),
    ("advance_dense", lambda n: "k_advance_dense" in n),
    ("clamp_all", lambda n: "k_clamp_all" in n),
    ("band_scalar", lambda n: "k_band_scalar" in n),
]
SUMMARY_METRICS = [
    "gpu__time_duration.sum", "dram__bytes_read.sum", "dram__bytes_write.sum", "smsp__inst_executed.sum",
    "gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed", "lts__throughput.avg.pct_of_peak_sustained_elapsed",
    "lts__t_sector_hit_rate.pct", "l1tex__throughput.avg.pct_of_peak_sustained_elapsed",
    "smsp__issue_active.avg.pct_of_peak_sustained_active", "sm__warps_active.avg.pct_of_peak_sustained_active",
    "sm__pipe_fma_cycles_active.avg.pct_of_peak_sustained_active", "sm__pipe_alu_cycles_active.avg.pct_of_peak_sustained_active",
    "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum", "l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum",
    "launch__registers_per_thread", "launch__grid_size", "launch__block_size", "launch__occupancy_limit_shared_mem",
    "launch__occupancy_limit_registers",
    "smsp__average_warps_issue_stalled_barrier_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_long_scoreboard_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_short_scoreboard_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_wait_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_math_pipe_throttle_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_not_selected_per_issue_active.ratio",
]


def _targs(name: str):
    """Template arguments of k_band_tile<T, ADV, K, CLAMP, RESIDUAL, EMIT_T, ...> as strings ('0' / '1' / ...)."""
    inner = name[name.index("<") + 1:]
    parts = [p.strip() for p in inner.split(">")[0].split(",")]
    return [p.replace("(bool)", "").replace("(int)", "") for p in parts]


def classify(name: str):
    for key, test in KEYS:
        try:
            if test(name):
                return key
        except (ValueError, IndexError):
            continue
    return None


def to_bytes(value: str, unit: str) -> float:
    v = float(value.replace(",", ""))
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}.get(unit)
    if scale is None:
        raise ValueError(f"unexpected byte unit {unit!r}")
    return v * scale


def to_us(value: str, unit: str) -> float:
    v = float(value.replace(",", ""))
    scale = {"ns": 1e-3, "us": 1.0, "ms": 1e3, "s": 1e6}.get(unit.replace("second", "s").replace("usecond", "us"))
    if scale is None:
        scale = {"nsecond": 1e-3, "usecond": 1.0, "msecond": 1e3, "second": 1e6}[unit]
    return v * scale


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("report")
    ap.add_argument("--workload", required=True, help="label stored in the rows, e.g. cfg4")
    ap.add_argument("--out", required=True, help="output prefix, e.g. profiles/r2_ncu")
    ap.add_argument("--append", action="store_true", help="keep the rows already in <out>_kernels.csv")
    args = ap.parse_args(argv)
    raw = subprocess.run(["ncu", "-i", args.report, "--page", "raw", "--csv"], capture_output=True, text=True, check=True).stdout
    rows = list(csv.reader(io.StringIO(raw)))
    hdr, units = rows[0], rows[1]
    col = {h: i for i, h in enumerate(hdr)}
    per_key = {}
    lines = [f"# {Path(args.report).name}: per-launch metrics (ncu --set full), workload {args.workload}, csrc {ls_build.source_sha()}"]
    for r in rows[2:]:
        name = r[col["Kernel Name"]]
        key = classify(name)
        lines.append(f"\n== {key or '?'}: {name[:140]}")
        for m in SUMMARY_METRICS:
            if m in col:
                lines.append(f"  {m} = {r[col[m]]} {units[col[m]]}")
        if key is None:
            continue
        d = per_key.setdefault(key, {"n": 0, "us": 0.0, "rd": 0.0, "wr": 0.0, "inst": 0.0})
        d["n"] += 1
        d["us"] += to_us(r[col["gpu__time_duration.sum"]], units[col["gpu__time_duration.sum"]])
        d["rd"] += to_bytes(r[col["dram__bytes_read.sum"]], units[col["dram__bytes_read.sum"]])
        d["wr"] += to_bytes(r[col["dram__bytes_write.sum"]], units[col["dram__bytes_write.sum"]])
        d["inst"] += float(r[col["smsp__inst_executed.sum"]].replace(",", ""))
    out_csv = Path(args.out + "_kernels.csv")
    fields = ["workload", "key", "launches_captured", "time_us", "dram_read_bytes", "dram_write_bytes", "warp_instructions", "csrc_sha"]
    old = []
    if args.append and out_csv.exists():
        old = [r for r in csv.DictReader(l for l in out_csv.read_text().splitlines() if l and not l.startswith("#"))
               if not (r["workload"] == args.workload and r["key"] in per_key)]
    with out_csv.open("w", newline="") as f:
        f.write("# per-launch averages from `ncu --set full` captures; written by python -m paper_1612_04040_b200.ncu_summary\n")
        w = csv.DictWriter(f, fieldnames=fields)
        w.writeheader()
        for r in old:
            w.writerow(r)
        for key, d in per_key.items():
            n = d["n"]
            w.writerow({"workload": args.workload, "key": key, "launches_captured": n, "time_us": round(d["us"] / n, 3),
                        "dram_read_bytes": round(d["rd"] / n), "dram_write_bytes": round(d["wr"] / n),
                        "warp_instructions": round(d["inst"] / n), "csrc_sha": ls_build.source_sha()})
    mode = "a" if args.append else "w"
    with Path(args.out + "_summary.txt").open(mode) as f:
        f.write("\n".join(lines) + "\n")
    print(f"{out_csv}: {sorted(per_key)}", file=sys.stderr)


if __name__ == "__main__":
    main()
