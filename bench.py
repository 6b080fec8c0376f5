#!/usr/bin/env python
"""bench.py — throughput of the narrow-band level-set hot path on B200 (contract: task prompt).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 4] [--n EDGE]
                    [--rebuild incremental|full]

One "step" = one narrow-band step (Step 1 band build -> Step 2 Advance -> `iters` Reinit sweeps ->
eq. 10 clamp) over the whole grid of the workload, default BASELINE.json configs[3]
(cfg 4: 1024^3 fp32 torus, the config north_star quotes its target on).  Metric: band grid-point
updates per second, GLUPS = 1e-9 * sum_steps(|T_s| + iters*|N_s|) / time.

our arm       W warm-up steps (one unchained ls_step call), then EXACTLY K steps as one chained
              ls_step call timed with CUDA events on the ctx stream (= torch's current stream),
              barrier + synchronize on both sides, max over ranks.  A second, identical K-step region
              runs with the library's per-kernel event brackets on (ls_profile_*) and feeds `roofline`
              and `kernels`.  `e2e` calls ls_step_host (HOST pinned buffers; H2D of phi and F and D2H
              of phi inside the timed region) once per step.
reference arm the CPU oracle (oracle/), as it stands, on the host cores, on a bounded z-slab sample of
              the same workload.  Rank 0 only.
N > 1         replicas only: every rank runs the same workload on its own GPU, no
              data-path collective; value = N * updates / max-over-ranks time; "scaling": "weak".
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

METRIC = "narrow-band grid-point updates/sec (GLUPS)"
UNIT = "GLUPS"
# Per launch of the dominant kernel (k_reinit_tma<float,0,0,0>, cfg 4), from the committed `ncu --set full`
# capture: dram__bytes_read.sum + dram__bytes_write.sum, and smsp__inst_executed.sum (warp instructions).
NCU_TRAFFIC_BYTES = {"reinit": 213.6e6 + 69.8e6}
NCU_WARP_INSTRUCTIONS = {"reinit": 70.23e6}
NCU_TRAFFIC_SOURCE = "profiles/r1b_ncu_full_summary.txt (cfg 4, one capture; not re-measured per run)"
# issue-slot peak: 148 SMs x 4 schedulers x 1 warp instruction / clock x SM clock
ISSUE_SLOTS_PER_CLOCK = 148 * 4


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json config (1-based); bench line = 4")
    ap.add_argument("--n", type=int, default=None, help="grid edge override (smoke runs of the bench itself)")
    ap.add_argument("--rebuild", default="incremental", choices=["incremental", "full"])
    ap.add_argument("--fuse", type=int, default=0, choices=[0, 1, 2],
                    help="reinit sweeps per launch: 0 = library default (1), 1 = one sweep per launch, 2 = temporal blocking")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    return ap.parse_args()


def peaks():
    """HBM GB/s roofline denominator: MEASURED_PEAKS.json (driver-written), else the guide's fallback."""
    f = ROOT / "MEASURED_PEAKS.json"
    if f.exists():
        try:
            return float(json.loads(f.read_text())["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 100 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.thr = [], None, None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thr = threading.Thread(target=self._read, daemon=True)
            self.thr.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.perf_counter(), [x.strip() for x in line.split(",")]))

    def stop(self, t0=None, t1=None):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        rows = [r for t, r in self.rows if (t0 is None or t >= t0 - 0.05) and (t1 is None or t <= t1 + 0.15)] \
            or [r for _, r in self.rows]
        sm, mx, reasons = [], [], set()
        for r in rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except Exception:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def aggregate_over_ranks(ms: float, updates: int, world: int, device: str = "cuda"):
    """N > 1 is replicas only: -> (max-over-ranks milliseconds, whole-job updates).
    The only collective of the bench: one MAX all-reduce of the timing (every rank does `updates`)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item()), world * updates


def make_workload(args):
    from paper_1612_04040_b200 import inputs
    w = inputs.config(args.config, n=args.n)
    if w.mode != "band":
        raise SystemExit("bench.py times the narrow-band step (configs 1, 3, 4); cfg 2 / cfg 5 are parity-test cases")
    return w


def workload_name(w):
    return f"{w.name} {w.nx}x{w.ny}x{w.nz} {w.dtype.name} (BASELINE.json configs[{int(w.name[3]) - 1}]): {w.note}"


def oracle_sample(w):
    """Bounded sample for the CPU oracle: a z-slab of the workload through the middle of the band."""
    nzs = min(w.nz, 64)
    k0 = (w.nz - nzs) // 2
    phi = np.ascontiguousarray(w.phi[k0:k0 + nzs])
    F = np.ascontiguousarray(w.F[k0:k0 + nzs])
    return phi, F, f"z-slab k in [{k0},{k0 + nzs}) of the workload ({w.nx}x{w.ny}x{nzs} points)"


def time_oracle(w, steps, warmup):
    """-> (GLUPS, seconds per step, threads, sample text).  The oracle as it stands (full-grid masked
    evaluation, OpenMP over all host threads)."""
    from oracle import ls_oracle as orc
    phi, F, what = oracle_sample(w)
    threads = orc.max_threads()
    cur = phi
    for _ in range(warmup):
        cur, _ = orc.step(cur, F, w.dx, w.dt, w.dtau, w.beta, w.gamma, w.iters, 1)
    t0 = time.perf_counter()
    upd = 0
    for _ in range(steps):
        cur, u = orc.step(cur, F, w.dx, w.dt, w.dtau, w.beta, w.gamma, w.iters, 1)
        upd += u
    dt = time.perf_counter() - t0
    return upd / dt * 1e-9, dt / max(steps, 1), threads, f"{steps} step(s) on a {what}"


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w = make_workload(args)
    glups, sps, threads, sample = time_oracle(w, args.steps, args.warmup)
    line = {
        "impl": "reference", "metric": METRIC, "value": glups, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": sps * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32" if w.dtype == np.float32 else "f64",
        "data": "synthetic", "gpu_launches": 0,
        "config": {"workload": workload_name(w), "sample": sample, "iters": w.iters,
                   "note": "CPU oracle (oracle/ls_oracle.cpp, -O2, no FMA contraction, OpenMP), not tuned"},
        "cpu_baseline": {"value": glups, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": glups, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line), flush=True)


def run_ours(args):
    import torch
    import torch.distributed as dist

    from paper_1612_04040_b200 import binding as ls
    from paper_1612_04040_b200 import build as ls_build

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --impl ours needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if rank == 0:
        ls_build.build()
    if world > 1:
        dist.barrier()
    ls.lib()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    w = make_workload(args)
    K, W = args.steps, args.warmup
    rebuild = ls.LS_REBUILD_INCREMENTAL if args.rebuild == "incremental" else ls.LS_REBUILD_FULL
    esz = w.dtype.itemsize
    # host buffers (pinned: the e2e leg copies from / to them)
    h_phi = torch.from_numpy(w.phi).pin_memory()
    h_F = torch.from_numpy(w.F).pin_memory()
    d_phi = h_phi.cuda(non_blocking=True)
    d_F = h_F.cuda(non_blocking=True)
    stream = torch.cuda.current_stream()
    ctx = ls.ls_create(w.nx, w.ny, w.nz, ls.LS_F32 if esz == 4 else ls.LS_F64, stream.cuda_stream)
    p0 = ls.make_params(w.dx, w.dt, w.dtau, w.beta, w.gamma, w.iters, rebuild, 0, args.fuse)
    p1 = ls.make_params(w.dx, w.dt, w.dtau, w.beta, w.gamma, w.iters, rebuild, 1, args.fuse)
    out = {}
    try:
        # ---- warm-up (unchained: resync copy + whole-grid scan + global clamp happen here, once) ----
        ls.ls_step(ctx, d_phi, d_F, p0, max(W, 1))
        barrier()
        # ---- timed region: exactly K steps, one chained call, CUDA events on the launching stream ----
        ls.ls_stats_reset(ctx)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        sampler = ClockSampler(local) if rank == 0 else None
        barrier()
        t0 = time.perf_counter()
        e0.record(stream)
        ls.ls_step(ctx, d_phi, d_F, p1, K)
        e1.record(stream)
        barrier()
        t1 = time.perf_counter()
        ms = e0.elapsed_time(e1)
        clocks = sampler.stop(t0, t1) if sampler else None
        updates, steps_done, launches = ls.ls_stats(ctx)
        assert steps_done == K
        nT, nN, bT, bN = ls.ls_band_counts(ctx)   # band of the last step
        ms_max, job_updates = aggregate_over_ranks(ms, updates, world)
        out.update(ms=ms_max, updates=updates, job_updates=job_updates, launches=launches, band=(nT, nN, bT, bN), clocks=clocks)

        # ---- same K-step region again with per-kernel event brackets (roofline / breakdown) ----
        if rank == 0:
            ls.ls_profile_reset(ctx)
            ls.ls_profile_enable(ctx, True)
            ls.ls_stats_reset(ctx)
            ls.ls_step(ctx, d_phi, d_F, p1, K)
            prof = {name: ls.ls_profile_read(ctx, k) for k, name in enumerate(ls.KERNEL_KINDS)}
            ls.ls_profile_enable(ctx, False)
            upd2, _, _ = ls.ls_stats(ctx)
            nT2, nN2, bT2, bN2 = ls.ls_band_counts(ctx)
            out.update(prof=prof, prof_updates=upd2, prof_band=(nT2, nN2, bT2, bN2))

        # ---- e2e: the C-ABI call with HOST buffers, one step per call, copies inside the timed region ----
        if rank == 0 and not args.no_e2e:
            Ke = min(K, 5)
            hp = h_phi.clone().pin_memory()
            ls.ls_step_host(ctx, hp.data_ptr(), h_F.data_ptr(), p0, 1)   # warm-up: allocates the staging fields
            ls.ls_stats_reset(ctx)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            for _ in range(Ke):
                ls.ls_step_host(ctx, hp.data_ptr(), h_F.data_ptr(), p0, 1)   # synchronises
            dt = time.perf_counter() - t0
            upd_e, _, _ = ls.ls_stats(ctx)
            out.update(e2e={"value": upd_e / dt * 1e-9, "unit": UNIT, "h2d_bytes_per_step": 2 * w.n_points * esz,
                            "d2h_bytes_per_step": w.n_points * esz, "steps": Ke, "ms_per_step": dt / Ke * 1e3,
                            "call": "ls_step_host(n_steps=1) per step, pinned host phi and F in, phi out"})
            del hp
    finally:
        ls.ls_destroy(ctx)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    value = out["job_updates"] / (out["ms"] * 1e-3) * 1e-9
    peak, peak_src = peaks()
    prof = out["prof"]
    total_prof_ms = sum(ms for ms, _ in prof.values()) or 1.0
    kernels = {name: {"ms_per_step": ms / K, "launches_per_step": n / K, "share": ms / total_prof_ms,
                      "us_per_launch": (ms / n * 1e3) if n else None}
               for name, (ms, n) in prof.items() if n}
    # dominant kernel: the reinit sweep.  Algorithmic bytes per launch: read + write of
    # every N point (2w), plus the brick list entry (4 B id + 64 B mask) per N brick.
    r_ms, r_n = prof["reinit"]
    nN_pts = out["prof_band"][1]   # |N| of the region's last step (the band moves < 1 cell per step)
    alg_bytes = 2 * esz * nN_pts + 68 * out["prof_band"][3]
    ach = alg_bytes / (r_ms / max(r_n, 1) * 1e-3) * 1e-9 if r_n else None
    is_cfg4 = w.name.startswith("cfg4") and w.nx == 1024
    traffic = NCU_TRAFFIC_BYTES["reinit"] if is_cfg4 else None
    sm_mhz = (out["clocks"] or {}).get("sm_mhz") or 1965.0
    us = r_ms / max(r_n, 1) * 1e3
    alu_peak = ISSUE_SLOTS_PER_CLOCK * sm_mhz * 1e6 * 1e-12          # T warp-instructions / s
    alu_ach = (NCU_WARP_INSTRUCTIONS["reinit"] / (us * 1e-6) * 1e-12) if (is_cfg4 and r_n) else None
    roofline_alu = {"bound": "alu", "kernel": "k_reinit_tma (one Step 3 sweep)", "achieved": alu_ach, "peak": alu_peak,
                    "unit": "T warp-instructions/s", "frac": (alu_ach / alu_peak) if alu_ach else None,
                    "note": "issue slots: executed warp instructions per launch (ncu capture) / live launch duration; "
                            "peak = 148 SMs x 4 schedulers x SM clock sampled during the run (DESIGN.md section 6)"}
    roofline = {"bound": "hbm", "kernel": "k_reinit_tma (one Step 3 sweep)", "achieved": ach, "peak": peak,
                "peak_source": peak_src, "unit": "GB/s", "frac": (ach / peak) if ach else None,
                "traffic": traffic, "traffic_source": NCU_TRAFFIC_SOURCE if traffic else None,
                "algorithmic_bytes_per_launch": alg_bytes, "us_per_launch": r_ms / max(r_n, 1) * 1e3,
                "frac_of_8TBps_nominal": (ach / 8000.0) if ach else None}
    cpu = None
    if not args.no_cpu_baseline:
        g, sps, threads, sample = time_oracle(w, 20, 1)   # ~10 s of CPU work on the GPU box (0.44 s per slab step)
        cpu = {"value": g, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample, "s_per_step": sps}
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": out["ms"] / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32" if esz == 4 else "f64", "data": "synthetic",
        "config": {"workload": workload_name(w), "iters": w.iters, "gamma_dx": w.gamma / w.dx,
                   "beta_dx": w.beta / w.dx, "dt_dx": w.dt / w.dx, "dtau_dx": w.dtau / w.dx,
                   "rebuild": args.rebuild, "parallelism": "replicas only" if world > 1 else "1 GPU",
                   "band_last_step": dict(zip(("T_points", "N_points", "T_bricks", "N_bricks"), out["band"])),
                   "updates_per_step": out["updates"] / K,
                   "l2": "inputs larger than L2 (fields 4 GiB each; one band sweep touches ~0.3 GB > 126 MB L2)"
                   if w.n_points * esz > 512e6 else "working set fits L2 (small config): not a bandwidth number"},
        "clocks": out["clocks"], "e2e": out.get("e2e"), "gpu_launches": out["launches"],
        "roofline": roofline, "roofline_alu": roofline_alu, "kernels": kernels, "cpu_baseline": cpu,
    }
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
