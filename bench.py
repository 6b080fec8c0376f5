#!/usr/bin/env python
"""bench.py — throughput of the narrow-band level-set hot path on B200 (contract: task prompt).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 1..5] [--edge EDGE]
                    [--rebuild incremental|full] [--fuse 0|1|2]

Workload: BASELINE.json configs[--config - 1]; default 4 (cfg 4: 1024^3 fp32 torus, the config north_star quotes its
target on) — THE bench line.  The other configs are the same driver on the other workloads:
  cfg 1, 3, 4   one "step" = one narrow-band step (Step 1 band build -> Step 2 Advance -> `iters` Reinit sweeps ->
                eq. 10 clamp) over the whole grid
  cfg 2         one "step" = one full-domain Advance (ls_advance, gamma = beta = inf), ping-pong between two fields
  cfg 5         one "step" = one Reinit sweep on the band of phi^0 (ls_reinit with K iterations), fp64
Metric: band grid-point updates per second, GLUPS = 1e-9 * sum_steps(|T_s| + iters*|N_s|) / time (cfg 2: grid points
per advance; cfg 5: |N| per sweep).

our arm       W warm-up steps (band: one unchained ls_step call), then EXACTLY K steps timed with CUDA events on the
              ctx stream (= torch's current stream), barrier + synchronize on both sides, max over ranks.  A second,
              identical K-step region runs with the library's per-kernel event brackets on (ls_profile_*) and feeds
              `roofline` (the dominant kernel), `roofline_advance` and `kernels`; a short third one with
              LS_REBUILD_FULL feeds `full_rebuild` (the paper's own Step 1).  `e2e` calls ls_step_host
              once per step: pinned HOST phi in and out inside the timed region (the static F is uploaded by the
              warm-up call and reused, R17).
reference arm the CPU oracle (oracle/), as it stands, on the host cores, on a bounded z-slab sample of the same
              workload.  Rank 0 only.
N > 1         replicas only: every rank runs the same workload on its own GPU, no data-path collective;
              value = N * updates / max-over-ranks time; "scaling": "weak".
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
# Per-launch ncu counters (dram__bytes_read/write.sum, smsp__inst_executed.sum) come from the tracked capture summary
# profiles/<NCU_KERNELS_CSV>, written by `python -m paper_1612_04040_b200.ncu_summary` from an `ncu --set full` report
# of this bench command (profiles/*.md name the commands).  Every row carries the hash of csrc/ it was captured from;
# rows from other sources are reported as stale and not used.
NCU_KERNELS_CSV = "r2_ncu_kernels.csv"
# issue-slot peak: 148 SMs x 4 schedulers x 1 warp instruction / clock x SM clock
ISSUE_SLOTS_PER_CLOCK = 148 * 4


def ncu_rows():
    """-> ({kernel key: row dict}, note).  Keys: 'reinit', 'reinit_last', 'advance', 'dilate', 'compact', 'classify', ..."""
    import csv
    from paper_1612_04040_b200 import build as ls_build
    f = ROOT / "profiles" / NCU_KERNELS_CSV
    if not f.exists():
        return {}, f"profiles/{NCU_KERNELS_CSV} absent"
    sha = ls_build.source_sha()
    rows, stale = {}, 0
    for r in csv.DictReader(l for l in f.read_text().splitlines() if l and not l.startswith("#")):
        if r.get("csrc_sha") != sha:
            stale += 1
            continue
        rows[(r["workload"], r["key"])] = r
    note = f"profiles/{NCU_KERNELS_CSV} (csrc {sha})" + (f"; {stale} stale row(s) from other sources ignored" if stale else "")
    if stale and not rows:
        print(f"bench.py: every row of profiles/{NCU_KERNELS_CSV} was captured from other kernel sources than csrc {sha}: "
              "roofline.traffic is null until the capture is redone", file=sys.stderr)
    return rows, note


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json config 1..5 (1-based); the bench line is 4; 2 = dense advance, 5 = fp64 reinit sweeps")
    ap.add_argument("--edge", "--n", dest="n", type=int, default=None,
                    help="grid edge override (smaller or paper-shaped grids; under torchrun spell it --edge: its own parser claims --n)")
    ap.add_argument("--rebuild", default="incremental", choices=["incremental", "full"])
    ap.add_argument("--fuse", type=int, default=0, choices=[0, 1, 2],
                    help="reinit sweeps per launch: 0 = library default (1), 1 = one sweep per launch, 2 = temporal blocking")
    ap.add_argument("--tile-min-cells", type=int, default=-1,
                    help="ls_tile_threshold: grids below it take the scalar band kernels (-1 = library default, 0 = tiled wherever possible)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-full-rebuild", action="store_true", help="skip the short LS_REBUILD_FULL run of the same workload")
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
    return inputs.config(args.config, n=args.n)


def workload_name(w):
    return f"{w.name} {w.nx}x{w.ny}x{w.nz} {w.dtype.name} (BASELINE.json configs[{int(w.name[3]) - 1}]): {w.note}"


def oracle_sample(w):
    """Bounded sample for the CPU oracle: a z-slab of the workload through the middle of the band."""
    nzs = min(w.nz, 64 if w.mode == "band" else 32)
    k0 = (w.nz - nzs) // 2
    phi = np.ascontiguousarray(w.phi[k0:k0 + nzs])
    F = np.ascontiguousarray(w.F[k0:k0 + nzs]) if w.F is not None else None
    return phi, F, f"z-slab k in [{k0},{k0 + nzs}) of the workload ({w.nx}x{w.ny}x{nzs} points)"


def oracle_unit(w, cur, F, Nm):
    """One unit of the oracle's work for this workload -> (next field, point updates)."""
    from oracle import ls_oracle as orc
    if w.mode == "band":
        return orc.step(cur, F, w.dx, w.dt, w.dtau, w.beta, w.gamma, w.iters, 1)
    if w.mode == "dense":
        return orc.advance(cur, F, None, w.dt, w.dx, w.beta, w.gamma), cur.size
    nxt, _ = orc.reinit_iter(cur, Nm, w.dtau, w.dx)      # cfg 5: one sweep on the tube N of phi^0
    return nxt, int(Nm.sum())


def time_oracle(w, steps, warmup, threads=None):
    """-> (GLUPS, seconds per step, threads, sample text).  The oracle as it stands (full-grid masked evaluation,
    OpenMP over `threads` host threads; None = all)."""
    from oracle import ls_oracle as orc
    phi, F, what = oracle_sample(w)
    all_threads = orc.max_threads()
    if threads is not None:
        orc.set_threads(threads)
    try:
        Nm = orc.band_masks(phi, w.gamma)[1] if w.mode == "reinit_tol" else None
        cur = phi
        for _ in range(warmup):
            cur, _ = oracle_unit(w, cur, F, Nm)
        t0 = time.perf_counter()
        upd = 0
        for _ in range(steps):
            cur, u = oracle_unit(w, cur, F, Nm)
            upd += u
        dt = time.perf_counter() - t0
    finally:
        if threads is not None:
            orc.set_threads(all_threads)
    unit = {"band": "step(s)", "dense": "full-domain advance(s)", "reinit_tol": "reinit sweep(s)"}[w.mode]
    return upd / dt * 1e-9, dt / max(steps, 1), threads or all_threads, f"{steps} {unit} on a {what}"


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
    h_F = torch.from_numpy(w.F).pin_memory() if w.F is not None else None      # cfg 5 has no F (reinit only)
    d_phi = h_phi.cuda(non_blocking=True)
    d_F = h_F.cuda(non_blocking=True) if h_F is not None else None
    stream = torch.cuda.current_stream()
    ctx = ls.ls_create(w.nx, w.ny, w.nz, ls.LS_F32 if esz == 4 else ls.LS_F64, stream.cuda_stream)
    ls.ls_tile_threshold(ctx, args.tile_min_cells)
    p0 = ls.make_params(w.dx, w.dt, w.dtau, w.beta, w.gamma, w.iters, rebuild, 0, args.fuse)
    p1 = ls.make_params(w.dx, w.dt, w.dtau, w.beta, w.gamma, w.iters, rebuild, 1, args.fuse)
    out = {}

    # One "step" of the workload, n times, on the ctx stream (no host synchronisation inside):
    #   band (cfg 1, 3, 4): n narrow-band steps, one chained ls_step call
    #   dense (cfg 2):      n full-domain ls_advance calls, ping-pong between two fields
    #   reinit (cfg 5):     ls_reinit with n sweeps on the band of phi^0 (band built before the timed region)
    d_alt = torch.empty_like(d_phi) if w.mode != "band" else None
    state = {"cur": d_phi, "alt": d_alt}

    def run_steps(n, params):
        if w.mode == "band":
            ls.ls_step(ctx, d_phi, d_F, params, n)
        elif w.mode == "dense":
            for _ in range(n):
                ls.ls_advance(ctx, state["cur"], d_F, w.dt, w.dx, w.beta, w.gamma, state["alt"])
                state["cur"], state["alt"] = state["alt"], state["cur"]
        else:
            ls.ls_reinit(ctx, d_alt, d_phi, w.dtau, w.dx, w.gamma, n)

    def timed(n, params):
        ls.ls_stats_reset(ctx)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        t0 = time.perf_counter()
        e0.record(stream)
        run_steps(n, params)
        e1.record(stream)
        barrier()
        t1 = time.perf_counter()
        upd, steps_done, launches = ls.ls_stats(ctx)
        if w.mode == "reinit_tol":
            upd = n * ls.ls_band_counts(ctx)[1]          # n sweeps over |N|
        return e0.elapsed_time(e1), upd, launches, t0, t1

    try:
        # ---- warm-up (band: unchained, so the resync copy, whole-grid scan and global clamp happen here, once) ----
        if w.mode == "reinit_tol":
            ls.ls_build_band(ctx, d_phi, w.dx, w.gamma)
        run_steps(max(W, 1), p0)
        barrier()
        # ---- timed region: exactly K steps, CUDA events on the launching stream ----
        sampler = ClockSampler(local) if rank == 0 else None
        ms, updates, launches, t0, t1 = timed(K, p1)
        clocks = sampler.stop(t0, t1) if sampler else None
        band = ls.ls_band_counts(ctx) if w.mode != "dense" else (w.n_points, w.n_points, 0, 0)
        ms_max, job_updates = aggregate_over_ranks(ms, updates, world)
        out.update(ms=ms_max, updates=updates, job_updates=job_updates, launches=launches, band=band, clocks=clocks)

        # ---- same K-step region again with per-kernel event brackets (roofline / breakdown) ----
        if rank == 0:
            ls.ls_profile_reset(ctx)
            ls.ls_profile_enable(ctx, True)
            timed(K, p1)
            prof = {name: ls.ls_profile_read(ctx, k) for k, name in enumerate(ls.KERNEL_KINDS)}
            ls.ls_profile_enable(ctx, False)
            out.update(prof=prof, prof_band=ls.ls_band_counts(ctx) if w.mode != "dense" else band)

        # ---- the paper's own Step 1 (every grid point scanned every step): --rebuild full, short ----
        if rank == 0 and w.mode == "band" and args.rebuild == "incremental" and not args.no_full_rebuild:
            pf = ls.make_params(w.dx, w.dt, w.dtau, w.beta, w.gamma, w.iters, ls.LS_REBUILD_FULL, 1, args.fuse)
            Kf = min(K, 5)
            run_steps(1, pf)
            msf, updf, _, _, _ = timed(Kf, pf)
            out.update(full_rebuild={"ms_per_step": msf / Kf, "value": updf / (msf * 1e-3) * 1e-9, "unit": UNIT, "steps": Kf,
                                     "what": "same workload with LS_REBUILD_FULL: the whole grid re-classified every step"})

        # ---- e2e: the C-ABI call with HOST buffers, one step per call, copies inside the timed region ----
        if rank == 0 and not args.no_e2e and w.mode == "band":
            Ke = min(K, 5)
            hp = h_phi.clone().pin_memory()
            ls.ls_step_host(ctx, hp.data_ptr(), h_F.data_ptr(), p0, 1)   # warm-up: allocates the staging fields, uploads F
            ls.ls_stats_reset(ctx)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            for _ in range(Ke):
                ls.ls_step_host(ctx, hp.data_ptr(), None, p0, 1)         # phi in, phi out; F is static (R17): on the device
            dt = time.perf_counter() - t0
            upd_e, _, _ = ls.ls_stats(ctx)
            out.update(e2e={"value": upd_e / dt * 1e-9, "unit": UNIT, "h2d_bytes_per_step": w.n_points * esz,
                            "d2h_bytes_per_step": w.n_points * esz, "steps": Ke, "ms_per_step": dt / Ke * 1e3,
                            "pcie_gbs": 2 * w.n_points * esz * Ke / dt * 1e-9,
                            "call": "ls_step_host(n_steps=1) per step: pinned host phi in, phi out; the static F was uploaded "
                                    "once by the warm-up call (F_host = NULL afterwards); fields >= 64 MiB go through the "
                                    "library's z-slab pipeline (H2D / kernels / D2H overlapped, every layer copied once each way)"})
            del hp
    finally:
        ls.ls_destroy(ctx)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    report(args, w, out, world, K, W, esz)
    if world > 1:
        dist.destroy_process_group()


def report(args, w, out, world, K, W, esz):
    """Assemble and print the JSON line (rank 0)."""
    value = out["job_updates"] / (out["ms"] * 1e-3) * 1e-9
    peak, peak_src = peaks()
    prof = out["prof"]
    total_prof_ms = sum(ms for ms, _ in prof.values()) or 1.0
    kernels = {name: {"ms_per_step": ms / K, "launches_per_step": n / K, "share": ms / total_prof_ms,
                      "us_per_launch": (ms / n * 1e3) if n else None}
               for name, (ms, n) in prof.items() if n}
    nT_pts, nN_pts, bT, bN = out["prof_band"]
    ncu, ncu_note = ncu_rows()
    wl = f"cfg{args.config}" if args.n is None else None       # captures are of the full-size workloads only
    sm_mhz = (out["clocks"] or {}).get("sm_mhz") or 1965.0

    def roof(kind, key, what, alg_bytes):
        """HBM roofline of one kernel class: algorithmic bytes per launch / live launch duration."""
        ms, n = prof[kind]
        if not n:
            return None
        us = ms / n * 1e3
        ach = alg_bytes / (us * 1e-6) * 1e-9
        row = ncu.get((wl, key)) if key else None   # scalar band kernels: one ncu class for Advance and sweeps, no per-kind traffic
        traffic = (float(row["dram_read_bytes"]) + float(row["dram_write_bytes"])) if row else None
        r = {"bound": "hbm", "kernel": what, "achieved": ach, "peak": peak, "peak_source": peak_src, "unit": "GB/s",
             "frac": ach / peak, "traffic": traffic, "traffic_source": ncu_note if row else None,
             "algorithmic_bytes_per_launch": alg_bytes, "us_per_launch": us, "frac_of_8TBps_nominal": ach / 8000.0,
             "overfetch": (traffic / alg_bytes) if traffic else None,
             "dram_gbs": (traffic / (us * 1e-6) * 1e-9) if traffic else None}
        if row:   # issue-slot view of the same launch (the band kernels are bound by instruction issue)
            alu_peak = ISSUE_SLOTS_PER_CLOCK * sm_mhz * 1e6 * 1e-12
            alu_ach = float(row["warp_instructions"]) / (us * 1e-6) * 1e-12
            r["issue"] = {"bound": "alu", "achieved": alu_ach, "peak": alu_peak, "unit": "T warp-instructions/s",
                          "frac": alu_ach / alu_peak, "warp_instructions_per_launch": float(row["warp_instructions"]),
                          "note": "executed warp instructions per launch (ncu capture) / live launch duration; peak = 148 SMs x 4 "
                                  "schedulers x the SM clock sampled during the run"}
        return r

    roofline = roofline_advance = None
    if w.mode == "band":
        # reinit sweep: read + write of every N point (2w) + the quad's item list (2 B per item ~ 0.6 B per point) and
        # list entry; Advance: phi, F read and phi-bar written on T (3w), halo read on N \ T (w), same lists
        # which band kernels ran: the library's rule (ls.h, ls_tile_threshold) restated for the label only
        thr = 4_000_000 if args.tile_min_cells < 0 else args.tile_min_cells
        tiled = w.n_points >= thr and (w.nx * esz) % 16 == 0
        kr, ka = ("k_band_tile<K=1>", "k_band_tile<ADV>") if tiled else ("k_band_scalar<kReinit>", "k_band_scalar<kAdvance>")
        roofline = roof("reinit", "reinit" if tiled else None, kr + " (one Step 3 sweep, eq. 12-13)", 2 * esz * nN_pts + 68 * bN)
        roofline_advance = roof("advance", "advance" if tiled else None, ka + " (Step 2, eq. 3-8)",
                                3 * esz * nT_pts + esz * (nN_pts - nT_pts) + 68 * bN)
    elif w.mode == "dense":
        roofline = roof("advance", "advance_dense", "k_advance_dense2 (full-domain Step 2, c == 1)", 3 * esz * w.n_points)
    else:
        roofline = roof("reinit", "reinit", "k_band_tile<double, K=1> (one Step 3 sweep, eq. 12-13)", 2 * esz * nN_pts + 68 * bN)

    cpu = None
    if not args.no_cpu_baseline:
        # ~10-20 s of CPU work on the GPU box: all host threads, then one thread on a shorter run
        n_all = {"band": 20, "dense": 40, "reinit_tol": 40}[w.mode]
        g, sps, threads, sample = time_oracle(w, n_all, 1)
        g1, sps1, _, sample1 = time_oracle(w, max(n_all // 10, 2), 0, threads=1)
        cpu = {"value": g, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample, "s_per_step": sps,
               "one_thread": {"value": g1, "unit": UNIT, "cores": 1, "sample": sample1, "ns_per_update": 1.0 / g1},
               "ns_per_update_per_core": threads / g}
    unit_name = {"band": "narrow-band step (build + advance + iters sweeps + clamp)", "dense": "full-domain advance (ls_advance)",
                 "reinit_tol": "reinit sweep (ls_reinit iteration on the band of phi^0)"}[w.mode]
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": out["ms"] / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32" if esz == 4 else "f64", "data": "synthetic",
        "config": {"workload": workload_name(w), "step": unit_name, "iters": w.iters, "gamma_dx": w.gamma / w.dx,
                   "beta_dx": w.beta / w.dx, "dt_dx": w.dt / w.dx, "dtau_dx": w.dtau / w.dx,
                   "rebuild": args.rebuild, "fuse": args.fuse or 1,
                   "tile_min_cells": "library default (4 M cells: smaller grids take the scalar band kernels)" if args.tile_min_cells < 0 else args.tile_min_cells, "parallelism": "replicas only" if world > 1 else "1 GPU",
                   "band_last_step": dict(zip(("T_points", "N_points", "T_bricks", "N_bricks"), out["band"])),
                   "updates_per_step": out["updates"] / K,
                   "l2": "inputs larger than L2 (fields >= 0.5 GiB each; one pass touches more than the 126 MB L2)"
                   if w.n_points * esz > 512e6 else "working set fits L2 (small config): not a bandwidth number"},
        "clocks": out["clocks"], "e2e": out.get("e2e"), "gpu_launches": out["launches"],
        "roofline": roofline, "roofline_advance": roofline_advance, "full_rebuild": out.get("full_rebuild"),
        "kernels": kernels, "cpu_baseline": cpu,
    }
    if w.mode == "band" and "band" in kernels:   # the whole-step figure with the build included and excluded
        line["ms_per_step_without_band_build"] = out["ms"] / K - kernels["band"]["ms_per_step"]
    print(json.dumps(line), flush=True)


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
