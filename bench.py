#!/usr/bin/env python
"""bench.py — grid-point updates/s and ms/step of the full dipolar SSCN step (BASELINE.json `metric`).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C4] [--impl ours|reference]

One "step" is one pass of the whole hot path: calcpsidd2 (density -> FFT -> x V_dd -> inverse FFT),
calcnu, calclux, calcluy, calcluz (+ calcnorm in imaginary time) on the workload's grid.  The default
workload is C4 (real3d, 256^3, complex128), the configuration the metric is quoted on.

Our arm prints ONE JSON line: `value` = whole-job grid-point updates/s with psi resident in HBM
(CUDA events on the library's stream, barrier + synchronize on both sides, max over ranks); `e2e` =
the same metric through the C ABI with HOST buffers (set_psi from pinned host memory, one step,
get_psi back to the host, every step); `roofline` for the dominant kernel from per-kernel CUDA event
pairs (dbec_step_profile); `cpu_baseline` = the CPU oracle timed on this box's host cores.

Multi-GPU: the step does not shard without all-to-all transposes: N ranks
run N independent replicas, no data-path collective, `scaling` = "weak".

`--impl reference` times the oracle (oracle/, as it stands) on the host cores, rank 0 only.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_1601_04640_b200.inputs import initial_psi, workload  # noqa: E402

METRIC = "grid_point_updates_per_s"
UNIT = "updates/s"

# Algorithmic bytes per grid point per launch of each pass (
# SURVEY.md §8(d)).  The half spectrum is half a complex value per grid point.  Keys = dbec_kernel_name.
ALG_BYTES_PER_POINT = {
    "density+fft_x": 16 + 8,
    "fft_y<fwd>": 8 + 8,
    "fft_last<fwd*Vdd*inv>": 8 + 8,          # the V_dd table (4 B/pt) is not counted as useful traffic
    "fft_y<inv>": 8 + 8,
    "ifft_x+calcnu+cn_x": 8 + 16 + 16,
    "cn_x": 32,
    "cn_y": 32,
    "cn_z": 32,
}
MODEL_BYTES_PER_POINT = {3: 208, 2: 144}    # SURVEY.md §8(d) "Model M": fixed reference accounting


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clock / throttle-reason samples while the timed region runs."""
    Q = ("timestamp,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows = []
        self.t0 = self.t1 = None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "50"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def mark_start(self):
        self.t0 = time.time()

    def mark_stop(self):
        self.t1 = time.time()

    def close(self):
        if self.proc:
            time.sleep(0.12)
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except Exception:
                self.proc.kill()

    def summary(self):
        sm, smax, reasons = [], [], set()
        rows = [r for t, r in self.rows if self.t0 is not None and self.t0 - 0.05 <= t <= (self.t1 or 1e30) + 0.1]
        if not rows:
            rows = [r for _, r in self.rows]
        for r in rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 8:
                continue
            try:
                sm.append(float(f[1]))
                smax.append(float(f[2]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[4:8]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(smax)), "reasons": sorted(reasons),
                "samples": len(sm)}


def oracle_time(w, steps, threads_hint=None):
    """Seconds per step of the CPU oracle on workload w (oracle as it stands)."""
    from oracle import binding as ob
    o = ob.Oracle(ob.params_of(w, G=w.G_run, D=w.D_run))
    o.set_psi(initial_psi(w))
    t0 = time.perf_counter()
    o.step(steps)
    dt = (time.perf_counter() - t0) / steps
    o.close()
    return dt, ob.threads()


def shrunk(w, n):
    """The same physical problem on a coarser grid of n points along the longest axis (oracle samples)."""
    from dataclasses import replace
    f = max(w.nx, w.ny, w.nz) // n
    if f <= 1:
        return w
    nz = max(w.nz // f, 1) if w.ndim == 3 else 1
    return replace(w, nx=w.nx // f, ny=w.ny // f, nz=nz, dx=w.dx * f, dy=w.dy * f, dz=w.dz * f)


def run_reference(args, w):
    """The reference arm: the oracle on the host cores; each step is one oracle SSCN step on a bounded
    sample (a coarser grid of the same box, same parameters) sized so that K+W steps end in minutes."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import binding as ob
    ob.build()
    probe = shrunk(w, 32)
    t_probe, threads = oracle_time(probe, 2)
    per_point = t_probe / probe.npoints
    budget = 120.0
    n = max(w.nx, w.ny, w.nz)
    while n > 32 and per_point * shrunk(w, n).npoints * (args.steps + args.warmup) * 1.3 > budget:
        n //= 2
    ws = shrunk(w, n)
    o = ob.Oracle(ob.params_of(ws, G=ws.G_run, D=ws.D_run))
    o.set_psi(initial_psi(ws))
    o.step(args.warmup)
    t0 = time.perf_counter()
    o.step(args.steps)
    dt = time.perf_counter() - t0
    o.close()
    value = ws.npoints * args.steps / dt
    sample = (f"{args.steps} oracle steps on a {ws.nx}x{ws.ny}x{ws.nz} grid of the same box and parameters "
              f"(1/{w.npoints // ws.npoints} of the {w.name} grid points)")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "grid": [w.nx, w.ny, w.nz], "sample_grid": [ws.nx, ws.ny, ws.nz],
                       "mode": "real" if w.time_mode else "imag"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def max_over_ranks(x, world, device="cpu"):
    """Max of a per-rank float over all ranks (the only collective of the benchmark; timing plumbing)."""
    if world <= 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(npoints, steps, world, seconds):
    """Replicas only: every rank advances its own npoints-grid `steps` times; the job took `seconds`."""
    return world * npoints * steps / seconds


def run_ours(args, w):
    import torch
    import torch.distributed as dist
    from paper_1601_04640_b200 import dbec

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = f"cuda:{local}"
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(dev))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    dbec.lib()
    sim = dbec.Dbec(dbec.params_of(w), device=dev)
    psi0 = initial_psi(w)
    sim.set_psi(psi0)
    if (w.G_run, w.D_run) != (w.G, w.D):
        sim.set_coupling(w.G_run, w.D_run)

    # ---- device-resident timing ----
    sampler = ClockSampler(local) if rank == 0 else None
    sim.step(args.warmup)
    barrier()
    l0 = sim.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    if sampler:
        sampler.mark_start()
    e0.record(sim.stream)
    sim.step(args.steps)
    e1.record(sim.stream)
    barrier()
    if sampler:
        sampler.mark_stop()
    ms = e0.elapsed_time(e1)
    launches = sim.launch_count() - l0
    ms = max_over_ranks(ms, world, dev)
    value = whole_job_value(w.npoints, args.steps, world, ms * 1e-3)
    obs = sim.observables()

    # ---- end to end through the C ABI with host buffers ----
    e2e_steps = max(3, min(args.steps, 10))
    host_in = torch.from_numpy(psi0.copy()).pin_memory()
    host_out = torch.empty_like(host_in).pin_memory()
    for _ in range(2):
        sim.set_psi(host_in.numpy())
        sim.step(1)
        sim.get_psi(host_out.numpy())
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        sim.set_psi(host_in.numpy())       # H2D of the step's input
        sim.step(1)
        sim.get_psi(host_out.numpy())      # D2H of the step's result (synchronises)
    barrier()
    e2e_s = time.perf_counter() - t0
    e2e_value = whole_job_value(w.npoints, e2e_steps, world, max_over_ranks(e2e_s, world, dev))

    # ---- per-kernel roofline (rank 0) ----
    line = None
    if rank == 0:
        sim.set_psi(psi0)
        sim.step_profile(3)
        prof_steps = max(5, min(args.steps, 50))
        prof = sim.step_profile(prof_steps)
        peak, peak_src = measured_peaks()
        per_kernel = {}
        kernels = sim.pass_kernels()
        for name, (tot_ms, cnt) in prof.items():
            avg_ms = tot_ms / cnt
            gbs = ALG_BYTES_PER_POINT[name] * w.npoints / (avg_ms * 1e-3) / 1e9
            per_kernel[name] = {"kernel": kernels.get(name, ""), "ms": avg_ms, "alg_GBps": gbs, "frac": gbs / peak}
        top = max(per_kernel, key=lambda k: per_kernel[k]["ms"])
        step_ms_prof = sum(v["ms"] for v in per_kernel.values())
        model = MODEL_BYTES_PER_POINT[w.ndim]
        model_gbs = model * w.npoints / (ms / args.steps * 1e-3) / 1e9
        roofline = {"bound": "hbm", "kernel": kernels.get(top, top), "pass": top, "achieved": per_kernel[top]["alg_GBps"], "peak": peak,
                    "unit": "GB/s", "frac": per_kernel[top]["frac"], "traffic": None, "peak_source": peak_src,
                    "kernel_ms": per_kernel[top]["ms"], "kernel_share_of_step": per_kernel[top]["ms"] / step_ms_prof,
                    "alg_bytes_per_launch": ALG_BYTES_PER_POINT[top] * w.npoints,
                    "per_kernel": per_kernel,
                    "step_model": {"bytes_per_point": model, "achieved_GBps": model_gbs, "frac": model_gbs / peak}}
        tr = os.path.join(ROOT, "profiles", "traffic.csv")      # ncu dram__bytes_{read,write}.sum per launch
        if os.path.exists(tr):
            import csv
            with open(tr) as f:
                for row in csv.DictReader(f):
                    if row["workload"] == w.name and row["pass"] == top:
                        roofline["traffic"] = int(row["dram_read_bytes"]) + int(row["dram_write_bytes"])
                        roofline["traffic_source"] = row["source"]

        # ---- CPU baseline: the oracle on this box's cores, bounded sample ----
        cpu = None
        if not args.no_cpu_baseline and world == 1:
            from oracle import binding as ob
            ob.build()
            small = shrunk(w, 64)
            t1, threads = oracle_time(small, 1)
            est_full = t1 * w.npoints / small.npoints          # seconds per full-grid oracle step
            ws = w if est_full < 40 else shrunk(w, max(w.nx, w.ny, w.nz) // 2)
            est = est_full * ws.npoints / w.npoints
            nsteps = int(min(5, max(1, round(20.0 / max(est, 1e-3)))))
            sec, threads = oracle_time(ws, nsteps)
            cpu = {"value": ws.npoints / sec, "unit": UNIT, "cores": threads, "kind": "oracle",
                   "ms_per_step": sec * 1e3,
                   "sample": f"{nsteps} oracle steps of {w.name} on a {ws.nx}x{ws.ny}x{ws.nz} grid"}

        sampler.close()
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "config": {"workload": w.name, "grid": [w.nx, w.ny, w.nz], "mode": "real" if w.time_mode else "imag",
                           "psi": "complex128", "parallelism": f"replicas x{world}",
                           "l2": f"psi is {16 * w.npoints / 2**20:.0f} MiB per field (L2 126 MB); no flush between steps",
                           "G": w.G_run, "D": w.D_run, "dt": w.dt},
                "clocks": sampler.summary(),
                "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": 16 * w.npoints,
                        "d2h_bytes_per_step": 16 * w.npoints, "steps": e2e_steps},
                "gpu_launches": launches,
                "roofline": roofline,
                "cpu_baseline": cpu,
                "observables_after_run": obs}
    sim.close()
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if line:
        print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=500)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--workload", default="C4", choices=["C1", "C2", "C3", "C4", "C5"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    w = workload(args.workload)
    if args.impl == "reference":
        run_reference(args, w)
    else:
        run_ours(args, w)


if __name__ == "__main__":
    main()
