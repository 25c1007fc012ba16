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

Beside the headline the line carries `configs` (all five BASELINE.json workloads: ms/step, updates/s, model
fraction, dominant kernel and its roofline fraction — `north_star` asks for the five), `observables` (one
calcmuen + calcrms evaluation, excluded from the step and reported separately) and `batch`
(dbec_create_batch: many small grids per launch against one of them alone).

`--impl reference` times the oracle (oracle/, as it stands) on the host cores, rank 0 only; `config.workload`
names the grid it really ran.
"""
from __future__ import annotations

import argparse
import datetime
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
    # the whole step of a small grid in one launch (kernels_small.cu): the fused pipeline's bytes per point,
    # filled in per workload by alg_bytes() — the data never leaves L2, so its HBM fraction only says how far
    # from a streaming grid the small one runs
    "sscn_step<cluster>": None,
}
MODEL_BYTES_PER_POINT = {3: 208, 2: 144}    # SURVEY.md §8(d) "Model M": fixed reference accounting
# What this repository's fused pipeline itself has to stream (x sweep inside the nonlinear kernel): the honest
# denominator beside M.
FUSED_BYTES_PER_POINT = {3: 176, 2: 112}
# One calcmuen + calcrms evaluation (reported separately): the forward passes and the spectral
# multiply as in a step, the last inverse writing Phi (8 + 8), the reduction pass reading psi and Phi (16 + 8).
OBS_BYTES_PER_POINT = {3: 24 + 16 + 16 + 16 + 16 + 24, 2: 24 + 16 + 16 + 24}
REF_BUDGET_S = 240.0                        # --impl reference: whole run (K + W oracle steps)


def alg_bytes(name, w):
    b = ALG_BYTES_PER_POINT[name]
    return FUSED_BYTES_PER_POINT[w.ndim] if b is None else b


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clock / throttle-reason samples.  Each line is stamped by nvidia-smi itself (`timestamp`
    field), so that the window [mark_start, mark_stop] selects the samples taken while the timed region ran,
    however late Python reads them from the pipe.  No fall-back to samples outside the window."""
    Q = ("timestamp,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows = []
        self.t0 = self.t1 = None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "20"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True, bufsize=1)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    @staticmethod
    def _stamp(text):
        try:
            return datetime.datetime.strptime(text.strip(), "%Y/%m/%d %H:%M:%S.%f").timestamp()
        except ValueError:
            return None

    def _read(self):
        for line in self.proc.stdout:
            f = [x.strip() for x in line.split(",")]
            t = self._stamp(f[0]) if f else None
            if t is not None and len(f) >= 8:
                self.rows.append((t, f))

    def mark_start(self):
        self.t0 = time.time()

    def mark_stop(self):
        self.t1 = time.time()

    def close(self):
        if self.proc:
            time.sleep(0.1)
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except Exception:
                self.proc.kill()

    def in_window(self):
        if self.t0 is None or self.t1 is None:
            return []
        return [f for t, f in self.rows if self.t0 <= t <= self.t1]

    def summary(self, note=""):
        sm, smax, reasons = [], [], set()
        for f in self.in_window():
            try:
                sm.append(float(f[1]))
                smax.append(float(f[2]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[4:8]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        out = {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": float(max(smax)) if smax else None,
               "reasons": sorted(reasons), "samples": len(sm),
               "window_s": None if self.t0 is None or self.t1 is None else self.t1 - self.t0}
        if note:
            out["window"] = note
        return out


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
    """The reference arm: the oracle on the host cores.  Each step is one oracle SSCN step of the named
    workload; if K + W steps of the full grid would take longer than REF_BUDGET_S, the grid is coarsened
    (same box and parameters) and `config.workload` / `config.grid` name the grid that really ran."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import binding as ob
    ob.build()
    probe = shrunk(w, 32)
    t_probe, threads = oracle_time(probe, 2)
    per_point = t_probe / probe.npoints
    n = max(w.nx, w.ny, w.nz)
    while n > 32 and per_point * shrunk(w, n).npoints * (args.steps + args.warmup) * 1.3 > REF_BUDGET_S:
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
    full = ws.npoints == w.npoints
    name = w.name if full else f"{w.name} coarsened to {ws.nx}x{ws.ny}x{ws.nz}"
    sample = (f"{args.steps} oracle steps on the full {ws.nx}x{ws.ny}x{ws.nz} grid" if full else
              f"{args.steps} oracle steps on a {ws.nx}x{ws.ny}x{ws.nz} grid of the same box and parameters "
              f"(1/{w.npoints // ws.npoints} of the {w.name} grid points: {args.steps + args.warmup} full-grid steps "
              f"would exceed the {REF_BUDGET_S:.0f} s budget)")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": name, "grid": [ws.nx, ws.ny, ws.nz], "named_grid": [w.nx, w.ny, w.nz],
                       "full_grid": full, "mode": "real" if w.time_mode else "imag"},
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


def timed_steps(torch, sim, steps):
    """Milliseconds for `steps` steps: CUDA events on the library's own stream, synchronised on both sides."""
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sim.synchronize()
    e0.record(sim.stream)
    sim.step(steps)
    e1.record(sim.stream)
    sim.synchronize()
    return e0.elapsed_time(e1)


def kernel_profile(sim, w, steps, peak):
    """Per-pass average milliseconds (CUDA event pairs around every launch, dbec_step_profile) and the roofline
    fraction of each pass by its algorithmic bytes."""
    sim.step_profile(2)
    prof = sim.step_profile(steps)
    kernels = sim.pass_kernels()
    per_kernel = {}
    for name, (tot_ms, cnt) in prof.items():
        avg_ms = tot_ms / cnt
        gbs = alg_bytes(name, w) * w.npoints / (avg_ms * 1e-3) / 1e9
        per_kernel[name] = {"kernel": kernels.get(name, ""), "ms": avg_ms, "alg_GBps": gbs, "frac": gbs / peak}
    return per_kernel


def observables_ms(torch, sim, reps=3):
    """One dbec_observables call (calcmuen + calcrms: a dipolar pass, Phi written, one reduction pass)."""
    sim.observables()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sim.synchronize()
    e0.record(sim.stream)
    for _ in range(reps):
        sim.observables()
    e1.record(sim.stream)
    sim.synchronize()
    return e0.elapsed_time(e1) / reps


def measure_config(torch, dbec, key, dev, peak, steps=None):
    """ms/step, updates/s, model fraction and dominant kernel of one BASELINE.json workload."""
    w = workload(key)
    sim = dbec.Dbec(dbec.params_of(w), device=dev)
    sim.set_psi(initial_psi(w))
    if (w.G_run, w.D_run) != (w.G, w.D):
        sim.set_coupling(w.G_run, w.D_run)
    sim.step(5)
    if steps is None:
        est = timed_steps(torch, sim, 5) / 5
        steps = int(min(2000, max(20, 150.0 / max(est, 1e-3))))      # ~0.15 s of steps
    ms = timed_steps(torch, sim, steps) / steps
    per_kernel = kernel_profile(sim, w, 5, peak)
    top = max(per_kernel, key=lambda k: per_kernel[k]["ms"])
    obs_ms = observables_ms(torch, sim)
    sim.close()
    model, fused = MODEL_BYTES_PER_POINT[w.ndim], FUSED_BYTES_PER_POINT[w.ndim]
    gb = w.npoints / (ms * 1e-3) / 1e9
    return {"workload": w.name, "grid": [w.nx, w.ny, w.nz], "mode": "real" if w.time_mode else "imag", "steps": steps,
            "ms_per_step": ms, "updates_per_s": w.npoints / (ms * 1e-3),
            "step_model": {"bytes_per_point": model, "frac": model * gb / peak},
            "fused_pipeline": {"bytes_per_point": fused, "frac": fused * gb / peak},
            "top_kernel": {"pass": top, "kernel": per_kernel[top]["kernel"], "ms": per_kernel[top]["ms"],
                           "frac": per_kernel[top]["frac"]},
            "field_MiB": 16 * w.npoints / 2 ** 20,
            "observables_ms": obs_ms}


def measure_batch(torch, dbec, key, nbatch, dev):
    """dbec_create_batch: nbatch members of workload `key` per launch against one member alone."""
    w = workload(key)
    psi0 = initial_psi(w)
    out = {}
    for nb in (1, nbatch):
        sim = dbec.Dbec(dbec.params_of(w), device=dev, nbatch=nb)
        sim.set_psi(psi0 if nb == 1 else np.broadcast_to(psi0, (nb,) + psi0.shape).copy())
        if (w.G_run, w.D_run) != (w.G, w.D):
            sim.set_coupling(w.G_run, w.D_run)
        sim.step(10)
        est = timed_steps(torch, sim, 10) / 10
        steps = int(min(2000, max(20, 100.0 / max(est, 1e-3))))
        ms = timed_steps(torch, sim, steps) / steps
        sim.close()
        out[nb] = {"ms_per_step": ms, "updates_per_s": nb * w.npoints / (ms * 1e-3)}
    return {"workload": w.name, "nbatch": nbatch, "single": out[1], "batched": out[nbatch],
            "throughput_ratio": out[nbatch]["updates_per_s"] / out[1]["updates_per_s"]}


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
    clock_note = "the timed region"
    if sampler and len(sampler.in_window()) < 3:
        # the region was too short for nvidia-smi's sampling period: keep the same load running for 0.5 s more
        # and report the clocks of that stretch (timing above is untouched)
        leg = max(args.steps, int(500.0 / max(ms / args.steps, 1e-3)))
        sampler.mark_start()
        sim.step(leg)
        sim.synchronize()
        sampler.mark_stop()
        clock_note = (f"{leg} further steps of the same workload right after the timed region "
                      f"(the region itself lasted {ms:.1f} ms, shorter than three sampling periods)")
    obs = sim.observables()

    # ---- end to end through the C ABI with host buffers ----
    # Every step's input comes from pinned host memory and its result goes back there, inside the timed region.
    # A single handle does this one copy after the other (`serial`).  The headline figure feeds the GPU the way a
    # serving loop would: three handles on three streams, dbec_set_psi_async / dbec_get_psi_async, so that the upload of
    # one step's input runs while another handle's result goes down (both directions of the host link busy) and
    # the steps hide behind the copies.  Every step is still one full upload, one dbec_step(1), one full download.
    e2e_steps = max(6, min(args.steps, 24)) // 3 * 3
    host_in = torch.from_numpy(psi0.copy()).pin_memory()
    NRING = 3                              # handles taking turns in the pipelined leg
    host_out = [torch.empty_like(host_in).pin_memory() for _ in range(NRING)]
    for _ in range(2):
        sim.set_psi(host_in.numpy())
        sim.step(1)
        sim.get_psi(host_out[0].numpy())
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        sim.set_psi(host_in.numpy())       # H2D of the step's input
        sim.step(1)
        sim.get_psi(host_out[0].numpy())   # D2H of the step's result (synchronises)
    barrier()
    e2e_serial_s = time.perf_counter() - t0
    e2e_serial = whole_job_value(w.npoints, e2e_steps, world, max_over_ranks(e2e_serial_s, world, dev))
    ref_out = host_out[0].clone()
    extra = [dbec.Dbec(dbec.params_of(w), device=dev) for _ in range(NRING - 1)]
    for s_ in extra:
        if (w.G_run, w.D_run) != (w.G, w.D):
            s_.set_coupling(w.G_run, w.D_run)
    ring = [sim] + extra

    def pipelined(nsteps):
        for i in range(nsteps):
            s_ = ring[i % NRING]
            if i >= NRING:
                s_.wait()                  # this handle's previous result has landed in its host buffer
            s_.set_psi_async(host_in)
            s_.step(1)
            s_.get_psi_async(host_out[i % NRING])
        for s_ in ring:
            s_.wait()

    pipelined(2 * NRING)
    assert all(torch.equal(h_, ref_out) for h_ in host_out), "pipelined e2e leg differs from the serial one"
    barrier()
    t0 = time.perf_counter()
    pipelined(e2e_steps)
    barrier()
    e2e_s = time.perf_counter() - t0
    e2e_value = whole_job_value(w.npoints, e2e_steps, world, max_over_ranks(e2e_s, world, dev))
    for s_ in extra:
        s_.close()
    del extra, ring

    # ---- per-kernel roofline (rank 0) ----
    line = None
    if rank == 0:
        sim.set_psi(psi0)
        peak, peak_src = measured_peaks()
        per_kernel = kernel_profile(sim, w, max(5, min(args.steps, 50)), peak)
        top = max(per_kernel, key=lambda k: per_kernel[k]["ms"])
        step_ms_prof = sum(v["ms"] for v in per_kernel.values())
        model, fused = MODEL_BYTES_PER_POINT[w.ndim], FUSED_BYTES_PER_POINT[w.ndim]
        pts_per_ns = w.npoints / (ms / args.steps * 1e-3) / 1e9
        roofline = {"bound": "hbm", "kernel": per_kernel[top]["kernel"], "pass": top, "achieved": per_kernel[top]["alg_GBps"],
                    "peak": peak, "unit": "GB/s", "frac": per_kernel[top]["frac"], "traffic": None, "peak_source": peak_src,
                    "kernel_ms": per_kernel[top]["ms"], "kernel_share_of_step": per_kernel[top]["ms"] / step_ms_prof,
                    "alg_bytes_per_launch": alg_bytes(top, w) * w.npoints,
                    "per_kernel": per_kernel,
                    "step_model": {"bytes_per_point": model, "achieved_GBps": model * pts_per_ns, "frac": model * pts_per_ns / peak,
                                   "note": "SURVEY 8(d) fixed accounting M (counts an x sweep pass the fused kernels never make)"},
                    "fused_pipeline": {"bytes_per_point": fused, "achieved_GBps": fused * pts_per_ns,
                                       "frac": fused * pts_per_ns / peak,
                                       "note": "algorithmic bytes of this repository's own seven-pass pipeline"}}
        # the x-line kernel (inverse FFT-x + calcnu + calclux) is the one pass whose time is set by the fp64 pipe rather
        # than by memory; its HBM fraction is still what the step pays for it
        roofline["secondary"] = ("fp64 pipe: 63 DFMA/clk/SM measured (profiles/r2_fp64_probe.md); the x-line kernel runs at about "
                                 "55 % of it with 79 DP instructions per grid point (profiles/r2_step_ncu_full.md)")
        tr = os.path.join(ROOT, "profiles", "traffic.csv")      # ncu dram__bytes_{read,write}.sum per launch
        if os.path.exists(tr):
            import csv
            with open(tr) as f:
                for row in csv.DictReader(f):
                    if row["workload"] == w.name and row["pass"] == top:
                        roofline["traffic"] = int(row["dram_read_bytes"]) + int(row["dram_write_bytes"])
                        roofline["traffic_source"] = f'{row["source"]} (ncu capture of commit {row.get("commit", "?")})'
        obs_ms = observables_ms(torch, sim)
        observables = {"ms": obs_ms, "dram_alg_bytes": OBS_BYTES_PER_POINT[w.ndim] * w.npoints,
                       "alg_GBps": OBS_BYTES_PER_POINT[w.ndim] * w.npoints / (obs_ms * 1e-3) / 1e9,
                       "what": "one dbec_observables call (calcmuen + calcrms), excluded from ms_per_step"}
        sim.close()

        # ---- the five BASELINE.json workloads and the batched small grids (1 GPU only) ----
        configs, batch = None, None
        if world == 1 and not args.headline_only:
            configs = {}
            for key in ("C1", "C2", "C3", "C4", "C5"):
                if workload(key).name == w.name:
                    configs[key] = {"workload": w.name, "grid": [w.nx, w.ny, w.nz], "mode": "real" if w.time_mode else "imag",
                                    "steps": args.steps, "ms_per_step": ms / args.steps, "updates_per_s": value,
                                    "step_model": {"bytes_per_point": model, "frac": model * pts_per_ns / peak},
                                    "fused_pipeline": {"bytes_per_point": fused, "frac": fused * pts_per_ns / peak},
                                    "top_kernel": {"pass": top, "kernel": per_kernel[top]["kernel"], "ms": per_kernel[top]["ms"],
                                                   "frac": per_kernel[top]["frac"]},
                                    "field_MiB": 16 * w.npoints / 2 ** 20, "observables_ms": obs_ms}
                else:
                    configs[key] = measure_config(torch, dbec, key, dev, peak)
            batch = [measure_batch(torch, dbec, "C1", 64, dev), measure_batch(torch, dbec, "C2", 16, dev)]

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
                           "l2": (f"inputs larger than L2: psi is {16 * w.npoints / 2**20:.0f} MiB per field (L2 126 MB), "
                                  "every pass streams it; no flush between steps"
                                  if 16 * w.npoints > 126e6 else
                                  f"psi is {16 * w.npoints / 2**20:.1f} MiB: the working set is L2-resident by nature, no flush"),
                           "G": w.G_run, "D": w.D_run, "dt": w.dt},
                "clocks": sampler.summary(clock_note),
                "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": 16 * w.npoints,
                        "d2h_bytes_per_step": 16 * w.npoints, "steps": e2e_steps,
                        "how": "three handles on three streams taking turns, dbec_set_psi_async / dbec_step(1) / dbec_get_psi_async "
                               "per step from / to pinned host buffers: uploads overlap the other handles' downloads",
                        "serial": {"value": e2e_serial, "unit": UNIT,
                                   "how": "one handle: dbec_set_psi, dbec_step(1), dbec_get_psi one after the other"}},
                "gpu_launches": launches,
                "roofline": roofline,
                "cpu_baseline": cpu,
                "observables": observables,
                "configs": configs,
                "batch": batch,
                "observables_after_run": obs}
    else:
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
    ap.add_argument("--headline-only", action="store_true", help="skip the `configs` and `batch` entries")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    w = workload(args.workload)
    if args.impl == "reference":
        run_reference(args, w)
    else:
        run_ours(args, w)


if __name__ == "__main__":
    main()
