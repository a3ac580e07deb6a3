#!/usr/bin/env python
"""bench.py — the LLG hot path on BASELINE.json's 3-D slab (configs[3]): one step = one fixed-dt
Dormand-Prince step (7 RHS evaluations: demag FFT convolution + local field + torque + RK stage
algebra) of a 512x512x16 mesh.  Metric: cell-updates/s per RHS evaluation = N * 7 * steps / seconds.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--prec f32|f64|both] [--workload cfg4|cfg5_<n>]
  python bench.py --impl reference ...      # the CPU oracle on a bounded sample of the same workload

One JSON line.  Its top-level fields are the fp32 run (the arithmetic the paper's throughput figure is quoted in,
PAPER.md:495); with --prec both (the default) the same line carries an "fp64" object with the fp64 run's value,
ms_per_step, roofline and e2e.  N > 1: independent replicas, one per GPU, no data-path collective ("replicas
only"); value = cells all ranks processed / max-over-ranks time.  Started without torchrun,
`--gpus N` launches the N ranks itself (torch.distributed.run on 127.0.0.1).
"""
import argparse
import csv
import ctypes
import json
import os
import socket
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "cell_updates_per_sec_per_rhs_eval"
UNIT = "cell-updates/s"
RHS_PER_STEP = 7
CLASSES = ["fwd_xz", "y_conv", "inv_zx", "llg_stage"]
TRAFFIC_CSV = os.path.join(ROOT, "profiles", "ncu_traffic.csv")


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured"
        except Exception:
            pass
    return 6650.0, "fallback"


def ncu_traffic(version, workload, prec, cls):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of kernel class `cls`, from the committed table of
    `ncu --set full` captures (profiles/ncu_traffic.csv).  A row counts only if it was captured from THIS library
    version (mm_version()), workload and precision; otherwise None — a stale capture is not a measurement."""
    try:
        with open(TRAFFIC_CSV) as f:
            for row in csv.DictReader(r for r in f if not r.startswith("#")):
                if (row["mm_version"], row["workload"], row["prec"], row["class"]) == (version, workload, prec, cls):
                    return float(row["dram_read_bytes"]) + float(row["dram_write_bytes"])
    except Exception:
        pass
    return None


def get_workload(name):
    from paper_2406_16064_b200 import workloads as wl
    if name == "cfg4":
        return wl.cfg4()
    if name.startswith("cfg4_"):
        nx, ny, nz = (int(v) for v in name.split("_")[1].split("x"))
        return wl.cfg4(nx, ny, nz)
    if name.startswith("cfg5_"):
        return wl.cfg5(int(name.split("_")[1]))
    raise SystemExit(f"unknown workload {name}")


class ClockSampler:
    """SM clock and throttle reasons of one GPU, polled through NVML every ~5 ms with a timestamp per sample
    (nvidia-smi -lms as the fallback), so that the samples inside the timed region can be picked out."""

    REASONS = {"hw_slowdown": 0x8, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20, "sw_power_cap": 0x4}

    def __init__(self, index):
        self.index, self.rows, self.stop_flag, self.th, self.mode = index, [], False, None, None

    def start(self):
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.mode = "nvml"
            self.th = threading.Thread(target=self._poll_nvml, daemon=True)
            self.th.start()
            return
        except Exception:
            self.mode = None
        q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={q}", "--format=csv,noheader,nounits", "-lms", "20",
                                          "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.mode = "smi"
            self.th = threading.Thread(target=self._read_smi, daemon=True)
            self.th.start()
        except Exception:
            self.mode = None

    def _poll_nvml(self):
        nv = self.nv
        while not self.stop_flag:
            try:
                mhz = float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    mask = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                except Exception:
                    mask = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                self.rows.append((time.perf_counter(), mhz, self.max_mhz, mask))
            except Exception:
                pass
            time.sleep(0.004)

    def _read_smi(self):
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.proc.stdout:
            r = [c.strip() for c in line.split(",")]
            try:
                mask = 0
                for n, v in zip(names, r[2:6]):
                    if v.lower().startswith("active"):
                        mask |= self.REASONS[n]
                self.rows.append((time.perf_counter(), float(r[0]), float(r[1]), mask))
            except Exception:
                pass

    def stop(self, t0=None, t1=None):
        """Summary of the samples with t0 <= timestamp <= t1 (all samples when the window holds none)."""
        self.stop_flag = True
        if self.mode == "smi":
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except Exception:
                self.proc.kill()
        if self.th is not None:
            self.th.join(timeout=1)
        if not self.mode:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["clock sampling unavailable"], "samples": 0}
        rows = [r for r in self.rows if t0 is None or (t0 <= r[0] <= t1)]
        window = "timed region"
        if not rows:
            rows, window = list(self.rows), "whole run (no sample fell inside the timed region)"
        sm = sorted(r[1] for r in rows)
        mask = 0
        for r in rows:
            mask |= r[3]
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max((r[2] for r in rows), default=None),
                "reasons": sorted(n for n, b in self.REASONS.items() if mask & b), "samples": len(sm), "window": window,
                "source": self.mode}


def aggregate_over_ranks(local_seconds, local_units, device=None):
    """max-over-ranks time and summed units; works with gloo (CPU) and nccl."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return local_seconds, local_units
    t = torch.tensor([local_seconds], dtype=torch.float64, device=device)
    u = torch.tensor([float(local_units)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def algorithmic_bytes(w, esize):
    """per RHS 39 N s (film) / 89 N s (3-D); DOPRI5 step = 7 RHS + 102 N s.
    Per kernel class (units of N s): pass B is SURVEY's "last forward + multiply + first inverse (+K^)" row,
    16 (film) / 30 (3-D); this build does z inside the x passes, so A = 4 + 6 / 4 + 12 and C = 6 + 3 / 12 + 3
    (DESIGN.md §5); the stage kernel reads H_d, m, Ms and writes k: 13, and a DOPRI5 stage s also reads the s earlier
    k_j (3 each), reads m0 and writes the next stage's input (3 + 3, stages that have one): over the seven launches of a
    step that is SURVEY's 102 = 3 (0+1+...+6) + 18 + 18 + 3 extra N s, so the AVERAGE stage launch moves (7*13 + 99)/7 =
    27.1 N s — the figure the per-class time (an average over all stage launches) is divided into."""
    N = w.N
    three_d = w.nz > 1
    per_class = {"fwd_xz": 16 if three_d else 10, "y_conv": 30 if three_d else 16, "inv_zx": 15 if three_d else 9, "llg_stage": (7 * 13 + 99) / 7.0}
    return {"rhs": (89 if three_d else 39) * N * esize, "step": (7 * (89 if three_d else 39) + 102) * N * esize,
            "class": {k: v * N * esize for k, v in per_class.items()}}


# ------------------------------------------------------------------------------------------------------------
# CPU legs: the oracle, as it stands, on the host cores
# ------------------------------------------------------------------------------------------------------------
def omp_set_threads(n):
    """Thread count of the oracle's OpenMP loops for the calls that follow (the runtime libmo.so is linked with)."""
    try:
        ctypes.CDLL("libgomp.so.1").omp_set_num_threads(int(n))
        return True
    except Exception:
        return False


def oracle_sample(w, shrink=0):
    """Bounded sample of the workload for the reference arm: same cells/material, fewer cells (shrink halves the
    in-plane size again)."""
    from paper_2406_16064_b200 import workloads as wl
    if w.nz > 1:
        n = max(16, 64 >> shrink)
        return wl.cfg4(n, n, w.nz)
    n = max(16, min(w.nx, 256) >> shrink)
    return wl.cfg5(n)


def time_oracle(ws, steps, warmup, per_step_rhs):
    import numpy as np
    import oracle
    from paper_2406_16064_b200 import workloads as wl
    o = oracle.Oracle(ws.nx, ws.ny, ws.nz, ws.dx, ws.dy, ws.dz)
    wl.apply(o, ws)
    m = np.ascontiguousarray(ws.m0)
    o.llg_rhs(m)                       # builds the cached spectrum (setup, untimed)
    for _ in range(warmup):
        for _ in range(per_step_rhs):
            o.llg_rhs(m)
    t0 = time.perf_counter()
    for _ in range(steps):
        if per_step_rhs == RHS_PER_STEP:
            o.step(m, ws.dt)
        else:
            o.llg_rhs(m)
    dt = time.perf_counter() - t0
    return dt, ws.N * per_step_rhs * steps


def cpu_baseline_full_mesh(w):
    """BASELINE.md's plan: the oracle's FFT-path RHS on the benchmark's OWN mesh (no sub-mesh), one evaluation with
    all host cores and one with a single thread.  `value` is the all-cores figure."""
    import numpy as np
    import oracle
    from paper_2406_16064_b200 import workloads as wl
    cores = os.cpu_count()
    t_setup = time.perf_counter()
    o = oracle.Oracle(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz)
    wl.apply(o, w)
    m = np.ascontiguousarray(w.m0)
    o.llg_rhs(m)                       # first call: builds the cached spectrum (setup, untimed) and warms up
    t_setup = time.perf_counter() - t_setup
    t0 = time.perf_counter()
    o.llg_rhs(m)
    t_all = time.perf_counter() - t0
    one = None
    # single thread only when it stays a bounded sample (~30 s): estimated from the all-cores time
    if omp_set_threads(1) and t_all * cores <= 60.0:
        t0 = time.perf_counter()
        o.llg_rhs(m)
        one = time.perf_counter() - t0
    omp_set_threads(cores)
    out = {"value": w.N / t_all, "unit": UNIT, "cores": cores, "kind": "oracle",
           "sample": f"1 RHS evaluation (oracle FFT path, fp64) on the full {w.nx}x{w.ny}x{w.nz} mesh, all {cores} host cores; "
                     f"setup (quad-precision tensor + spectrum) {t_setup:.1f} s untimed",
           "seconds_per_rhs": t_all}
    if one is not None:
        out["single_thread"] = {"value": w.N / one, "unit": UNIT, "cores": 1, "seconds_per_rhs": one}
    return out


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w = get_workload(args.workload)
    cores = os.cpu_count()
    # bound the whole run to a few minutes on whatever host this is: one probe step decides the sample size
    budget = float(os.environ.get("MM_REF_BUDGET_S", "150"))
    for shrink in range(3):
        ws = oracle_sample(w, shrink)
        probe, _ = time_oracle(ws, 1, 0, RHS_PER_STEP)
        if probe * (args.steps + args.warmup) <= budget or shrink == 2:
            break
    sec, units = time_oracle(ws, args.steps, args.warmup, RHS_PER_STEP)
    value = units / sec
    sample = f"{ws.nx}x{ws.ny}x{ws.nz} sub-mesh of the workload (same cells and material), {args.steps} DOPRI5 steps"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * sec / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "sample": sample, "integrator": "dopri5_fixed_dt", "rhs_per_step": RHS_PER_STEP},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------------------
# The CUDA path
# ------------------------------------------------------------------------------------------------------------
def measure(args, w, prec_name, rank, world, local, barrier, dev, sample_clocks):
    """One precision: warm-up, K timed steps (device events, max over ranks), a profiled pass for the per-kernel
    times, and the end-to-end leg through mm_run_host.  Returns the fields of the JSON line for this precision."""
    import numpy as np
    import torch
    from paper_2406_16064_b200 import Sim, F32, F64, workloads as wl
    from paper_2406_16064_b200.binding import load_library

    prec = F64 if prec_name == "f64" else F32
    esize = 8 if prec == F64 else 4
    s = Sim(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, prec=prec, device=local)
    wl.apply(s, w)
    dm = s.to_device(w.m0)
    host_m = torch.from_numpy(np.ascontiguousarray(w.m0)).to(s.dtype).pin_memory()
    warm = max(args.warmup, 3)

    # which kernel class dominates: every class bracketed by events over the warm-up steps
    s.set_profiling(True)
    for _ in range(warm):
        s.step(dm, w.dt, sync=False)
    barrier()
    warm_ms, warm_cnt = s.get_profile()
    dom = max(range(4), key=lambda i: warm_ms[i])
    # Timed region: K steps through the public call exactly as a user issues them — no events inside, so the library
    # replays each step as one captured CUDA graph (its default path; two untimed steps first: eager + capture).
    s.set_profiling(0)
    for _ in range(2):
        s.step(dm, w.dt, sync=False)
    sampler = ClockSampler(local) if sample_clocks else None
    if sampler:
        sampler.start()
        time.sleep(0.02)
    l0 = s.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    t_host0 = time.perf_counter()
    e0.record()
    for _ in range(args.steps):
        s.step(dm, w.dt, sync=False)
    e1.record()
    barrier()
    sec = e0.elapsed_time(e1) * 1e-3
    launches = s.launch_count() - l0

    # Kernel-time region, directly after it: the same K steps with the dominant class bracketed by CUDA events on the
    # library's stream (events switch the graph off: kernel-by-kernel launches; 2 stream operations per bracketed
    # kernel).  --no-kernel-events skips it (the dominant kernel's time then comes from the warm-up profile).
    if args.no_kernel_events:
        dom_ms, dom_cnt, ev_sec = warm_ms, warm_cnt, None
    else:
        s.set_profiling(2 << dom)
        v0, v1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        v0.record()
        for _ in range(args.steps):
            s.step(dm, w.dt, sync=False)
        v1.record()
        barrier()
        ev_sec = v0.elapsed_time(v1) * 1e-3
        dom_ms, dom_cnt = s.get_profile()
    t_host1 = time.perf_counter()
    clocks = sampler.stop(t_host0, t_host1) if sampler else None
    assert bool(torch.isfinite(dm).all()), "non-finite magnetisation after the timed region"

    # per-kernel times of every class: a separate profiled pass over the same number of steps (not part of `value`)
    s.set_profiling(True)
    for _ in range(min(args.steps, 20)):
        s.step(dm, w.dt, sync=False)
    barrier()
    prof_ms, prof_cnt = s.get_profile()
    s.set_profiling(False)

    # end to end: host buffers through the C ABI, H2D + step + D2H inside the timed region
    e2e_steps = max(1, min(args.steps, 5))
    s.run_host(host_m, 1, w.dt)
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        s.run_host(host_m, 1, w.dt)
    torch.cuda.synchronize()
    e2e_sec = time.perf_counter() - t0

    # sustained: the run length BASELINE.json configs[3] specifies (1000 fixed-dt steps), with the clocks of that window
    sus = None
    if args.sustained_steps > 0:
        sus_sampler = ClockSampler(local) if sample_clocks else None
        if sus_sampler:
            sus_sampler.start()
            time.sleep(0.02)
        u0, u1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        th0 = time.perf_counter()
        u0.record()
        for _ in range(args.sustained_steps):
            s.step(dm, w.dt, sync=False)
        u1.record()
        barrier()
        th1 = time.perf_counter()
        sus_sec, sus_units = aggregate_over_ranks(u0.elapsed_time(u1) * 1e-3, w.N * RHS_PER_STEP * args.sustained_steps, dev)
        sus = {"steps": args.sustained_steps, "seconds": sus_sec, "units": sus_units, "clocks": sus_sampler.stop(th0, th1) if sus_sampler else None}
        assert bool(torch.isfinite(dm).all()), "non-finite magnetisation after the sustained run"

    units = w.N * RHS_PER_STEP * args.steps
    ev_max = aggregate_over_ranks(ev_sec, units, dev)[0] if ev_sec is not None else None
    sec_max, units_all = aggregate_over_ranks(sec, units, dev)
    e2e_max, e2e_units = aggregate_over_ranks(e2e_sec, w.N * RHS_PER_STEP * e2e_steps, dev)
    version = load_library().mm_version().decode()
    del s, dm
    torch.cuda.empty_cache()
    if rank != 0:
        return None
    peak, peak_kind = measured_peaks()
    ab = algorithmic_bytes(w, esize)
    per = {n: (prof_ms[i] / prof_cnt[i] if prof_cnt[i] else None) for i, n in enumerate(CLASSES)}
    dom_name = CLASSES[dom]
    dom_avg = dom_ms[dom] / dom_cnt[dom]      # the dominant kernel's average launch, measured inside the timed region
    per[dom_name] = dom_avg
    dom_bytes = ab["class"][dom_name]
    achieved = dom_bytes / (dom_avg * 1e-3) / 1e9
    step_gbs = ab["step"] * args.steps / sec / 1e9
    tot = sum(prof_ms)
    if sus is not None:
        sus_gbs = ab["step"] * sus["steps"] / sus["seconds"] / 1e9
        sus = {"steps": sus["steps"], "value": sus["units"] / sus["seconds"], "unit": UNIT, "ms_per_step": 1e3 * sus["seconds"] / sus["steps"],
               "seconds": sus["seconds"], "step_frac": sus_gbs / peak, "step_frac_nominal_8TBs": sus_gbs / 8000.0, "clocks": sus["clocks"],
               "note": "BASELINE.json configs[3]'s own run length (fixed-dt DOPRI5 steps, one CUDA graph launch each), timed with CUDA events "
                       "after the short region above; reported beside `value`, not instead of it"}
    return {
        "sustained": sus,
        "value": units_all / sec_max, "ms_per_step": 1e3 * sec_max / args.steps, "dtype": prec_name,
        "e2e": {"value": e2e_units / e2e_max, "unit": UNIT, "h2d_bytes_per_step": 3 * w.N * esize, "d2h_bytes_per_step": 3 * w.N * esize,
                "api": "mm_run_host (pinned host m in, one DOPRI5 step, m out)"},
        "gpu_launches": launches, "clocks": clocks,
        "events_region": (None if ev_max is None else
                          {"value": units_all / ev_max, "ms_per_step": 1e3 * ev_max / args.steps, "unit": UNIT,
                           "note": "the same K steps directly after the timed region with the dominant kernel bracketed by CUDA events "
                                   "(kernel-by-kernel launches instead of the step graph): where roofline.avg_launch_ms is measured"}),
        "roofline": {"bound": "hbm", "kernel": dom_name, "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "peak_kind": peak_kind, "traffic": ncu_traffic(version, w.name, prec_name, dom_name),
                     "traffic_source": "profiles/ncu_traffic.csv row of this mm_version / workload / precision, else null",
                     "algorithmic_bytes_per_launch": dom_bytes, "avg_launch_ms": dom_avg, "kernel_ms": per,
                     "kernel_frac": {n: (ab["class"][n] / (per[n] * 1e-3) / 1e9 / peak if per[n] else None) for n in CLASSES},
                     "kernel_share": {n: prof_ms[i] / tot for i, n in enumerate(CLASSES)},
                     "kernel_ms_source": (f"{dom_name}: CUDA events over the warm-up steps (--no-kernel-events)" if args.no_kernel_events else
                                          f"{dom_name}: CUDA events around every launch of it in the K steps that directly follow the timed region "
                                          "(events_region; the timed region itself runs each step as one CUDA graph launch)") +
                                         "; the other classes and kernel_share: a profiled pass of the same steps after it (all classes bracketed)",
                     "step_algorithmic_gbs": step_gbs, "step_frac": step_gbs / peak, "step_frac_nominal_8TBs": step_gbs / 8000.0,
                     "mm_version": version},
    }


def film_point(n, prec_name, local, steps=15, warm=3):
    """One point of BASELINE.json configs[4] (N x N x 1 film, demag + exchange + Zeeman): `steps` fixed-dt DOPRI5 steps
    (15 steps = 105 RHS evaluations; configs[4] asks for 100) timed with CUDA events as one graph launch per step, then a
    profiled pass for the per-kernel averages.  Fractions are against the measured HBM peak with the film byte model
    of SURVEY 8(d) — for N = 1024 the working set (about 45 MB in fp32) fits the 126 MB L2, so that point is not HBM-bound
    by construction and its fraction is a comparison figure only."""
    import torch
    from paper_2406_16064_b200 import Sim, F32, F64, workloads as wl
    w = wl.cfg5(n)
    prec = F64 if prec_name == "f64" else F32
    esize = 8 if prec == F64 else 4
    s = Sim(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, prec=prec, device=local)
    wl.apply(s, w)
    dm = s.to_device(w.m0)
    for _ in range(warm + 2):
        s.step(dm, w.dt, sync=False)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(steps):
        s.step(dm, w.dt, sync=False)
    e1.record()
    torch.cuda.synchronize()
    sec = e0.elapsed_time(e1) * 1e-3
    s.set_profiling(True)
    for _ in range(5):
        s.step(dm, w.dt, sync=False)
    torch.cuda.synchronize()
    ms, cnt = s.get_profile()
    s.set_profiling(False)
    assert bool(torch.isfinite(dm).all())
    del s, dm
    torch.cuda.empty_cache()
    peak, _ = measured_peaks()
    ab = algorithmic_bytes(w, esize)
    per = {c: ms[i] / cnt[i] for i, c in enumerate(CLASSES) if cnt[i]}
    frac = {c: ab["class"][c] / (per[c] * 1e-3) / 1e9 / peak for c in per}
    dom = max(per, key=lambda c: per[c] * cnt[CLASSES.index(c)])
    weakest = min(frac, key=frac.get)
    gbs = ab["step"] * steps / sec / 1e9
    return {"n": n, "dtype": prec_name, "value": w.N * RHS_PER_STEP * steps / sec, "unit": UNIT, "ms_per_step": 1e3 * sec / steps,
            "us_per_rhs": 1e6 * sec / steps / RHS_PER_STEP, "step_frac": gbs / peak, "step_frac_nominal_8TBs": gbs / 8000.0,
            "kernel": dom, "frac": frac[dom], "weakest_kernel": weakest, "weakest_frac": frac[weakest],
            "kernel_us": {c: 1e3 * v for c, v in per.items()}, "kernel_frac": frac}


def run_mm(args):
    import torch
    import torch.distributed as dist

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device("cuda", local))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    w = get_workload(args.workload)
    w.seed += rank

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    precs = ["f32", "f64"] if args.prec == "both" else [args.prec]
    res = {p: measure(args, w, p, rank, world, local, barrier, dev, sample_clocks=(rank == 0)) for p in precs}
    if rank == 0:
        top = res[precs[0]]
        cpu = None
        if not args.no_cpu_baseline:
            cpu = cpu_baseline_full_mesh(w)
        line = {
            "metric": METRIC, "value": top["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": top["ms_per_step"], "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": top["dtype"], "data": "synthetic",
            "config": {"workload": w.name, "mesh": [w.nx, w.ny, w.nz], "integrator": "dopri5_fixed_dt", "dt": w.dt,
                       "rhs_per_step": RHS_PER_STEP, "parallelism": f"replicas x{world}",
                       "l2": "working set (spectra + stage vectors > 1 GB) exceeds the 126 MB L2; no explicit flush",
                       "launch": "each step = one CUDA graph launch of the step's kernels (the library's default path)"},
            "e2e": top["e2e"], "gpu_launches": top["gpu_launches"], "clocks": top["clocks"], "roofline": top["roofline"],
            "events_region": top["events_region"],
            "cpu_baseline": cpu,
        }
        line["sustained"] = top["sustained"]
        if len(precs) > 1:
            o = res["f64"]
            line["fp64"] = {k: o[k] for k in ("value", "ms_per_step", "dtype", "e2e", "gpu_launches", "clocks", "roofline", "events_region", "sustained")}
            line["fp64"]["unit"] = UNIT
        if args.films and world == 1 and args.workload == "cfg4":
            # BASELINE.json configs[4], the paper's own throughput shape: the weakest numbers of this build
            line["films"] = [film_point(n, p, local) for n in (1024, 4096) for p in precs]
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="mm", choices=["mm", "reference"])
    ap.add_argument("--prec", default="both", choices=["f32", "f64", "both"])
    ap.add_argument("--workload", default="cfg4")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-kernel-events", action="store_true", help="no CUDA events inside the timed region (whole-step CUDA graphs stay on)")
    ap.add_argument("--sustained-steps", type=int, default=1000, help="length of the `sustained` leg (configs[3]: 1000 steps); 0 skips it")
    ap.add_argument("--no-films", dest="films", action="store_false", help="skip the N x N x 1 film points (configs[4]) of the default line")
    args = ap.parse_args()
    world_env = os.environ.get("WORLD_SIZE")
    if world_env is None and args.gpus > 1:
        # not under torchrun: start the N ranks ourselves, one process per GPU
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", str(free_port()), os.path.abspath(__file__)] + sys.argv[1:]
        raise SystemExit(subprocess.run(cmd).returncode)
    if world_env is not None and int(world_env) != args.gpus:
        print(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world_env}: launch one rank per GPU", file=sys.stderr)
        raise SystemExit(2)
    if args.impl == "reference":
        run_reference(args)
    else:
        run_mm(args)


if __name__ == "__main__":
    main()
