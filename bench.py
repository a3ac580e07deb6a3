#!/usr/bin/env python
"""bench.py — the LLG hot path on BASELINE.json's 3-D slab (configs[3]): one step = one fixed-dt
Dormand-Prince step (7 RHS evaluations: demag FFT convolution + local field + torque + RK stage
algebra) of a 512x512x16 mesh.  Metric: cell-updates/s per RHS evaluation = N * 7 * steps / seconds.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--prec f32|f64] [--workload cfg4|cfg5_<n>]
  python bench.py --impl reference ...      # the CPU oracle on a bounded sample of the same workload

N > 1 (torchrun): independent replicas, one per GPU, no data-path collective ("replicas only",
DESIGN.md); value = cells all ranks processed / max-over-ranks time.
"""
import argparse
import json
import os
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


# dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed `ncu --set full` capture
# (profiles/r01_ncu_full_v6.md); None where no capture of that kernel / workload / precision exists.
NCU_TRAFFIC = {("cfg4_slab_512x512x16", "f32", "y_conv"): 520.2e6 + 187.2e6,
               ("cfg4_slab_512x512x16", "f32", "fwd_xz"): 68.2e6 + 159.6e6,
               ("cfg4_slab_512x512x16", "f32", "inv_zx"): 202.9e6 + 31.4e6}


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured"
        except Exception:
            pass
    return 6650.0, "fallback"


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
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md)."""

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={q}", "--format=csv,noheader,nounits", "-lms", "100",
                                          "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
                for n, v in zip(names, r[2:6]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                pass
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


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
    Pass B ("last forward + multiply + first inverse"): 16 N s (film) / 30 N s (3-D)."""
    N = w.N
    three_d = w.nz > 1
    return {"rhs": (89 if three_d else 39) * N * esize, "step": (7 * (89 if three_d else 39) + 102) * N * esize,
            "passB": (30 if three_d else 16) * N * esize}


def oracle_sample(w, shrink=0):
    """Bounded sample of the workload for the CPU legs: same cells/material, fewer cells (shrink halves the
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


def run_mm(args):
    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_2406_16064_b200 import Sim, F32, F64, workloads as wl

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device("cuda", local))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    prec = F64 if args.prec == "f64" else F32
    esize = 8 if prec == F64 else 4
    w = get_workload(args.workload)
    w.seed += rank
    s = Sim(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, prec=prec, device=local)
    wl.apply(s, w)
    dm = s.to_device(w.m0)
    host_m = torch.from_numpy(np.ascontiguousarray(w.m0)).to(s.dtype).pin_memory()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # warm-up with every kernel class bracketed by events: per-class times, and which class dominates
    s.set_profiling(True)
    for _ in range(max(args.warmup, 3)):
        s.step(dm, w.dt, sync=False)
    barrier()
    warm_ms, warm_cnt = s.get_profile()
    dom = max(range(4), key=lambda i: warm_ms[i])
    # timed region: only the dominant class keeps its events (2 stream operations per bracketed kernel)
    s.set_profiling(2 << dom)
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    l0 = s.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        s.step(dm, w.dt, sync=False)
    e1.record()
    barrier()
    sec = e0.elapsed_time(e1) * 1e-3
    launches = s.launch_count() - l0
    prof_ms, prof_cnt = s.get_profile()
    s.set_profiling(False)
    clocks = sampler.stop() if rank == 0 else None
    assert bool(torch.isfinite(dm).all()), "non-finite magnetisation after the timed region"

    # end to end: host buffers through the C ABI, H2D + step + D2H inside the timed region
    e2e_steps = max(1, min(args.steps, 5))
    s.run_host(host_m, 1, w.dt)
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        s.run_host(host_m, 1, w.dt)
    torch.cuda.synchronize()
    e2e_sec = time.perf_counter() - t0

    units = w.N * RHS_PER_STEP * args.steps
    sec_max, units_all = aggregate_over_ranks(sec, units, dev)
    e2e_max, e2e_units = aggregate_over_ranks(e2e_sec, w.N * RHS_PER_STEP * e2e_steps, dev)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    peak, peak_kind = measured_peaks()
    ab = algorithmic_bytes(w, esize)
    names = ["fwd_xz", "y_conv", "inv_zx", "llg_stage"]
    # the dominant class is timed in the timed region, the others come from the warm-up steps
    per = {n: ((prof_ms[i] / prof_cnt[i]) if prof_cnt[i] else (warm_ms[i] / warm_cnt[i] if warm_cnt[i] else None)) for i, n in enumerate(names)}
    # algorithmic bytes of each kernel class per launch (units of N*s): SURVEY.md §8(d) rows
    three_d = w.nz > 1
    # y_conv is SURVEY's "last forward + multiply + first inverse (+K^)" row; the other rows are DESIGN.md §5's
    # (this build does z inside the x passes: A = 4 + 12 (film 4 + 6), C = 12 + 3 (film 6 + 3))
    alg_units = {"fwd_xz": 16 if three_d else 10, "y_conv": 30 if three_d else 16,
                 "inv_zx": 15 if three_d else 9, "llg_stage": 13}
    dom_name = names[dom]
    dom_bytes = alg_units[dom_name] * w.N * esize
    achieved = dom_bytes / (per[dom_name] * 1e-3) / 1e9
    step_gbs = ab["step"] * args.steps / sec / 1e9
    cpu = None
    if not args.no_cpu_baseline:
        ws = oracle_sample(w)
        csec, cunits = time_oracle(ws, 1, 0, 1)
        reps = 1
        while csec < 5.0 and reps < 64:
            reps *= 2
            csec, cunits = time_oracle(ws, reps, 0, 1)
        cpu = {"value": cunits / csec, "unit": UNIT, "cores": os.cpu_count(), "kind": "oracle",
               "sample": f"{reps} RHS evaluation(s) (oracle FFT path, fp64) on a {ws.nx}x{ws.ny}x{ws.nz} sub-mesh of the workload"}
    line = {
        "metric": METRIC, "value": units_all / sec_max, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": 1e3 * sec_max / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": args.prec, "data": "synthetic",
        "config": {"workload": w.name, "mesh": [w.nx, w.ny, w.nz], "integrator": "dopri5_fixed_dt", "dt": w.dt,
                   "rhs_per_step": RHS_PER_STEP, "parallelism": f"replicas x{world}",
                   "l2": "working set (spectra + stage vectors > 1 GB) exceeds the 126 MB L2; no explicit flush"},
        "e2e": {"value": e2e_units / e2e_max, "unit": UNIT, "h2d_bytes_per_step": 3 * w.N * esize, "d2h_bytes_per_step": 3 * w.N * esize,
                "api": "mm_run_host (pinned host m in, one DOPRI5 step, m out)"},
        "gpu_launches": launches,
        "clocks": clocks,
        "roofline": {"bound": "hbm", "kernel": dom_name, "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "peak_kind": peak_kind, "traffic": NCU_TRAFFIC.get((w.name, args.prec, dom_name)), "algorithmic_bytes_per_launch": dom_bytes,
                     "avg_launch_ms": per[dom_name], "kernel_ms": per,
                     "kernel_share": {n: warm_ms[i] / sum(warm_ms) for i, n in enumerate(names)},
                     "kernel_ms_source": f"{dom_name}: CUDA events in the timed region; other classes and kernel_share: the warm-up steps",
                     "step_algorithmic_gbs": step_gbs, "step_frac": step_gbs / peak,
                     "step_frac_nominal_8TBs": step_gbs / 8000.0},
        "cpu_baseline": cpu,
    }
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="mm", choices=["mm", "reference"])
    ap.add_argument("--prec", default="f32", choices=["f32", "f64"])
    ap.add_argument("--workload", default="cfg4")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_mm(args)


if __name__ == "__main__":
    main()
