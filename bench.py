#!/usr/bin/env python
"""bench.py -- throughput of the radiation-integral hot path on B200 (one JSON line on stdout).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg2|cfg1|cfg3|cfg4|cfg5]
    python bench.py --impl reference ...     # the CPU oracle on the host cores, same metric

A "step" is one pass of the whole hot path -- pack, main kernel, ordered reduction (SURVEY.md
section 8(a) rows a0-a7) -- over one synthetic batch: by default BASELINE.json configs[1]
(classical, 5 GeV planar-channeling positron, N = 14287 samples, 256 x 32 x 32 grid).
metric = FP64 radiation-integral evals/s (grid points x time steps), BASELINE.json `metric`.

  value      device-resident inputs, CUDA events on the launching stream, L2 flushed between steps
  e2e        same step through the C-ABI host-buffer call (pinned host memory, H2D + D2H inside)
  roofline   main kernel only: algorithmic flops (flops per eval x evals per launch)
             / its own event-timed duration, against the FP64 FMA peak measured in this run
  cpu_baseline  the CPU oracle (oracle/, double build of the same source) on a bounded sample

N > 1 (torchrun, one rank per GPU): each rank evaluates its own trajectory of the workload
(independent problems, no data-path collective; weak scaling); value = all ranks' evals / max time.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

METRIC = "fp64_radiation_integral_evals_per_s"
UNIT = "evals/s"
# algorithmic FP64 flops per eval, enumerated there operation by operation.
# Direct kernel: phase 2, exact range reduction 1 (+ one FRND beside the FP64 pipe), quarter-angle
# polynomials 21, two doublings 7, complex accumulation 8 [+4 for spin-1/2's J], integrand geometry
# 34 [37] per 8 omegas -> 43.25 [47.6] flops, 24.6 [26.9] FP64 instructions (SURVEY.md 8(d) estimated 52-60).
# The separable-phasor kernel needs far fewer: per eval one complex multiply (6) and
# the accumulation (8 [12]), plus per 16 [8] evals one T and one [half a] Y phasor and one [half an]
# integrand entry (36 + 35 + 28 [31] flops) -> 20.19 [26.63] flops, 11.75 [15.19] FP64 instructions.
# Both are checked against ncu's 2*DFMA + DMUL + DADD count (profiles/).
KERNELS = {1: "rad_main_kernel (direct phasor)", 2: "rad_sep_kernel (separable phasor)"}
FLOPS_PER_EVAL = {1: {0: 43.25, 1: 43.25, 2: 47.6}, 2: {0: 20.19, 1: 20.19, 2: 26.63}}
FP64_INSTR_PER_EVAL = {1: {0: 24.6, 1: 24.6, 2: 26.9}, 2: {0: 11.75, 1: 11.75, 2: 15.19}}
# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the main kernel, from the ncu --set full
# captures under profiles/ (r01_*_ncu_full.txt); bench.py cannot run ncu itself, other workloads report null.
NCU_TRAFFIC_BYTES = {("cfg2", 2): 1.256704e6 + 75.79136e6, ("cfg2", 1): 1.2224e6 + 8.14976e6,
                     ("cfg3", 2): 16.3904e6 + 10496.0, ("cfg3", 1): 16.240128e6 + 6144.0}
FP64_SPEC_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12      # 148 SM x 64 FMA lanes x 2 x 1.965 GHz


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["b200", "reference"], default="b200")
    ap.add_argument("--workload", default="cfg2")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cfg4-count", type=int, default=1000)
    ap.add_argument("--kernel", choices=["auto", "direct", "separable"], default="auto",
                    help="main kernel of the timed steps (auto: the library's own choice by grid shape)")
    ap.add_argument("--spin", choices=["0", "1/2"], default="1/2",
                    help="semi-classical variant of cfg3 / cfg5 (BASELINE.json configs[4] asks for both)")
    return ap.parse_args()


def make_workload(name: str, rank: int, cfg4_count: int, spin: str = "1/2"):
    import workloads
    model = workloads.SPIN0 if spin == "0" else workloads.SPIN_HALF
    if name == "cfg2":
        return workloads.make("cfg2", seed=2 + 1000 * rank)
    if name == "cfg1":
        return workloads.make("cfg1")
    if name == "cfg3":
        return workloads.make("cfg3", seed=3 + 1000 * rank, model=model)
    if name == "cfg4":
        return workloads.make("cfg4", count=cfg4_count, seed0=4000 + 100000 * rank)
    if name == "cfg5":
        return workloads.make("cfg5", seed=5 + 1000 * rank, model=model)
    raise SystemExit(f"unknown workload {name}")


# ----------------------------------------------------------------------------- clocks
class ClockSampler:
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""
    BAD = {"hw_slowdown": 0x8, "sw_thermal_slowdown": 0x20, "hw_thermal_slowdown": 0x40,
           "hw_power_brake_slowdown": 0x80}
    NOTED = {"sw_power_cap": 0x4}

    def __init__(self, index: int):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thread = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nv = None

    def _run(self):
        nv = self.nv
        while not self._stop.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                mask = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for name, bit in {**self.BAD, **self.NOTED}.items():
                    if mask & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            self._stop.wait(0.02)

    def __enter__(self):
        if self.nv is not None:
            self._thread = threading.Thread(target=self._run, daemon=True)
            self._thread.start()
        return self

    def __exit__(self, *exc):
        self._stop.set()
        if self._thread is not None:
            self._thread.join()

    def summary(self):
        return {"sm_mhz": float(np.median(self.samples)) if self.samples else None,
                "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


# ----------------------------------------------------------------------------- CPU oracle legs
def oracle_sample_rate(wl, n_points: int, variant: str, repeats: int = 1):
    """evals/s of the CPU oracle on a seeded subset of the workload's grid points."""
    import oracle
    import workloads
    idx = workloads.sample_points(wl, n_points, seed=777)
    w, nx, ny = workloads.points_of(wl, idx)
    best = None
    for _ in range(repeats):
        t0 = time.perf_counter()
        if wl.batch is not None:
            oracle.ensemble_points(wl.batch, wl.n, w, nx, ny, wl.model,
                                   wl.hbarc_over_E if wl.model else None, variant=variant)
            samples = int(np.sum(wl.n))
        else:
            oracle.points(wl.traj, w, nx, ny, wl.model, wl.hbarc_over_E, variant=variant)
            samples = len(wl.traj["t"])
        dt = time.perf_counter() - t0
        best = dt if best is None else min(best, dt)
    return len(idx) * samples / best, len(idx), best


def cpu_baseline(wl):
    import oracle
    samples = int(np.sum(wl.n)) if wl.batch is not None else len(wl.traj["t"])
    # size the sample for roughly 10-20 s of wall time on this box
    rate_guess = 2.0e7 * oracle.threads("f64")
    npts = int(min(wl.n_points, max(256, 12.0 * rate_guess / samples)))
    oracle_sample_rate(wl, min(npts, 512), "f64")                      # page in / warm up
    rate, got, secs = oracle_sample_rate(wl, npts, "f64")
    npts_ld = max(64, npts // 16)
    rate_ld, got_ld, secs_ld = oracle_sample_rate(wl, npts_ld, "ld")
    return {"value": rate, "unit": UNIT, "cores": oracle.threads("f64"), "kind": "oracle",
            "sample": (f"{got} seeded grid points x {samples} samples of {wl.name}, double build of "
                       f"oracle/rad_oracle.c (-O2, OpenMP), {secs:.1f} s; long-double build (the parity "
                       f"truth): {rate_ld:.3e} evals/s on {got_ld} points, {secs_ld:.1f} s"),
            "value_long_double": rate_ld}


def run_reference(args):
    """--impl reference: the CPU oracle as it stands (double build = the timed baseline of
    BASELINE.md section 3), on the host cores, bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import oracle
    oracle.build_all()
    wl = make_workload(args.workload, 0, min(args.cfg4_count, 8), args.spin)
    samples = int(np.sum(wl.n)) if wl.batch is not None else len(wl.traj["t"])
    cores = oracle.threads("f64")
    budget_s = 90.0 / max(1, args.steps + args.warmup)
    npts = int(min(wl.n_points, max(64, budget_s * 2.0e7 * cores / samples)))
    for _ in range(args.warmup):
        oracle_sample_rate(wl, npts, "f64")
    total_t = 0.0
    got = 0
    for _ in range(args.steps):
        _, got, dt = oracle_sample_rate(wl, npts, "f64")
        total_t += dt
    value = args.steps * got * samples / total_t
    sample = f"{got} seeded grid points x {samples} samples of {wl.name} per step, double build, OpenMP"
    line = {"metric": METRIC, "value": value, "unit": UNIT, "impl": "reference", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total_t / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": {"workload": wl.name, "sample_points_per_step": got},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


# ----------------------------------------------------------------------------- the B200 arm
def run_b200(args):
    import torch
    import torch.distributed as dist

    import paper_1910_10391_b200 as rad

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the CUDA path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    rad.build_library()
    rad.load_library()

    wl = make_workload(args.workload, rank, args.cfg4_count, args.spin)
    model, lam = wl.model, wl.hbarc_over_E
    grid = [torch.from_numpy(np.ascontiguousarray(a)).to(dev) for a in (wl.omega, wl.thx, wl.thy)]
    src = wl.batch if wl.batch is not None else wl.traj
    pinned = {k: torch.from_numpy(np.ascontiguousarray(v)).pin_memory() for k, v in src.items()}
    dtr = {k: v.to(dev) for k, v in pinned.items()}
    count = len(wl.n) if wl.batch is not None else 1
    n_max = int(np.max(wl.n)) if wl.batch is not None else len(wl.traj["t"])
    ws = torch.empty(rad.rad_workspace_bytes(count, n_max, len(wl.omega), len(wl.thx), len(wl.thy)),
                     dtype=torch.uint8, device=dev)
    out = torch.empty((len(wl.omega), len(wl.thy), len(wl.thx)), dtype=torch.float64, device=dev)
    lam_vec = np.full(count, lam) if model else None

    def step():
        if wl.batch is not None:
            rad.rad_ensemble_sum(dtr, wl.n, *grid, model=model, hbarc_over_E=lam_vec, out=out, workspace=ws)
        elif model == 0:
            rad.rad_classical(dtr, *grid, out=out, workspace=ws)
        else:
            rad.rad_semiclassical(dtr, *grid, 0 if model == 1 else 1, lam, out=out, workspace=ws)

    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)      # > 126 MB L2

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    peak = rad.rad_measure_fp64_peak(300.0)                            # FLOP/s, measured here
    rad.rad_profile_enable(True)
    rad.rad_set_kernel({"auto": 0, "direct": 1, "separable": 2}[args.kernel])
    kernel = rad.rad_plan_kernel(len(wl.omega), len(wl.thx), len(wl.thy), model)

    def timed_steps(n_steps):
        """W untimed steps, then n_steps timed ones: (sum of step ms, per-step main-kernel ms, launches, clocks)."""
        for _ in range(max(args.warmup, 3)):
            flush.zero_()
            step()
        barrier()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
              for _ in range(n_steps)]
        kernel_ms = []
        launches0 = rad.rad_launch_count()
        with ClockSampler(local) as clk:
            for a, b in ev:
                flush.zero_()
                a.record()
                step()
                b.record()
                kernel_ms.append(rad.rad_profile_last()[1])            # waits for this step
            torch.cuda.synchronize()
        n_launch = rad.rad_launch_count() - launches0
        barrier()
        return sum(a.elapsed_time(b) for a, b in ev), kernel_ms, n_launch, clk

    total_ms, main_ms, launches, clocks = timed_steps(args.steps)

    # the same workload through the other (direct-phasor) kernel, for the record: the north_star
    # target (>= 60 % of FP64 peak) is stated for the kernel that evaluates one phasor per eval
    direct = None
    if kernel == 2 and args.kernel == "auto" and rank == 0 and world == 1 and total_ms / args.steps < 2000.0:
        rad.rad_set_kernel(1)
        d_total, d_main, _, _ = timed_steps(min(args.steps, 5))
        rad.rad_set_kernel(0)
        d_s = float(np.mean(d_main)) * 1e-3
        d_flops = FLOPS_PER_EVAL[1][model] * wl.evals / d_s
        direct = {"kernel": KERNELS[1], "value": wl.evals * min(args.steps, 5) / (d_total * 1e-3), "unit": UNIT,
                  "main_kernel_ms": d_s * 1e3, "flops_per_eval": FLOPS_PER_EVAL[1][model],
                  "achieved": d_flops / 1e12, "frac": d_flops / peak,
                  "fp64_issue_frac": FP64_INSTR_PER_EVAL[1][model] * wl.evals / d_s / (peak / 2.0)}
    if world > 1:
        t = torch.tensor([total_ms], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = float(t.item())
    evals_step = wl.evals
    value = world * evals_step * args.steps / (total_ms * 1e-3)

    # ---- end to end through the host-buffer C-ABI call (pinned inputs, H2D + D2H inside)
    host_out = torch.empty(out.shape, dtype=torch.float64).pin_memory()
    host_grid = [torch.from_numpy(np.ascontiguousarray(a)).pin_memory() for a in (wl.omega, wl.thx, wl.thy)]

    def e2e_step():
        if wl.batch is not None:
            rad.rad_ensemble_sum_host(pinned, wl.n, *host_grid, model=model, hbarc_over_E=lam_vec, out=host_out)
        else:
            rad.rad_eval_host(pinned, *host_grid, model, lam, out=host_out)

    e2e_steps = max(3, min(args.steps, 10))
    for _ in range(2):
        e2e_step()
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        flush.zero_()
        torch.cuda.synchronize()
        e2e_step()                                                     # returns after D2H completed
    e2e_wall = time.perf_counter() - t0
    # subtract nothing: the flush is inside this wall-clock region, so time it separately
    torch.cuda.synchronize()
    t1 = time.perf_counter()
    for _ in range(e2e_steps):
        flush.zero_()
        torch.cuda.synchronize()
    flush_wall = time.perf_counter() - t1
    e2e_t = torch.tensor([e2e_wall - flush_wall], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(e2e_t, op=dist.ReduceOp.MAX)
    e2e_value = world * evals_step * e2e_steps / float(e2e_t.item())
    h2d = sum(v.numel() * 8 for v in pinned.values()) + sum(g.numel() * 8 for g in host_grid)
    d2h = host_out.numel() * 8

    if rank == 0:
        main_s = float(np.mean(main_ms)) * 1e-3
        achieved = FLOPS_PER_EVAL[kernel][model] * evals_step / main_s
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": total_ms / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": wl.name, "model": ["classical", "spin0", "spin1/2"][model],
                       "samples": n_max, "trajectories": count,
                       "grid": [len(wl.omega), len(wl.thy), len(wl.thx)], "evals_per_step": evals_step,
                       "l2": "flushed between steps (256 MiB memset)",
                       "parallelism": f"replicas x{world}, one trajectory per rank, no collective"},
            "clocks": clocks.summary(),
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "steps": e2e_steps, "call": "rad_eval_host / rad_ensemble_sum_host (pinned host buffers)"},
            "gpu_launches": int(launches),
            "roofline": {"bound": "alu", "kernel": KERNELS[kernel],
                         "achieved": achieved / 1e12, "peak": peak / 1e12, "unit": "TFLOP/s",
                         "frac": achieved / peak,
                         "traffic": NCU_TRAFFIC_BYTES.get((args.workload, kernel)) if args.spin == "1/2" else None,
                         "traffic_unit": "bytes per main-kernel launch (ncu capture in profiles/, not this run)",
                         "peak_kind": "FP64 FMA microbenchmark measured in this run (rad_measure_fp64_peak)",
                         "peak_spec": FP64_SPEC_TFLOPS, "frac_of_spec": achieved / 1e12 / FP64_SPEC_TFLOPS,
                         "flops_per_eval": FLOPS_PER_EVAL[kernel][model],
                         "fp64_issue_frac": FP64_INSTR_PER_EVAL[kernel][model] * evals_step / main_s / (peak / 2.0),
                         "main_kernel_ms": main_s * 1e3,
                         "main_kernel_share_of_step": main_s * 1e3 / (total_ms / args.steps)},
        }
        if direct is not None:
            line["roofline"]["direct_kernel_same_run"] = direct
        if not args.no_cpu_baseline and world == 1:
            line["cpu_baseline"] = cpu_baseline(wl)
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    args = parse()
    if args.impl == "reference":
        return run_reference(args)
    return run_b200(args)


if __name__ == "__main__":
    sys.exit(main())
