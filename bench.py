#!/usr/bin/env python
"""bench.py -- throughput of the radiation-integral hot path on B200 (one JSON line on stdout).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg5|cfg1|cfg2|cfg3|cfg4|paper_typical]
    python bench.py --impl reference ...     # the CPU oracle on the host cores, same metric and workload

A "step" is one pass of the whole hot path -- pack, main kernel(s), ordered reduction (SURVEY.md section 8(a)
rows a0-a7) -- over one synthetic batch.  Default workload: BASELINE.json configs[4] with the spin-1/2 model
(50 GeV axial channeling, N = 1e6 samples, 1024 x 64 x 64 grid: the largest single-GPU configuration, which
BASELINE.json's `metric` -- it names no config -- is therefore quoted on).  metric = FP64 radiation-integral
evals/s (grid points x time steps), BASELINE.json `metric`.

  value        device-resident inputs, CUDA events on the launching stream, L2 flushed between steps
  e2e          same step through the C-ABI host-buffer call (pinned host memory, H2D + D2H inside)
  roofline     main kernel(s) only: algorithmic flops (flops per eval x evals per launch) / their own
               event-timed duration (rad_options.profile), against the FP64 FMA peak measured in this run
  per_config   the other target configurations (cfg2 classical, cfg3 spin-1/2, cfg4 ensemble, cfg5 spin-0), config 1
               and the paper's typical 50 x 50 x 100 grid, each with its own value / roofline / clocks, and the
               direct (one phasor per eval) kernel beside the default one where the time budget allows
  cpu_baseline the CPU oracle (oracle/, double build of the same source) on a bounded sample

N > 1 (torchrun, one rank per GPU): the SAME job sharded (paper_1910_10391_b200/sharding.py) --
the headline grid cut into omega slabs (no exchange in the computation; the optional gather of the cube is outside
the metric), and in per_config the cfg4 ensemble dealt out by trajectories with ONE exchange (all-gather of the
partial cubes + ordered sum) inside the timed region.  Strong scaling: value = the whole job's evals / max-over-ranks
device time.
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
# algorithmic FP64 flops per eval, enumerated there operation by operation and checked against
# ncu's 2*DFMA + DMUL + DADD count (profiles/).  Direct kernel (also the fused single-launch kernel, which runs
# the same per-sample body): phase 2, exact range reduction 1 (+ one FRND beside the FP64 pipe), quarter-angle
# polynomials 21, two doublings 7, complex accumulation 8 [+4 for spin-1/2's J], integrand geometry 34 [37] per
# 8 omegas -> 43.25 [47.6] flops, 24.6 [26.9] FP64 instructions (SURVEY.md 8(d) estimated 52-60).  Separable-phasor
# kernel: per eval one complex multiply (6) and the accumulation (8 [12]), plus per 16 [8] evals one T and one
# [half a] Y phasor and one [half an] integrand entry (36 + 35 + 28 [31] flops) -> 20.19 [26.63] flops, 11.75 [15.19]
# FP64 instructions.  When the separable kernel runs as cluster pairs (plan["cluster"] == 2: every BASELINE config but
# cfg4, whose 16 x 16 angles are one tile) each CTA computes only half of the T table: 19.06 [24.38] flops, 11.09
# [13.88] FP64 instructions per eval -- the constants below marked '2c'.  cfg4's single angle tile pairs along omega
# instead and halves the F table (plan["cluster"] == 3, classical only): 19.31 flops, 11.19 instructions -- '2w'.
KERNELS = {1: "rad_main_kernel (direct phasor)", 2: "rad_sep_kernel (separable phasor)",
           3: "rad_fused_kernel (single launch: pack + direct phasor + grid-wide ordered reduction)"}
FLOPS_PER_EVAL = {1: {0: 43.25, 1: 43.25, 2: 47.6}, 2: {0: 20.19, 1: 20.19, 2: 26.63}, 3: {0: 43.25, 1: 43.25, 2: 47.6},
                  "2c": {0: 19.06, 1: 19.06, 2: 24.38}, "2w": {0: 19.31, 1: 19.31}}
FP64_INSTR_PER_EVAL = {1: {0: 24.6, 1: 24.6, 2: 26.9}, 2: {0: 11.75, 1: 11.75, 2: 15.19}, 3: {0: 24.6, 1: 24.6, 2: 26.9},
                       "2c": {0: 11.09, 1: 11.09, 2: 13.88}, "2w": {0: 11.19, 1: 11.19}}


def work_key(plan):
    """Key into the two tables above for the kernel of a plan's first part."""
    if plan["kernel"] == 2 and plan.get("cluster", 1) >= 2:
        return "2c" if plan["cluster"] == 2 else "2w"
    return plan["kernel"]
FP64_SPEC_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12      # 148 SM x 64 FMA lanes x 2 x 1.965 GHz
MODELS = ["classical", "spin0", "spin1/2"]
# dram__bytes_read.sum + dram__bytes_write.sum per main-kernel launch from the committed ncu --set full captures
# (bench.py cannot run ncu itself): profiles/r02_ncu_traffic.csv (workload, kernel code, bytes, capture file), written
# next to the captures it summarises.
TRAFFIC_FILE = ROOT / "profiles" / "r02_ncu_traffic.csv"


def read_traffic(path=TRAFFIC_FILE):
    """{"<workload name>|<kernel code>": dram bytes per main-kernel launch} from the committed table; {} if absent."""
    table = {}
    try:
        for ln in Path(path).read_text().splitlines():
            f = [x.strip() for x in ln.split(",")]
            if len(f) >= 3 and f[0] and not f[0].startswith("#") and f[0] != "workload":
                table[f"{f[0]}|{f[1]}"] = float(f[2])
    except OSError:
        pass
    return table


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["b200", "reference"], default="b200")
    ap.add_argument("--workload", default="cfg5")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-per-config", action="store_true", help="headline workload only")
    ap.add_argument("--cfg4-count", type=int, default=1000)
    ap.add_argument("--kernel", choices=["auto", "direct", "separable", "fused"], default="auto",
                    help="main kernel of the timed steps (auto: the library's own choice by shape)")
    ap.add_argument("--spin", choices=["0", "1/2"], default="1/2",
                    help="semi-classical variant of cfg3 / cfg5 (BASELINE.json configs[4] asks for both)")
    return ap.parse_args()


def inputs_hash(wl) -> str:
    """blake2b-64 over the arrays this process evaluates (trajectory fields in rad_traj order, n, grid): the arrays, not
    the recipe, are the inputs of record.  Under torchrun a cfg4 rank hashes its own block."""
    import hashlib
    h = hashlib.blake2b(digest_size=8)
    src = wl.batch if wl.batch is not None else wl.traj
    for k in ("t", "dz", "x", "y", "vx", "vy", "dvz", "ax", "ay", "az", "gamma"):
        h.update(np.ascontiguousarray(src[k]).view(np.uint8).reshape(-1).data)
    if wl.batch is not None:
        h.update(np.ascontiguousarray(wl.n, dtype=np.int64).view(np.uint8).data)
    for a in (wl.omega, wl.thx, wl.thy):
        h.update(np.ascontiguousarray(a).view(np.uint8).data)
    return h.hexdigest()


def job_evals(wl) -> int:
    """evals of the WHOLE job: a rank of a sharded cfg4 run holds only its own block of the trajectories."""
    if wl.batch is not None and "global_count" in wl.meta:
        return wl.n_points * wl.meta["global_count"] * int(wl.n[0])
    return wl.evals


def make_workload(name: str, cfg4_count: int = 1000, spin: str = "1/2", rank: int = 0, world: int = 1):
    """rank / world: under torchrun a rank generates only ITS block of cfg4's trajectories (seed of trajectory p is
    4000 + p wherever it is generated), not the whole 8.8 GB ensemble on every rank."""
    import workloads
    model = workloads.SPIN0 if spin == "0" else workloads.SPIN_HALF
    if name in ("cfg1", "cfg2", "paper_typical"):
        return workloads.make(name)
    if name in ("cfg3", "cfg5"):
        return workloads.make(name, model=model)
    if name == "cfg4":
        if world > 1:
            from paper_1910_10391_b200.sharding import shard_range
            lo, hi = shard_range(cfg4_count, rank, world)
            wl = workloads.make("cfg4", count=max(hi - lo, 1), seed0=4000 + lo)
            wl.meta.update(global_count=cfg4_count, block=(lo, hi))
            return wl
        return workloads.make("cfg4", count=cfg4_count)
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
def oracle_sample_rate(wl, n_points: int, variant: str, repeats: int = 1, keep: dict | None = None):
    """evals/s of the CPU oracle on a seeded subset of the workload's grid points."""
    import oracle
    import workloads
    idx = workloads.sample_points(wl, n_points, seed=777)
    w, nx, ny = workloads.points_of(wl, idx)
    best = None
    for _ in range(repeats):
        t0 = time.perf_counter()
        if wl.batch is not None:
            vals = oracle.ensemble_points(wl.batch, wl.n, w, nx, ny, wl.model,
                                          wl.hbarc_over_E if wl.model else None, variant=variant)
            samples = int(np.sum(wl.n))
        else:
            vals = oracle.points(wl.traj, w, nx, ny, wl.model, wl.hbarc_over_E, variant=variant)
            samples = len(wl.traj["t"])
        dt = time.perf_counter() - t0
        best = dt if best is None else min(best, dt)
    if keep is not None:
        keep["idx"], keep["values"] = idx, np.asarray(vals, dtype=np.float64)
    return len(idx) * samples / best, len(idx), best


def cpu_baseline(wl, gpu_cube=None):
    """gpu_cube: the cube the timed steps wrote (numpy): the long-double oracle values computed here anyway are then
    also a parity check of THIS run (BASELINE.json tolerance), reported under "parity_in_this_run"."""
    import oracle
    samples = int(np.sum(wl.n)) if wl.batch is not None else len(wl.traj["t"])
    # size the sample for roughly 10-20 s of wall time on this box
    rate_guess = 2.0e7 * oracle.threads("f64")
    npts = int(min(wl.n_points, max(64, 12.0 * rate_guess / samples)))
    oracle_sample_rate(wl, min(npts, 64), "f64")                       # page in / warm up
    rate, got, secs = oracle_sample_rate(wl, npts, "f64")
    npts_ld = max(16, npts // 16)
    kept = {}
    rate_ld, got_ld, secs_ld = oracle_sample_rate(wl, npts_ld, "ld", keep=kept)
    parity = None
    if gpu_cube is not None:
        flat = np.asarray(gpu_cube, dtype=np.float64).ravel()
        got, ref = flat[kept["idx"]], kept["values"].ravel()
        tol = np.maximum(1e-9 * np.abs(ref), 1e-12 * float(np.max(flat)))
        parity = {"points": int(len(ref)), "worst_err_over_tol": float(np.max(np.abs(got - ref) / tol)),
                  "tolerance": "max(1e-9 |oracle|, 1e-12 max(cube)), long-double oracle", "ok": bool(np.all(np.abs(got - ref) <= tol))}
    return {"value": rate, "unit": UNIT, "cores": oracle.threads("f64"), "kind": "oracle", "parity_in_this_run": parity,
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
    wl = make_workload(args.workload, min(args.cfg4_count, 8), args.spin)
    samples = int(np.sum(wl.n)) if wl.batch is not None else len(wl.traj["t"])
    cores = oracle.threads("f64")
    budget_s = 90.0 / max(1, args.steps + args.warmup)
    npts = int(min(wl.n_points, max(16, budget_s * 2.0e7 * cores / samples)))
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
            "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": wl.name, "model": MODELS[wl.model], "samples": int(np.max(wl.n)) if wl.batch is not None else samples,
                       "trajectories": len(wl.n) if wl.batch is not None else 1,
                       "grid": [len(wl.omega), len(wl.thy), len(wl.thx)], "evals_per_step": got * samples,
                       "sample_points_per_step": got, "inputs_blake2b64": inputs_hash(wl),
                       "note": "same workload as the b200 arm; each step evaluates a seeded sample of its grid points"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


# ----------------------------------------------------------------------------- the B200 arm
class Bench:
    def __init__(self, args):
        import torch
        import torch.distributed as dist

        import paper_1910_10391_b200 as rad
        self.torch, self.dist, self.rad, self.args = torch, dist, rad, args
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.rank = int(os.environ.get("RANK", "0"))
        self.local = int(os.environ.get("LOCAL_RANK", "0"))
        if not torch.cuda.is_available():
            raise SystemExit("bench.py needs a CUDA device: the CUDA path has no CPU fallback")
        torch.cuda.set_device(self.local)
        self.dev = torch.device("cuda", self.local)
        if self.world > 1:
            dist.init_process_group("nccl", device_id=self.dev)     # NCCL_DEBUG is left to the caller's environment
        rad.build_library()
        rad.load_library()
        self.flush = torch.empty(256 << 20, dtype=torch.uint8, device=self.dev)      # > 126 MB L2
        self.peak = rad.rad_measure_fp64_peak(300.0)                                 # FLOP/s, measured here
        self.prof = rad.RadProfile()
        self.traffic = read_traffic()

    def barrier(self):
        if self.world > 1:
            self.dist.barrier()
        self.torch.cuda.synchronize()

    def to_dev(self, a):
        return self.torch.from_numpy(np.ascontiguousarray(a)).to(self.dev)

    # ---- one workload, device-resident: W untimed steps, K timed ones
    def run(self, wl, steps, warmup, kernel=0, shard=None):
        """shard: None (whole job on this rank), "omega" (grid sharded across ranks), "ensemble" (trajectories dealt
        out, one exchange inside the timed region)."""
        torch, rad = self.torch, self.rad
        from paper_1910_10391_b200.sharding import shard_range
        model, lam = wl.model, wl.hbarc_over_E
        omega, thx, thy = (self.to_dev(a) for a in (wl.omega, wl.thx, wl.thy))
        n_w = len(wl.omega)
        if shard == "omega":
            lo, hi = shard_range(n_w, self.rank, self.world)
            omega = omega[lo:hi].contiguous()
            n_w = hi - lo
        if wl.batch is not None:
            p_lo, p_hi = shard_range(len(wl.n), self.rank, self.world) if shard == "ensemble" else (0, len(wl.n))
            if "block" in wl.meta:                                     # already this rank's block (make_workload)
                p_lo, p_hi = 0, wl.meta["block"][1] - wl.meta["block"][0]
            dtr = {k: self.to_dev(v[p_lo:p_hi]) for k, v in wl.batch.items()}
            n_vec = np.ascontiguousarray(wl.n[p_lo:p_hi])
            count, n_max = len(n_vec), int(np.max(n_vec)) if len(n_vec) else 2
        else:
            dtr = {k: self.to_dev(v) for k, v in wl.traj.items()}
            n_vec, count, n_max = None, 1, len(wl.traj["t"])
        ws = torch.empty(max(256, rad.rad_workspace_bytes(max(count, 1), n_max, max(n_w, 1), len(wl.thx), len(wl.thy))),
                         dtype=torch.uint8, device=self.dev)
        out = torch.empty((max(n_w, 1), len(wl.thy), len(wl.thx)), dtype=torch.float64, device=self.dev)
        lam_vec = np.full(max(count, 1), lam) if model else None
        parts = torch.empty((self.world, *out.shape), dtype=torch.float64, device=self.dev) if shard == "ensemble" else None
        total = torch.empty_like(out) if shard == "ensemble" else None

        def step():
            if n_w == 0 or count == 0:
                out.zero_()
            elif wl.batch is not None:
                rad.rad_ensemble_sum(dtr, n_vec, omega, thx, thy, model=model, hbarc_over_E=lam_vec, out=out, workspace=ws,
                                     kernel=kernel, profile=self.prof)
            elif model == 0:
                rad.rad_classical(dtr, omega, thx, thy, out=out, workspace=ws, kernel=kernel, profile=self.prof)
            else:
                rad.rad_semiclassical(dtr, omega, thx, thy, 0 if model == 1 else 1, lam, out=out, workspace=ws,
                                      kernel=kernel, profile=self.prof)
            if shard == "ensemble" and self.world > 1:                 # the ONE exchange of SURVEY.md 8(e)(ii)
                self.dist.all_gather_into_tensor(parts.view(-1), out.view(-1))
                rad.rad_sum_cubes(parts, out=total)

        for _ in range(warmup):
            self.flush.zero_()
            step()
        self.barrier()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        launches0 = rad.rad_launch_count()
        with ClockSampler(self.local) as clk:
            for a, b in ev:                                            # no host synchronisation inside the timed region
                self.flush.zero_()
                a.record()
                step()
                b.record()
            torch.cuda.synchronize()
        launches = rad.rad_launch_count() - launches0
        self.barrier()
        total_ms = sum(a.elapsed_time(b) for a, b in ev)
        main_ms = []                                                   # the main kernel's own duration: a few extra
        for _ in range(min(steps, 3) if n_w and count else 0):         # steps, each read back (this synchronises)
            self.flush.zero_()
            step()
            main_ms.append(self.prof.read()[1])
        rank_ms = total_ms
        if self.world > 1:
            t = torch.tensor([total_ms], dtype=torch.float64, device=self.dev)
            all_t = [torch.empty_like(t) for _ in range(self.world)]
            self.dist.all_gather(all_t, t)
            rank_ms = [float(x.item()) / steps for x in all_t]
            total_ms = max(float(x.item()) for x in all_t)
        plan = rad.rad_plan_describe(max(count, 1), n_max, max(n_w, 1), len(wl.thx), len(wl.thy), model, kernel)
        self.last_cube = out if shard is None else None
        return {"wl": wl, "steps": steps, "warmup": warmup, "total_ms": total_ms, "main_ms": main_ms, "launches": launches,
                "clocks": clk.summary(), "plan": plan, "rank_ms_per_step": rank_ms, "local_points": n_w * len(wl.thx) * len(wl.thy),
                "local_samples": int(np.sum(n_vec)) if n_vec is not None else n_max, "shard": shard}

    # ---- small problems: the same step captured ONCE in a CUDA graph and replayed (the single-trajectory calls only
    # enqueue kernels when the caller passes a workspace, tests/test_gpu_parity.py::test_single_trajectory_call_is_
    # graph_capturable): what remains is the kernels' own time without the per-launch gap of the eager call
    def graph_replay(self, wl, steps):
        torch, rad = self.torch, self.rad
        if wl.batch is not None:
            return None
        omega, thx, thy = (self.to_dev(a) for a in (wl.omega, wl.thx, wl.thy))
        dtr = {k: self.to_dev(v) for k, v in wl.traj.items()}
        ws = torch.empty(max(256, rad.rad_workspace_bytes(1, len(wl.traj["t"]), len(wl.omega), len(wl.thx), len(wl.thy))),
                         dtype=torch.uint8, device=self.dev)
        out = torch.empty((len(wl.omega), len(wl.thy), len(wl.thx)), dtype=torch.float64, device=self.dev)

        def step():
            if wl.model == 0:
                rad.rad_classical(dtr, omega, thx, thy, out=out, workspace=ws)
            else:
                rad.rad_semiclassical(dtr, omega, thx, thy, 0 if wl.model == 1 else 1, wl.hbarc_over_E, out=out, workspace=ws)
        for _ in range(3):
            step()
        graph, side = torch.cuda.CUDAGraph(), torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(side):
            with torch.cuda.graph(graph, stream=side):
                step()
        torch.cuda.current_stream().wait_stream(side)
        for _ in range(3):
            graph.replay()
        torch.cuda.synchronize()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        for a, b in ev:
            self.flush.zero_()
            a.record()
            graph.replay()
            b.record()
        torch.cuda.synchronize()
        ms = sum(a.elapsed_time(b) for a, b in ev) / steps
        return {"ms_per_step": ms, "value": wl.evals / (ms * 1e-3), "unit": UNIT, "steps": steps,
                "how": "one step captured in a CUDA graph (caller workspace), replayed; L2 flushed between replays"}

    # ---- roofline of a run: algorithmic flops of the kernels that ran / the main kernels' own time
    def roofline(self, r):
        wl, plan = r["wl"], r["plan"]
        model = wl.model
        evals = float(r["local_points"]) * r["local_samples"]          # this rank's evals per step
        if not r["main_ms"] or evals == 0:
            return None
        main_s = float(np.mean(r["main_ms"])) * 1e-3
        k, wk = plan["kernel"], work_key(plan)
        if plan["parts"] == 2:                                         # separable interior + direct rest
            frac_sep = plan["interior_x"] * plan["interior_y"] / (len(wl.thx) * len(wl.thy))
            flops = evals * (frac_sep * FLOPS_PER_EVAL[wk][model] + (1 - frac_sep) * FLOPS_PER_EVAL[1][model])
            instr = evals * (frac_sep * FP64_INSTR_PER_EVAL[wk][model] + (1 - frac_sep) * FP64_INSTR_PER_EVAL[1][model])
            name = f"{KERNELS[2]} on {plan['interior_x']} x {plan['interior_y']} angles + {KERNELS[1]} on the rest"
        else:
            flops, instr, name = evals * FLOPS_PER_EVAL[wk][model], evals * FP64_INSTR_PER_EVAL[wk][model], KERNELS[k]
        if wk in ("2c", "2w"):
            name += ", cluster pairs sharing the T table" if wk == "2c" else ", cluster pairs sharing the F table"
        achieved = flops / main_s
        key = f"{wl.name}|{k}"
        return {"bound": "alu", "kernel": name, "achieved": achieved / 1e12, "peak": self.peak / 1e12, "unit": "TFLOP/s",
                "frac": achieved / self.peak,
                "traffic": self.traffic.get(key),
                "traffic_unit": "bytes per main-kernel launch (ncu --set full capture under profiles/, not this run)",
                "peak_kind": "FP64 FMA microbenchmark measured in this run (rad_measure_fp64_peak)",
                "peak_spec": FP64_SPEC_TFLOPS, "frac_of_spec": achieved / 1e12 / FP64_SPEC_TFLOPS,
                "flops_per_eval": flops / evals, "fp64_issue_frac": instr / main_s / (self.peak / 2.0),
                "main_kernel_ms": main_s * 1e3,
                "main_kernel_share_of_step": main_s * 1e3 / (float(np.mean(r["rank_ms_per_step"])) if isinstance(r["rank_ms_per_step"], list)
                                                             else r["total_ms"] / r["steps"])}

    def entry(self, r, with_direct=None):
        """per_config record of a run (value = whole-job evals/s)."""
        wl = r["wl"]
        e = {"workload": wl.name, "model": MODELS[wl.model], "evals_per_step": job_evals(wl), "inputs_blake2b64": inputs_hash(wl),
             "value": job_evals(wl) * r["steps"] / (r["total_ms"] * 1e-3), "unit": UNIT,
             "ms_per_step": r["total_ms"] / r["steps"], "steps": r["steps"], "warmup": r["warmup"],
             "launches_per_step": r["launches"] / r["steps"], "plan": r["plan"], "roofline": self.roofline(r),
             "clocks": r["clocks"]}
        if r["shard"]:
            e["sharding"] = r["shard"]
            e["rank_ms_per_step"] = r["rank_ms_per_step"]
        if with_direct is not None:
            d = with_direct
            e["direct_kernel_same_run"] = {"value": wl.evals * d["steps"] / (d["total_ms"] * 1e-3), "unit": UNIT,
                                           "ms_per_step": d["total_ms"] / d["steps"], "steps": d["steps"],
                                           "warmup": d["warmup"], "roofline": self.roofline(d)}
        return e

    # ---- end to end through the host-buffer C-ABI call (pinned inputs, H2D + D2H inside)
    def e2e(self, wl, steps, kernel):
        torch, rad = self.torch, self.rad
        src = wl.batch if wl.batch is not None else wl.traj
        # ONE pinned allocation for the eleven SoA arrays (field order of rad_traj) followed by the grid: the library
        # then needs one H2D transfer instead of fourteen
        fields = list(rad.FIELDS)
        per = int(np.prod(np.shape(src[fields[0]])))
        ng = len(wl.omega) + len(wl.thx) + len(wl.thy)
        flat = torch.empty(len(fields) * per + ng, dtype=torch.float64).pin_memory()
        pinned = {}
        for i, k in enumerate(fields):
            pinned[k] = flat[i * per:(i + 1) * per].view(np.shape(src[k]))
            pinned[k].copy_(torch.from_numpy(np.ascontiguousarray(src[k])))
        gflat = flat[len(fields) * per:]
        gflat.copy_(torch.from_numpy(np.concatenate([wl.omega, wl.thx, wl.thy])))
        host_grid = [gflat[:len(wl.omega)], gflat[len(wl.omega):len(wl.omega) + len(wl.thx)], gflat[len(wl.omega) + len(wl.thx):]]
        host_out = torch.empty((len(wl.omega), len(wl.thy), len(wl.thx)), dtype=torch.float64).pin_memory()
        lam_vec = np.full(len(wl.n), wl.hbarc_over_E) if wl.batch is not None and wl.model else None

        def step():
            if wl.batch is not None:
                rad.rad_ensemble_sum_host(pinned, wl.n, *host_grid, model=wl.model, hbarc_over_E=lam_vec, out=host_out,
                                          kernel=kernel)
            else:
                rad.rad_eval_host(pinned, *host_grid, wl.model, wl.hbarc_over_E, out=host_out, kernel=kernel)

        for _ in range(2 if wl.evals < 1e12 else 1):
            step()
        self.barrier()
        wall = 0.0
        for _ in range(steps):
            self.flush.zero_()
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            step()                                                     # returns after D2H completed
            wall += time.perf_counter() - t0
        h2d = sum(v.numel() * 8 for v in pinned.values()) + sum(g.numel() * 8 for g in host_grid)
        return wl.evals * steps / wall, h2d, host_out.numel() * 8, steps


def generator_throughput(B):
    """rad_generate_trajectories on its own -- 2000 particles (the paper's ensembles: up to
    2000 particles) x 20 000 steps in each of the three synthetic wells, device time by CUDA events.
    One thread per particle and a serial recurrence per step (stores staged through shared memory and written
    transposed, rad_traj.cuh): the bound is the latency of that dependent chain, not HBM; the HBM figure (88 B written
    per particle and step against the measured copy bandwidth) is reported so that this is visible."""
    import math
    torch, rad = B.torch, B.rad
    try:
        hbm = json.loads((ROOT / "MEASURED_PEAKS.json").read_text())["hbm_gbs"] * 1e9
        hbm_kind = "measured (MEASURED_PEAKS.json)"
    except Exception:
        hbm, hbm_kind = 6.65e12, "fallback (B200_PROFILING.md)"
    wells = {"cosine (cfg3)": (0, math.pi * 5e-5 ** 2 / (2 * 1.92e-10), 1.92e-10, 39139.0, 1e-9, 0.0),
             "axial exp (cfg5)": (1, 3e-5 ** 2 / (2 * 0.3e-10), 0.3e-10, 97847.0, 1e-9, 0.0),
             "harmonic + kicks (cfg2/4)": (2, (2 * math.pi / 7e-6) ** 2, 1.0, 9784.7, 7e-9, 2e-7)}
    count, n = 2000, 20000
    rng = np.random.Generator(np.random.PCG64(99))
    ini = [B.to_dev(a) for a in (rng.uniform(-4e-11, 4e-11, count), rng.uniform(-4e-11, 4e-11, count),
                                 rng.uniform(-1e-5, 1e-5, count), rng.uniform(-1e-5, 1e-5, count))]
    out = {k: torch.empty((count, n), dtype=torch.float64, device=B.dev) for k in rad.FIELDS}
    res = {}
    for name, (well, kappa, length, gamma, dt, sigma) in wells.items():
        def call():
            rad.rad_generate_trajectories(well, kappa, length, gamma, dt, n, *ini, out=out, sigma=sigma, seed=7)
        for _ in range(2):
            call()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(3):
            call()
        b.record()
        torch.cuda.synchronize()
        sec = a.elapsed_time(b) * 1e-3 / 3
        res[name] = {"particle_steps_per_s": count * n / sec, "ms": sec * 1e3, "bytes_written_per_s": 88.0 * count * n / sec,
                     "frac_of_hbm": 88.0 * count * n / sec / hbm}
    return {"particles": count, "steps": n, "hbm_peak_kind": hbm_kind, "bound": "latency of the per-particle recurrence",
            "wells": res}


def run_b200(args):
    B = Bench(args)
    world, rank = B.world, B.rank
    kopt = {"auto": 0, "direct": 1, "separable": 2, "fused": 3}[args.kernel]
    wl = make_workload(args.workload, args.cfg4_count, args.spin, rank, world)
    shard = None
    if world > 1:
        shard = "ensemble" if wl.batch is not None else "omega"
    warmup = max(args.warmup, 3)
    head = B.run(wl, args.steps, warmup, kopt, shard)
    head_cube = B.last_cube.cpu().numpy() if B.last_cube is not None else None
    step_ms = head["total_ms"] / args.steps
    value = job_evals(wl) * args.steps / (head["total_ms"] * 1e-3)

    # the same workload through the direct (one phasor per eval) kernel, for the record: the north_star target
    # (>= 60 % of FP64 peak) is stated for that kernel
    direct = None
    if head["plan"]["kernel"] == 2 and args.kernel == "auto" and world == 1:
        few = 5 if step_ms < 500 else 2
        direct = B.run(wl, few, 3 if step_ms < 500 else 1, 1)

    e2e_value = e2e_info = None
    if world == 1:
        e2e_steps = max(3, min(args.steps, 10)) if step_ms < 1000 else 3
        e2e_value, h2d, d2h, e2e_steps = B.e2e(wl, e2e_steps, kopt)
        e2e_info = {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "steps": e2e_steps, "call": "rad_eval_host / rad_ensemble_sum_host (pinned host buffers)"}
    else:
        e2e_info = {"value": None, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0,
                    "note": "host-buffer entry points are single-GPU calls; measured at --gpus 1"}

    per_config = []
    if not args.no_per_config and args.workload == "cfg5" and args.spin == "1/2" and args.kernel == "auto":
        # (workload, spin, timed steps, warm-up, also time the direct kernel?)
        todo = [("cfg2", "1/2", 20, 3, True), ("cfg3", "1/2", 5, 3, True), ("cfg4", "1/2", 2, 1, False),
                ("cfg5", "0", 2, 1, False), ("cfg1", "1/2", 50, 5, True), ("paper_typical", "1/2", 20, 3, True)]
        for name, spin, k, w, with_direct in todo:
            w2 = make_workload(name, args.cfg4_count, spin, rank, world)
            sh = None
            if world > 1:
                sh = "ensemble" if w2.batch is not None else "omega"
            r = B.run(w2, k, w, 0, sh)
            d = B.run(w2, min(k, 5), min(w, 3), 1) if with_direct and world == 1 and r["plan"]["kernel"] != 1 else None
            per_config.append(B.entry(r, d))
            if world == 1 and r["total_ms"] / r["steps"] < 1.0:         # launch-gap-sensitive problems (cfg1, the paper's grid)
                per_config[-1]["graph_replay"] = B.graph_replay(w2, k)
            del w2, r, d
            B.torch.cuda.empty_cache()

    if rank == 0:
        n_max = int(np.max(wl.n)) if wl.batch is not None else len(wl.traj["t"])
        count = wl.meta.get("global_count", len(wl.n)) if wl.batch is not None else 1
        roof = B.roofline(head)
        if direct is not None and roof is not None:
            roof["direct_kernel_same_run"] = {"kernel": KERNELS[1], "value": wl.evals * direct["steps"] / (direct["total_ms"] * 1e-3),
                                              "unit": UNIT, "steps": direct["steps"], "warmup": direct["warmup"],
                                              **{k: v for k, v in B.roofline(direct).items()
                                                 if k in ("achieved", "frac", "flops_per_eval", "fp64_issue_frac", "main_kernel_ms")}}
        par = {None: "one GPU", "omega": f"grid sharded in {world} omega slabs, whole trajectory on every rank, no exchange in the computation",
               "ensemble": f"trajectories dealt out to {world} ranks; all-gather of partial cubes + ordered sum inside the timed region"}[shard]
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": warmup, "ms_per_step": step_ms,
            "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": wl.name, "model": MODELS[wl.model], "samples": n_max, "trajectories": count,
                       "grid": [len(wl.omega), len(wl.thy), len(wl.thx)], "evals_per_step": job_evals(wl),
                       "inputs_blake2b64": inputs_hash(wl),
                       "l2": "flushed between steps (256 MiB memset)", "parallelism": par, "plan": head["plan"]},
            "clocks": head["clocks"],
            "e2e": e2e_info,
            "gpu_launches": int(head["launches"]),
            "roofline": roof,
        }
        if world > 1:
            line["rank_ms_per_step"] = head["rank_ms_per_step"]
        if per_config:
            line["per_config"] = per_config
            if world == 1:
                line["trajectory_generator"] = generator_throughput(B)
        if not args.no_cpu_baseline and world == 1:
            line["cpu_baseline"] = cpu_baseline(wl, head_cube)
        print(json.dumps(line))
    if world > 1:
        B.dist.destroy_process_group()
    return 0


def main():
    args = parse()
    if args.impl == "reference":
        return run_reference(args)
    return run_b200(args)


if __name__ == "__main__":
    sys.exit(main())
