"""bench.py's contract and the constants its roofline rests on (run with -m gpu on the B200 box)."""
import json
import subprocess
import sys
from pathlib import Path

import numpy as np
import pytest

import workloads

ROOT = Path(__file__).resolve().parent.parent
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def rad():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the CUDA path has no CPU fallback")
    import paper_1910_10391_b200 as rad
    rad.build_library()
    rad.load_library()
    return rad


@pytest.mark.parametrize("kernel,model", [(1, 0), (1, 2), (2, 0), (2, 2), (3, 0)])
def test_flop_constants_are_consistent_with_the_issue_rate(rad, kernel, model):
    """bench.py multiplies evals by DESIGN.md's enumerated flops / FP64 instructions per eval.  Whatever the kernel
    does, it cannot issue more than one FP64 instruction per lane and cycle: with the main kernel timed by the
    library's own events and the FMA peak measured in the same process,
        flops/eval * evals / t / peak  <=  instr/eval * evals / t / (peak / 2)  <=  1.
    A stale constant (a kernel that got cheaper per eval than the table says) breaks the right-hand inequality; the
    lower bound catches a run that did not execute the kernel it claims (achieved fraction absurdly low)."""
    import torch
    sys.path.insert(0, str(ROOT))
    import bench
    if kernel == 3:
        wl = workloads.make("cfg1")
    else:
        wl = workloads.make("cfg3", n=20000, n_omega=256, n_th=32, model=model) if model else workloads.make("cfg2")
    tr = {k: torch.from_numpy(np.ascontiguousarray(v)).cuda() for k, v in wl.traj.items()}
    g = [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (wl.omega, wl.thx, wl.thy)]
    prof = rad.RadProfile()
    peak = rad.rad_measure_fp64_peak(100.0)

    def call():
        if model == 0:
            rad.rad_classical(tr, *g, kernel=kernel, profile=prof)
        else:
            rad.rad_semiclassical(tr, *g, 1, wl.hbarc_over_E, kernel=kernel, profile=prof)
    for _ in range(3):
        call()
    ms = []
    for _ in range(5):
        call()
        ms.append(prof.read()[1])
    t = float(np.median(ms)) * 1e-3
    plan = rad.rad_plan_describe(1, len(wl.traj["t"]), len(wl.omega), len(wl.thx), len(wl.thy), model, kernel)
    assert plan["kernel"] == kernel and plan["parts"] == 1
    wk = bench.work_key(plan)                                          # "2c": separable kernel as cluster pairs
    frac = bench.FLOPS_PER_EVAL[wk][model] * wl.evals / t / peak
    issue = bench.FP64_INSTR_PER_EVAL[wk][model] * wl.evals / t / (peak / 2)
    assert frac <= issue <= 1.0, (frac, issue)
    assert frac >= (0.2 if kernel == 3 else 0.45), frac               # cfg1 is a 30 us problem: launch + tail dominate
    assert 0.9 * bench.FP64_SPEC_TFLOPS <= peak / 1e12 <= 1.05 * bench.FP64_SPEC_TFLOPS


def test_bench_line_contract_on_a_small_workload():
    """One JSON line with the keys the driver reads; cfg1 keeps this to seconds."""
    out = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--workload", "cfg1", "--steps", "5", "--warmup", "3",
                          "--no-cpu-baseline"], capture_output=True, text=True, check=True, cwd=ROOT).stdout
    lines = [ln for ln in out.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                "vs_baseline", "dtype", "data", "config", "clocks", "e2e", "gpu_launches", "roofline"):
        assert key in d, key
    assert d["config"]["workload"].startswith("cfg1") and d["dtype"] == "f64" and d["steps"] == 5
    assert d["gpu_launches"] == 5                                       # one fused launch per step
    assert d["roofline"]["bound"] == "alu" and 0 < d["roofline"]["frac"] <= d["roofline"]["fp64_issue_frac"] <= 1
    assert d["e2e"]["h2d_bytes_per_step"] == 11 * 4000 * 8 + (64 + 8 + 8) * 8 and d["e2e"]["d2h_bytes_per_step"] == 4096 * 8
    assert d["e2e"]["value"] < d["value"]                              # copies are inside the timed region


def test_traffic_table_names_kernels_that_exist():
    """profiles/r02_ncu_traffic.csv (dram bytes per main-kernel launch from the committed ncu captures) is keyed by
    workload name and kernel code; every row must name a workload bench.py can build."""
    import bench
    if not bench.TRAFFIC_FILE.exists():
        pytest.skip("no traffic table committed yet")
    names = {workloads.make(n, **kw).name for n, kw in (("cfg1", {}), ("cfg2", {}), ("paper_typical", {}),
                                                       ("cfg3", dict(n=10, n_omega=1, n_th=1)),
                                                       ("cfg5", dict(n=10, n_omega=1, n_th=1)),
                                                       ("cfg5", dict(n=10, n_omega=1, n_th=1, model=1)),
                                                       ("cfg4", dict(count=1, n=10, n_omega=1, n_th=1)))}
    table = bench.read_traffic()
    assert table
    for key, val in table.items():
        name, code = key.split("|")
        assert name in names and code in ("1", "2", "3") and val > 0
