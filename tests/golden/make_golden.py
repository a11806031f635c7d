"""Writes the fixtures of tests/golden/.  Calls ONLY oracle/ and workloads/ (never the CUDA path).

  weak_undulator_peak.txt   textbook closed form, no oracle involved: on-axis first-harmonic peak of a
                            weak planar undulator, d2I/dw dOmega = e^2 gamma^2 K^2 N_u^2  (
                            the paper's own validation idea, in the K -> 0 limit
                            where the expression is elementary).  Pure arithmetic in mpmath.
  oracle_regression.txt     long-double oracle outputs on a tiny seeded case, all three variants and an
                            ensemble: a drift alarm for the oracle itself (any later change of the
                            oracle's arithmetic must regenerate this file and say why in its commit).

Usage: python tests/golden/make_golden.py
"""
import sys
from pathlib import Path

import mpmath as mp
import numpy as np

HERE = Path(__file__).resolve().parent
sys.path.insert(0, str(HERE.parent.parent))


def weak_undulator_peak():
    mp.mp.dps = 30
    lines = ["# gamma  K  N_u  peak = gamma^2 K^2 N_u^2  (units of e^2; SURVEY.md P5, PAPER.md:163-167)"]
    for gamma, K, Nu in ((1000, "3e-4", 4), (1000, "1e-4", 10), (5000, "2e-4", 7), (200, "5e-4", 3)):
        peak = mp.mpf(gamma) ** 2 * mp.mpf(K) ** 2 * Nu ** 2
        lines.append(f"{gamma} {K} {Nu} {mp.nstr(peak, 17)}")
    (HERE / "weak_undulator_peak.txt").write_text("\n".join(lines) + "\n")


def oracle_regression():
    import oracle
    import workloads
    wl = workloads.make("cfg2", n=257, n_omega=3, n_th=2, seed=123)
    lam = 0.5 / wl.omega.max()
    lines = ["# workloads.make('cfg2', n=257, n_omega=3, n_th=2, seed=123), lam = 0.5/omega.max(); "
             "cube order (i_w, i_y, i_x); long-double oracle",
             "# model  flat_index  value"]
    for model in (0, 1, 2):
        cube = oracle.grid(wl.traj, wl.omega, wl.thx, wl.thy, model, lam).ravel()
        lines += [f"{model} {i} {v.hex()}" for i, v in enumerate(cube)]
    we = workloads.make("cfg4", count=3, n=130, n_omega=2, n_th=2, seed0=321)
    w, nx, ny = oracle.grid_points(we.omega, we.thx, we.thy)
    ens = oracle.ensemble_points(we.batch, np.array([130, 2, 77]), w, nx, ny)
    lines.append("# ensemble: workloads.make('cfg4', count=3, n=130, n_omega=2, n_th=2, seed0=321), n = [130, 2, 77]")
    lines += [f"9 {i} {v.hex()}" for i, v in enumerate(ens)]
    (HERE / "oracle_regression.txt").write_text("\n".join(lines) + "\n")


if __name__ == "__main__":
    weak_undulator_peak()
    oracle_regression()
