"""Fixtures of tests/golden/ (written by tests/golden/make_golden.py, which never touches the CUDA path)."""
import math
from pathlib import Path

import numpy as np
import pytest

import workloads

GOLD = Path(__file__).resolve().parent / "golden"


def _rows(name):
    return [ln.split() for ln in (GOLD / name).read_text().splitlines() if ln and not ln.startswith("#")]


@pytest.mark.parametrize("row", _rows("weak_undulator_peak.txt"))
def test_weak_undulator_peak_value(oracle_mod, row):
    """Textbook weak-undulator peak gamma^2 K^2 N_u^2 (PAPER.md:163-167 in the K -> 0
    limit): the oracle at w = w_1 on axis reproduces it to O(K^2) + O((w0 dt)^2)."""
    gamma, K, Nu, peak = float(row[0]), float(row[1]), int(row[2]), float(row[3])
    lam_u = 2e-6
    w0 = 2 * math.pi / lam_u
    tr = workloads.sinusoid_trajectory(gamma, K / (gamma * w0), lam_u, Nu, 1000 * Nu + 1)
    w1 = 2 * gamma ** 2 * w0
    out = oracle_mod.points(tr, [w1], [0.0], [0.0])[0]
    assert out == pytest.approx(peak, rel=2e-5)


def test_oracle_regression(oracle_mod):
    rows = _rows("oracle_regression.txt")
    wl = workloads.make("cfg2", n=257, n_omega=3, n_th=2, seed=123)
    lam = 0.5 / wl.omega.max()
    for model in (0, 1, 2):
        want = np.array([float.fromhex(r[2]) for r in rows if r[0] == str(model)])
        got = oracle_mod.grid(wl.traj, wl.omega, wl.thx, wl.thy, model, lam).ravel()
        np.testing.assert_allclose(got, want, rtol=1e-15)
    we = workloads.make("cfg4", count=3, n=130, n_omega=2, n_th=2, seed0=321)
    w, nx, ny = oracle_mod.grid_points(we.omega, we.thx, we.thy)
    got = oracle_mod.ensemble_points(we.batch, np.array([130, 2, 77]), w, nx, ny)
    want = np.array([float.fromhex(r[2]) for r in rows if r[0] == "9"])
    np.testing.assert_allclose(got, want, rtol=1e-15)
