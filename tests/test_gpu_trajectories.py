"""GPU trajectory generator (NEXT row N4) against the trajectory oracle, and the device-resident pipeline
generator -> rad_ensemble_sum against the spectrum oracle (run with -m gpu on the B200 box).

Tolerance of the trajectory comparison: the kernel integrates in double, the oracle in
long double; every Verlet step commits O(10) roundings of relative size eps = 2^-53 to a bounded
oscillation, whose phase error therefore grows linearly: |gpu - oracle| <= 64 n eps max|array|
(1.4e-10 of the array's scale at n = 20 000), checked for all eleven arrays."""
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

EPS = 2.0 ** -53
WELLS = {0: dict(kappa=math.pi * 5e-5 ** 2 / (2 * 1.92e-10), L=1.92e-10, gamma=39139.0, th=5e-5),     # config 3
         1: dict(kappa=3e-5 ** 2 / (2 * 0.3e-10), L=0.3e-10, gamma=97847.0, th=3e-5),                  # config 5
         2: dict(kappa=(2 * math.pi / 7e-6) ** 2, L=1.0, gamma=9784.7, th=0.0, sigma=2e-7, dt=7e-9)}   # configs 2, 4


@pytest.fixture(scope="module")
def rad():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the CUDA path has no CPU fallback")
    import paper_1910_10391_b200 as rad
    rad.build_library()
    rad.load_library()
    return rad


def initial_conditions(well, count, seed):
    rng = np.random.Generator(np.random.PCG64(seed))
    w = WELLS[well]
    if well == 2:                                      # amplitude uniform in [0, 0.96 A], phase uniform
        amp, ph = rng.uniform(0, 0.96e-10, count), rng.uniform(0, 2 * np.pi, count)
        return amp * np.sin(ph), np.zeros(count), amp * math.sqrt(w["kappa"]) * np.cos(ph), np.zeros(count)
    if well == 0:
        return (rng.uniform(-0.5 * w["L"], 0.5 * w["L"], count), np.zeros(count),
                rng.uniform(-w["th"], w["th"], count), np.zeros(count))
    r, a = 1e-10 * np.sqrt(rng.uniform(size=count)), rng.uniform(0, 2 * np.pi, count)
    v, b = 0.5 * w["th"] * np.sqrt(rng.uniform(size=count)), rng.uniform(0, 2 * np.pi, count)
    return r * np.cos(a), r * np.sin(a), v * np.cos(b), v * np.sin(b)


@pytest.mark.parametrize("well", [0, 1, 2])
def test_generator_matches_oracle(rad, oracle_mod, well):
    import torch
    w = WELLS[well]
    count, n, stride, dt = 300, 20000, 20003, w.get("dt", 1e-9)
    sigma, seed = w.get("sigma", 0.0), 4242
    ini = initial_conditions(well, count, seed=40 + well)
    dev = [torch.from_numpy(a).cuda() for a in ini]
    out = {k: torch.full((count, stride), -7.0, dtype=torch.float64, device="cuda") for k in rad.FIELDS}
    rad.rad_generate_trajectories(well, w["kappa"], w["L"], w["gamma"], dt, n, *dev, out=out, sigma=sigma, seed=seed)
    ref = oracle_mod.generate(well, w["kappa"], w["L"], w["gamma"], dt, n, *ini, sigma=sigma, seed=seed)
    worst = 0.0
    for k in rad.FIELDS:
        got = out[k].cpu().numpy()
        assert np.all(got[:, n:] == -7.0), f"{k}: wrote past n"
        scale = np.max(np.abs(ref[k]))
        err = np.max(np.abs(got[:, :n] - ref[k]))
        tol = 64 * n * EPS * scale
        worst = max(worst, err / tol if tol > 0 else (0.0 if err == 0 else np.inf))
        assert err <= tol, f"well {well} array {k}: error {err:.3e} > {tol:.3e} (scale {scale:.3e})"
    print(f"well {well}: worst error / tolerance = {worst:.3e}")


def test_generator_edge_cases(rad):
    import torch
    w = WELLS[1]
    z = torch.zeros(1, dtype=torch.float64, device="cuda")
    out = rad.rad_generate_trajectories(1, w["kappa"], w["L"], w["gamma"], 1e-9, 2, z, z, z, z)       # r = 0, n = 2
    assert all(torch.all(out[k] == 0) for k in ("x", "y", "vx", "vy", "ax", "ay", "az", "dz", "dvz"))
    assert out["t"].cpu().tolist() == [[0.0, 1e-9]] and torch.all(out["gamma"] == w["gamma"])
    with pytest.raises(rad.RadError):
        rad.rad_generate_trajectories(3, 1.0, 1.0, 10.0, 1e-9, 10, z, z, z, z)
    with pytest.raises(rad.RadError):
        rad.rad_generate_trajectories(2, 1.0, 1.0, 10.0, 1e-9, 10, z, z, z, z, sigma=-1.0)
    with pytest.raises(rad.RadError):
        rad.rad_generate_trajectories(0, 1.0, 1.0, 10.0, 1e-9, 1, z, z, z, z)
    with pytest.raises(rad.RadError):
        rad.rad_generate_trajectories(0, 1.0, 1.0, 10.0, -1e-9, 10, z, z, z, z)


@pytest.mark.parametrize("well,model", [(0, 2), (1, 1), (2, 0)])
def test_generated_ensemble_feeds_the_spectrum_on_the_device(rad, oracle_mod, well, model):
    """Trajectories generated on the device go straight into rad_ensemble_sum (no host round trip); the
    spectrum is compared with the oracle evaluated on a host copy of the same trajectories."""
    import torch
    import workloads
    from test_gpu_parity import assert_parity
    w = WELLS[well]
    count, n = 24, 6000
    ini = initial_conditions(well, count, seed=50 + well)
    batch = rad.rad_generate_trajectories(well, w["kappa"], w["L"], w["gamma"], w.get("dt", 1e-9), n,
                                          *[torch.from_numpy(a).cuda() for a in ini],
                                          sigma=w.get("sigma", 0.0), seed=99)
    E = w["gamma"] * workloads.ME_EV
    lam = workloads.HBARC_EV_M / E
    omega = 0.6 * E * (np.arange(16) + 1.0) / 16 / workloads.HBARC_EV_M
    half = w["th"] + 3.0 / w["gamma"]
    if well == 2:                                      # config-2 style grid: classical, around 2 gamma^2 w_p
        omega = 2 * w["gamma"] ** 2 * math.sqrt(w["kappa"]) * np.geomspace(0.05, 10, 16)
    th = -half + 2 * half * np.arange(16) / 15
    g = [torch.from_numpy(a).cuda() for a in (omega, th, th)]
    nvec = np.full(count, n, dtype=np.int64)
    cube = rad.rad_ensemble_sum(batch, nvec, *g, model=model, hbarc_over_E=lam).cpu().numpy()
    host = {k: v.cpu().numpy() for k, v in batch.items()}
    wv, nx, ny = oracle_mod.grid_points(omega, th, th)
    ref = oracle_mod.ensemble_points(host, nvec, wv, nx, ny, model, lam)
    assert_parity(cube, ref, label=f"generated ensemble well {well} model {model}")
