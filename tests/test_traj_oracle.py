"""Pins of the trajectory oracle (oracle/traj_oracle.c, NEXT row N4) against things other than itself:
closed forms, conservation laws of the velocity-Verlet scheme, and the independent double-precision
Python integrator of workloads/ (written separately, used as the input generator of configs 3 and 5)."""
import math

import numpy as np
import pytest

import workloads

KAPPA3, DP = math.pi * 5e-5 ** 2 / (2 * 1.92e-10), 1.92e-10          # config 3: cosine well
KAPPA5, AW = 3e-5 ** 2 / (2 * 0.3e-10), 0.3e-10                      # config 5: axial exponential well
GAMMA = 39139.0


def test_free_particle_is_a_straight_line(oracle_mod):
    """kappa = 0: x = x0 + vx0 t, accelerations 0, dvz constant, dz = dvz t (closed form)."""
    o = oracle_mod.generate(0, 0.0, DP, GAMMA, 1e-9, 500, [1e-11], [-2e-11], [3e-5], [-1e-5])
    t = o["t"][0]
    np.testing.assert_allclose(o["x"][0], 1e-11 + 3e-5 * t, rtol=1e-14)
    np.testing.assert_allclose(o["y"][0], -2e-11 - 1e-5 * t, rtol=1e-14)
    assert np.all(o["ax"] == 0) and np.all(o["ay"] == 0) and np.all(o["az"] == 0)
    dvz = -(3e-5 ** 2 + 1e-5 ** 2) / 2
    np.testing.assert_allclose(o["dvz"][0], dvz, rtol=1e-15)
    np.testing.assert_allclose(o["dz"][0], dvz * t, rtol=1e-13, atol=0)
    assert np.all(o["gamma"] == GAMMA) and t[1] == 1e-9 and t[-1] == pytest.approx(499e-9, rel=1e-15)


def test_harmonic_limit_of_the_cosine_well(oracle_mod):
    """Small amplitude: x'' = -kappa (2 pi / L) x, so x(t) = x0 cos(w t) with w^2 = 2 pi kappa / L; Verlet's
    phase error is (w dt)^2 / 24 per radian, the anharmonic correction (2 pi x0 / L)^2 / 16."""
    w = math.sqrt(2 * math.pi * KAPPA3 / DP)
    dt, n, x0 = 1e-9, 8000, 1e-13
    o = oracle_mod.generate(0, KAPPA3, DP, GAMMA, dt, n, [x0], [0.0], [0.0], [0.0])
    t = o["t"][0]
    phase_slip = (w * t[-1]) * ((w * dt) ** 2 / 24 + (2 * math.pi * x0 / DP) ** 2 / 16)
    assert np.max(np.abs(o["x"][0] - x0 * np.cos(w * t))) <= 1.5 * phase_slip * x0 + 1e-12 * x0
    assert w * t[-1] > 2 * math.pi                                   # more than one full oscillation


@pytest.mark.parametrize("well", [0, 1])
def test_energy_error_is_second_order_and_does_not_drift(oracle_mod, well):
    """H = v^2/2 + U with U = -(kappa L / 2 pi) cos(2 pi x / L) resp. -kappa L exp(-r / L): velocity Verlet
    keeps it to O(dt^2) -- halving dt divides the worst deviation by 4."""
    kappa, L = (KAPPA3, DP) if well == 0 else (KAPPA5, AW)
    ini = ([0.3 * L], [0.0 if well == 0 else 0.5 * L], [1e-5], [0.0 if well == 0 else -0.7e-5])

    def worst(dt, n):
        o = oracle_mod.generate(well, kappa, L, GAMMA, dt, n, *ini)
        v2 = o["vx"][0].astype(np.longdouble) ** 2 + o["vy"][0].astype(np.longdouble) ** 2
        if well == 0:
            U = -(kappa * L / (2 * math.pi)) * np.cos(2 * np.pi * o["x"][0] / L)
        else:
            U = -kappa * L * np.exp(-np.hypot(o["x"][0], o["y"][0]) / L)
        H = v2 / 2 + U
        return float(np.max(np.abs(H - H[0]))), float(abs(H[0]))

    e1, h0 = worst(4e-9, 5000)
    e2, _ = worst(2e-9, 10000)
    assert e1 < 1e-3 * h0
    assert 3.5 < e1 / e2 < 4.5


def test_angular_momentum_and_time_reversal(oracle_mod):
    """Central force: x vy - y vx is conserved by Verlet to rounding.  Reversing the velocities retraces the path."""
    n = 4000
    o = oracle_mod.generate(1, KAPPA5, AW, GAMMA, 1e-9, n, [0.8e-10], [0.1e-10], [0.4e-5], [1.2e-5])
    lz = o["x"][0] * o["vy"][0] - o["y"][0] * o["vx"][0]
    assert np.max(np.abs(lz - lz[0])) <= 1e-13 * abs(lz[0])
    back = oracle_mod.generate(1, KAPPA5, AW, GAMMA, 1e-9, n, [o["x"][0, -1]], [o["y"][0, -1]],
                               [-o["vx"][0, -1]], [-o["vy"][0, -1]])
    np.testing.assert_allclose(back["x"][0, -1], 0.8e-10, rtol=1e-11)
    np.testing.assert_allclose(back["y"][0, -1], 0.1e-10, rtol=1e-10)
    np.testing.assert_allclose(back["vx"][0, -1], -0.4e-5, rtol=1e-10)


def test_longitudinal_bookkeeping(oracle_mod):
    """dvz = -(vx^2 + vy^2)/2 (PAPER.md:28 leading order), dz = cumulative trapezoid of dvz, az = d(dvz)/dt."""
    o = oracle_mod.generate(1, KAPPA5, AW, GAMMA, 1e-9, 3000, [0.5e-10], [0.2e-10], [1e-5], [0.5e-5])
    vx, vy, dvz, dz, az = (o[k][0] for k in ("vx", "vy", "dvz", "dz", "az"))
    np.testing.assert_allclose(dvz, -(vx * vx + vy * vy) / 2, rtol=1e-15)
    ref = np.concatenate([[0.0], np.cumsum((dvz[1:] + dvz[:-1]) * 0.5e-9)])
    np.testing.assert_allclose(dz, ref, rtol=1e-12)
    np.testing.assert_allclose(az, -(vx * o["ax"][0] + vy * o["ay"][0]), rtol=1e-14, atol=1e-30)
    fd = (dvz[2:] - dvz[:-2]) / 2e-9
    assert np.max(np.abs(fd - az[1:-1])) <= 1e-4 * np.max(np.abs(az))


def test_against_the_independent_python_integrator(oracle_mod):
    """workloads.config3 / config5 integrate the same wells with their own double-precision Python loop
    (written separately; it generates the benchmark inputs).  Same initial conditions -> same trajectory to
    the rounding accumulated by the double version."""
    wl = workloads.make("cfg3", n=3000, n_omega=2, n_th=2, seed=3)
    tr = wl.traj
    o = oracle_mod.generate(0, KAPPA3, DP, wl.meta["gamma"], 1e-9, 3000, [tr["x"][0]], [0.0], [tr["vx"][0]], [0.0])
    for k in ("x", "vx", "ax", "dvz", "dz", "az"):
        np.testing.assert_allclose(o[k][0], tr[k], rtol=2e-10, atol=1e-12 * np.max(np.abs(tr[k])), err_msg=k)
    wl = workloads.make("cfg5", n=3000, n_omega=2, n_th=2, seed=5)
    tr = wl.traj
    o = oracle_mod.generate(1, KAPPA5, AW, wl.meta["gamma"], 1e-9, 3000, [tr["x"][0]], [tr["y"][0]],
                            [tr["vx"][0]], [tr["vy"][0]])
    for k in ("x", "y", "vx", "vy", "ax", "ay", "dz"):
        np.testing.assert_allclose(o[k][0], tr[k], rtol=2e-10, atol=1e-12 * np.max(np.abs(tr[k])), err_msg=k)


# --------------------------------------------------------------------------- well 2: harmonic + scattering kicks
WP = 2 * math.pi / 7e-6                                               # configs 2 / 4: 7 um period


def test_philox_known_answers(oracle_mod):
    """tests/golden/philox4x32_10_kat.txt: the published known-answer vectors of Philox4x32-10."""
    from pathlib import Path
    rows = [ln.split() for ln in (Path(__file__).parent / "golden" / "philox4x32_10_kat.txt").read_text().splitlines()
            if ln and not ln.startswith("#")]
    assert len(rows) == 3
    for r in rows:
        v = [int(w, 16) for w in r]
        assert [int(o) for o in oracle_mod.philox4x32_10(v[:4], v[4:6])] == v[6:]


def test_kick_normals_are_standard_normal(oracle_mod):
    a, b = oracle_mod.kick_normals(seed=11, particle=5, n=400000)
    for v in (a, b):
        assert abs(v.mean()) < 5e-3 and abs(v.std() - 1) < 5e-3
        assert abs(np.mean(np.abs(v) > 2) - 0.0455) < 2e-3               # two-sigma tail of a Gaussian
        assert abs(np.mean(v ** 4) - 3) < 0.05                           # kurtosis
    assert abs(np.corrcoef(a, b)[0, 1]) < 5e-3 and abs(np.corrcoef(a[1:], a[:-1])[0, 1]) < 5e-3
    c, _ = oracle_mod.kick_normals(seed=11, particle=6, n=1000)          # another particle: another stream
    assert not np.allclose(c, a[:1000])


def test_scattering_well_without_kicks_is_exact_harmonic_motion(oracle_mod):
    """sigma = 0: the step is an exact rotation, so x = A sin(w t + phi) to rounding, for any dt."""
    A, ph = 0.7e-10, 1.1
    o = oracle_mod.generate(2, WP * WP, 1.0, 9784.7, 7e-9, 5000, [A * math.sin(ph)], [0.0],
                            [A * WP * math.cos(ph)], [1e-6], sigma=0.0, seed=1)
    t = o["t"][0]
    np.testing.assert_allclose(o["x"][0], A * np.sin(WP * t + ph), rtol=0, atol=1e-12 * A)
    np.testing.assert_allclose(o["vx"][0], A * WP * np.cos(WP * t + ph), rtol=0, atol=1e-12 * A * WP)
    np.testing.assert_allclose(o["ax"][0], -WP * WP * o["x"][0], rtol=1e-14)
    np.testing.assert_allclose(o["y"][0], 1e-6 * t, rtol=1e-13)
    assert np.all(o["ay"] == 0)


def test_scattering_well_against_numpy_recurrence(oracle_mod):
    """The kicked recurrence re-implemented in numpy longdouble from the recipe,
    fed with the oracle's own normals: pins the bookkeeping (kick / dt in the acceleration of the kicked
    sample, Q15; trapezoid y and dz; az)."""
    LD = np.longdouble
    n, dt, sig, seed = 3000, 7e-9, 2e-7, 21
    x0, v0, vy0 = 0.3e-10, 0.5e-10 * WP, -1e-7
    o = oracle_mod.generate(2, WP * WP, 1.0, 9784.7, dt, n, [x0, -x0], [0.0, 1e-11], [v0, v0], [vy0, 0.0],
                            sigma=sig, seed=seed)
    for p, (xi, vi, yi, vyi) in enumerate([(x0, v0, 0.0, vy0), (-x0, v0, 1e-11, 0.0)]):
        a, b = (v.astype(LD) for v in oracle_mod.kick_normals(seed, p, n + 1))
        a[0] = b[0] = 0
        wp, h = LD(WP), LD(dt)
        c, s = np.cos(wp * h), np.sin(wp * h)
        x, u = np.empty(n, LD), np.empty(n, LD)
        x[0], u[0] = xi, LD(vi) / wp
        for k in range(1, n):
            x[k] = c * x[k - 1] + s * u[k - 1]
            u[k] = c * u[k - 1] - s * x[k - 1] + LD(sig) / wp * a[k]
        vx = u * wp
        vy = LD(vyi) + LD(sig) * np.cumsum(b[:n])
        y = LD(yi) + np.concatenate([[LD(0)], np.cumsum((vy[1:] + vy[:-1]) / 2 * h)])
        ax = -wp * wp * x + LD(sig) * a[:n] / h
        ay = LD(sig) * b[:n] / h
        dvz = -(vx * vx + vy * vy) / 2
        dz = np.concatenate([[LD(0)], np.cumsum((dvz[1:] + dvz[:-1]) / 2 * h)])
        ref = dict(x=x, vx=vx, vy=vy, y=y, ax=ax, ay=ay, dvz=dvz, dz=dz, az=-(vx * ax + vy * ay))
        for k, v in ref.items():
            np.testing.assert_allclose(o[k][p], v.astype(np.float64), rtol=1e-11,
                                       atol=1e-13 * float(np.max(np.abs(v))), err_msg=f"particle {p} {k}")
    # Q15: the accelerations reproduce the velocity change sample-wise to O(dt): sum(ay dt) = vy - vy0 exactly
    np.testing.assert_allclose(np.cumsum(o["ay"][0]) * dt, o["vy"][0] - vy0, rtol=1e-9, atol=1e-18)
