"""Pins of the CPU oracle against what the paper and the mathematics fix.

None of these tests compares the oracle with itself or with the CUDA path.
Pin numbering follows DESIGN.md "Oracle pins".
Each tolerance is derived in the docstring of its test.
"""
import math

import numpy as np
import pytest

import workloads
from physics_ref import (LD, exact_amplitudes, exact_integrands, planar_2d_trajectory,
                         trapezoid_weights)

CL, S0, SH = 0, 1, 2
W0 = 2 * math.pi / 2e-6


def _undulator(gamma, K, periods, n, B_over_A=0.0):
    A = K / (gamma * W0)
    return planar_2d_trajectory(gamma, A, B_over_A * A, W0, periods, n)


# --------------------------------------------------------------------------- P1
@pytest.mark.parametrize("model", [CL, S0, SH])
def test_p1_straight_line_emits_nothing(oracle_mod, model):
    """f is linear in beta_dot (eq. 2): a straight line radiates exactly 0."""
    n = 500
    t = np.linspace(0.0, 1e-6, n)
    tr = {k: np.zeros(n) for k in workloads.FIELDS}
    tr["t"] = t
    tr["vx"] = np.full(n, 3e-5)
    tr["vy"] = np.full(n, -1e-5)
    tr["x"], tr["y"] = tr["vx"] * t, tr["vy"] * t
    tr["dvz"] = np.full(n, -0.5 * (9e-10 + 1e-10))
    tr["dz"] = tr["dvz"] * t
    tr["gamma"] = np.full(n, 5000.0)
    out = oracle_mod.points(tr, [1e12, 5e13], [1e-4, -2e-5], [0.0, 7e-5], model, 1e-18)
    assert np.all(out == 0.0)


# --------------------------------------------------------------------------- P2
def test_p2_transversality_identity(oracle_mod):
    """n.f = 0 for eq. (2); at leading order A_z + n_x A_x + n_y A_y = 0 for eqs. (3)-(5)
    as printed.  Only rounding remains: << 1e-12 of sum |w f|."""
    wl = workloads.make("cfg2", n=3000, n_omega=6, n_th=5)
    w, nx, ny = oracle_mod.grid_points(wl.omega, wl.thx, wl.thy)
    _, amp = oracle_mod.points(wl.traj, w, nx, ny, return_amplitudes=True)
    resid = amp[:, 2] + nx * amp[:, 0] + ny * amp[:, 1]
    scale = np.abs(nx * amp[:, 0]) + np.abs(ny * amp[:, 1]) + np.abs(amp[:, 2])
    assert np.all(np.abs(resid) <= 1e-12 * scale.max())
    assert np.abs(amp[:, 2]).max() > 0  # f_z is not trivially zero


# --------------------------------------------------------------------------- P3
@pytest.mark.parametrize("nxg,nyg", [(0.0, 0.0), (0.4, 0.3), (-0.9, 0.5)])
def test_p3_parseval_per_angle(oracle_mod, nxg, nyg):
    """With tau = t - n.r monotone, A(w) = int (f/kappa) e^{i w tau} d tau, so
    int_0^inf |A|^2 dw = pi int |f|^2/kappa dt (kappa = 1 - n.beta), i.e.
    int_0^inf out dw = (1/4pi) int |f|^2/kappa dt  -- Jackson's dI/dOmega.  Same for J.
    RHS uses the UNEXPANDED f of eq. (2) (differs by O(1/gamma^2) = 1e-6).  |A|^2 is
    band-limited to |tau| <= tau_N - tau_0, so a uniform sum with step < 2pi/span is
    exact up to the cut-off at 60 w_1 (harmonics ~K^(2n), negligible).  Pins 1/4pi^2,
    g, |f| and the phase scale jointly.  Tolerance 2e-5."""
    gamma = 1000.0
    tr = _undulator(gamma, 0.3142, 4, 4001, B_over_A=0.35)
    nx, ny = nxg / gamma, nyg / gamma
    f, hJ, tau, kappa = exact_integrands(tr, nx, ny)
    w = trapezoid_weights(tr["t"])
    rhs = float((w * (f ** 2).sum(0) / kappa).sum() / (4 * LD(math.pi)))
    rhs_j = float((w * hJ ** 2 / kappa).sum() * LD(math.pi))
    dw = 2 * math.pi / float(tau[-1] - tau[0]) / 4
    om = np.arange(0, int(60 * 2 * gamma ** 2 * W0 / dw) + 1) * dw
    out, amp = oracle_mod.points(tr, om, np.full_like(om, nx), np.full_like(om, ny),
                                 return_amplitudes=True)
    lhs = (out[1:].sum() + 0.5 * out[0]) * dw
    j2 = np.abs(amp[:, 3]) ** 2
    lhs_j = (j2[1:].sum() + 0.5 * j2[0]) * dw
    assert lhs == pytest.approx(rhs, rel=2e-5)
    assert lhs_j == pytest.approx(rhs_j, rel=2e-5)


def test_p3b_lienard_total_energy(oracle_mod):
    """north_star (c): int dw dOmega out = int (2/3) gamma^6 [bdot^2 - (beta x bdot)^2] dt
    (e^2 = 1).  Coarse: angles on a 33 x 33 grid to +-5/gamma miss the tail of
    dI/dOmega ~ (1+gamma^2 theta^2)^-3..-5  (few %) -> tolerance 5 %."""
    gamma, K = 200.0, 0.2
    tr = _undulator(gamma, K, 2, 801)
    na = 33
    th = np.linspace(-5 / gamma, 5 / gamma, na)
    dth = th[1] - th[0]
    w1 = 2 * gamma ** 2 * W0
    om = np.linspace(0, 8 * w1, 161)
    W, Y, X = np.meshgrid(om, th, th, indexing="ij")
    out = oracle_mod.points(tr, W.ravel(), X.ravel(), Y.ravel()).reshape(W.shape)
    wt = np.full(len(om), om[1] - om[0])
    wt[0] *= 0.5
    total = float((out * wt[:, None, None]).sum() * dth * dth)
    g = LD(gamma)
    beta0 = 1 - 1 / (2 * g * g)
    b = np.stack([tr["vx"], tr["vy"], beta0 + tr["dvz"]]).astype(LD)
    bd = np.stack([tr["ax"], tr["ay"], tr["az"]]).astype(LD)
    cr = np.stack([b[1] * bd[2] - b[2] * bd[1], b[2] * bd[0] - b[0] * bd[2],
                   b[0] * bd[1] - b[1] * bd[0]])
    power = (2 / LD(3)) * g ** 6 * ((bd ** 2).sum(0) - (cr ** 2).sum(0))
    lien = float((trapezoid_weights(tr["t"]) * power).sum())
    assert total == pytest.approx(lien, rel=0.05)


# --------------------------------------------------------------------------- P4
@pytest.mark.parametrize("gth", [0.0, 0.8])
def test_p4_harmonic_position(oracle_mod, gth):
    """w_1 = 2 gamma^2 w_0 / (1 + gamma^2 theta^2 + K^2/2) (north_star (b); PAPER.md:177:
    peak positions are kinematic).  20 periods: the finite-train pull is O(1/N_u^2);
    scan step 0.05 % -> tolerance 0.3 %."""
    gamma, K = 1000.0, 0.3142
    tr = _undulator(gamma, K, 20, 4001)
    w1 = 2 * gamma ** 2 * W0 / (1 + gth ** 2 + K ** 2 / 2)
    om = w1 * np.linspace(0.9, 1.1, 401)
    # emission in the plane perpendicular to the oscillation keeps f_x on its maximum
    out = oracle_mod.points(tr, om, np.zeros_like(om), np.full_like(om, gth / gamma))
    assert om[np.argmax(out)] == pytest.approx(w1, rel=3e-3)
    # without the K^2/2 term the prediction would be off by (K^2/2)/(1+gth^2) = 3.0-4.9 %
    assert abs(om[np.argmax(out)] / (2 * gamma ** 2 * W0 / (1 + gth ** 2)) - 1) > 0.02


# --------------------------------------------------------------------------- P5
def test_p5_weak_undulator_closed_form_on_axis(oracle_mod):
    """K -> 0, on axis: out = (1/4pi^2) 4 gamma^4 A^2 w0^6 * 4 sin^2(Om T/2)/(w0^2-Om^2)^2,
    Om = w/(2 gamma^2); peak = gamma^2 K^2 N_u^2 (textbook weak-undulator peak, e^2 = 1).
    Corrections are O(K^2) = 1e-7 and O((w0 dt)^2/12) = 3e-6 -> tolerance 2e-5 of peak."""
    gamma, K, Nu = 1000.0, 3e-4, 4
    tr = _undulator(gamma, K, Nu, 4001)
    A = K / (gamma * W0)
    T = Nu * 2 * math.pi / W0
    w1 = 2 * gamma ** 2 * W0
    om = w1 * np.linspace(0.3, 1.7, 57)
    Om = om / (2 * gamma ** 2)
    with np.errstate(invalid="ignore", divide="ignore"):
        shape = 4 * np.sin(Om * T / 2) ** 2 / (W0 ** 2 - Om ** 2) ** 2
    shape = np.where(np.isclose(Om, W0, rtol=1e-12), T ** 2 / (4 * W0 ** 2), shape)
    expect = 4 * gamma ** 4 * A ** 2 * W0 ** 6 * shape / (4 * math.pi ** 2)
    peak = gamma ** 2 * K ** 2 * Nu ** 2
    out = oracle_mod.points(tr, om, np.zeros_like(om), np.zeros_like(om))
    assert np.max(np.abs(out - expect)) <= 2e-5 * peak
    assert out.max() == pytest.approx(peak, rel=1e-4)      # the grid contains w = w_1


def test_p5_weak_undulator_closed_form_off_axis(oracle_mod):
    """K -> 0, off axis: f_x = -[(ny^2-nx^2)/2 + 1/2g^2] g0 ax, f_y = nx ny g0 ax,
    f_z = (1/2g^2 - th^2/2) nx g0 ax, g0 = 4 g^4/(1+g^2 th^2)^2, Om = w (1+g^2 th^2)/(2 g^2).
    The dropped n_x x(t) phase term is O(K) -> tolerance 3 K of the peak."""
    gamma, K, Nu = 1000.0, 3e-4, 4
    tr = _undulator(gamma, K, Nu, 4001)
    A = K / (gamma * W0)
    T = Nu * 2 * math.pi / W0
    nx, ny = 0.5 / gamma, -0.7 / gamma
    th2 = nx * nx + ny * ny
    g0 = 4 * gamma ** 4 / (1 + gamma ** 2 * th2) ** 2
    a = 1 / (2 * gamma ** 2)
    coef = (((ny * ny - nx * nx) / 2 + a) ** 2 + (nx * ny) ** 2 + ((a - th2 / 2) * nx) ** 2) * g0 ** 2
    w1 = 2 * gamma ** 2 * W0 / (1 + gamma ** 2 * th2)
    om = w1 * np.linspace(0.3, 1.7, 56)
    Om = om * (1 + gamma ** 2 * th2) / (2 * gamma ** 2)
    time_int2 = (A * W0 ** 2) ** 2 * W0 ** 2 * 4 * np.sin(Om * T / 2) ** 2 / (W0 ** 2 - Om ** 2) ** 2
    expect = coef * time_int2 / (4 * math.pi ** 2)
    out = oracle_mod.points(tr, om, np.full_like(om, nx), np.full_like(om, ny))
    assert np.max(np.abs(out - expect)) <= 3 * K * expect.max()


# --------------------------------------------------------------------------- P6
def test_p6_brute_force_unexpanded(oracle_mod):
    """Brute force of the UNEXPANDED eqs. (1)-(2), (11)-(12) (exact n_z, beta_z) in numpy
    longdouble on tiny inputs.  The expansion drops terms two orders in 1/gamma higher
    (PAPER.md:28), so every component -- A_x, A_y, A_z and J -- must agree to
    C/gamma^2 and improve x100 per decade of gamma at fixed K and gamma*theta.
    A wrong sign, a dropped term or a swapped index gives an O(1) mismatch."""
    pts = [(0.5, 0.3, 0.2), (0.9, -0.6, 0.4), (1.7, 0.1, -0.8), (2.6, 0.7, 0.7)]
    worst = {}
    for gamma in (30.0, 300.0, 3000.0):
        tr = _undulator(gamma, 0.3, 3, 1501, B_over_A=0.4)
        w1 = 2 * gamma ** 2 * W0
        errs = []
        for wf, gx, gy in pts:
            om, nx, ny = wf * w1, gx / gamma, gy / gamma
            _, amp = oracle_mod.points(tr, [om], [nx], [ny], return_amplitudes=True)
            A_ex, J_ex = exact_amplitudes(tr, om, nx, ny)
            perp = math.hypot(abs(A_ex[0]), abs(A_ex[1]))
            errs.append([abs(amp[0, 0] - A_ex[0]) / perp, abs(amp[0, 1] - A_ex[1]) / perp,
                         abs(amp[0, 2] - A_ex[2]) / abs(A_ex[2]), abs(amp[0, 3] - J_ex) / abs(J_ex)])
        worst[gamma] = np.max(errs, axis=0)
    assert np.all(worst[30.0] < 0.2)
    assert np.all(worst[300.0] < 2e-3)
    assert np.all(worst[3000.0] < 2e-5)
    assert np.all(worst[300.0] / worst[3000.0] > 80) and np.all(worst[300.0] / worst[3000.0] < 120)


# --------------------------------------------------------------------------- P7
def test_p7_variant_identities(oracle_mod):
    """(i) Lambda -> 0: both semi-classical variants reduce to classical;
    (ii) spin-0(w) = (1-u) classical(w*)                       (eq. 9);
    (iii) spin-1/2 - (1+(1-u)^2)/(2(1-u)) spin-0 = u^2 |J|^2 / (8 pi^2 gamma^2) >= 0
          (eq. 10).  Rounding level: 1e-15 relative."""
    wl = workloads.make("cfg3", n=4000, n_omega=12, n_th=3)
    lam = wl.hbarc_over_E
    w, nx, ny = oracle_mod.grid_points(wl.omega, wl.thx, wl.thy)
    u = w * lam
    cl = oracle_mod.points(wl.traj, w, nx, ny, CL)
    assert np.array_equal(oracle_mod.points(wl.traj, w, nx, ny, S0, 0.0), cl)
    assert np.array_equal(oracle_mod.points(wl.traj, w, nx, ny, SH, 0.0), cl)
    s0 = oracle_mod.points(wl.traj, w, nx, ny, S0, lam)
    sh, amp = oracle_mod.points(wl.traj, w, nx, ny, SH, lam, return_amplitudes=True)
    # w* rounded to double here, while the oracle keeps it in long double:
    # the phase w* psi (<= 1e5 rad on this input) moves by <= 1e-11 -> 1e-9 relative
    cl_star = oracle_mod.points(wl.traj, w / (1 - u), nx, ny, CL)
    np.testing.assert_allclose(s0, (1 - u) * cl_star, rtol=1e-9)
    extra = sh - (1 + (1 - u) ** 2) / (2 * (1 - u)) * s0
    g0 = wl.traj["gamma"][0]
    expect = u ** 2 * np.abs(amp[:, 3]) ** 2 / (8 * math.pi ** 2 * g0 ** 2)
    np.testing.assert_allclose(extra, expect, rtol=0, atol=4e-16 * sh.max())
    # the bracket of eq. 10 also directly, to rounding
    S = (np.abs(amp[:, :3]) ** 2).sum(1)
    direct = ((1 + (1 - u) ** 2) / 2 * S + u ** 2 / (2 * g0 ** 2) * np.abs(amp[:, 3]) ** 2) / (4 * math.pi ** 2)
    np.testing.assert_allclose(sh, direct, rtol=1e-14)


def test_p7b_semi_classical_domain(oracle_mod):
    """u = hbar w / E >= 1 has no photon (E* <= 0): rejected (Q10)."""
    wl = workloads.make("cfg1", n=100, n_omega=2, n_th=1)
    with pytest.raises(ValueError):
        oracle_mod.points(wl.traj, [2.0], [0.0], [0.0], S0, 0.5)


# --------------------------------------------------------------------------- P8
def test_p8_J_by_parts(oracle_mod):
    """With az = d(dvz)/dt:  dq/dt = -(az + nx ax + ny ay) = -h/g, hence
    int e^{i w psi} dt = [e^{i w psi}/(i w q)] - J/(i w)  =>  J = [e^{i w psi}/q] - i w int e^{i w psi} dt.
    Pins the definition, sign and 1/q^2 of the J integrand independently of eq. (12).
    Trapezoid error O((w q dt)^2) ~ 1e-5 at 4000 samples, 4x smaller... tolerance 1e-4."""
    gamma = 1000.0
    tr = _undulator(gamma, 0.3142, 4, 16001, B_over_A=0.35)
    nx, ny = 0.4 / gamma, -0.3 / gamma
    om = 0.8 * 2 * gamma ** 2 * W0
    _, amp = oracle_mod.points(tr, [om], [nx], [ny], return_amplitudes=True)
    t = tr["t"].astype(LD)
    a = 1 / (2 * LD(gamma) ** 2)
    th2 = LD(nx) ** 2 + LD(ny) ** 2
    q = a + th2 / 2 - tr["dvz"] - LD(nx) * tr["vx"] - LD(ny) * tr["vy"]
    psi = (a + th2 / 2) * t - tr["dz"] - LD(nx) * tr["x"] - LD(ny) * tr["y"]
    ph = LD(om) * psi
    w = trapezoid_weights(t)
    plain = complex((w * np.cos(ph)).sum(), (w * np.sin(ph)).sum())
    edge = (complex(np.cos(ph[-1]), np.sin(ph[-1])) / float(q[-1])
            - complex(np.cos(ph[0]), np.sin(ph[0])) / float(q[0]))
    J_expect = edge - 1j * om * plain
    assert abs(amp[0, 3] - J_expect) <= 1e-4 * abs(J_expect)


# --------------------------------------------------------------------------- P10
def test_p10_independent_reimplementation(oracle_mod):
    """A second implementation, written vectorised in numpy longdouble from PAPER.md
    eqs. (3)-(7), on a non-uniform time grid with varying gamma (catches C-level slips:
    weights, indexing, operand order).  Not a pin by itself; agreement 1e-15."""
    rng = np.random.Generator(np.random.PCG64(7))
    n = 257
    t = np.sort(rng.uniform(0, 3e-6, n))
    tr = {k: rng.normal(0, 1, n) * s for k, s in
          [("x", 1e-10), ("y", 1e-10), ("vx", 2e-5), ("vy", 2e-5), ("ax", 30.0), ("ay", 30.0),
           ("az", 1e-3), ("dz", 1e-15), ("dvz", 1e-10)]}
    tr["dvz"] = -np.abs(tr["dvz"])
    tr["t"] = t
    tr["gamma"] = 8000.0 + 50.0 * rng.uniform(size=n)
    om, nx, ny, lam = 3.1e13, 7e-5, -4e-5, 1.1e-15
    L = {k: v.astype(LD) for k, v in tr.items()}
    a = 1 / (2 * L["gamma"] ** 2)
    nxl, nyl = LD(nx), LD(ny)
    th2 = nxl ** 2 + nyl ** 2
    br = -th2 / 2 - L["dvz"] + a
    g = (a + th2 / 2 - L["dvz"] - nxl * L["vx"] - nyl * L["vy"]) ** -2
    fx = ((L["az"] + nyl * L["ay"]) * (nxl - L["vx"]) - (nyl * (nyl - L["vy"]) + br) * L["ax"]) * g
    fy = ((L["az"] + nxl * L["ax"]) * (nyl - L["vy"]) - (nxl * (nxl - L["vx"]) + br) * L["ay"]) * g
    fz = (br * (nxl * L["ax"] + nyl * L["ay"])
          - (nxl * (nxl - L["vx"]) + nyl * (nyl - L["vy"])) * L["az"]) * g
    hj = (nxl * L["ax"] + nyl * L["ay"] + L["az"]) * g
    u = LD(om) * LD(lam)
    wst = LD(om) / (1 - u)
    ph = wst * ((a + th2 / 2) * L["t"] - L["dz"] - nxl * L["x"] - nyl * L["y"])
    w = trapezoid_weights(t)
    c, s = np.cos(ph), np.sin(ph)
    S = sum((w * f * c).sum() ** 2 + (w * f * s).sum() ** 2 for f in (fx, fy, fz))
    J2 = (w * hj * c).sum() ** 2 + (w * hj * s).sum() ** 2
    four_pi2 = 4 * (4 * np.arctan(LD(1))) ** 2      # pi in long double
    expect = {
        CL: None,
        S0: (1 - u) * S / four_pi2,
        SH: ((1 + (1 - u) ** 2) / 2 * S + u ** 2 / (2 * L["gamma"][0] ** 2) * J2) / four_pi2,
    }
    for model in (S0, SH):
        got = oracle_mod.points(tr, [om], [nx], [ny], model, lam)[0]
        assert got == pytest.approx(float(expect[model]), rel=1e-15)
    phc = LD(om) * ((a + th2 / 2) * L["t"] - L["dz"] - nxl * L["x"] - nyl * L["y"])
    cc, sc = np.cos(phc), np.sin(phc)
    Sc = sum((w * f * cc).sum() ** 2 + (w * f * sc).sum() ** 2 for f in (fx, fy, fz))
    got = oracle_mod.points(tr, [om], [nx], [ny], CL)[0]
    assert got == pytest.approx(float(Sc / four_pi2), rel=1e-15)


# --------------------------------------------------------------- precision of the truth
def test_long_double_is_accurate_enough(oracle_mod):
    """The parity truth is the long-double build.  Against the __float128 build of the same
    source on a large-phase input (cfg3-like, |phi| up to ~1e6 rad) it must sit far inside
    the parity tolerance max(1e-9 |S|, 1e-12 S_max): here <= 1e-11 |S| + 1e-14 S_max."""
    wl = workloads.make("cfg3", n=200000, n_omega=512, n_th=64)
    idx = workloads.sample_points(wl, 24, seed=99)
    idx = np.concatenate([idx, [wl.n_points - 1]])
    w, nx, ny = workloads.points_of(wl, idx)
    ld = oracle_mod.points(wl.traj, w, nx, ny, SH, wl.hbarc_over_E, variant="ld")
    qd = oracle_mod.points(wl.traj, w, nx, ny, SH, wl.hbarc_over_E, variant="quad")
    assert np.all(np.abs(ld - qd) <= 1e-11 * np.abs(qd) + 1e-14 * qd.max())


# --------------------------------------------------------------- ensemble
def test_ensemble_is_sum_of_members(oracle_mod):
    """spectrum of sections / particles = sum of their spectra.
    Ragged lengths; accumulate adds to a previous partial ensemble."""
    wl = workloads.make("cfg4", count=5, n=600, n_omega=4, n_th=3)
    nvec = np.array([600, 431, 2, 600, 77], dtype=np.int64)
    w, nx, ny = oracle_mod.grid_points(wl.omega, wl.thx, wl.thy)
    tot = oracle_mod.ensemble_points(wl.batch, nvec, w, nx, ny, CL)
    ref = np.zeros_like(tot)
    for p in range(5):
        tr = {k: wl.batch[k][p, : nvec[p]] for k in workloads.FIELDS}
        ref += oracle_mod.points(tr, w, nx, ny, CL)
    np.testing.assert_allclose(tot, ref, rtol=1e-14)
    first = oracle_mod.ensemble_points({k: v[:2] for k, v in wl.batch.items()}, nvec[:2], w, nx, ny, CL)
    rest = oracle_mod.ensemble_points({k: v[2:] for k, v in wl.batch.items()}, nvec[2:], w, nx, ny, CL,
                                      accumulate_into=first)
    np.testing.assert_allclose(rest, tot, rtol=1e-14)
    lam = np.linspace(1e-17, 3e-17, 5)
    sh = oracle_mod.ensemble_points(wl.batch, nvec, w, nx, ny, SH, lam)
    ref = np.zeros_like(sh)
    for p in range(5):
        tr = {k: wl.batch[k][p, : nvec[p]] for k in workloads.FIELDS}
        ref += oracle_mod.points(tr, w, nx, ny, SH, lam[p])
    np.testing.assert_allclose(sh, ref, rtol=1e-14)


def test_grid_order(oracle_mod):
    """Cube order (Q11): out[i_w, i_y, i_x]; x fastest."""
    wl = workloads.make("cfg1", n=300, n_omega=3, n_th=4)
    cube = oracle_mod.grid(wl.traj, wl.omega, wl.thx[:4], wl.thy[:2])
    assert cube.shape == (3, 2, 4)
    one = oracle_mod.points(wl.traj, [wl.omega[2]], [wl.thx[3]], [wl.thy[1]])[0]
    assert cube[2, 1, 3] == one


# --------------------------------------------------------------------------- symmetries of eq. (1)
def _sym_workload():
    import workloads
    wl = workloads.make("cfg5", n=1500, n_omega=5, n_th=4, seed=9)
    rng = np.random.Generator(np.random.PCG64(4))
    nx = rng.uniform(-5e-5, 5e-5, 12)
    ny = rng.uniform(-5e-5, 5e-5, 12)
    om = np.repeat(wl.omega[1:4], 4)
    return wl, om, nx, ny


@pytest.mark.parametrize("model", [0, 2])
def test_translation_and_time_shift_invariance(oracle_mod, model):
    """A constant shift of x, y or of the time origin multiplies every amplitude of eq. (1) by one common
    phase factor: the spectrum does not change (catches a wrong sign or coefficient in eq. 7)."""
    wl, om, nx, ny = _sym_workload()
    lam = wl.hbarc_over_E
    base = oracle_mod.points(wl.traj, om, nx, ny, model, lam)
    tr = {k: v.copy() for k, v in wl.traj.items()}
    tr["x"] += 3e-10
    tr["y"] -= 1e-10
    np.testing.assert_allclose(oracle_mod.points(tr, om, nx, ny, model, lam), base, rtol=2e-9)
    tr = {k: v.copy() for k, v in wl.traj.items()}
    tr["t"] += 2.5e-7
    np.testing.assert_allclose(oracle_mod.points(tr, om, nx, ny, model, lam), base, rtol=2e-9)


@pytest.mark.parametrize("model", [0, 2])
def test_mirror_and_axis_swap_symmetry(oracle_mod, model):
    """Mirroring the trajectory in x (x, vx, ax -> -x, -vx, -ax) maps the spectrum at n_x to the one at
    -n_x; exchanging the roles of x and y maps (n_x, n_y) to (n_y, n_x).  The second one pins eq. (4)
    against eq. (3): they must be each other's image under x <-> y."""
    wl, om, nx, ny = _sym_workload()
    lam = wl.hbarc_over_E
    base = oracle_mod.points(wl.traj, om, nx, ny, model, lam)
    tr = {k: v.copy() for k, v in wl.traj.items()}
    for k in ("x", "vx", "ax"):
        tr[k] = -tr[k]
    np.testing.assert_allclose(oracle_mod.points(tr, om, -nx, ny, model, lam), base, rtol=1e-12)
    tr = {k: v.copy() for k, v in wl.traj.items()}
    for a, b in (("x", "y"), ("vx", "vy"), ("ax", "ay")):
        tr[a], tr[b] = wl.traj[b].copy(), wl.traj[a].copy()
    np.testing.assert_allclose(oracle_mod.points(tr, om, ny, nx, model, lam), base, rtol=1e-12)


# --------------------------------------------------------------------------- P9
@pytest.mark.parametrize("xi,u", [(0.3, 0.0), (1.0, 0.0), (0.5, 0.3), (1.5, 0.6)])
def test_p9_quantum_synchrotron_limit(oracle_mod, xi, u):
    """Circular arc (constant v'_x = a0, deflection +-10/gamma), central in-plane direction n_x = 0, spectrum
    integrated over n_y: the energy per frequency and per in-plane angle is (dP/dw)/a0 with the textbook
    (Baier-Katkov) synchrotron spectrum
        dP/dw = w / (sqrt(3) pi gamma^2) [ int_xi^inf K_5/3 + u^2/(1-u) K_2/3(xi) ]      (units of e^2, c = 1),
    xi = w*/w_c, w_c = 3 gamma^3 a0 / 2; spin-0: the first term only; u = 0: classical (Jackson 14.91).
    Pins eq. (10) with its J term and coefficient u^2/2gamma^2 (reading Q4), the substitution w -> w*
    (eqs. 8-9, reading Q3) and the absolute normalisation against a result the oracle does not contain."""
    from scipy.integrate import quad
    from scipy.special import kv
    gamma, a0, n = 1000.0, 1.0, 40001
    t = np.linspace(-10.0 / gamma / a0, 10.0 / gamma / a0, n)
    vx = a0 * t
    z = np.zeros(n)
    tr = dict(t=t, x=a0 * t * t / 2, y=z.copy(), vx=vx, vy=z.copy(), ax=np.full(n, a0), ay=z.copy(),
              dvz=-vx * vx / 2, dz=-a0 * a0 * t ** 3 / 6, az=-a0 * a0 * t, gamma=np.full(n, gamma))
    w_star = xi * 1.5 * gamma ** 3 * a0
    om = w_star * (1 - u)
    lam = u / om
    ny = np.linspace(-8 / gamma, 8 / gamma, 321)
    i53 = quad(lambda x: kv(5 / 3, x), xi, np.inf)[0]
    pref = om / (math.sqrt(3) * math.pi * gamma ** 2) / a0
    want = {0: None, 1: pref * i53, 2: pref * (i53 + u * u / (1 - u) * kv(2 / 3, xi))}
    for model in (1, 2):
        out = oracle_mod.points(tr, np.full(ny.size, om), np.zeros(ny.size), ny, model, lam)
        got = np.trapezoid(out, ny)
        assert got == pytest.approx(want[model], rel=1e-3), f"model {model}"
    if u == 0.0:
        out = oracle_mod.points(tr, np.full(ny.size, om), np.zeros(ny.size), ny, 0, 0.0)
        assert np.trapezoid(out, ny) == pytest.approx(want[1], rel=1e-3)
    else:                                             # the spin term is not small here: it must be there
        assert want[2] / want[1] - 1 > 0.05


# --------------------------------------------------------------------------- quadrature rule (Q1) and gamma reading (Q6)
def _zero_phase_trajectory(t, ax, gamma):
    """A trajectory whose eq. (3) integrand at omega = 0, n = (0, 0) is the closed form -2 gamma^2 ax:
    with n = 0, vx = vy = dvz = az = 0 eqs. (3), (6) give D = q = 1/(2 gamma^2), g = 4 gamma^4 and
    f_x = -D ax g = -2 gamma^2 ax; the phase of eq. (7) is 0 at omega = 0."""
    tr = {k: np.zeros(len(t)) for k in workloads.FIELDS}
    tr["t"] = np.asarray(t, dtype=np.float64)
    tr["ax"] = np.asarray(ax, dtype=np.float64)
    tr["gamma"] = np.broadcast_to(np.asarray(gamma, dtype=np.float64), tr["t"].shape).copy()
    return tr


def _ragged_times(n, seed):
    """Non-uniform abscissae with dyadic spacings (exact in double), different first and last steps."""
    rng = np.random.default_rng(seed)
    steps = rng.integers(1, 9, size=n - 1).astype(np.float64) * 2.0 ** -10
    steps[0], steps[-1] = 5 * 2.0 ** -10, 3 * 2.0 ** -10
    return np.concatenate([[0.25], 0.25 + np.cumsum(steps)])


def test_q1_trapezoid_weights_are_exact_for_a_linear_integrand(oracle_mod):
    """Reading Q1 (the paper only says "points in time"): composite trapezoid on the
    given t_k.  That rule integrates a LINEAR integrand exactly on any grid, end intervals included:
    with ax = c0 + c1 t, non-zero at both ends, A_x = -2 gamma^2 [c0 (t_N - t_0) + c1 (t_N^2 - t_0^2)/2].
    Inputs are dyadic rationals, so the closed form is exact in double and the oracle's long-double sum
    has no rounding to speak of: tolerance 1e-15 relative.  A wrong end weight (un-halved, or dropped)
    changes the sum by O(h/T) ~ 1e-3 and fails; so does any interior weight that is not (t_{k+1}-t_{k-1})/2."""
    gamma = 64.0
    for n, seed in ((2, 1), (3, 2), (57, 3), (400, 4)):
        t = _ragged_times(n, seed)
        c0, c1 = 0.75, -0.5
        tr = _zero_phase_trajectory(t, c0 + c1 * t, gamma)
        _, amp = oracle_mod.points(tr, [0.0], [0.0], [0.0], return_amplitudes=True)
        expect = -2 * gamma ** 2 * (c0 * (t[-1] - t[0]) + c1 * (t[-1] ** 2 - t[0] ** 2) / 2)
        assert amp[0, 0].imag == 0.0
        assert abs(amp[0, 0].real - expect) <= 1e-15 * abs(expect), (n, amp[0, 0].real, expect)
        assert amp[0, 1] == 0 and amp[0, 2] == 0 and amp[0, 3] == 0     # ay = az = 0, n = 0


def test_q1_rule_is_the_trapezoid_not_a_higher_order_one(oracle_mod):
    """For a QUADRATIC integrand the composite trapezoid rule has the closed-form excess
    sum_i h_i^3 / 6 per unit of curvature over the exact integral (interval error h^3 f''/12 with f'' = 2);
    Simpson-type rules would be exact and a midpoint/rectangle rule has a different excess.  1e-14 relative."""
    gamma = 64.0
    t = _ragged_times(200, 7)
    tr = _zero_phase_trajectory(t, t * t, gamma)
    _, amp = oracle_mod.points(tr, [0.0], [0.0], [0.0], return_amplitudes=True)
    h = np.diff(t)
    expect = -2 * gamma ** 2 * ((t[-1] ** 3 - t[0] ** 3) / 3 + (h ** 3).sum() / 6)
    assert abs(amp[0, 0].real - expect) <= 1e-14 * abs(expect)


def test_q6_gamma_is_used_sample_wise_in_the_integrand(oracle_mod):
    """Reading Q6, first half: 1/(2 gamma_k^2) enters eqs. (3)-(7) with the sample's own gamma_k.  With
    gamma_k^2 linear in t and constant ax, f_x = -2 gamma_k^2 ax is linear, so the trapezoid sum is exact:
    A_x = -2 ax [g2_0 T + s (t_N^2 - t_0^2)/2 - s t_0 T].  A single gamma (first, last or mean) for the whole
    trajectory gives a different number at the 10 % level."""
    t = _ragged_times(120, 11)
    g2 = 4096.0 + 2048.0 * (t - t[0])                      # gamma^2, dyadic
    gam = np.sqrt(g2)
    tr = _zero_phase_trajectory(t, np.full_like(t, 0.5), gam)
    _, amp = oracle_mod.points(tr, [0.0], [0.0], [0.0], return_amplitudes=True)
    T = t[-1] - t[0]
    expect = -2 * 0.5 * (4096.0 * T + 2048.0 * ((t[-1] ** 2 - t[0] ** 2) / 2 - t[0] * T))
    # gamma_k = sqrt(g2) is rounded to double before the oracle squares it again: 2 ulp per sample
    assert abs(amp[0, 0].real - expect) <= 1e-15 * abs(expect) * 4


def test_q6_j_coefficient_uses_the_first_gamma(oracle_mod):
    """Reading Q6, second half: the coefficient w^2/(2 E^2 gamma^2) of eq. (10) is taken with
    gamma_0 = gamma[0] (E is fixed "to the value at entering the section").  On a trajectory whose
    gamma falls by a factor 2, identity P7(iii) isolates the coefficient:
        [spin-1/2 - (1+(1-u)^2)/(2(1-u)) spin-0] * 8 pi^2 / (u^2 |J|^2) = 1/gamma_0^2,
    which differs by 4x from the last sample's gamma and by ~2x from the mean."""
    wl = workloads.make("cfg3", n=3000, n_omega=6, n_th=3)
    tr = {k: v.copy() for k, v in wl.traj.items()}
    g0 = tr["gamma"][0]
    tr["gamma"] = g0 * np.linspace(1.0, 0.5, len(tr["t"]))
    lam = wl.hbarc_over_E
    w, nx, ny = oracle_mod.grid_points(wl.omega[-3:], wl.thx, wl.thy)      # u = 0.79 ... 0.8: J term matters
    u = w * lam
    s0 = oracle_mod.points(tr, w, nx, ny, S0, lam)
    sh, amp = oracle_mod.points(tr, w, nx, ny, SH, lam, return_amplitudes=True)
    j2 = np.abs(amp[:, 3]) ** 2
    coeff = (sh - (1 + (1 - u) ** 2) / (2 * (1 - u)) * s0) * 8 * math.pi ** 2 / (u ** 2 * j2)
    # the difference cancels ~ S/(u^2 J^2/gamma^2) digits: keep points where the J term is not negligible
    keep = u ** 2 * j2 / g0 ** 2 > 1e-6 * sh * 8 * math.pi ** 2
    assert keep.sum() >= 5
    np.testing.assert_allclose(coeff[keep], 1 / g0 ** 2, rtol=1e-8)
    assert np.all(np.abs(coeff[keep] * tr["gamma"][-1] ** 2 - 1) > 0.5)
