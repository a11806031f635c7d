"""Independent references the oracle is pinned against (tests only).

Nothing here is the paper's EXPANDED form (eqs. 3-7): these are the UNEXPANDED
eqs. (1)-(2), (11)-(12) of PAPER.md:23-28, 66-68 with exact n_z and beta_z,
textbook closed forms, and plain numpy quadrature -- all in numpy longdouble.
"""
from __future__ import annotations

import numpy as np

LD = np.longdouble


def trapezoid_weights(t):
    t = np.asarray(t, dtype=LD)
    w = np.empty_like(t)
    w[0] = (t[1] - t[0]) / 2
    w[-1] = (t[-1] - t[-2]) / 2
    w[1:-1] = (t[2:] - t[:-2]) / 2
    return w


def exact_vectors(traj, nx, ny):
    """beta, beta_dot, r, n as exact 3-vectors from the SoA arrays.

    beta_z = beta0 + dvz and z = beta0 t + dz with beta0 = 1 - 1/(2 gamma^2)
    (definitions of PAPER.md:28), n_z = sqrt(1 - nx^2 - ny^2)."""
    g = np.asarray(traj["gamma"], dtype=LD)
    beta0 = 1 - 1 / (2 * g * g)
    t = np.asarray(traj["t"], dtype=LD)
    beta = np.stack([np.asarray(traj["vx"], dtype=LD), np.asarray(traj["vy"], dtype=LD),
                     beta0 + np.asarray(traj["dvz"], dtype=LD)])
    bdot = np.stack([np.asarray(traj[k], dtype=LD) for k in ("ax", "ay", "az")])
    r = np.stack([np.asarray(traj["x"], dtype=LD), np.asarray(traj["y"], dtype=LD),
                  beta0 * t + np.asarray(traj["dz"], dtype=LD)])
    nx, ny = LD(nx), LD(ny)
    n = np.array([nx, ny, np.sqrt(1 - nx * nx - ny * ny)], dtype=LD)
    return t, beta, bdot, r, n


def _cross(a, b):
    return np.stack([a[1] * b[2] - a[2] * b[1], a[2] * b[0] - a[0] * b[2], a[0] * b[1] - a[1] * b[0]])


def exact_integrands(traj, nx, ny):
    """f = n x [(n - beta) x beta_dot] / (1 - n.beta)^2   (eq. 2, brackets as in eq. 11),
    hJ = n.beta_dot / (1 - n.beta)^2                      (eq. 12),
    tau = t - n.r                                         (phase / omega, eq. 1),
    kappa = 1 - n.beta."""
    t, beta, bdot, r, n = exact_vectors(traj, nx, ny)
    nb = n[:, None] - beta
    kappa = 1 - (n[:, None] * beta).sum(0)
    inner = _cross(nb, bdot)
    f = _cross(np.broadcast_to(n[:, None], inner.shape), inner) / kappa ** 2
    hJ = (n[:, None] * bdot).sum(0) / kappa ** 2
    tau = t - (n[:, None] * r).sum(0)
    return f, hJ, tau, kappa


def exact_amplitudes(traj, omega_ph, nx, ny):
    """Trapezoid sums of the UNEXPANDED integrands: complex A (3,), J."""
    f, hJ, tau, _ = exact_integrands(traj, nx, ny)
    w = trapezoid_weights(traj["t"])
    ph = LD(omega_ph) * tau
    c, s = np.cos(ph), np.sin(ph)
    A = np.array([complex((w * f[i] * c).sum(), (w * f[i] * s).sum()) for i in range(3)])
    J = complex((w * hJ * c).sum(), (w * hJ * s).sum())
    return A, J


def planar_2d_trajectory(gamma, A, B, w0, periods, n):
    """x = A sin(w0 t), y = B sin(2 w0 t): analytic v, a; dvz = -(vx^2+vy^2)/2 with its
    analytic time integral dz; az = d(dvz)/dt.  Acceleration vanishes at both ends when
    `periods` is an integer."""
    t = (periods * 2 * np.pi / w0) * np.arange(n) / (n - 1)
    vx = A * w0 * np.cos(w0 * t)
    vy = 2 * B * w0 * np.cos(2 * w0 * t)
    ax = -A * w0 ** 2 * np.sin(w0 * t)
    ay = -4 * B * w0 ** 2 * np.sin(2 * w0 * t)
    dz = -0.5 * ((A * w0) ** 2 * (t / 2 + np.sin(2 * w0 * t) / (4 * w0))
                 + (2 * B * w0) ** 2 * (t / 2 + np.sin(4 * w0 * t) / (8 * w0)))
    return {"t": t, "x": A * np.sin(w0 * t), "y": B * np.sin(2 * w0 * t), "vx": vx, "vy": vy,
            "ax": ax, "ay": ay, "dvz": -0.5 * (vx ** 2 + vy ** 2), "dz": dz,
            "az": -(vx * ax + vy * ay), "gamma": np.full(n, float(gamma))}
