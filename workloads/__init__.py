"""Seeded synthetic inputs shaped like the paper's channeling workloads.

This module serves BOTH the CPU oracle (``oracle/``) and the CUDA path
(``paper_1910_10391_b200``) and therefore holds none of the method's arithmetic:
it only integrates toy equations of motion and lays out grids.  It imports
neither side.  numpy only; deterministic (single-threaded PCG64 streams, fixed
operation order).

The five configurations are BASELINE.json ``configs[0..4]`` with the open choices
fixed as in SURVEY.md section 8(d) / DESIGN.md "Input recipe".  They stand in for
the paper's own trajectories (Doyle-Turner potentials + RK45 + Monte-Carlo
scattering), whose coefficient tables are not available.
Shapes and scales follow the paper: ~3e3-sample integrals,
50 x 50 x 100 grids, <= 2000 particles, GeV e+/e-
in ~0.1 mm crystals.

Units: c = 1, lengths and times in metres, omega in rad/m.
Trajectory = dict of the 11 SoA arrays named in BASELINE.json ``north_star``:
t, dz, x, y, vx, vy, dvz, ax, ay, az, gamma.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

HBARC_EV_M = 1.973269804e-7      # hbar*c in eV*m
ME_EV = 0.51099895e6             # electron mass in eV
FIELDS = ("t", "dz", "x", "y", "vx", "vy", "dvz", "ax", "ay", "az", "gamma")
CLASSICAL, SPIN0, SPIN_HALF = 0, 1, 2


@dataclass
class Workload:
    name: str
    model: int
    omega: np.ndarray               # (n_omega,)
    thx: np.ndarray                 # (n_thx,)  n_x values
    thy: np.ndarray                 # (n_thy,)  n_y values
    traj: dict | None = None        # single trajectory: FIELDS -> (n,)
    batch: dict | None = None       # ensemble: FIELDS -> (count, stride)
    n: np.ndarray | None = None     # ensemble: (count,) samples per trajectory
    hbarc_over_E: float = 0.0       # Lambda = hbar c / E  [m]; 0 for classical
    meta: dict = field(default_factory=dict)

    @property
    def n_points(self) -> int:
        return len(self.omega) * len(self.thx) * len(self.thy)

    @property
    def evals(self) -> int:
        if self.batch is not None:
            return self.n_points * int(np.sum(self.n))
        return self.n_points * len(self.traj["t"])


# ----------------------------------------------------------------------------
# helpers (trajectory bookkeeping only)
# ----------------------------------------------------------------------------
def _cumtrapz(f: np.ndarray, dt: float) -> np.ndarray:
    out = np.zeros_like(f)
    np.cumsum(0.5 * (f[..., 1:] + f[..., :-1]) * dt, axis=-1, out=out[..., 1:])
    return out


def _longitudinal(tr: dict, dt: float) -> dict:
    """Leading-order longitudinal bookkeeping shared by configs 2-5:
    dvz = -(vx^2+vy^2)/2, dz = int dvz dt (trapezoid), az = -(vx ax + vy ay)."""
    tr["dvz"] = -0.5 * (tr["vx"] ** 2 + tr["vy"] ** 2)
    tr["dz"] = _cumtrapz(tr["dvz"], dt)
    tr["az"] = -(tr["vx"] * tr["ax"] + tr["vy"] * tr["ay"])
    return tr


def _logspace(lo: float, hi: float, n: int) -> np.ndarray:
    if n == 1:
        return np.array([math.sqrt(lo * hi)])
    return lo * (hi / lo) ** (np.arange(n) / (n - 1))


def _uniform_sym(half_width: float, n: int) -> np.ndarray:
    if n == 1:
        return np.array([0.37 * half_width])
    return -half_width + 2.0 * half_width * np.arange(n) / (n - 1)


# ----------------------------------------------------------------------------
# config 1: ideal planar sinusoid
# ----------------------------------------------------------------------------
def sinusoid_trajectory(gamma: float, amplitude: float, wavelength: float,
                        periods: float, n: int) -> dict:
    """x = A sin(w0 t), analytic derivatives, leading-order dvz, dz (config 1)."""
    w0 = 2.0 * math.pi / wavelength
    t = (periods * wavelength) * np.arange(n) / (n - 1)
    s, c = np.sin(w0 * t), np.cos(w0 * t)
    vx = amplitude * w0 * c
    ax = -amplitude * w0 * w0 * s
    z = np.zeros(n)
    return {
        "t": t, "x": amplitude * s, "y": z.copy(), "vx": vx, "vy": z.copy(),
        "ax": ax, "ay": z.copy(),
        "dvz": -0.5 * vx * vx,
        "dz": -0.5 * (amplitude * w0) ** 2 * (0.5 * t + np.sin(2.0 * w0 * t) / (4.0 * w0)),
        "az": -vx * ax,
        "gamma": np.full(n, float(gamma)),
    }


def config1(n: int = 4000, n_omega: int = 64, n_th: int = 8) -> Workload:
    gamma, A, lam = 1000.0, 1e-10, 2e-6
    w0 = 2.0 * math.pi / lam
    K = gamma * A * w0
    w1 = 2.0 * gamma ** 2 * w0 / (1.0 + 0.5 * K * K)
    tr = sinusoid_trajectory(gamma, A, lam, 4.0, n)
    return Workload(
        name="cfg1_sinusoid_classical", model=CLASSICAL,
        omega=_logspace(0.1 * w1, 4.0 * w1, n_omega),
        thx=_uniform_sym(1.0 / gamma, n_th), thy=_uniform_sym(1.0 / gamma, n_th),
        traj=tr, meta={"gamma": gamma, "K": K, "omega1": w1, "omega0": w0})


# ----------------------------------------------------------------------------
# configs 2 and 4: harmonic planar channeling with Gaussian scattering kicks
# ----------------------------------------------------------------------------
def _harmonic_ms(seeds, n: int, dt: float, gamma: float, w_p: float,
                 a_max: float, sigma: float) -> dict:
    """`len(seeds)` independent trajectories, vectorised over trajectories.

    State at sample k is (x_k, vx_k, vy_k).  Step k -> k+1: exact harmonic rotation
    of (x, vx/w_p) by w_p*dt, then vx += sigma*xi1[k+1], vy += sigma*xi2[k+1].
    ax_k = -w_p^2 x_k + sigma*xi1[k]/dt, ay_k = sigma*xi2[k]/dt (xi[0] = 0), so that
    sum(ax*dt) reproduces the velocity change sample-wise (Q15).
    """
    P = len(seeds)
    amp = np.empty(P)
    ph = np.empty(P)
    xi1 = np.empty((P, n))
    xi2 = np.empty((P, n))
    for p, seed in enumerate(seeds):
        rng = np.random.Generator(np.random.PCG64(int(seed)))
        amp[p] = rng.uniform(0.0, a_max)
        ph[p] = rng.uniform(0.0, 2.0 * math.pi)
        xi1[p] = rng.standard_normal(n)
        xi2[p] = rng.standard_normal(n)
    xi1[:, 0] = 0.0
    xi2[:, 0] = 0.0

    cs, sn = math.cos(w_p * dt), math.sin(w_p * dt)
    x = np.empty((P, n))
    vx = np.empty((P, n))
    xk = amp * np.sin(ph)
    uk = amp * np.cos(ph)            # u = vx / w_p
    x[:, 0] = xk
    vx[:, 0] = uk * w_p
    kick = sigma / w_p
    for k in range(1, n):
        xn = cs * xk + sn * uk
        un = cs * uk - sn * xk + kick * xi1[:, k]
        xk, uk = xn, un
        x[:, k] = xk
        vx[:, k] = uk * w_p
    vy = sigma * np.cumsum(xi2, axis=1)
    tr = {
        "t": np.broadcast_to(dt * np.arange(n), (P, n)).copy(),
        "x": x, "vx": vx, "vy": vy, "y": _cumtrapz(vy, dt),
        "ax": -w_p * w_p * x + (sigma / dt) * xi1,
        "ay": (sigma / dt) * xi2,
        "gamma": np.full((P, n), float(gamma)),
    }
    return _longitudinal(tr, dt)


def config2(n: int = 14287, n_omega: int = 256, n_th: int = 32, seed: int = 2) -> Workload:
    E = 5e9
    gamma = E / ME_EV
    w_p = 2.0 * math.pi / 7e-6
    dt = 7e-9
    b = _harmonic_ms([seed], n, dt, gamma, w_p, 0.96e-10, 2e-7)
    tr = {k: v[0] for k, v in b.items()}
    w_c = 2.0 * gamma ** 2 * w_p
    return Workload(
        name="cfg2_planar_positron_classical", model=CLASSICAL,
        omega=_logspace(0.05 * w_c, 10.0 * w_c, n_omega),
        thx=_uniform_sym(3.0 / gamma, n_th), thy=_uniform_sym(3.0 / gamma, n_th),
        traj=tr, meta={"gamma": gamma, "E_eV": E, "seed": seed})


def config4(count: int = 1000, n: int = 100000, n_omega: int = 128, n_th: int = 16,
            seed0: int = 4000) -> Workload:
    E = 5e9
    gamma = E / ME_EV
    w_p = 2.0 * math.pi / 7e-6
    dt = 7e-9
    b = _harmonic_ms([seed0 + p for p in range(count)], n, dt, gamma, w_p, 0.96e-10, 2e-7)
    w_c = 2.0 * gamma ** 2 * w_p
    return Workload(
        name="cfg4_ensemble_classical", model=CLASSICAL,
        omega=_logspace(0.05 * w_c, 10.0 * w_c, n_omega),
        thx=_uniform_sym(2.0 / gamma, n_th), thy=_uniform_sym(2.0 / gamma, n_th),
        batch=b, n=np.full(count, n, dtype=np.int64),
        meta={"gamma": gamma, "E_eV": E, "seed0": seed0})


# ----------------------------------------------------------------------------
# config 3: anharmonic cosine well (planar electron), spin-1/2
# ----------------------------------------------------------------------------
def _verlet(acc, r0, v0, n: int, dt: float):
    """Velocity Verlet, fixed step; r, v are python tuples of floats (1-D or 2-D)."""
    dim = len(r0)
    r = np.empty((dim, n))
    v = np.empty((dim, n))
    a = np.empty((dim, n))
    rk, vk = list(r0), list(v0)
    ak = acc(rk)
    for k in range(n):
        for d in range(dim):
            r[d, k], v[d, k], a[d, k] = rk[d], vk[d], ak[d]
        vh = [vk[d] + 0.5 * dt * ak[d] for d in range(dim)]
        rk = [rk[d] + dt * vh[d] for d in range(dim)]
        ak = acc(rk)
        vk = [vh[d] + 0.5 * dt * ak[d] for d in range(dim)]
    return r, v, a


def config3(n: int = 200000, n_omega: int = 512, n_th: int = 64, seed: int = 3,
            model: int = SPIN_HALF) -> Workload:
    E = 20e9
    gamma = E / ME_EV
    d_p, th_L = 1.92e-10, 5e-5
    kappa = math.pi * th_L ** 2 / (2.0 * d_p)
    dt = 1e-9
    rng = np.random.Generator(np.random.PCG64(seed))
    x0 = rng.uniform(-0.5 * d_p, 0.5 * d_p)
    v0 = rng.uniform(-th_L, th_L)
    kk = 2.0 * math.pi / d_p
    r, v, a = _verlet(lambda r_: [-kappa * math.sin(kk * r_[0])], [x0], [v0], n, dt)
    z = np.zeros(n)
    tr = _longitudinal({
        "t": dt * np.arange(n), "x": r[0], "y": z.copy(), "vx": v[0], "vy": z.copy(),
        "ax": a[0], "ay": z.copy(), "gamma": np.full(n, gamma)}, dt)
    hw = 0.8 * E * (np.arange(n_omega) + 1.0) / n_omega       # photon energies, eV
    half = th_L + 3.0 / gamma
    return Workload(
        name="cfg3_cosine_well_spin_half" if model == SPIN_HALF else f"cfg3_cosine_well_model{model}",
        model=model, omega=hw / HBARC_EV_M,
        thx=_uniform_sym(half, n_th), thy=_uniform_sym(half, n_th),
        traj=tr, hbarc_over_E=HBARC_EV_M / E,
        meta={"gamma": gamma, "E_eV": E, "seed": seed})


# ----------------------------------------------------------------------------
# config 5: axial (2-D) exponential well, spin-0 and spin-1/2
# ----------------------------------------------------------------------------
def config5(n: int = 1000000, n_omega: int = 1024, n_th: int = 64, seed: int = 5,
            model: int = SPIN_HALF) -> Workload:
    E = 50e9
    gamma = E / ME_EV
    a_w, th_L = 0.3e-10, 3e-5
    kappa = th_L ** 2 / (2.0 * a_w)
    dt = 1e-9
    rng = np.random.Generator(np.random.PCG64(seed))
    rr = 1e-10 * math.sqrt(rng.uniform())
    pa = rng.uniform(0.0, 2.0 * math.pi)
    vr = 0.5 * th_L * math.sqrt(rng.uniform())
    va = rng.uniform(0.0, 2.0 * math.pi)

    def acc(r_):
        rad = math.hypot(r_[0], r_[1])
        if rad == 0.0:
            return [0.0, 0.0]
        s = -kappa * math.exp(-rad / a_w) / rad
        return [s * r_[0], s * r_[1]]

    r, v, a = _verlet(acc, [rr * math.cos(pa), rr * math.sin(pa)],
                      [vr * math.cos(va), vr * math.sin(va)], n, dt)
    tr = _longitudinal({
        "t": dt * np.arange(n), "x": r[0], "y": r[1], "vx": v[0], "vy": v[1],
        "ax": a[0], "ay": a[1], "gamma": np.full(n, gamma)}, dt)
    hw = 0.8 * E * (np.arange(n_omega) + 1.0) / n_omega
    half = th_L + 3.0 / gamma
    return Workload(
        name=f"cfg5_axial_well_model{model}", model=model, omega=hw / HBARC_EV_M,
        thx=_uniform_sym(half, n_th), thy=_uniform_sym(half, n_th),
        traj=tr, hbarc_over_E=HBARC_EV_M / E,
        meta={"gamma": gamma, "E_eV": E, "seed": seed})


def paper_typical(n: int = 3000, n_omega: int = 100, n_th: int = 50, seed: int = 6, model: int = CLASSICAL) -> Workload:
    """The grid the paper calls typical "when multiple scattering is included" (N_x = N_y = 50,
    N_omega = 100) over its benchmark trajectory length (3000 time points): the config-2 recipe
    (5 GeV e+, harmonic well, scattering kicks), 50 uniform angles in +-3/gamma, 100 log-spaced omegas.  Not a
    BASELINE.json config: a shape whose angle counts are not multiples of the kernels' tiles."""
    E = 5e9
    gamma = E / ME_EV
    w_p = 2.0 * math.pi / 7e-6
    dt = 7e-9
    b = _harmonic_ms([seed], n, dt, gamma, w_p, 0.96e-10, 2e-7)
    tr = {k: v[0] for k, v in b.items()}
    w_c = 2.0 * gamma ** 2 * w_p
    return Workload(
        name=f"paper_typical_50x50x100_model{model}", model=model,
        omega=_logspace(0.05 * w_c, 10.0 * w_c, n_omega),
        thx=_uniform_sym(3.0 / gamma, n_th), thy=_uniform_sym(3.0 / gamma, n_th),
        traj=tr, hbarc_over_E=0.0 if model == CLASSICAL else HBARC_EV_M / E,
        meta={"gamma": gamma, "E_eV": E, "seed": seed})


CONFIGS = {"cfg1": config1, "cfg2": config2, "cfg3": config3, "cfg4": config4, "cfg5": config5,
           "paper_typical": paper_typical}


def make(name: str, **overrides) -> Workload:
    """Build a configuration by name; keyword overrides shrink it for tests
    (e.g. ``make("cfg3", n=20000, n_omega=16, n_th=8)``)."""
    return CONFIGS[name](**overrides)


def sample_points(wl: Workload, n_random: int, lattice: tuple[int, int, int] = (0, 0, 0),
                  seed: int = 12345) -> np.ndarray:
    """Flat cube indices for sampled parity: a seeded random subset plus an optional
    coarse strided lattice (n_w, n_y, n_x points per axis).  Index order (Q11):
    (i_omega * n_thy + i_y) * n_thx + i_x."""
    nw, ny, nx = len(wl.omega), len(wl.thy), len(wl.thx)
    rng = np.random.Generator(np.random.PCG64(seed))
    idx = [rng.integers(0, nw * ny * nx, size=n_random)]
    lw, ly, lx = lattice
    if lw and ly and lx:
        iw = np.unique(np.linspace(0, nw - 1, lw).round().astype(np.int64))
        iy = np.unique(np.linspace(0, ny - 1, ly).round().astype(np.int64))
        ix = np.unique(np.linspace(0, nx - 1, lx).round().astype(np.int64))
        W, Y, X = np.meshgrid(iw, iy, ix, indexing="ij")
        idx.append(((W * ny + Y) * nx + X).ravel())
    return np.unique(np.concatenate(idx))


def points_of(wl: Workload, flat_idx: np.ndarray):
    """(omega, n_x, n_y) values of flat cube indices."""
    ny, nx = len(wl.thy), len(wl.thx)
    iw, rem = np.divmod(flat_idx, ny * nx)
    iy, ix = np.divmod(rem, nx)
    return wl.omega[iw], wl.thx[ix], wl.thy[iy]
