"""CPU oracle for the radiation integral of arXiv 1910.10391 -- TEST INFRASTRUCTURE.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It never imports the CUDA
path (``paper_1910_10391_b200``) and shares no code or constants with it.

The arithmetic lives in ``rad_oracle.c`` (plain C, one literal loop nest of
PAPER.md eqs. 3-7, 1, 9, 10-12).  This module only compiles it with gcc and
marshals numpy arrays through ctypes.  Three builds of the same source:

  ``ld``    long double (64-bit significand)  -- the parity truth
  ``f64``   double                            -- the timed CPU baseline (mirrors the
                                                 paper's CPU build)
  ``quad``  __float128                        -- checks that ``ld`` is accurate enough
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_BUILD = _HERE / "build"
_VARIANTS = {
    "ld": [],
    "f64": ["-DRAD_ORACLE_DOUBLE"],
    "quad": ["-DRAD_ORACLE_QUAD"],
}
_LIBS: dict[str, ctypes.CDLL] = {}
_LOCK = threading.Lock()

CLASSICAL, SPIN0, SPIN_HALF = 0, 1, 2
FIELDS = ("t", "dz", "x", "y", "vx", "vy", "dvz", "ax", "ay", "az", "gamma")

_dp = ctypes.POINTER(ctypes.c_double)
_ip = ctypes.POINTER(ctypes.c_int64)


def build(variant: str = "ld", force: bool = False) -> Path:
    """Compile ``rad_oracle.c`` into ``oracle/build/librad_oracle_<variant>.so``."""
    flags = _VARIANTS[variant]
    _BUILD.mkdir(exist_ok=True)
    so = _BUILD / f"librad_oracle_{variant}.so"
    srcs = [_HERE / "rad_oracle.c", _HERE / "rad_oracle.h"]
    if not force and so.exists() and all(so.stat().st_mtime >= s.stat().st_mtime for s in srcs):
        return so
    tmp = so.with_suffix(f".tmp{os.getpid()}.so")
    cmd = ["gcc", "-std=c11", "-O2", "-fopenmp", "-fPIC", "-shared", "-fno-fast-math",
           "-ffp-contract=off", *flags, "-o", str(tmp), str(srcs[0]), "-lm"]
    if variant == "quad":
        cmd.append("-lquadmath")
    subprocess.run(cmd, check=True)
    os.replace(tmp, so)
    return so


def build_traj(force: bool = False) -> Path:
    """Compile ``traj_oracle.c`` (synthetic-well trajectory generator, long double)."""
    _BUILD.mkdir(exist_ok=True)
    so = _BUILD / "libtraj_oracle.so"
    src = _HERE / "traj_oracle.c"
    if not force and so.exists() and so.stat().st_mtime >= src.stat().st_mtime:
        return so
    tmp = so.with_suffix(f".tmp{os.getpid()}.so")
    subprocess.run(["gcc", "-std=c11", "-O2", "-fopenmp", "-fPIC", "-shared", "-fno-fast-math",
                    "-ffp-contract=off", "-o", str(tmp), str(src), "-lm"], check=True)
    os.replace(tmp, so)
    return so


def build_all() -> None:
    for v in _VARIANTS:
        build(v)
    build_traj()


WELL_COSINE, WELL_AXIAL_EXP, WELL_HARMONIC_MS = 0, 1, 2


def _traj_lib():
    generate(0, 0.0, 1.0, 1.0, 1.0, 2, [0.0], [0.0], [0.0], [0.0])       # builds and loads on first use
    return _LIBS["traj"]


def philox4x32_10(counter, key):
    """Philox4x32-10 block (for the known-answer pin): 4 + 2 uint32 in, 4 uint32 out."""
    c = np.ascontiguousarray(counter, dtype=np.uint32)
    k = np.ascontiguousarray(key, dtype=np.uint32)
    out = np.zeros(4, dtype=np.uint32)
    u32p = ctypes.POINTER(ctypes.c_uint32)
    _traj_lib().traj_oracle_philox(c.ctypes.data_as(u32p), k.ctypes.data_as(u32p), out.ctypes.data_as(u32p))
    return out


def kick_normals(seed: int, particle: int, n: int):
    """The standard normals (xi1, xi2) of steps 0..n-1 of one particle of the scattering well."""
    a, b = np.zeros(n), np.zeros(n)
    _traj_lib().traj_oracle_normals(int(seed), int(particle), int(n), _ptr(a), _ptr(b))
    return a, b


def generate(well: int, kappa: float, length: float, gamma: float, dt: float, n: int,
             x0, y0, vx0, vy0, sigma: float = 0.0, seed: int = 0) -> dict:
    """Oracle trajectories of ``len(x0)`` particles in a synthetic well: FIELDS -> (count, n) arrays."""
    with _LOCK:
        if "traj" not in _LIBS:
            lib = ctypes.CDLL(str(build_traj()))
            lib.traj_oracle_generate.restype = ctypes.c_int
            lib.traj_oracle_generate.argtypes = ([ctypes.c_int] + [ctypes.c_double] * 5 + [ctypes.c_uint64]
                                                 + [ctypes.c_int32, ctypes.c_int64, ctypes.c_int64]
                                                 + [_dp] * 15)
            u32p = ctypes.POINTER(ctypes.c_uint32)
            lib.traj_oracle_philox.argtypes = [u32p, u32p, u32p]
            lib.traj_oracle_philox.restype = None
            lib.traj_oracle_normals.argtypes = [ctypes.c_uint64, ctypes.c_int32, ctypes.c_int64, _dp, _dp]
            lib.traj_oracle_normals.restype = None
            _LIBS["traj"] = lib
        lib = _LIBS["traj"]
    ini = [_f64(a).ravel() for a in (x0, y0, vx0, vy0)]
    count = ini[0].shape[0]
    out = {k: np.zeros((count, n)) for k in FIELDS}
    rc = lib.traj_oracle_generate(int(well), float(kappa), float(length), float(gamma), float(dt), float(sigma),
                                  int(seed), count, n, n,
                                  *[_ptr(a) for a in ini], *[_ptr(out[k]) for k in FIELDS])
    if rc != 0:
        raise ValueError("traj_oracle_generate: invalid arguments")
    return out


def _lib(variant: str) -> ctypes.CDLL:
    with _LOCK:
        if variant not in _LIBS:
            lib = ctypes.CDLL(str(build(variant)))
            lib.rad_oracle_points.restype = ctypes.c_int
            lib.rad_oracle_points.argtypes = (
                [ctypes.c_int64] + [_dp] * 11 + [ctypes.c_int64, _dp, _dp, _dp,
                                                 ctypes.c_int, ctypes.c_double, _dp, _dp])
            lib.rad_oracle_ensemble_points.restype = ctypes.c_int
            lib.rad_oracle_ensemble_points.argtypes = (
                [ctypes.c_int32, ctypes.c_int64, _ip] + [_dp] * 11
                + [ctypes.c_int64, _dp, _dp, _dp, ctypes.c_int, _dp, ctypes.c_int, _dp])
            lib.rad_oracle_real_digits.restype = ctypes.c_int
            lib.rad_oracle_threads.restype = ctypes.c_int
            _LIBS[variant] = lib
        return _LIBS[variant]


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def _ptr(a: np.ndarray):
    return a.ctypes.data_as(_dp)


def threads(variant: str = "ld") -> int:
    return int(_lib(variant).rad_oracle_threads())


def real_digits(variant: str = "ld") -> int:
    return int(_lib(variant).rad_oracle_real_digits())


def points(traj: dict, omega, nx, ny, model: int = CLASSICAL, hbarc_over_E: float = 0.0,
           variant: str = "ld", return_amplitudes: bool = False):
    """Spectrum at a list of points.  ``traj`` maps FIELDS -> 1-D arrays of one length.

    Returns ``out`` (npts,) and, if asked, ``amp`` (npts, 4) complex: A_x, A_y, A_z, J.
    """
    arrs = [_f64(traj[k]) for k in FIELDS]
    n = arrs[0].shape[0]
    if any(a.ndim != 1 or a.shape[0] != n for a in arrs):
        raise ValueError("trajectory arrays must be 1-D and of one length")
    omega, nx, ny = _f64(omega).ravel(), _f64(nx).ravel(), _f64(ny).ravel()
    npts = omega.shape[0]
    if nx.shape[0] != npts or ny.shape[0] != npts:
        raise ValueError("omega, nx, ny must have one length")
    out = np.empty(npts, dtype=np.float64)
    amp = np.empty((npts, 8), dtype=np.float64) if return_amplitudes else None
    rc = _lib(variant).rad_oracle_points(
        n, *[_ptr(a) for a in arrs], npts, _ptr(omega), _ptr(nx), _ptr(ny),
        int(model), float(hbarc_over_E), _ptr(out),
        _ptr(amp) if amp is not None else None)
    if rc != 0:
        raise ValueError(f"rad_oracle_points: invalid arguments (rc={rc})")
    if return_amplitudes:
        return out, amp[:, 0::2] + 1j * amp[:, 1::2]
    return out


def grid_points(omega, thx, thy):
    """Flatten a tensor grid to point lists in the cube order of DESIGN.md (Q11):
    index = (i_omega * n_thy + i_y) * n_thx + i_x."""
    omega, thx, thy = _f64(omega), _f64(thx), _f64(thy)
    W, Y, X = np.meshgrid(omega, thy, thx, indexing="ij")
    return W.ravel(), X.ravel(), Y.ravel()


def grid(traj: dict, omega, thx, thy, model: int = CLASSICAL, hbarc_over_E: float = 0.0,
         variant: str = "ld"):
    """Full cube, shape (n_omega, n_thy, n_thx)."""
    w, nx, ny = grid_points(omega, thx, thy)
    out = points(traj, w, nx, ny, model, hbarc_over_E, variant)
    return out.reshape(len(np.atleast_1d(omega)), len(np.atleast_1d(thy)), len(np.atleast_1d(thx)))


def ensemble_points(batch: dict, n, omega, nx, ny, model: int = CLASSICAL, hbarc_over_E=None,
                    accumulate_into=None, variant: str = "ld"):
    """Sum over trajectories.  ``batch`` maps FIELDS -> (count, stride) arrays; ``n`` (count,)."""
    arrs = [_f64(batch[k]) for k in FIELDS]
    count, stride = arrs[0].shape
    if any(a.shape != (count, stride) for a in arrs):
        raise ValueError("batch arrays must share one (count, stride) shape")
    n = np.ascontiguousarray(n, dtype=np.int64)
    if n.shape != (count,):
        raise ValueError("n must have shape (count,)")
    omega, nx, ny = _f64(omega).ravel(), _f64(nx).ravel(), _f64(ny).ravel()
    npts = omega.shape[0]
    lam = None if hbarc_over_E is None else _f64(np.broadcast_to(hbarc_over_E, (count,)))
    if accumulate_into is not None:
        out = _f64(accumulate_into).ravel().copy()
    else:
        out = np.empty(npts, dtype=np.float64)
    rc = _lib(variant).rad_oracle_ensemble_points(
        count, stride, n.ctypes.data_as(_ip), *[_ptr(a) for a in arrs],
        npts, _ptr(omega), _ptr(nx), _ptr(ny), int(model),
        _ptr(lam) if lam is not None else None,
        1 if accumulate_into is not None else 0, _ptr(out))
    if rc != 0:
        raise ValueError(f"rad_oracle_ensemble_points: invalid arguments (rc={rc})")
    return out
