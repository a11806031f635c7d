"""ctypes binding of ``include/rad.h`` (argument marshalling only; see package docstring)."""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

import numpy as np
import torch

_PKG = Path(__file__).resolve().parent
_SRC = _PKG / "csrc"
_SO = _PKG / "librad_b200.so"

CLASSICAL, SPIN0, SPIN_HALF = 0, 1, 2
FIELDS = ("t", "dz", "x", "y", "vx", "vy", "dvz", "ax", "ay", "az", "gamma")

EXPORTS = ("rad_classical", "rad_semiclassical", "rad_ensemble_sum", "rad_sections_sum", "rad_angular_sum", "rad_sum_cubes",
           "rad_workspace_bytes", "rad_eval_host", "rad_ensemble_sum_host",
           "rad_measure_fp64_peak", "rad_launch_count", "rad_strerror",
           "rad_profile_create", "rad_profile_destroy", "rad_profile_read", "rad_plan_kernel",
           "rad_generate_trajectories", "rad_plan_describe", "rad_angular_spectrum",
           "rad_angular_spectrum_workspace_bytes", "rad_formation_length", "rad_sections_check",
           "rad_number_spectrum", "rad_eval_static", "rad_static_scratch_bytes")

KERNEL_AUTO, KERNEL_DIRECT, KERNEL_SEPARABLE, KERNEL_FUSED = 0, 1, 2, 3

_dp = ctypes.POINTER(ctypes.c_double)
_lib = None


class RadError(RuntimeError):
    def __init__(self, code: int, text: str):
        super().__init__(f"rad status {code}: {text}")
        self.code = code


class _Traj(ctypes.Structure):
    _fields_ = [("n", ctypes.c_int64)] + [(k, ctypes.c_void_p) for k in FIELDS]


class _Batch(ctypes.Structure):
    _fields_ = ([("count", ctypes.c_int32), ("stride", ctypes.c_int64), ("n", ctypes.c_void_p)]
                + [(k, ctypes.c_void_p) for k in FIELDS])


class _TrajBuffers(ctypes.Structure):
    _fields_ = [(k, ctypes.c_void_p) for k in FIELDS]


class _Options(ctypes.Structure):
    _fields_ = [("kernel", ctypes.c_int32), ("reserved", ctypes.c_int32), ("profile", ctypes.c_void_p)]


class _Grid(ctypes.Structure):
    _fields_ = [("n_omega", ctypes.c_int32), ("n_thx", ctypes.c_int32), ("n_thy", ctypes.c_int32),
                ("omega", ctypes.c_void_p), ("thx", ctypes.c_void_p), ("thy", ctypes.c_void_p)]


def library_path() -> Path:
    return _SO


def build_library(force: bool = False, verbose: bool = False) -> Path:
    """Compile csrc/rad.cu for sm_100a into the in-tree shared library (nvcc cross-compiles
    without a GPU)."""
    srcs = [_SRC / "rad.cu", _SRC / "rad_device.cuh", _SRC / "rad_sep.cuh", _SRC / "rad_traj.cuh",
            _SRC / "rad_fused.cuh", _SRC / "rad_plan.h", _SRC / "sincos_coeffs.h",
            _PKG.parent / "include" / "rad.h"]
    if not force and _SO.exists() and all(_SO.stat().st_mtime >= s.stat().st_mtime for s in srcs):
        return _SO
    tmp = _SO.with_suffix(f".tmp{os.getpid()}.so")
    cmd = ["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
           "-shared", "-Xcompiler", "-fPIC", "-o", str(tmp), str(srcs[0])]
    if verbose:
        cmd[1:1] = ["-Xptxas", "-v"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, _SO)
    return _SO


def load_library() -> ctypes.CDLL:
    """Load the C-ABI library.  Fails loudly if it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not _SO.exists():
        raise FileNotFoundError(
            f"{_SO} is missing: run __graft_entry__.build() (nvcc) first; there is no CPU fallback")
    lib = ctypes.CDLL(str(_SO))
    vp, sz, i32, i64, dbl = ctypes.c_void_p, ctypes.c_size_t, ctypes.c_int32, ctypes.c_int64, ctypes.c_double
    P = ctypes.POINTER
    op = P(_Options)
    sig = {
        "rad_classical": (ctypes.c_int, [P(_Traj), P(_Grid), vp, vp, sz, op, vp]),
        "rad_semiclassical": (ctypes.c_int, [P(_Traj), P(_Grid), ctypes.c_int, dbl, vp, vp, sz, op, vp]),
        "rad_ensemble_sum": (ctypes.c_int, [P(_Batch), P(_Grid), ctypes.c_int, vp, ctypes.c_int, vp, vp, sz, op, vp]),
        "rad_sections_sum": (ctypes.c_int, [P(_Traj), i32, vp, P(_Grid), ctypes.c_int, vp, ctypes.c_int, vp, vp, sz,
                                            op, vp]),
        "rad_sections_check": (ctypes.c_int, [i32, vp, vp, vp, dbl, vp, i32]),
        "rad_angular_sum": (ctypes.c_int, [vp, P(_Grid), dbl, dbl, vp, vp]),
        "rad_angular_spectrum": (ctypes.c_int, [P(_Batch), P(_Grid), ctypes.c_int, vp, dbl, dbl, vp, vp, sz, op, vp]),
        "rad_angular_spectrum_workspace_bytes": (sz, [i32, i64, i32, i32, i32]),
        "rad_number_spectrum": (ctypes.c_int, [vp, vp, i32, dbl, vp, vp]),
        "rad_sum_cubes": (ctypes.c_int, [vp, i32, i64, ctypes.c_int, vp, vp]),
        "rad_plan_kernel": (ctypes.c_int, [i32, i64, i32, i32, i32, ctypes.c_int, i32]),
        "rad_plan_describe": (ctypes.c_int, [i32, i64, i32, i32, i32, ctypes.c_int, i32, P(ctypes.c_int32)]),
        "rad_formation_length": (dbl, [dbl, dbl, dbl]),
        "rad_generate_trajectories": (ctypes.c_int, [ctypes.c_int] + [dbl] * 5 + [ctypes.c_uint64, i32, i64, i64]
                                      + [vp] * 4 + [P(_TrajBuffers), vp]),
        "rad_workspace_bytes": (sz, [i32, i64, i32, i32, i32]),
        "rad_eval_host": (ctypes.c_int, [P(_Traj), P(_Grid), ctypes.c_int, dbl, vp, op, vp]),
        "rad_eval_static": (ctypes.c_int, [P(_Traj), P(_Grid), ctypes.c_int, dbl, vp, op, vp]),
        "rad_static_scratch_bytes": (sz, []),
        "rad_ensemble_sum_host": (ctypes.c_int, [P(_Batch), P(_Grid), ctypes.c_int, vp, ctypes.c_int, vp, op, vp]),
        "rad_measure_fp64_peak": (dbl, [dbl, vp]),
        "rad_launch_count": (i64, []),
        "rad_profile_create": (vp, []),
        "rad_profile_destroy": (None, [vp]),
        "rad_profile_read": (ctypes.c_int, [vp, P(ctypes.c_float)]),
        "rad_strerror": (ctypes.c_char_p, [ctypes.c_int]),
    }
    assert set(sig) == set(EXPORTS)
    for name, (res, args) in sig.items():
        fn = getattr(lib, name)
        fn.restype, fn.argtypes = res, args
    _lib = lib
    return lib


def _check(rc: int) -> None:
    if rc != 0:
        raise RadError(rc, load_library().rad_strerror(rc).decode())


def _dev(t: torch.Tensor, name: str) -> torch.Tensor:
    if not isinstance(t, torch.Tensor) or not t.is_cuda or t.dtype != torch.float64 or not t.is_contiguous():
        raise TypeError(f"{name}: expected a contiguous float64 CUDA tensor")
    return t


def _stream_ptr(stream) -> int:
    if stream is None:
        if not torch.cuda.is_available():
            return 0           # the library itself then reports RAD_ECUDA: no CPU fallback
        stream = torch.cuda.current_stream()
    return int(stream.cuda_stream)


def _grid_struct(omega, thx, thy) -> _Grid:
    return _Grid(omega.numel(), thx.numel(), thy.numel(), omega.data_ptr(), thx.data_ptr(), thy.data_ptr())


def _traj_struct(traj: dict) -> _Traj:
    ts = [_dev(traj[k], k) for k in FIELDS]
    n = ts[0].numel()
    if any(t.ndim != 1 or t.numel() != n for t in ts):
        raise ValueError("trajectory tensors must be 1-D and of one length")
    return _Traj(n, *[t.data_ptr() for t in ts])


class RadProfile:
    """Per-kernel timing of one call (include/rad.h rad_profile): pass as ``profile=`` to a compute call, then
    ``read()`` -> (pack_ms, main_ms, reduction_ms).  Owns CUDA events of the current device."""

    def __init__(self):
        self._h = load_library().rad_profile_create()
        if not self._h:
            raise RadError(-3, "rad_profile_create failed (no CUDA device?)")

    def read(self):
        ms = (ctypes.c_float * 3)()
        _check(load_library().rad_profile_read(self._h, ms))
        return float(ms[0]), float(ms[1]), float(ms[2])

    def close(self):
        if self._h:
            load_library().rad_profile_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def _opt(kernel: int, profile):
    """rad_options for a call (NULL when everything is default)."""
    if not kernel and profile is None:
        return None
    return ctypes.byref(_Options(int(kernel), 0, profile._h if profile is not None else None))


def _ws_args(workspace):
    if workspace is None:
        return None, 0
    if not workspace.is_cuda or not workspace.is_contiguous():
        raise TypeError("workspace: expected a contiguous CUDA tensor")
    return workspace.data_ptr(), workspace.numel() * workspace.element_size()


def _out_cube(out, omega, thx, thy):
    shape = (omega.numel(), thy.numel(), thx.numel())
    if out is None:
        return torch.empty(shape, dtype=torch.float64, device=omega.device)
    _dev(out, "out")
    if out.numel() != shape[0] * shape[1] * shape[2]:
        raise ValueError("out has the wrong number of elements")
    return out


def rad_workspace_bytes(count: int, n_max: int, n_omega: int, n_thx: int, n_thy: int) -> int:
    return int(load_library().rad_workspace_bytes(count, n_max, n_omega, n_thx, n_thy))


def rad_classical(traj: dict, omega, thx, thy, out=None, workspace=None, stream=None, kernel: int = 0, profile=None):
    """Classical cube (n_omega, n_thy, n_thx); eq. (1) with eqs. (3)-(7)."""
    g = _grid_struct(_dev(omega, "omega"), _dev(thx, "thx"), _dev(thy, "thy"))
    t = _traj_struct(traj)
    out = _out_cube(out, omega, thx, thy)
    ws, nb = _ws_args(workspace)
    _check(load_library().rad_classical(ctypes.byref(t), ctypes.byref(g), out.data_ptr(), ws, nb,
                                        _opt(kernel, profile), _stream_ptr(stream)))
    return out


def rad_semiclassical(traj: dict, omega, thx, thy, spin: int, hbarc_over_E: float, out=None,
                      workspace=None, stream=None, kernel: int = 0, profile=None):
    """spin=0: substitution model, eq. (9); spin=1: spin-1/2 BCK, eq. (10) PAPER.md:62."""
    g = _grid_struct(_dev(omega, "omega"), _dev(thx, "thx"), _dev(thy, "thy"))
    t = _traj_struct(traj)
    out = _out_cube(out, omega, thx, thy)
    ws, nb = _ws_args(workspace)
    _check(load_library().rad_semiclassical(ctypes.byref(t), ctypes.byref(g), int(spin), float(hbarc_over_E),
                                            out.data_ptr(), ws, nb, _opt(kernel, profile), _stream_ptr(stream)))
    return out


def rad_eval_static(traj: dict, omega, thx, thy, model: int = CLASSICAL, hbarc_over_E: float = 0.0, out=None,
                    stream=None, kernel: int = 0, profile=None):
    """Cube of one trajectory through the entry point that allocates nothing (include/rad.h rad_eval_static): the
    scratch is the library's 16 MiB static device array; RadError(RAD_ETOOBIG = -5) beyond it.  Pass ``out`` to keep
    this wrapper from allocating the result tensor either."""
    g = _grid_struct(_dev(omega, "omega"), _dev(thx, "thx"), _dev(thy, "thy"))
    t = _traj_struct(traj)
    out = _out_cube(out, omega, thx, thy)
    _check(load_library().rad_eval_static(ctypes.byref(t), ctypes.byref(g), int(model), float(hbarc_over_E),
                                          out.data_ptr(), _opt(kernel, profile), _stream_ptr(stream)))
    return out


def rad_static_scratch_bytes() -> int:
    return int(load_library().rad_static_scratch_bytes())


def rad_ensemble_sum(batch: dict, n, omega, thx, thy, model: int = CLASSICAL, hbarc_over_E=None,
                     accumulate: bool = False, out=None, workspace=None, stream=None, kernel: int = 0,
                     profile=None):
    """Sum of the spectra of `count` trajectories.  batch: FIELDS -> (count, stride)
    CUDA tensors; n: host int64 (count,)."""
    ts = [_dev(batch[k], k) for k in FIELDS]
    count, stride = ts[0].shape
    if any(tuple(t.shape) != (count, stride) for t in ts):
        raise ValueError("batch tensors must share one (count, stride) shape")
    n_host = np.ascontiguousarray(n, dtype=np.int64)
    if n_host.shape != (count,):
        raise ValueError("n must have shape (count,)")
    lam = None
    if hbarc_over_E is not None:
        lam = np.ascontiguousarray(np.broadcast_to(np.asarray(hbarc_over_E, dtype=np.float64), (count,)))
    b = _Batch(count, stride, n_host.ctypes.data, *[t.data_ptr() for t in ts])
    g = _grid_struct(_dev(omega, "omega"), _dev(thx, "thx"), _dev(thy, "thy"))
    if accumulate and out is None:
        raise ValueError("accumulate needs an existing out")
    out = _out_cube(out, omega, thx, thy)
    ws, nb = _ws_args(workspace)
    _check(load_library().rad_ensemble_sum(ctypes.byref(b), ctypes.byref(g), int(model),
                                           lam.ctypes.data if lam is not None else None,
                                           1 if accumulate else 0, out.data_ptr(), ws, nb,
                                           _opt(kernel, profile), _stream_ptr(stream)))
    return out


def rad_sections_sum(traj: dict, start, omega, thx, thy, model: int = CLASSICAL, hbarc_over_E=None,
                     accumulate: bool = False, out=None, workspace=None, stream=None, kernel: int = 0,
                     profile=None):
    """Sum of the spectra of the sections start[s]..start[s+1] (both included) of one trajectory, each with
    its own hbar c / E."""
    t = _traj_struct(traj)
    st = np.ascontiguousarray(start, dtype=np.int64)
    if st.ndim != 1 or st.size < 2:
        raise ValueError("start needs at least two indices")
    lam = None
    if hbarc_over_E is not None:
        lam = np.ascontiguousarray(np.broadcast_to(np.asarray(hbarc_over_E, dtype=np.float64), (st.size - 1,)))
    g = _grid_struct(_dev(omega, "omega"), _dev(thx, "thx"), _dev(thy, "thy"))
    if accumulate and out is None:
        raise ValueError("accumulate needs an existing out")
    out = _out_cube(out, omega, thx, thy)
    ws, nb = _ws_args(workspace)
    _check(load_library().rad_sections_sum(ctypes.byref(t), st.size - 1, st.ctypes.data, ctypes.byref(g), int(model),
                                           lam.ctypes.data if lam is not None else None,
                                           1 if accumulate else 0, out.data_ptr(), ws, nb, _opt(kernel, profile),
                                           _stream_ptr(stream)))
    return out


def rad_sections_check(t_start, gamma0, omega_min: float, hbarc_over_E=None):
    """Indices of the sections not longer than the formation length at omega_min.  Host arrays:
    t_start (n_sections + 1 boundary times), gamma0 and hbarc_over_E (n_sections each; None: classical)."""
    t = np.ascontiguousarray(t_start, dtype=np.float64)
    g = np.ascontiguousarray(gamma0, dtype=np.float64)
    ns = g.size
    if t.shape != (ns + 1,):
        raise ValueError("t_start needs n_sections + 1 entries")
    lam = None
    if hbarc_over_E is not None:
        lam = np.ascontiguousarray(np.broadcast_to(np.asarray(hbarc_over_E, dtype=np.float64), (ns,)))
    idx = np.empty(ns, dtype=np.int32)
    rc = load_library().rad_sections_check(ns, t.ctypes.data, g.ctypes.data, lam.ctypes.data if lam is not None else None,
                                           float(omega_min), idx.ctypes.data, ns)
    if rc < 0:
        _check(rc)
    return idx[:rc].copy()


def rad_number_spectrum(spectrum, omega, hbar_c: float, out=None, stream=None):
    """dN/dw = (dI/dw) / (hbar_c * omega)."""
    _dev(spectrum, "spectrum"), _dev(omega, "omega")
    if spectrum.numel() != omega.numel():
        raise ValueError("spectrum and omega must have one length")
    if out is None:
        out = torch.empty_like(spectrum)
    _check(load_library().rad_number_spectrum(spectrum.data_ptr(), omega.data_ptr(), omega.numel(), float(hbar_c),
                                              _dev(out, "out").data_ptr(), _stream_ptr(stream)))
    return out


def rad_angular_sum(cube, omega, thx, thy, d_solid_angle: float, theta_cut: float = 0.0, out=None,
                    stream=None):
    """dI/dw = sum over angles of cube * dOmega, optional collimator cut."""
    g = _grid_struct(_dev(omega, "omega"), _dev(thx, "thx"), _dev(thy, "thy"))
    _dev(cube, "cube")
    if out is None:
        out = torch.empty(omega.numel(), dtype=torch.float64, device=cube.device)
    _check(load_library().rad_angular_sum(cube.data_ptr(), ctypes.byref(g), float(d_solid_angle),
                                          float(theta_cut), _dev(out, "out").data_ptr(), _stream_ptr(stream)))
    return out


WELL_COSINE, WELL_AXIAL_EXP, WELL_HARMONIC_MS = 0, 1, 2


def rad_generate_trajectories(well: int, kappa: float, length: float, gamma: float, dt: float, n: int,
                              x0, y0, vx0, vy0, out: dict | None = None, stream=None, sigma: float = 0.0,
                              seed: int = 0) -> dict:
    """`count` particles in a synthetic well, generated on the device (PAPER.md:233 outlook): FIELDS ->
    (count, n) CUDA tensors ready for rad_ensemble_sum."""
    ini = [_dev(a, name) for a, name in ((x0, "x0"), (y0, "y0"), (vx0, "vx0"), (vy0, "vy0"))]
    count = ini[0].numel()
    if any(a.numel() != count for a in ini):
        raise ValueError("x0, y0, vx0, vy0 must have one length")
    if out is None:
        out = {k: torch.empty((count, n), dtype=torch.float64, device=ini[0].device) for k in FIELDS}
    ts = [_dev(out[k], k) for k in FIELDS]
    stride = ts[0].shape[1]
    if any(tuple(t.shape) != (count, stride) for t in ts):
        raise ValueError("out tensors must share one (count, stride) shape")
    bufs = _TrajBuffers(*[t.data_ptr() for t in ts])
    _check(load_library().rad_generate_trajectories(int(well), float(kappa), float(length), float(gamma), float(dt),
                                                    float(sigma), int(seed), count,
                                         int(n), int(stride), *[a.data_ptr() for a in ini], ctypes.byref(bufs),
                                         _stream_ptr(stream)))
    return out


def rad_sum_cubes(cubes, accumulate: bool = False, out=None, stream=None):
    """Sum of ``cubes[c]`` over the leading axis in ascending order (ensemble shards)."""
    _dev(cubes, "cubes")
    count, m = cubes.shape[0], cubes[0].numel()
    if out is None:
        if accumulate:
            raise ValueError("accumulate needs an existing out")
        out = torch.empty(cubes.shape[1:], dtype=torch.float64, device=cubes.device)
    if _dev(out, "out").numel() != m:
        raise ValueError("out has the wrong number of elements")
    _check(load_library().rad_sum_cubes(cubes.data_ptr(), count, m, 1 if accumulate else 0, out.data_ptr(),
                                        _stream_ptr(stream)))
    return out


def rad_angular_spectrum(batch: dict, n, omega, thx, thy, d_solid_angle: float, theta_cut: float = 0.0,
                         model: int = CLASSICAL, hbarc_over_E=None, out=None, workspace=None, stream=None,
                         kernel: int = 0, profile=None):
    """dI/dw of an ensemble, formed in the main kernel's epilogue without a cube where the grid fills the GPU."""
    ts = [_dev(batch[k], k) for k in FIELDS]
    count, stride = ts[0].shape
    if any(tuple(t.shape) != (count, stride) for t in ts):
        raise ValueError("batch tensors must share one (count, stride) shape")
    n_host = np.ascontiguousarray(n, dtype=np.int64)
    if n_host.shape != (count,):
        raise ValueError("n must have shape (count,)")
    lam = None
    if hbarc_over_E is not None:
        lam = np.ascontiguousarray(np.broadcast_to(np.asarray(hbarc_over_E, dtype=np.float64), (count,)))
    b = _Batch(count, stride, n_host.ctypes.data, *[t.data_ptr() for t in ts])
    g = _grid_struct(_dev(omega, "omega"), _dev(thx, "thx"), _dev(thy, "thy"))
    lib = load_library()
    if workspace is None:
        need = lib.rad_angular_spectrum_workspace_bytes(count, int(n_host.max()), omega.numel(), thx.numel(), thy.numel())
        workspace = torch.empty(need, dtype=torch.uint8, device=omega.device)
    ws, nb = _ws_args(workspace)
    if out is None:
        out = torch.empty(omega.numel(), dtype=torch.float64, device=omega.device)
    _check(lib.rad_angular_spectrum(ctypes.byref(b), ctypes.byref(g), int(model),
                                    lam.ctypes.data if lam is not None else None, float(d_solid_angle),
                                    float(theta_cut), _dev(out, "out").data_ptr(), ws, nb, _opt(kernel, profile),
                                    _stream_ptr(stream)))
    return out


def _host(a, name: str) -> np.ndarray:
    if isinstance(a, torch.Tensor):
        if a.is_cuda or a.dtype != torch.float64 or not a.is_contiguous():
            raise TypeError(f"{name}: expected a contiguous float64 CPU tensor")
        return a.numpy()
    a = np.asarray(a)
    if a.dtype != np.float64 or not a.flags.c_contiguous:
        raise TypeError(f"{name}: expected a C-contiguous float64 array")
    return a


def _host_ptr(a, name: str):
    """(address, shape, keep-alive object) of a contiguous float64 host array or CPU tensor.  The host-buffer calls
    marshal fifteen arrays per call and a small problem is ~50 us of GPU work: torch's data_ptr() and numpy's
    __array_interface__ cost a fraction of a microsecond each, `tensor.numpy().ctypes.data` several."""
    if isinstance(a, torch.Tensor):
        if a.is_cuda or a.dtype != torch.float64 or not a.is_contiguous():
            raise TypeError(f"{name}: expected a contiguous float64 CPU tensor")
        return a.data_ptr(), tuple(a.shape), a
    a = np.asarray(a)
    if a.dtype != np.float64 or not a.flags.c_contiguous:
        raise TypeError(f"{name}: expected a C-contiguous float64 array")
    return a.__array_interface__["data"][0], a.shape, a


def _host_grid_and_out(omega, thx, thy, out, need_out: bool):
    (pw, sw, kw), (px, sx, kx), (py, sy, ky) = _host_ptr(omega, "omega"), _host_ptr(thx, "thx"), _host_ptr(thy, "thy")
    if len(sw) != 1 or len(sx) != 1 or len(sy) != 1:
        raise ValueError("omega, thx, thy must be 1-D")
    g = _Grid(sw[0], sx[0], sy[0], pw, px, py)
    if out is None:
        if need_out:
            raise ValueError("accumulate needs an existing out")
        out = np.empty((sw[0], sy[0], sx[0]), dtype=np.float64)
    po, so, ko = _host_ptr(out, "out")
    if int(np.prod(so)) != sw[0] * sx[0] * sy[0]:
        raise ValueError("out has the wrong number of elements")
    return g, out, po, (kw, kx, ky, ko)


def rad_eval_host(traj: dict, omega, thx, thy, model: int = CLASSICAL, hbarc_over_E: float = 0.0,
                  out=None, stream=None, kernel: int = 0, profile=None):
    """Host-buffer call: H2D, evaluate, D2H inside the C library."""
    hs = [_host_ptr(traj[k], k) for k in FIELDS]
    shape = hs[0][1]
    if len(shape) != 1 or any(h[1] != shape for h in hs):
        raise ValueError("trajectory arrays must be 1-D and of one length")
    t = _Traj(shape[0], *[h[0] for h in hs])
    g, out, po, keep = _host_grid_and_out(omega, thx, thy, out, False)
    _check(load_library().rad_eval_host(ctypes.byref(t), ctypes.byref(g), int(model), float(hbarc_over_E),
                                        po, _opt(kernel, profile), _stream_ptr(stream)))
    return out


def rad_ensemble_sum_host(batch: dict, n, omega, thx, thy, model: int = CLASSICAL, hbarc_over_E=None,
                          accumulate: bool = False, out=None, stream=None, kernel: int = 0, profile=None):
    hs = [_host_ptr(batch[k], k) for k in FIELDS]
    shape = hs[0][1]
    if len(shape) != 2:
        raise ValueError("batch arrays must be 2-D (count, stride)")
    count, stride = shape
    if any(h[1] != shape for h in hs):
        raise ValueError("batch arrays must share one (count, stride) shape")
    n_host = np.ascontiguousarray(n, dtype=np.int64)
    if n_host.shape != (count,):
        raise ValueError("n must have shape (count,)")
    lam = None
    if hbarc_over_E is not None:
        lam = np.ascontiguousarray(np.broadcast_to(np.asarray(hbarc_over_E, dtype=np.float64), (count,)))
    b = _Batch(count, stride, n_host.ctypes.data, *[h[0] for h in hs])
    g, out, po, keep = _host_grid_and_out(omega, thx, thy, out, bool(accumulate))
    _check(load_library().rad_ensemble_sum_host(ctypes.byref(b), ctypes.byref(g), int(model),
                                                lam.ctypes.data if lam is not None else None,
                                                1 if accumulate else 0, po, _opt(kernel, profile),
                                                _stream_ptr(stream)))
    return out


def rad_measure_fp64_peak(millis: float = 200.0, stream=None) -> float:
    """Measured FP64 FMA peak of the current device in FLOP/s."""
    v = float(load_library().rad_measure_fp64_peak(float(millis), _stream_ptr(stream)))
    if v <= 0:
        raise RadError(-3, "rad_measure_fp64_peak failed (no CUDA device?)")
    return v


def rad_launch_count() -> int:
    return int(load_library().rad_launch_count())


def rad_plan_kernel(n_omega: int, n_thx: int, n_thy: int, model: int = CLASSICAL, kernel: int = 0, count: int = 1,
                    n_max: int = 1 << 20) -> int:
    """1 direct, 2 separable, 3 fused: the kernel that takes (the largest part of) a grid of this shape for
    `count` trajectories of at most n_max samples under the option `kernel`."""
    rc = load_library().rad_plan_kernel(count, n_max, n_omega, n_thx, n_thy, int(model), int(kernel))
    if rc < 0:
        _check(rc)
    return rc


def rad_plan_describe(count: int, n_max: int, n_omega: int, n_thx: int, n_thy: int, model: int = CLASSICAL,
                      kernel: int = 0) -> dict:
    """Launch plan of a call of this shape (include/rad.h rad_plan_describe)."""
    plan = (ctypes.c_int32 * 11)()
    _check(load_library().rad_plan_describe(count, n_max, n_omega, n_thx, n_thy, int(model), int(kernel), plan))
    keys = ("kernel", "mode", "tiles", "slices", "t_slices", "chunks", "parts", "interior_x", "interior_y", "launches",
            "cluster")
    return dict(zip(keys, (int(v) for v in plan)))


def rad_formation_length(gamma: float, omega: float, hbarc_over_E: float) -> float:
    """l_f = 2 gamma^2 (E - w)/(E w), in the length unit of omega; ValueError outside the domain."""
    v = float(load_library().rad_formation_length(float(gamma), float(omega), float(hbarc_over_E)))
    if v < 0:
        raise ValueError("rad_formation_length: need gamma >= 1, omega > 0 and hbar omega < E")
    return v
