"""CPU-side checks of the boundary: the C-ABI library builds for sm_100a, loads, exports every
symbol include/rad.h declares, and its host logic (argument validation, workspace plan) works
without a GPU.  No compute is attempted here."""
import ctypes
import re
from pathlib import Path

import numpy as np
import pytest

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module")
def radlib():
    import paper_1910_10391_b200 as rad
    rad.build_library()
    return rad


def test_exports_match_header(radlib):
    header = (ROOT / "include" / "rad.h").read_text()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(rad_[a-z0-9_]+)\s*\(", header))
    assert declared, "no declarations found in include/rad.h"
    lib = ctypes.CDLL(str(radlib.library_path()))
    missing = [n for n in sorted(declared) if not hasattr(lib, n)]
    assert not missing, f"declared in rad.h but not exported: {missing}"
    assert declared == set(radlib.binding.EXPORTS)


def test_library_is_sm100a_with_tma(radlib):
    """The fat binary holds sm_100a code and the main kernel stages chunks with TMA bulk
    copies (SASS UBLKCP) completing on an mbarrier (SYNCS)."""
    import subprocess
    sass = subprocess.run(["cuobjdump", "-sass", str(radlib.library_path())], capture_output=True,
                          text=True, check=True).stdout
    assert "sm_100a" in sass
    assert "UBLKCP" in sass and "SYNCS" in sass
    assert "DFMA" in sass and "FRND.F64" in sass
    assert "USETMAXREG" in sass                      # the separable kernel's producer / consumer register split


def test_strerror_and_launch_count(radlib):
    lib = radlib.load_library()
    assert lib.rad_strerror(0) == b"ok"
    assert b"invalid" in lib.rad_strerror(-1)
    assert b"workspace" in lib.rad_strerror(-4)
    assert radlib.rad_launch_count() >= 0


def test_workspace_plan_without_gpu(radlib):
    """The plan is a pure function of the shapes; grows with n and count; 0 on bad shapes."""
    f = radlib.rad_workspace_bytes
    assert f(0, 100, 4, 4, 4) == 0 and f(1, 1, 4, 4, 4) == 0 and f(1, 100, 0, 4, 4) == 0
    small, big = f(1, 4000, 64, 8, 8), f(1, 400000, 64, 8, 8)
    assert 0 < small < big
    assert f(1000, 100000, 128, 16, 16) > 8 * 1000 * 100000 * 10      # packed records: 80 B/sample
    assert f(1, 1000000, 1024, 64, 64) < 2 * 8 * 10 * 1000000 + (1 << 20)   # direct mode: no partials


def test_validation_happens_before_any_cuda_call(radlib):
    """Null pointers, bad spin / model, n < 2, negative hbar c / E are rejected on the host."""
    lib = radlib.load_library()
    B = radlib.binding
    buf = np.zeros(16)
    p = buf.ctypes.data
    grid = B._Grid(2, 2, 2, p, p, p)
    traj = B._Traj(8, *([p] * 11))
    out = np.zeros(8).ctypes.data
    assert lib.rad_classical(None, ctypes.byref(grid), out, None, 0, None, None) == -1
    assert lib.rad_classical(ctypes.byref(traj), None, out, None, 0, None, None) == -1
    assert lib.rad_classical(ctypes.byref(traj), ctypes.byref(grid), None, None, 0, None, None) == -1
    assert lib.rad_semiclassical(ctypes.byref(traj), ctypes.byref(grid), 3, 1e-15, out, None, 0, None, None) == -1
    assert lib.rad_semiclassical(ctypes.byref(traj), ctypes.byref(grid), 1, -1.0, out, None, 0, None, None) == -2
    assert lib.rad_classical(ctypes.byref(B._Traj(1, *([p] * 11))), ctypes.byref(grid), out, None, 0, None, None) == -1
    assert lib.rad_classical(ctypes.byref(B._Traj(8, *([p] * 10 + [None]))), ctypes.byref(grid), out,
                             None, 0, None, None) == -1
    assert lib.rad_classical(ctypes.byref(traj), ctypes.byref(B._Grid(0, 2, 2, p, p, p)), out, None, 0, None, None) == -1
    misaligned = B._Traj(8, *([p + 4] + [p] * 10))
    assert lib.rad_classical(ctypes.byref(misaligned), ctypes.byref(grid), out, None, 0, None, None) == -1
    n = np.array([8, 1], dtype=np.int64)
    batch = B._Batch(2, 8, n.ctypes.data, *([p] * 11))
    assert lib.rad_ensemble_sum(ctypes.byref(batch), ctypes.byref(grid), 0, None, 0, out, None, 0, None, None) == -1
    n[1] = 9                                                          # n[p] > stride
    assert lib.rad_ensemble_sum(ctypes.byref(batch), ctypes.byref(grid), 0, None, 0, out, None, 0, None, None) == -1
    n[1] = 8
    assert lib.rad_ensemble_sum(ctypes.byref(batch), ctypes.byref(grid), 2, None, 0, out, None, 0, None, None) == -1
    assert lib.rad_angular_sum(None, ctypes.byref(grid), 1.0, 0.0, out, None) == -1
    start = np.array([0, 4, 4], dtype=np.int64)                       # empty section
    assert lib.rad_sections_sum(ctypes.byref(traj), 2, start.ctypes.data, ctypes.byref(grid), 0, None, 0, out,
                                None, 0, None, None) == -1
    start = np.array([0, 4, 8], dtype=np.int64)                       # runs past the last sample (n = 8)
    assert lib.rad_sections_sum(ctypes.byref(traj), 2, start.ctypes.data, ctypes.byref(grid), 0, None, 0, out,
                                None, 0, None, None) == -1
    assert lib.rad_sections_sum(ctypes.byref(traj), 0, start.ctypes.data, ctypes.byref(grid), 0, None, 0, out,
                                None, 0, None, None) == -1
    bad = B._Options(9, 0, None)                                      # unknown kernel option; reserved must be 0
    assert lib.rad_classical(ctypes.byref(traj), ctypes.byref(grid), out, None, 0, ctypes.byref(bad), None) == -1
    bad = B._Options(0, 1, None)
    assert lib.rad_classical(ctypes.byref(traj), ctypes.byref(grid), out, None, 0, ctypes.byref(bad), None) == -1
    fused = B._Options(3, 0, None)                                    # fused kernel: single trajectory only
    assert lib.rad_ensemble_sum(ctypes.byref(batch), ctypes.byref(grid), 0, None, 0, out, None, 0,
                                ctypes.byref(fused), None) == -1


def test_no_cpu_fallback(radlib):
    """Without a CUDA device a compute call fails loudly with RAD_ECUDA (and the Python
    binding refuses CPU tensors)."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(radlib.RadError) as e:
        radlib.rad_eval_host({k: np.zeros(8) + 1.0 for k in radlib.FIELDS}, np.ones(2), np.zeros(2), np.zeros(2))
    assert e.value.code == -3
    with pytest.raises(TypeError):
        radlib.rad_classical({k: torch.zeros(8, dtype=torch.float64) for k in radlib.FIELDS},
                             torch.ones(2, dtype=torch.float64), torch.zeros(2, dtype=torch.float64),
                             torch.zeros(2, dtype=torch.float64))


def test_kernel_choice_is_a_pure_function_of_the_shape(radlib):
    """rad_plan_kernel without a device: separable kernel where the grid fills its 16 x 16 x 16 (8) point
    tiles (BASELINE.json configs 2-5), direct kernel on small angle grids with long trajectories, the fused
    single-launch kernel on small problems (config 1); the per-call option overrides."""
    f = radlib.rad_plan_kernel
    assert f(256, 32, 32, 0) == 2 and f(512, 64, 64, 2) == 2 and f(128, 16, 16, 0) == 2 and f(1024, 64, 64, 1) == 2
    assert f(64, 8, 8, 0) == 1 and f(5, 3, 3, 2) == 1                 # n_max defaults to 2^20: too long to fuse
    assert f(64, 8, 8, 0, n_max=4000) == 3                            # BASELINE config 1
    assert f(64, 8, 8, 0, n_max=4000, count=3) == 1                   # ensembles are never fused
    assert f(256, 32, 32, 0, kernel=1) == 1 and f(64, 8, 8, 0, kernel=2) == 2
    assert f(64, 8, 8, 2, kernel=3, n_max=100000) == 3                # forced: any single trajectory that fits
    with pytest.raises(radlib.RadError):
        f(0, 4, 4, 0)
    with pytest.raises(radlib.RadError):
        f(1024, 64, 64, 0, kernel=3)                                  # more tiles than the GPU holds at once


def test_launch_plans_of_the_baseline_configs(radlib):
    """The plan is host logic: a pure function of the shapes (148 SMs assumed without a device).  The five
    BASELINE.json configs get whole waves of CTAs: separable kernel 1 CTA/SM, direct kernel 2 CTAs/SM, fused
    kernel 4 CTAs/SM all resident at once."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("plan depends on the visible device's SM count; this checks the 148-SM default")
    d = radlib.rad_plan_describe
    p = d(1, 4000, 64, 8, 8, 0)                      # cfg 1: fused kernel, 8 tiles of 64 threads x 74 time slices = 592 resident CTAs, ONE launch
    assert (p["kernel"], p["tiles"], p["slices"], p["launches"]) == (3, 8, 74, 1)
    assert p["tiles"] * p["slices"] <= 4 * 148
    p = d(1, 4000, 64, 8, 8, 0, kernel=1)            # the three-launch direct path: 4 tiles x 32 one-chunk time slices
    assert (p["kernel"], p["mode"], p["tiles"], p["slices"], p["chunks"], p["launches"]) == (1, 2, 4, 32, 32, 3)
    p = d(1, 14287, 256, 32, 32, 0)                  # cfg 2: 64 tiles x 16 time slices = 6.92 waves of 148
    assert (p["kernel"], p["mode"], p["tiles"], p["slices"], p["parts"]) == (2, 2, 64, 16, 1)
    p = d(1, 200000, 512, 64, 64, 2)                 # cfg 3 spin-1/2: 16 x 16 x 8 point tiles -> 1024 CTAs = 6.92 waves
    assert (p["kernel"], p["mode"], p["tiles"], p["slices"]) == (2, 0, 1024, 1)
    p = d(1, 200000, 512, 64, 64, 1)                 # cfg 3 spin-0: 16 x 16 x 16 tiles -> 512 tiles x 2 time slices
    assert (p["kernel"], p["mode"], p["tiles"], p["slices"]) == (2, 2, 512, 2)
    p = d(1000, 100000, 128, 16, 16, 0)              # cfg 4: 8 tiles x 37 trajectory slices = 2 waves
    assert (p["kernel"], p["mode"], p["tiles"], p["slices"]) == (2, 1, 8, 37)
    p = d(1, 1000000, 1024, 64, 64, 1)               # cfg 5 spin-0: 1024 tiles, one CTA per tile
    assert (p["kernel"], p["mode"], p["tiles"], p["slices"]) == (2, 0, 1024, 1)
    p = d(1, 1000000, 1024, 64, 64, 2)               # cfg 5 spin-1/2: 2048 tiles = 13.8 waves
    assert (p["kernel"], p["mode"], p["tiles"], p["slices"], p["launches"]) == (2, 0, 2048, 1, 2)
    p = d(1, 14287, 256, 32, 32, 0, kernel=1)        # direct kernel on cfg 2: 256 tiles x 8 = 6.92 waves of 296
    assert (p["kernel"], p["mode"], p["tiles"], p["slices"]) == (1, 2, 256, 8)
    for k in range(1, 60):                           # slices never exceed the work there is
        p = d(k, 300, 16, 16, 16, 0)
        assert p["slices"] <= k * p["chunks"] and p["slices"] >= 1


def test_the_papers_typical_grid_is_split_in_two_parts(radlib):
    """N_x = N_y = 50, N_w = 100 "when multiple scattering is included".  50 is 3 tiles of 16 + 2:
    the separable kernel takes the 48 x 48 interior (63 tiles for 100 -> 112 omegas, 441 CTAs = 2.98 waves), the
    direct kernel the L-shaped rest of 196 angles; padding to 64 x 64 (fill 0.55) or the direct kernel alone
    would both be slower.  Grids that fill whole tiles, and small problems, stay in one part."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("plan depends on the visible device's SM count; this checks the 148-SM default")
    d = radlib.rad_plan_describe
    p = d(1, 3000, 100, 50, 50, 0)
    assert (p["kernel"], p["parts"], p["interior_x"], p["interior_y"], p["tiles"], p["slices"]) == (2, 2, 48, 48, 63, 7)
    assert p["launches"] == 4                         # pack, separable main + reduction, fused single launch on the rest
    p = d(1, 3000, 100, 50, 50, 2)                   # spin-1/2: 16 x 16 x 8 tiles, 48 = 6 x 8 rows
    assert (p["parts"], p["interior_x"], p["interior_y"]) == (2, 48, 48)
    assert d(1, 14287, 256, 32, 32, 0)["parts"] == 1 and d(1, 3000, 100, 64, 48, 0)["parts"] == 1
    assert d(1, 3000, 100, 60, 60, 0)["parts"] == 1  # remainder 12 of 16: padding is cheaper than a second launch
    p = d(1, 3000, 100, 50, 64, 0)                   # only the x axis leaves a rest
    assert (p["parts"], p["interior_x"], p["interior_y"]) == (2, 48, 64)
    assert d(1, 3000, 17, 17, 17, 0)["kernel"] == 3  # 1.5e7 evals: the fused single-launch kernel


def test_sections_check(radlib):
    """every section must be longer than the formation length l_f = 2 gamma^2 (E - w)/(E w) at the
    lowest frequency of interest.  Golden numbers: the paper's own example (50 GeV, 5 GeV photon: 680 nm by the
    formula) and its 0.1 mm sections."""
    rows = [ln.split() for ln in (ROOT / "tests" / "golden" / "formation_length.txt").read_text().splitlines()
            if ln and not ln.startswith("#")]
    E_eV, w_eV, formula_m, _ = (float(v) for v in rows[0])
    me, hbarc = 0.51099895e6, 1.973269804e-7
    gamma, omega, lam = E_eV / me, w_eV / hbarc, hbarc / E_eV
    # boundaries: 0.1 mm sections and two short ones, just below and just above l_f
    t = np.array([0.0, 1e-4, 1e-4 + 0.999 * formula_m, 2e-4, 2e-4 + 1.001 * formula_m, 3e-4])
    g = np.full(5, gamma)
    assert list(radlib.rad_sections_check(t, g, omega, lam)) == [1]
    # classical (no recoil): l_f = 2 gamma^2 / w is longer by E/(E - w) = 1/0.9 -> section 3 is now too short as well
    assert list(radlib.rad_sections_check(t, g, omega)) == [1, 3]
    # a lower frequency lengthens l_f ~ 1/w: at w/1000 the 0.1 mm sections themselves are too short
    assert list(radlib.rad_sections_check(t, g, omega / 1000, lam)) == [0, 1, 2, 3, 4]
    # per-section energy: halving gamma quarters l_f
    g2 = g.copy()
    g2[1] = gamma / 2
    assert list(radlib.rad_sections_check(t, g2, omega, lam * np.array([1, 2, 1, 1, 1]))) == []
    with pytest.raises(radlib.RadError):
        radlib.rad_sections_check(t, g, 0.0, lam)                     # omega_min must be positive
    with pytest.raises(radlib.RadError):
        radlib.rad_sections_check(t[::-1].copy(), g, omega, lam)      # boundaries must ascend
    lib = radlib.load_library()                                       # raw ABI: count returned even when cap is too small
    idx = np.zeros(1, dtype=np.int32)
    lamv = np.full(5, lam)
    assert lib.rad_sections_check(5, t.ctypes.data, g.ctypes.data, lamv.ctypes.data, omega / 1000, idx.ctypes.data, 1) == 5
    assert idx[0] == 0


def test_formation_length_of_the_papers_example(radlib):
    """l_f = 2 gamma^2 (E - w)/(E w); "in the case of a 50 GeV positron emitting a 5 GeV photon
    l_f = 71 nm".  The formula gives 680 nm for those numbers (tests/golden/formation_length.txt): the paper's
    printed value is off by a factor 9.6 from its own formula, which DESIGN.md lists as a reading; the library
    implements the formula."""
    rows = [ln.split() for ln in (ROOT / "tests" / "golden" / "formation_length.txt").read_text().splitlines()
            if ln and not ln.startswith("#")]
    E_eV, w_eV, formula_m, printed_m = (float(v) for v in rows[0])
    me, hbarc = 0.51099895e6, 1.973269804e-7
    got = radlib.rad_formation_length(E_eV / me, w_eV / hbarc, hbarc / E_eV)
    assert got == pytest.approx(formula_m, rel=1e-6)
    assert got == pytest.approx(2 * (E_eV / me) ** 2 * (E_eV - w_eV) / (E_eV * w_eV) * hbarc, rel=1e-12)
    assert 9 < got / printed_m < 10                                   # the discrepancy, on record
    with pytest.raises(ValueError):
        radlib.rad_formation_length(1e5, 1e18, 1e-17)                 # hbar w >= E
