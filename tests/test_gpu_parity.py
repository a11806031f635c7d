"""GPU-vs-oracle parity (run with -m gpu on the B200 box).  Every call goes through the C ABI.

Tolerance (BASELINE.json north_star, Q14): at every compared point
|gpu - oracle| <= max(1e-9 |oracle|, 1e-12 S_max), S_max = maximum of the GPU cube;
the GPU arg-max point is always among the compared points.
"""
import os

import numpy as np
import pytest

import workloads

pytestmark = pytest.mark.gpu

RTOL, FLOOR = 1e-9, 1e-12
CL, S0, SH = 0, 1, 2


@pytest.fixture(scope="module")
def rad():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the CUDA path has no CPU fallback")
    import paper_1910_10391_b200 as rad
    rad.build_library()
    rad.load_library()
    return rad


def dev_dict(d):
    import torch
    return {k: torch.from_numpy(np.ascontiguousarray(v)).cuda() for k, v in d.items()}


def dev_grid(wl):
    import torch
    return [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (wl.omega, wl.thx, wl.thy)]


def assert_parity(gpu_cube, ref, idx=None, label=""):
    """gpu_cube: full GPU cube (numpy); ref: oracle values at flat indices idx (or full cube)."""
    flat = gpu_cube.ravel()
    assert np.all(np.isfinite(flat)), f"{label}: non-finite GPU output"
    s_max = flat.max()
    got = flat if idx is None else flat[idx]
    ref = np.asarray(ref).ravel()
    tol = np.maximum(RTOL * np.abs(ref), FLOOR * s_max)
    ratio = np.abs(got - ref) / tol
    worst = int(np.argmax(ratio))
    if os.environ.get("RAD_PARITY_LOG"):                     # optional record for profiles/ 
        with open(os.environ["RAD_PARITY_LOG"], "a") as f:
            f.write(f"{label}\t{len(ref)} points\tworst |err|/tol = {ratio[worst]:.3e}\t"
                    f"max rel err = {np.max(np.abs(got - ref) / np.maximum(np.abs(ref), 1e-300)):.3e}\n")
    assert ratio[worst] <= 1.0, (f"{label}: worst |err|/tol = {ratio[worst]:.3g} at compared point {worst} "
                                 f"(gpu {got[worst]:.17g}, oracle {ref[worst]:.17g}, S_max {s_max:.6g})")
    return float(ratio[worst])


def run_single(rad, wl, model, lam, kernel=0):
    """kernel: rad_options.kernel of the call (0 auto, 1 direct, 2 separable, 3 fused single-launch)."""
    tr, g = dev_dict(wl.traj), dev_grid(wl)
    if model == CL:
        return rad.rad_classical(tr, *g, kernel=kernel).cpu().numpy()
    return rad.rad_semiclassical(tr, *g, 0 if model == S0 else 1, lam, kernel=kernel).cpu().numpy()


def sampled_reference(oracle_mod, wl, cube, n_random, lattice, model, lam, seed=1):
    idx = workloads.sample_points(wl, n_random, lattice, seed=seed)
    idx = np.unique(np.concatenate([idx, [int(np.argmax(cube))]]))      # Q14: include the arg-max
    w, nx, ny = workloads.points_of(wl, idx)
    return idx, oracle_mod.points(wl.traj, w, nx, ny, model, lam)


# ------------------------------------------------------------------ small, full-grid comparisons
def test_cfg1_full_grid(rad, oracle_mod):
    """BASELINE.json configs[0] exactly, full grid (time-split path: 4 tiles only)."""
    wl = workloads.make("cfg1")
    cube = run_single(rad, wl, CL, 0.0)
    ref = oracle_mod.grid(wl.traj, wl.omega, wl.thx, wl.thy)
    assert_parity(cube, ref, label="cfg1")


@pytest.mark.parametrize("model", [CL, S0, SH])
@pytest.mark.parametrize("shape", [dict(n=2, n_omega=1, n_th=1), dict(n=129, n_omega=9, n_th=3),
                                   dict(n=1037, n_omega=13, n_th=5)])
def test_ragged_shapes_all_models(rad, oracle_mod, model, shape):
    """Ragged tails everywhere: n not a multiple of the 128-sample chunk (incl. the minimum n = 2),
    n_omega not a multiple of the 8-omega register tile, angle count not a multiple of 128."""
    wl = workloads.make("cfg2", seed=11, **shape)
    lam = 0.6 / wl.omega.max()
    cube = run_single(rad, wl, model, lam)
    ref = oracle_mod.grid(wl.traj, wl.omega, wl.thx, wl.thy, model, lam)
    assert_parity(cube, ref, label=f"ragged {shape} model {model}")


def test_rectangular_grid_order(rad, oracle_mod):
    """n_thx != n_thy: cube order (i_w, i_y, i_x), x fastest (Q11)."""
    wl = workloads.make("cfg2", n=700, n_omega=5, n_th=6, seed=5)
    wl.thx = wl.thx[:4].copy()
    wl.thy = (wl.thy * 0.7).copy()
    cube = run_single(rad, wl, SH, 0.3 / wl.omega.max())
    assert cube.shape == (5, 6, 4)
    ref = oracle_mod.grid(wl.traj, wl.omega, wl.thx, wl.thy, SH, 0.3 / wl.omega.max())
    assert_parity(cube, ref, label="rectangular")


def test_nonuniform_time_and_varying_gamma(rad, oracle_mod):
    """Trapezoid weights on a non-uniform t (Q1) and sample-wise 1/2gamma_k^2 (Q6)."""
    wl = workloads.make("cfg2", n=900, n_omega=10, n_th=4, seed=8)
    rng = np.random.Generator(np.random.PCG64(3))
    t = np.sort(rng.uniform(0, wl.traj["t"][-1], 900))
    tr = {k: np.interp(t, wl.traj["t"], v) for k, v in wl.traj.items()}
    tr["t"] = t
    tr["gamma"] = wl.traj["gamma"] * (1 - 1e-3 * np.linspace(0, 1, 900))
    wl.traj = tr
    lam = 0.5 / wl.omega.max()
    for model in (CL, SH):
        cube = run_single(rad, wl, model, lam)
        ref = oracle_mod.grid(tr, wl.omega, wl.thx, wl.thy, model, lam)
        assert_parity(cube, ref, label=f"nonuniform model {model}")


def test_straight_line_is_exact_zero(rad):
    """P1 on the GPU path: zero acceleration gives exactly 0, all variants."""
    wl = workloads.make("cfg2", n=500, n_omega=8, n_th=4)
    for k in ("ax", "ay", "az"):
        wl.traj[k] = np.zeros(500)
    for model in (CL, S0, SH):
        cube = run_single(rad, wl, model, 1e-16)
        assert np.all(cube == 0.0)


def test_domain_u_ge_1_gives_nan_only_there(rad, oracle_mod):
    """u = hbar w / E >= 1: NaN at those points only (include/rad.h), the rest in parity."""
    wl = workloads.make("cfg1", n=600, n_omega=8, n_th=2)
    lam = 1.0000001 / wl.omega[5]                 # u >= 1 from i_w = 5 on
    cube = run_single(rad, wl, S0, lam)
    assert np.all(np.isnan(cube[5:])) and np.all(np.isfinite(cube[:5]))
    ref = oracle_mod.grid(wl.traj, wl.omega[:5], wl.thx, wl.thy, S0, lam)
    assert_parity(cube[:5], ref, label="domain")


def test_deterministic(rad):
    wl = workloads.make("cfg2", n=2000, n_omega=16, n_th=8)
    a = run_single(rad, wl, SH, 1e-17)
    b = run_single(rad, wl, SH, 1e-17)
    assert np.array_equal(a, b)


# ------------------------------------------------------------------ launch-plan coverage
def test_direct_mode_many_tiles(rad, oracle_mod):
    """Grid large enough (>= 8 CTAs per SM) for the no-split path; sampled + lattice."""
    wl = workloads.make("cfg2", n=300, n_omega=40, n_th=200, seed=21)
    cube = run_single(rad, wl, CL, 0.0, kernel=1)      # the direct-phasor kernel (auto would pick the separable one)
    idx, ref = sampled_reference(oracle_mod, wl, cube, 3000, (5, 9, 9), CL, 0.0)
    assert_parity(cube, ref, idx, label="direct")


def test_workspace_argument(rad, oracle_mod):
    """Caller-provided workspace gives the same bits as pool-allocated scratch; too small -> error."""
    import torch
    wl = workloads.make("cfg2", n=1500, n_omega=16, n_th=8)
    tr, g = dev_dict(wl.traj), dev_grid(wl)
    nb = rad.rad_workspace_bytes(1, 1500, 16, 8, 8)
    assert nb > 0
    ws = torch.empty(nb, dtype=torch.uint8, device="cuda")
    a = rad.rad_classical(tr, *g, workspace=ws).cpu().numpy()
    b = rad.rad_classical(tr, *g).cpu().numpy()
    assert np.array_equal(a, b)
    with pytest.raises(rad.RadError) as e:
        rad.rad_classical(tr, *g, workspace=ws[:1024])
    assert e.value.code == -4


def test_invalid_arguments(rad):
    import torch
    wl = workloads.make("cfg1", n=100, n_omega=4, n_th=2)
    tr, g = dev_dict(wl.traj), dev_grid(wl)
    with pytest.raises(rad.RadError) as e:
        rad.rad_semiclassical(tr, *g, 2, 1e-15)
    assert e.value.code == -1
    with pytest.raises(rad.RadError) as e:
        rad.rad_semiclassical(tr, *g, 1, -1.0)
    assert e.value.code == -2
    short = {k: v[:1].contiguous() for k, v in tr.items()}
    with pytest.raises(rad.RadError):
        rad.rad_classical(short, *g)
    with pytest.raises(TypeError):
        rad.rad_classical({k: v.cpu() for k, v in tr.items()}, *g)
    del torch


# ------------------------------------------------------------------ ensembles
@pytest.mark.parametrize("model", [CL, SH])
def test_ensemble_small_ragged(rad, oracle_mod, model):
    """Few ragged trajectories (time-split path), per-trajectory hbar c / E."""
    we = workloads.make("cfg4", count=6, n=700, n_omega=9, n_th=5)
    nvec = np.array([700, 512, 129, 2, 700, 333], dtype=np.int64)
    lam = np.linspace(0.2, 0.7, 6) / we.omega.max() if model != CL else None
    cube = rad.rad_ensemble_sum(dev_dict(we.batch), nvec, *dev_grid(we), model=model,
                                hbarc_over_E=lam).cpu().numpy()
    w, nx, ny = oracle_mod.grid_points(we.omega, we.thx, we.thy)
    ref = oracle_mod.ensemble_points(we.batch, nvec, w, nx, ny, model, lam)
    assert_parity(cube, ref, label=f"ensemble small model {model}")


def test_ensemble_many_trajectories_and_accumulate(rad, oracle_mod):
    """Many short trajectories on a tiny grid (trajectory-split path), then accumulate=1
    continuing a partial ensemble (sum of section spectra)."""
    we = workloads.make("cfg4", count=400, n=300, n_omega=8, n_th=4, seed0=900)
    rng = np.random.Generator(np.random.PCG64(1))
    nvec = rng.integers(2, 301, size=400).astype(np.int64)
    b, g = dev_dict(we.batch), dev_grid(we)
    full = rad.rad_ensemble_sum(b, nvec, *g).cpu().numpy()
    w, nx, ny = oracle_mod.grid_points(we.omega, we.thx, we.thy)
    ref = oracle_mod.ensemble_points(we.batch, nvec, w, nx, ny)
    assert_parity(full, ref, label="ensemble many")
    first = rad.rad_ensemble_sum({k: v[:150].contiguous() for k, v in b.items()}, nvec[:150], *g)
    both = rad.rad_ensemble_sum({k: v[150:].contiguous() for k, v in b.items()}, nvec[150:], *g,
                                accumulate=True, out=first).cpu().numpy()
    assert_parity(both, ref, label="ensemble accumulate")


# ------------------------------------------------------------------ host-buffer entry points
def test_host_entry_points(rad, oracle_mod):
    wl = workloads.make("cfg2", n=1200, n_omega=12, n_th=6)
    lam = 0.4 / wl.omega.max()
    cube = rad.rad_eval_host(wl.traj, wl.omega, wl.thx, wl.thy, SH, lam)
    ref = oracle_mod.grid(wl.traj, wl.omega, wl.thx, wl.thy, SH, lam)
    assert_parity(cube, ref, label="host single")
    we = workloads.make("cfg4", count=4, n=500, n_omega=6, n_th=3)
    cube = rad.rad_ensemble_sum_host(we.batch, we.n, we.omega, we.thx, we.thy)
    w, nx, ny = oracle_mod.grid_points(we.omega, we.thx, we.thy)
    ref = oracle_mod.ensemble_points(we.batch, we.n, w, nx, ny)
    assert_parity(cube, ref, label="host ensemble")
    # accumulate on the host path: first two trajectories, then the other two added to the same cube
    part = rad.rad_ensemble_sum_host({k: np.ascontiguousarray(v[:2]) for k, v in we.batch.items()}, we.n[:2],
                                     we.omega, we.thx, we.thy)
    both = rad.rad_ensemble_sum_host({k: np.ascontiguousarray(v[2:]) for k, v in we.batch.items()}, we.n[2:],
                                     we.omega, we.thx, we.thy, accumulate=True, out=part)
    assert_parity(both, ref, label="host ensemble accumulate")
    # SoA arrays that follow one another in one host allocation go over in one transfer (partly adjacent: the first
    # seven fields in one block, the rest separate; grid arrays in one block): bit-identical results
    block = np.empty((7,) + we.batch["t"].shape)
    mixed = {}
    for i, k in enumerate(rad.FIELDS):
        if i < 7:
            block[i] = we.batch[k]
            mixed[k] = block[i]
        else:
            mixed[k] = we.batch[k].copy()
    gb = np.concatenate([we.omega, we.thx, we.thy])
    nw, nx_ = len(we.omega), len(we.thx)
    again = rad.rad_ensemble_sum_host(mixed, we.n, gb[:nw], gb[nw:nw + nx_], gb[nw + nx_:])
    assert np.array_equal(again, cube)
    # everything -- eleven fields and the grid behind them -- in ONE allocation: one transfer
    per = we.batch["t"].size
    flat = np.empty(11 * per + gb.size)
    whole = {}
    for i, k in enumerate(rad.FIELDS):
        whole[k] = flat[i * per:(i + 1) * per].reshape(we.batch[k].shape)
        whole[k][...] = we.batch[k]
    flat[11 * per:] = gb
    gf = flat[11 * per:]
    once = rad.rad_ensemble_sum_host(whole, we.n, gf[:nw], gf[nw:nw + nx_], gf[nw + nx_:])
    assert np.array_equal(once, cube)


# ------------------------------------------------------------------ angular sum (NEXT-1)
def test_angular_sum(rad):
    import torch
    wl = workloads.make("cfg2", n=800, n_omega=12, n_th=20)
    g = dev_grid(wl)
    cube = rad.rad_classical(dev_dict(wl.traj), *g)
    d_om = (wl.thx[1] - wl.thx[0]) * (wl.thy[1] - wl.thy[0])
    cut = 2.0 / wl.meta["gamma"]
    got = rad.rad_angular_sum(cube, *g, d_om, cut).cpu().numpy()
    c = cube.cpu().numpy()
    X, Y = np.meshgrid(wl.thx, wl.thy)
    mask = X * X + Y * Y <= cut * cut
    np.testing.assert_allclose(got, (c * mask).sum((1, 2)) * d_om, rtol=1e-13)
    got_all = rad.rad_angular_sum(cube, *g, d_om).cpu().numpy()
    np.testing.assert_allclose(got_all, c.sum((1, 2)) * d_om, rtol=1e-13)
    del torch


# ------------------------------------------------------------------ full-size configs, sampled
@pytest.fixture(params=[0, 1, 2], ids=["auto", "direct", "separable"])
def each_kernel(request):
    """The full-size configs run through the kernel the library picks (what bench.py times) and through
    each of the two kernels forced (include/rad.h rad_options.kernel)."""
    return request.param


def test_cfg2_full_size_sampled(rad, each_kernel, oracle_mod):
    """BASELINE.json configs[1] at full size, in the launch configuration bench.py times."""
    wl = workloads.make("cfg2")
    cube = run_single(rad, wl, CL, 0.0, each_kernel)
    idx, ref = sampled_reference(oracle_mod, wl, cube, 3000, (8, 6, 6), CL, 0.0)
    assert_parity(cube, ref, idx, label="cfg2 full")


def test_cfg3_full_size_sampled(rad, each_kernel, oracle_mod):
    """BASELINE.json configs[2]: spin-1/2, N = 2e5, |phase| up to ~1e6 rad; 512 x 64 x 64 grid."""
    wl = workloads.make("cfg3")
    cube = run_single(rad, wl, SH, wl.hbarc_over_E, each_kernel)
    idx, ref = sampled_reference(oracle_mod, wl, cube, 160, (4, 3, 3), SH, wl.hbarc_over_E)
    assert_parity(cube, ref, idx, label="cfg3 full")


def test_cfg4_reduced_ensemble_sampled(rad, each_kernel, oracle_mod):
    """configs[3] shape (128 x 16 x 16 grid, batched trajectories) with 48 x 20000 samples."""
    we = workloads.make("cfg4", count=48, n=20000)
    cube = rad.rad_ensemble_sum(dev_dict(we.batch), we.n, *dev_grid(we), kernel=each_kernel).cpu().numpy()
    idx = workloads.sample_points(we, 100, (4, 3, 3))
    idx = np.unique(np.concatenate([idx, [int(np.argmax(cube))]]))
    w, nx, ny = workloads.points_of(we, idx)
    ref = oracle_mod.ensemble_points(we.batch, we.n, w, nx, ny)
    assert_parity(cube, ref, idx, label="cfg4 reduced")


@pytest.mark.parametrize("model", [S0, SH])
def test_cfg5_reduced_sampled(rad, each_kernel, oracle_mod, model):
    """configs[4] (axial well, both spin variants) at N = 2e5 on the full 1024 x 64 x 64 grid."""
    wl = workloads.make("cfg5", n=200000, model=model)
    cube = run_single(rad, wl, model, wl.hbarc_over_E, each_kernel)
    idx, ref = sampled_reference(oracle_mod, wl, cube, 120, (4, 3, 3), model, wl.hbarc_over_E)
    assert_parity(cube, ref, idx, label=f"cfg5 model {model}")


# ------------------------------------------------------------------ sharding on one GPU
def test_sum_cubes_ordered(rad):
    import torch
    rng = np.random.Generator(np.random.PCG64(9))
    parts = rng.standard_normal((5, 7, 3, 11)) * 10.0 ** rng.integers(-8, 8, size=(5, 1, 1, 1))
    d = torch.from_numpy(parts).cuda()
    got = rad.rad_sum_cubes(d).cpu().numpy()
    want = parts[0].copy()
    for c in range(1, 5):
        want += parts[c]                                   # same order => same bits
    assert np.array_equal(got, want)
    again = rad.rad_sum_cubes(d, accumulate=True, out=torch.from_numpy(want).cuda()).cpu().numpy()
    acc = want.copy()
    for c in range(5):
        acc += parts[c]
    assert np.array_equal(again, acc)


def test_shards_run_sequentially_equal_unsharded(rad, oracle_mod):
    """Grid shards (omega slabs) reproduce the unsharded cube bit for bit when the launch plan is the
    same per point, and within tolerance otherwise; ensemble shards + rad_sum_cubes match the oracle."""
    import torch
    from paper_1910_10391_b200.sharding import shard_range
    wl = workloads.make("cfg2", n=900, n_omega=11, n_th=6, seed=14)
    tr, g = dev_dict(wl.traj), dev_grid(wl)
    ref = oracle_mod.grid(wl.traj, wl.omega, wl.thx, wl.thy)
    slabs = []
    for r in range(3):
        lo, hi = shard_range(11, r, 3)
        slabs.append(rad.rad_classical(tr, g[0][lo:hi].contiguous(), g[1], g[2]))
    assert_parity(torch.cat(slabs).cpu().numpy(), ref, label="grid shards")

    we = workloads.make("cfg4", count=7, n=400, n_omega=6, n_th=4, seed0=50)
    b, ge = dev_dict(we.batch), dev_grid(we)
    parts = []
    for r in range(3):
        lo, hi = shard_range(7, r, 3)
        parts.append(rad.rad_ensemble_sum({k: v[lo:hi].contiguous() for k, v in b.items()}, we.n[lo:hi], *ge))
    total = rad.rad_sum_cubes(torch.stack(parts)).cpu().numpy()
    w, nx, ny = oracle_mod.grid_points(we.omega, we.thx, we.thy)
    assert_parity(total, oracle_mod.ensemble_points(we.batch, we.n, w, nx, ny), label="ensemble shards")


# ------------------------------------------------------------------ separable-phasor kernel (N2), forced
class _Forced:
    """The binding with one kernel forced on every compute call (rad_options.kernel is per call)."""

    def __init__(self, rad, kernel):
        self._rad, self._kernel = rad, kernel

    def __getattr__(self, name):
        fn = getattr(self._rad, name)
        if name in ("rad_classical", "rad_semiclassical", "rad_ensemble_sum", "rad_sections_sum", "rad_eval_host",
                    "rad_ensemble_sum_host", "rad_angular_spectrum"):
            return lambda *a, **k: fn(*a, **{**k, "kernel": self._kernel})
        return fn


@pytest.fixture
def sep_kernel(rad):
    return _Forced(rad, 2)


@pytest.mark.parametrize("model", [CL, S0, SH])
@pytest.mark.parametrize("shape", [dict(n=2, n_omega=1, n_th=1), dict(n=131, n_omega=17, n_th=5),
                                   dict(n=1037, n_omega=33, n_th=19)])
def test_sep_ragged_shapes_all_models(sep_kernel, oracle_mod, model, shape):
    """Separable kernel on grids that are not multiples of its 16 x 16 x 16 (8) tiles, n not a multiple
    of the 4-sample sub-block or the 128-sample chunk (time-split plan)."""
    wl = workloads.make("cfg2", seed=12, **shape)
    lam = 0.6 / wl.omega.max()
    cube = run_single(sep_kernel, wl, model, lam)
    ref = oracle_mod.grid(wl.traj, wl.omega, wl.thx, wl.thy, model, lam)
    assert_parity(cube, ref, label=f"sep ragged {shape} model {model}")


def test_sep_rectangular_and_nonuniform(sep_kernel, oracle_mod):
    wl = workloads.make("cfg2", n=900, n_omega=10, n_th=21, seed=8)
    wl.thx = wl.thx[:18].copy()
    wl.thy = (wl.thy[:9] * 0.7).copy()
    rng = np.random.Generator(np.random.PCG64(3))
    t = np.sort(rng.uniform(0, wl.traj["t"][-1], 900))
    tr = {k: np.interp(t, wl.traj["t"], v) for k, v in wl.traj.items()}
    tr["t"] = t
    tr["gamma"] = wl.traj["gamma"] * (1 - 1e-3 * np.linspace(0, 1, 900))
    wl.traj = tr
    lam = 0.5 / wl.omega.max()
    for model in (CL, SH):
        cube = run_single(sep_kernel, wl, model, lam)
        assert cube.shape == (10, 9, 18)
        ref = oracle_mod.grid(tr, wl.omega, wl.thx, wl.thy, model, lam)
        assert_parity(cube, ref, label=f"sep rectangular nonuniform model {model}")


def test_sep_direct_mode_and_determinism(sep_kernel, oracle_mod):
    """Enough tiles for the no-split plan (>= 8 per SM); two runs give the same bits."""
    wl = workloads.make("cfg2", n=300, n_omega=80, n_th=256, seed=21)
    cube = run_single(sep_kernel, wl, CL, 0.0)
    idx, ref = sampled_reference(oracle_mod, wl, cube, 3000, (5, 9, 9), CL, 0.0)
    assert_parity(cube, ref, idx, label="sep direct")
    assert np.array_equal(cube, run_single(sep_kernel, wl, CL, 0.0))


@pytest.mark.parametrize("model", [CL, SH])
def test_sep_ensembles(sep_kernel, oracle_mod, model):
    """Few ragged trajectories (time split) and many short ones (trajectory split) + accumulate."""
    we = workloads.make("cfg4", count=6, n=700, n_omega=9, n_th=5)
    nvec = np.array([700, 512, 129, 2, 700, 333], dtype=np.int64)
    lam = np.linspace(0.2, 0.7, 6) / we.omega.max() if model != CL else None
    cube = sep_kernel.rad_ensemble_sum(dev_dict(we.batch), nvec, *dev_grid(we), model=model,
                                       hbarc_over_E=lam).cpu().numpy()
    w, nx, ny = oracle_mod.grid_points(we.omega, we.thx, we.thy)
    assert_parity(cube, oracle_mod.ensemble_points(we.batch, nvec, w, nx, ny, model, lam),
                  label=f"sep ensemble small model {model}")
    we = workloads.make("cfg4", count=400, n=300, n_omega=8, n_th=4, seed0=900)
    rng = np.random.Generator(np.random.PCG64(1))
    nvec = rng.integers(2, 301, size=400).astype(np.int64)
    lam = np.full(400, 0.4 / we.omega.max()) if model != CL else None
    b, g = dev_dict(we.batch), dev_grid(we)
    ref = oracle_mod.ensemble_points(we.batch, nvec, *oracle_mod.grid_points(we.omega, we.thx, we.thy), model, lam)
    full = sep_kernel.rad_ensemble_sum(b, nvec, *g, model=model, hbarc_over_E=lam).cpu().numpy()
    assert_parity(full, ref, label=f"sep ensemble many model {model}")
    first = sep_kernel.rad_ensemble_sum({k: v[:150].contiguous() for k, v in b.items()}, nvec[:150], *g,
                                        model=model, hbarc_over_E=None if lam is None else lam[:150])
    both = sep_kernel.rad_ensemble_sum({k: v[150:].contiguous() for k, v in b.items()}, nvec[150:], *g,
                                       model=model, hbarc_over_E=None if lam is None else lam[150:],
                                       accumulate=True, out=first).cpu().numpy()
    assert_parity(both, ref, label=f"sep ensemble accumulate model {model}")


def test_sep_cluster_pairs_time_and_trajectory_split(sep_kernel, oracle_mod):
    """The separable kernel as thread-block cluster pairs (an even number of theta_y tiles: the two CTAs of a pair
    share their T table through distributed shared memory) in the two split modes the full-size
    configs do not reach with ragged input: a time split of one short trajectory (classical, 2 y tiles of 16) and a
    trajectory split of a ragged ensemble with empty-ish members (spin-1/2, 2 y tiles of 8); an odd tile count next
    to it runs as single CTAs.  Bit-identical from run to run."""
    import torch
    rad = sep_kernel
    wl = workloads.make("cfg2", n=1500, n_omega=20, n_th=20, seed=31)
    thx = wl.thx[:5].copy()
    g = [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (wl.omega, thx, wl.thy)]
    plan = rad.rad_plan_describe(1, 1500, 20, 5, 20, CL, 2)
    assert plan["cluster"] == 2 and plan["mode"] == 2 and plan["kernel"] == 2
    tr = dev_dict(wl.traj)
    cube = rad.rad_classical(tr, *g)
    again = rad.rad_classical(tr, *g)
    assert torch.equal(cube, again)
    w, nx, ny = oracle_mod.grid_points(wl.omega, thx, wl.thy)
    assert_parity(cube.cpu().numpy(), oracle_mod.points(wl.traj, w, nx, ny, CL, 0.0), label="cluster time split")
    # 3 y tiles: no y neighbour for every tile.  Classical / spin-0 grids with an even number of omega tiles then pair
    # along omega and share the F table (cluster code 3); spin-1/2 and odd omega tile counts run as single CTAs.
    assert rad.rad_plan_describe(1, 1500, 20, 5, 40, CL, 2)["cluster"] == 3
    assert rad.rad_plan_describe(1, 1500, 20, 5, 40, SH, 2)["cluster"] == 1
    assert rad.rad_plan_describe(1, 1500, 40, 5, 40, CL, 2)["cluster"] == 1
    thy3 = np.linspace(wl.thy[0], wl.thy[-1], 40)
    g3 = [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (wl.omega, thx, thy3)]
    for spin in (None, 0):                             # time split through the omega pairs, classical and spin-0
        lam3 = 0.4 / wl.omega.max()
        cube = rad.rad_classical(tr, *g3) if spin is None else rad.rad_semiclassical(tr, *g3, 0, lam3)
        again = rad.rad_classical(tr, *g3) if spin is None else rad.rad_semiclassical(tr, *g3, 0, lam3)
        assert torch.equal(cube, again)
        w, nx, ny = oracle_mod.grid_points(wl.omega, thx, thy3)
        assert_parity(cube.cpu().numpy(), oracle_mod.points(wl.traj, w, nx, ny, CL if spin is None else S0,
                                                            0.0 if spin is None else lam3), label="omega pairs time split")

    we = workloads.make("cfg4", count=40, n=260, n_omega=9, n_th=11, seed0=1234)
    thx = we.thx[:6].copy()
    rng = np.random.Generator(np.random.PCG64(5))
    nvec = rng.integers(2, 261, size=40).astype(np.int64)
    nvec[[0, 7, 39]] = 2
    lam = np.linspace(0.1, 0.6, 40) / we.omega.max()
    plan = rad.rad_plan_describe(40, 260, 9, 6, 11, SH, 2)
    assert plan["cluster"] == 2 and plan["mode"] == 1
    ge = [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (we.omega, thx, we.thy)]
    b = dev_dict(we.batch)
    cube = rad.rad_ensemble_sum(b, nvec, *ge, model=SH, hbarc_over_E=lam)
    assert torch.equal(cube, rad.rad_ensemble_sum(b, nvec, *ge, model=SH, hbarc_over_E=lam))
    w, nx, ny = oracle_mod.grid_points(we.omega, thx, we.thy)
    assert_parity(cube.cpu().numpy(), oracle_mod.ensemble_points(we.batch, nvec, w, nx, ny, SH, lam),
                  label="cluster trajectory split")
    # the same ragged ensemble, classical, on 20 omegas x one angle tile: omega pairs in the trajectory split
    we2 = workloads.make("cfg4", count=40, n=260, n_omega=20, n_th=7, seed0=1234)
    plan = rad.rad_plan_describe(40, 260, 20, 7, 7, CL, 2)
    assert plan["cluster"] == 3 and plan["mode"] == 1
    cube = rad.rad_ensemble_sum(dev_dict(we2.batch), nvec, *dev_grid(we2))
    w, nx, ny = oracle_mod.grid_points(we2.omega, we2.thx, we2.thy)
    assert_parity(cube.cpu().numpy(), oracle_mod.ensemble_points(we2.batch, nvec, w, nx, ny),
                  label="omega pairs trajectory split")


# ------------------------------------------------------------------ edge cases through the separable kernel too
def test_sep_straight_line_domain_and_workspace(sep_kernel, oracle_mod):
    """P1 (zero acceleration -> exactly 0), u >= 1 -> NaN only there, caller workspace == pool scratch,
    all through the separable kernel (the same checks above run through the direct one)."""
    import torch
    rad = sep_kernel
    wl = workloads.make("cfg2", n=500, n_omega=8, n_th=4)
    for k in ("ax", "ay", "az"):
        wl.traj[k] = np.zeros(500)
    for model in (CL, S0, SH):
        assert np.all(run_single(rad, wl, model, 1e-16) == 0.0)

    wl = workloads.make("cfg1", n=600, n_omega=8, n_th=2)
    lam = 1.0000001 / wl.omega[5]
    cube = run_single(rad, wl, SH, lam)
    assert np.all(np.isnan(cube[5:])) and np.all(np.isfinite(cube[:5]))
    assert_parity(cube[:5], oracle_mod.grid(wl.traj, wl.omega[:5], wl.thx, wl.thy, SH, lam), label="sep domain")

    wl = workloads.make("cfg2", n=1500, n_omega=16, n_th=8)
    tr, g = dev_dict(wl.traj), dev_grid(wl)
    ws = torch.empty(rad.rad_workspace_bytes(1, 1500, 16, 8, 8), dtype=torch.uint8, device="cuda")
    a = rad.rad_classical(tr, *g, workspace=ws).cpu().numpy()
    b = rad.rad_classical(tr, *g).cpu().numpy()
    assert np.array_equal(a, b)


def test_plan_kernel_choice(rad):
    """rad_plan_kernel: separable where the grid fills its tiles (BASELINE configs 2-5), direct on small angle
    grids with long trajectories, the fused single-launch kernel on small problems (config 1); the per-call
    option overrides; a bad option is rejected by the call itself."""
    assert rad.rad_plan_kernel(256, 32, 32, CL) == 2 and rad.rad_plan_kernel(512, 64, 64, SH) == 2
    assert rad.rad_plan_kernel(128, 16, 16, CL) == 2 and rad.rad_plan_kernel(1024, 64, 64, S0) == 2
    assert rad.rad_plan_kernel(64, 8, 8, CL) == 1 and rad.rad_plan_kernel(5, 3, 3, SH) == 1       # n_max = 2^20
    assert rad.rad_plan_kernel(64, 8, 8, CL, n_max=4000) == 3 and rad.rad_plan_kernel(5, 3, 3, SH, n_max=900) == 3
    assert rad.rad_plan_kernel(64, 8, 8, CL, n_max=4000, count=2) == 1
    assert rad.rad_plan_kernel(256, 32, 32, CL, kernel=1) == 1
    assert rad.rad_plan_kernel(5, 3, 3, SH, kernel=2) == 2
    wl = workloads.make("cfg1", n=100, n_omega=4, n_th=2)
    with pytest.raises(rad.RadError) as e:
        rad.rad_classical(dev_dict(wl.traj), *dev_grid(wl), kernel=7)
    assert e.value.code == -1


def test_sep_matches_direct_kernel(rad, oracle_mod):
    """Both kernels on the same input agree far inside the tolerance (they share only the packed records)."""
    wl = workloads.make("cfg3", n=5000, n_omega=32, n_th=32)
    a = run_single(rad, wl, SH, wl.hbarc_over_E, kernel=1)
    b = run_single(rad, wl, SH, wl.hbarc_over_E, kernel=2)
    tol = np.maximum(RTOL * np.abs(a), FLOOR * a.max())
    assert np.max(np.abs(a - b) / tol) <= 1.0


# ------------------------------------------------------------------ sectioned trajectory (NEXT row N3)
@pytest.mark.parametrize("kernel", [1, 2])
def test_sections_sum(rad, oracle_mod, kernel):
    """one trajectory cut into sections with their own energy; spectrum = sum of the
    section spectra.  Oracle: the sections copied out as an ensemble (shared boundary samples)."""
    wl = workloads.make("cfg3", n=3000, n_omega=12, n_th=10, seed=17)
    start = np.array([0, 700, 701, 1500, 2999], dtype=np.int64)          # one 2-sample section, ragged lengths
    lam = wl.hbarc_over_E * np.array([1.0, 1.02, 1.05, 1.1])             # energy drops from section to section
    tr = {k: v.copy() for k, v in wl.traj.items()}
    for s in range(4):                                                   # per-section gamma, as the paper fixes E per section
        tr["gamma"][start[s] + (s > 0):start[s + 1] + 1] = wl.meta["gamma"] / (lam[s] / lam[0])
    nvec = np.diff(start) + 1
    batch = {k: np.zeros((4, nvec.max())) for k in tr}
    for s in range(4):
        for k in tr:
            batch[k][s, :nvec[s]] = tr[k][start[s]:start[s + 1] + 1]
    # the shared boundary sample is ONE array entry read by both neighbours (include/rad.h, boundary-sample rule):
    # it carries the NEW section's gamma here, and the oracle batch is cut from the same arrays
    trs = {k: v.copy() for k, v in tr.items()}
    w, nx, ny = oracle_mod.grid_points(wl.omega, wl.thx, wl.thy)
    for model in (CL, SH):
        ref = oracle_mod.ensemble_points(batch, nvec, w, nx, ny, model, lam if model else None)
        cube = rad.rad_sections_sum(dev_dict(trs), start, *dev_grid(wl), model=model,
                                    hbarc_over_E=lam if model else None, kernel=kernel).cpu().numpy()
        assert_parity(cube, ref, label=f"sections kernel {kernel} model {model}")
    half = rad.rad_sections_sum(dev_dict(trs), start[:3], *dev_grid(wl), model=SH, hbarc_over_E=lam[:2], kernel=kernel)
    both = rad.rad_sections_sum(dev_dict(trs), start[2:], *dev_grid(wl), model=SH, hbarc_over_E=lam[2:],
                                accumulate=True, out=half, kernel=kernel).cpu().numpy()
    assert_parity(both, ref, label=f"sections accumulate kernel {kernel}")
    # ONE section that starts inside the trajectory: a single short trajectory at an offset -- the shape the fused
    # single-launch kernel takes (regression: its plan overlays the partial amplitudes on the unused packed buffer, so
    # falling through to the multi-launch path with that plan corrupted the records)
    one = np.array([701, 1500], dtype=np.int64)
    b1 = {k: tr[k][None, 701:1501].copy() for k in tr}
    for model in (CL, S0, SH):
        ref1 = oracle_mod.ensemble_points(b1, np.array([800]), w, nx, ny, model, lam[2:3] if model else None)
        c1 = rad.rad_sections_sum(dev_dict(trs), one, *dev_grid(wl), model=model, hbarc_over_E=lam[2:3] if model else None,
                                  kernel=kernel).cpu().numpy()
        assert_parity(c1, ref1, label=f"one section kernel {kernel} model {model}")
    with pytest.raises(rad.RadError):
        rad.rad_sections_sum(dev_dict(trs), [0, 10, 10], *dev_grid(wl))
    with pytest.raises(rad.RadError):
        rad.rad_sections_sum(dev_dict(trs), [0, 3000], *dev_grid(wl))


def test_concurrent_host_threads_with_different_options(rad):
    """include/rad.h: no process-wide switch, per-call options, "two threads may call with different options".  Four
    host threads (ctypes releases the GIL during the call), each on its own stream with its own kernel option, model
    and grid, 25 calls each; every result equals the serial one bit for bit."""
    import threading
    import torch
    jobs = []
    for i, (kernel, model, shape) in enumerate([(1, CL, dict(n=900, n_omega=24, n_th=9)), (2, SH, dict(n=1100, n_omega=32, n_th=16)),
                                                (3, S0, dict(n=1500, n_omega=20, n_th=6)), (0, SH, dict(n=700, n_omega=40, n_th=20))]):
        wl = workloads.make("cfg2", seed=50 + i, **shape)
        lam = 0.4 / wl.omega.max()
        tr, g = dev_dict(wl.traj), dev_grid(wl)
        call = (lambda tr=tr, g=g, kernel=kernel, model=model, lam=lam, **kw:
                rad.rad_classical(tr, *g, kernel=kernel, **kw) if model == CL
                else rad.rad_semiclassical(tr, *g, 0 if model == S0 else 1, lam, kernel=kernel, **kw))
        jobs.append((call, call().clone()))
    torch.cuda.synchronize()
    errors = []

    def worker(call, ref):
        try:
            st = torch.cuda.Stream()
            with torch.cuda.stream(st):
                for _ in range(25):
                    out = call(stream=st)
                    st.synchronize()
                    if not torch.equal(out, ref):
                        errors.append("result differs from the serial call")
                        return
        except Exception as e:                                   # noqa: BLE001 -- reported below
            errors.append(repr(e))

    threads = [threading.Thread(target=worker, args=j) for j in jobs]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    assert not errors, errors


# ------------------------------------------------------------------ seeded random shapes
@pytest.mark.parametrize("seed", [11, 12, 13])
def test_random_shapes_models_kernels_and_entry_points(rad, oracle_mod, seed):
    """120 seeded random cases per seed: grid shapes around the tile edges (1 ... 51 angles per axis, 1 ... 69 omegas),
    trajectory lengths around the chunk edges, all three models, the library's kernel choice and each kernel forced,
    single trajectories, ragged ensembles (with and without accumulate in two calls) and single sections at an offset --
    the launch plans this reaches include time and trajectory splits, cluster pairs along theta_y and along omega, and
    the fused kernel.  Sampled points (always the arg-max and both corners) against the oracle.  (A longer unseeded
    run of the same generator found the single-section bug fixed in rad.cu's run_batch.)"""
    import torch
    rng = np.random.Generator(np.random.PCG64(seed))
    for case in range(120):
        model = int(rng.integers(0, 3)); kernel = int(rng.choice([0, 0, 0, 1, 2]))
        n = int(rng.choice([2, 3, 127, 128, 129, 500, 1025, 2600]))
        nw, nx, ny = int(rng.integers(1, 70)), int(rng.integers(1, 52)), int(rng.integers(1, 52))
        kind = str(rng.choice(["single", "single", "ensemble", "section"]))
        cnt = int(rng.integers(1, 6)) if kind == "ensemble" else 1
        we = workloads.make("cfg4", count=cnt, n=n, n_omega=nw, n_th=max(nx, ny), seed0=int(rng.integers(1, 5000)))
        thx, thy = we.thx[:nx].copy(), we.thy[max(nx, ny) - ny:].copy()
        g = [torch.from_numpy(a).cuda() for a in (we.omega, thx, thy)]
        lam = rng.uniform(0.05, 0.8, size=cnt) / we.omega.max() if model else None
        nvec = rng.integers(2, n + 1, size=cnt).astype(np.int64) if kind == "ensemble" else np.array([n], dtype=np.int64)
        batch = we.batch
        if kind == "single":
            tr = {k: v[0] for k, v in batch.items()}
            cube = run_single(rad, types_workload(tr, we.omega, thx, thy), model, None if lam is None else float(lam[0]), kernel)
        elif kind == "section":
            lo = int(rng.integers(0, n - 1)); hi = int(rng.integers(lo + 1, n))
            tr = {k: v[0] for k, v in batch.items()}
            cube = rad.rad_sections_sum(dev_dict(tr), [lo, hi], *g, model=model, hbarc_over_E=lam, kernel=kernel).cpu().numpy()
            batch = {k: v[:, lo:hi + 1].copy() for k, v in batch.items()}
            nvec = np.array([hi - lo + 1], dtype=np.int64)
        else:
            b = dev_dict(batch)
            cut = int(rng.integers(0, cnt + 1))
            if 0 < cut < cnt:
                first = rad.rad_ensemble_sum({k: v[:cut].contiguous() for k, v in b.items()}, nvec[:cut], *g, model=model,
                                             hbarc_over_E=None if lam is None else lam[:cut], kernel=kernel)
                cube = rad.rad_ensemble_sum({k: v[cut:].contiguous() for k, v in b.items()}, nvec[cut:], *g, model=model,
                                            hbarc_over_E=None if lam is None else lam[cut:], accumulate=True, out=first,
                                            kernel=kernel).cpu().numpy()
            else:
                cube = rad.rad_ensemble_sum(b, nvec, *g, model=model, hbarc_over_E=lam, kernel=kernel).cpu().numpy()
        flat = cube.ravel()
        idx = np.unique(np.concatenate([rng.integers(0, flat.size, size=min(flat.size, 20)), [int(np.argmax(flat)), 0, flat.size - 1]]))
        iw, iy, ix = np.unravel_index(idx, cube.shape)
        ref = oracle_mod.ensemble_points(batch, nvec, we.omega[iw], thx[ix], thy[iy], model, lam)
        assert_parity(cube, ref, idx, label=f"random seed {seed} case {case}: {kind} n={n} grid {nw}x{ny}x{nx} model {model} kernel {kernel}")


def types_workload(traj, omega, thx, thy):
    """The few attributes run_single reads, for a trajectory that did not come from workloads.make."""
    import types
    return types.SimpleNamespace(traj=traj, omega=omega, thx=thx, thy=thy)


# ------------------------------------------------------------------ extreme shapes the paper names
def test_three_thousand_squared_angles(rad, oracle_mod):
    """"more than 3000^2" angular points without multiple scattering.  2 omegas x 3000 x 3000
    angles = 1.8e7 integrals (144 MB cube) over a short trajectory; sampled against the oracle."""
    wl = workloads.make("cfg2", n=150, n_omega=2, n_th=3000, seed=33)
    cube = run_single(rad, wl, CL, 0.0)
    assert cube.shape == (2, 3000, 3000)
    idx, ref = sampled_reference(oracle_mod, wl, cube, 4000, (2, 7, 7), CL, 0.0)
    assert_parity(cube, ref, idx, label="3000^2 angles")


@pytest.mark.parametrize("kernel", [1, 2])
def test_million_samples_on_a_small_grid(rad, oracle_mod, kernel):
    """configs[4]'s trajectory length (N = 1e6, phases to 3.8e6 rad) on a grid small enough that the time
    axis is split across the whole GPU (7813 chunks), both kernels, spin-1/2."""
    wl = workloads.make("cfg5", n=1000000, n_omega=16, n_th=16)
    cube = run_single(rad, wl, SH, wl.hbarc_over_E, kernel=kernel)
    idx, ref = sampled_reference(oracle_mod, wl, cube, 40, (3, 3, 3), SH, wl.hbarc_over_E)
    assert_parity(cube, ref, idx, label=f"N=1e6 kernel {kernel}")


# ------------------------------------------------------------------ configs[3] and configs[4] at FULL size
@pytest.mark.parametrize("model", [S0, SH])
def test_cfg5_full_size_sampled(rad, oracle_mod, model):
    """BASELINE.json configs[4] exactly (N = 1e6, 1024 x 64 x 64, phases to 3.8e6 rad), both spin variants,
    in the launch configuration bench.py times (the library's own kernel choice); sampled outputs."""
    wl = workloads.make("cfg5", model=model)
    cube = run_single(rad, wl, model, wl.hbarc_over_E)
    idx, ref = sampled_reference(oracle_mod, wl, cube, 48, (3, 3, 3), model, wl.hbarc_over_E)
    assert_parity(cube, ref, idx, label=f"cfg5 FULL model {model}")


def test_cfg4_full_size_sampled(rad, oracle_mod):
    """BASELINE.json configs[3] exactly: 1000 trajectories x 1e5 samples (8.8 GB of trajectories) summed on the
    128 x 16 x 16 grid, as bench.py --workload cfg4 times it; a dozen sampled points (1e8 samples each)."""
    we = workloads.make("cfg4")
    cube = rad.rad_ensemble_sum(dev_dict(we.batch), we.n, *dev_grid(we)).cpu().numpy()
    idx = workloads.sample_points(we, 10, (0, 0, 0))
    idx = np.unique(np.concatenate([idx, [int(np.argmax(cube))]]))
    w, nx, ny = workloads.points_of(we, idx)
    ref = oracle_mod.ensemble_points(we.batch, we.n, w, nx, ny)
    assert_parity(cube, ref, idx, label="cfg4 FULL")


def test_angular_spectrum_in_slabs(rad, oracle_mod):
    """rad_angular_spectrum without the 460 MB cube of the whole grid (the sums come out of the main kernel's
    epilogue); equals cube + rad_angular_sum, and the oracle's sum on a small grid (cube path inside the workspace)."""
    import torch
    wl = workloads.make("cfg2", n=120, n_omega=40, n_th=1200, seed=19)
    g = dev_grid(wl)
    d_om = (wl.thx[1] - wl.thx[0]) * (wl.thy[1] - wl.thy[0])
    cut = 2.5 / wl.meta["gamma"]
    b = {k: v[None, :].contiguous() for k, v in dev_dict(wl.traj).items()}
    n = np.array([120], dtype=np.int64)
    assert rad.load_library().rad_angular_spectrum_workspace_bytes(1, 120, 40, 1200, 1200) < 1200 * 1200 * 8 * 20
    assert rad.rad_plan_describe(1, 120, 40, 1200, 1200)["mode"] == 0      # one CTA per tile: sums in the epilogue
    got = rad.rad_angular_spectrum(b, n, *g, d_om, cut).cpu().numpy()
    cube = rad.rad_classical(dev_dict(wl.traj), *g)
    want = rad.rad_angular_sum(cube, *g, d_om, cut).cpu().numpy()
    np.testing.assert_allclose(got, want, rtol=1e-12)
    del cube
    torch.cuda.empty_cache()
    ws = workloads.make("cfg3", n=800, n_omega=9, n_th=7, seed=23)          # small: against the oracle, spin-1/2
    gs = dev_grid(ws)
    bs = {k: v[None, :].contiguous() for k, v in dev_dict(ws.traj).items()}
    got = rad.rad_angular_spectrum(bs, np.array([800]), *gs, 1.0, 0.0, model=SH, hbarc_over_E=ws.hbarc_over_E)
    ref = oracle_mod.grid(ws.traj, ws.omega, ws.thx, ws.thy, SH, ws.hbarc_over_E).sum((1, 2))
    np.testing.assert_allclose(got.cpu().numpy(), ref, rtol=1e-9)
    with pytest.raises(rad.RadError) as e:
        rad.rad_angular_spectrum(bs, np.array([800]), *gs, 1.0, workspace=torch.empty(1024, dtype=torch.uint8, device="cuda"))
    assert e.value.code == -4


def test_single_trajectory_call_is_graph_capturable(rad):
    """With a caller workspace a single-trajectory call only enqueues kernels (no host sync, no allocation, no
    host copy), so it can be captured in a CUDA graph and replayed; replays reproduce the eager bits."""
    import torch
    for shape, kernel in ((dict(n=900, n_omega=16, n_th=6), 1), (dict(n=900, n_omega=32, n_th=16), 2),
                          (dict(n=900, n_omega=16, n_th=6), 3)):
        wl = workloads.make("cfg2", seed=4, **shape)
        tr, g = dev_dict(wl.traj), dev_grid(wl)
        lam = 0.4 / wl.omega.max()
        ws = torch.empty(rad.rad_workspace_bytes(1, 900, len(wl.omega), len(wl.thx), len(wl.thy)),
                         dtype=torch.uint8, device="cuda")
        out = torch.zeros((len(wl.omega), len(wl.thy), len(wl.thx)), dtype=torch.float64, device="cuda")
        eager = rad.rad_semiclassical(tr, *g, 1, lam, workspace=ws, kernel=kernel).clone()   # also warms up the kernels
        graph = torch.cuda.CUDAGraph()
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(side):
            with torch.cuda.graph(graph, stream=side):
                rad.rad_semiclassical(tr, *g, 1, lam, out=out, workspace=ws, kernel=kernel)
        torch.cuda.current_stream().wait_stream(side)
        for _ in range(3):
            out.zero_()
            graph.replay()
            torch.cuda.synchronize()
            assert torch.equal(out, eager)


# ------------------------------------------------------------------ fused single-launch kernel (row a6, small problems)
def test_fused_kernel_is_what_cfg1_runs(rad, oracle_mod):
    """BASELINE configs[0] through the library's own choice: ONE launch (pack, time split over all SMs, grid-wide
    ordered reduction, epilogue), full grid against the oracle, deterministic, accumulate adds."""
    wl = workloads.make("cfg1")
    plan = rad.rad_plan_describe(1, 4000, 64, 8, 8)
    assert plan["kernel"] == 3 and plan["launches"] == 1
    tr, g = dev_dict(wl.traj), dev_grid(wl)
    n0 = rad.rad_launch_count()
    cube = rad.rad_classical(tr, *g)
    assert rad.rad_launch_count() - n0 == 1
    ref = oracle_mod.grid(wl.traj, wl.omega, wl.thx, wl.thy)
    assert_parity(cube.cpu().numpy(), ref, label="cfg1 fused")
    assert np.array_equal(cube.cpu().numpy(), rad.rad_classical(tr, *g).cpu().numpy())
    direct = rad.rad_classical(tr, *g, kernel=1).cpu().numpy()          # the three-launch path, same arithmetic per sample
    tol = np.maximum(RTOL * np.abs(direct), FLOOR * direct.max())
    assert np.max(np.abs(direct - cube.cpu().numpy()) / tol) <= 1e-3


@pytest.mark.parametrize("model", [CL, S0, SH])
@pytest.mark.parametrize("shape", [dict(n=2, n_omega=1, n_th=1), dict(n=63, n_omega=3, n_th=2), dict(n=129, n_omega=9, n_th=3),
                                   dict(n=1037, n_omega=13, n_th=5), dict(n=5000, n_omega=17, n_th=17)])
def test_fused_kernel_ragged_shapes_all_models(rad, oracle_mod, model, shape):
    """Forced fused kernel: n below / not a multiple of its 64-sample rounds, omega count not a multiple of 8,
    thread count not a multiple of 64, more time slices than samples allow."""
    wl = workloads.make("cfg2", seed=13, **shape)
    lam = 0.6 / wl.omega.max()
    cube = run_single(rad, wl, model, lam, kernel=3)
    ref = oracle_mod.grid(wl.traj, wl.omega, wl.thx, wl.thy, model, lam)
    assert_parity(cube, ref, label=f"fused ragged {shape} model {model}")


def test_fused_kernel_edges(rad, oracle_mod):
    """Straight line -> exactly 0; u >= 1 -> NaN only there; non-uniform t and varying gamma; long trajectory on a tiny
    grid (forced: auto would take the TMA-pipelined path); refused where it does not apply."""
    wl = workloads.make("cfg2", n=500, n_omega=8, n_th=4)
    for k in ("ax", "ay", "az"):
        wl.traj[k] = np.zeros(500)
    for model in (CL, S0, SH):
        assert np.all(run_single(rad, wl, model, 1e-16, kernel=3) == 0.0)
    wl = workloads.make("cfg1", n=600, n_omega=8, n_th=2)
    lam = 1.0000001 / wl.omega[5]
    cube = run_single(rad, wl, SH, lam, kernel=3)
    assert np.all(np.isnan(cube[5:])) and np.all(np.isfinite(cube[:5]))
    assert_parity(cube[:5], oracle_mod.grid(wl.traj, wl.omega[:5], wl.thx, wl.thy, SH, lam), label="fused domain")
    wl = workloads.make("cfg2", n=900, n_omega=10, n_th=4, seed=8)
    rng = np.random.Generator(np.random.PCG64(3))
    t = np.sort(rng.uniform(0, wl.traj["t"][-1], 900))
    tr = {k: np.interp(t, wl.traj["t"], v) for k, v in wl.traj.items()}
    tr["t"] = t
    tr["gamma"] = wl.traj["gamma"] * (1 - 1e-3 * np.linspace(0, 1, 900))
    wl.traj = tr
    lam = 0.5 / wl.omega.max()
    assert_parity(run_single(rad, wl, SH, lam, kernel=3), oracle_mod.grid(tr, wl.omega, wl.thx, wl.thy, SH, lam),
                  label="fused nonuniform")
    wl = workloads.make("cfg5", n=100000, n_omega=8, n_th=4)
    cube = run_single(rad, wl, SH, wl.hbarc_over_E, kernel=3)
    assert_parity(cube, oracle_mod.grid(wl.traj, wl.omega, wl.thx, wl.thy, SH, wl.hbarc_over_E), label="fused N=1e5")
    big = workloads.make("cfg2", n=200, n_omega=64, n_th=128)
    with pytest.raises(rad.RadError) as e:
        run_single(rad, big, CL, 0.0, kernel=3)                         # 2048 tiles of 64 threads: more CTAs than fit at once
    assert e.value.code == -1
    we = workloads.make("cfg4", count=2, n=300, n_omega=4, n_th=2)
    with pytest.raises(rad.RadError):
        rad.rad_ensemble_sum(dev_dict(we.batch), we.n, *dev_grid(we), kernel=3)


# ------------------------------------------------------------------ two-part plan: separable interior + direct L-shaped rest
@pytest.mark.parametrize("model", [CL, SH])
def test_papers_typical_grid_in_two_parts(rad, oracle_mod, model):
    """PAPER.md:149's typical grid with multiple scattering, N_x = N_y = 50, N_w = 100, N = 3000: the
    library's own plan (separable kernel on 48 x 48 angles, direct kernel on the other 196), full grid against the
    oracle; the output of both parts lands in the one cube with the right strides."""
    wl = workloads.make("paper_typical", model=model)
    plan = rad.rad_plan_describe(1, len(wl.traj["t"]), 100, 50, 50, model)
    assert (plan["parts"], plan["interior_x"], plan["interior_y"]) == (2, 48, 48)
    lam = wl.hbarc_over_E
    cube = run_single(rad, wl, model, lam)
    assert cube.shape == (100, 50, 50)
    ref = oracle_mod.grid(wl.traj, wl.omega, wl.thx, wl.thy, model, lam)
    assert_parity(cube, ref, label=f"paper typical model {model}")


@pytest.mark.parametrize("kernel", [0, 1, 2, 3])
def test_seventeen_cubed_through_every_kernel(rad, oracle_mod, kernel):
    """17 x 17 x 17: one more than a tile in every direction (the separable kernel pads to 32 x 32 x 32, fill 0.15; the
    direct kernel has a ragged last omega group of 1; the library's own choice is the fused kernel), spin-1/2, full grid
    against the oracle through the library's choice and through each kernel forced."""
    wl = workloads.make("cfg2", n=3000, n_omega=17, n_th=17, seed=21)
    lam = 0.45 / wl.omega.max()
    if kernel == 0:
        assert rad.rad_plan_kernel(17, 17, 17, SH, n_max=3000) == 3
    cube = run_single(rad, wl, SH, lam, kernel=kernel)
    assert_parity(cube, oracle_mod.grid(wl.traj, wl.omega, wl.thx, wl.thy, SH, lam), label=f"17^3 kernel {kernel}")


def test_two_parts_rectangular_rest_on_one_axis_and_ensemble(rad, oracle_mod):
    """Only one axis leaves a rest (50 x 32: columns 48, 49), n_thx != n_thy, an ensemble with accumulate; against the
    oracle on a sample of points that covers interior, rest and the corners."""
    we = workloads.make("cfg4", count=3, n=2500, n_omega=40, n_th=50, seed0=77)
    we.thy = we.thy[:32].copy()
    plan = rad.rad_plan_describe(3, 2500, 40, 50, 32)
    assert (plan["parts"], plan["interior_x"], plan["interior_y"]) == (2, 48, 32)
    b, g = dev_dict(we.batch), dev_grid(we)
    first = rad.rad_ensemble_sum({k: v[:1].contiguous() for k, v in b.items()}, we.n[:1], *g)
    cube = rad.rad_ensemble_sum({k: v[1:].contiguous() for k, v in b.items()}, we.n[1:], *g, accumulate=True,
                                out=first).cpu().numpy()
    assert cube.shape == (40, 32, 50)
    rng = np.random.Generator(np.random.PCG64(5))
    iw, iy, ix = rng.integers(0, 40, 600), rng.integers(0, 32, 600), rng.integers(0, 50, 600)
    ix[:200] = rng.integers(48, 50, 200)                                # the rest columns
    idx = np.unique(np.concatenate([(iw * 32 + iy) * 50 + ix, [0, 49, 31 * 50, 40 * 32 * 50 - 1, int(np.argmax(cube))]]))
    W_, Y_, X_ = np.unravel_index(idx, cube.shape)
    ref = oracle_mod.ensemble_points(we.batch, we.n, we.omega[W_], we.thx[X_], we.thy[Y_])
    assert_parity(cube, ref, idx, label="two parts ensemble")


# ------------------------------------------------------------------ angular spectrum from the epilogue (NEXT row N1)
@pytest.mark.parametrize("kernel", [1, 2])
@pytest.mark.parametrize("model", [CL, SH])
def test_angular_spectrum_fused_against_the_oracle(rad, oracle_mod, kernel, model):
    """dI/dw = dOmega * sum over the angles inside the collimator of the ORACLE's cube, with a real solid-angle element
    and an active theta cut whose mask is computed here from the grid arrays; grid big enough (400 x 400 angles x 32
    omegas) that the sums come out of the main kernel's epilogue, through both kernels."""
    wl = workloads.make("cfg3" if model == SH else "cfg2", n=90, n_omega=32, n_th=400, seed=29)
    lam = wl.hbarc_over_E if model == SH else 0.0
    plan = rad.rad_plan_describe(1, 90, 32, 400, 400, model, kernel)
    assert plan["mode"] == 0 and plan["kernel"] == kernel
    d_om = (wl.thx[1] - wl.thx[0]) * (wl.thy[1] - wl.thy[0])
    cut = 0.6 * wl.thx.max()
    b = {k: v[None, :].contiguous() for k, v in dev_dict(wl.traj).items()}
    got = rad.rad_angular_spectrum(b, np.array([90]), *dev_grid(wl), d_om, cut, model=model,
                                   hbarc_over_E=lam if model else None, kernel=kernel).cpu().numpy()
    X, Y = np.meshgrid(wl.thx, wl.thy)
    mask = X * X + Y * Y <= cut * cut
    assert 0.2 < mask.mean() < 0.4                                       # the cut is active
    ref_cube = oracle_mod.grid(wl.traj, wl.omega, wl.thx, wl.thy, model, lam)
    ref = (ref_cube * mask).sum((1, 2)) * d_om
    # every term is >= 0, so the sum of N terms each within 1e-9 relative / 1e-12 S_max absolute stays within that
    tol = np.maximum(RTOL * np.abs(ref), FLOOR * ref_cube.max() * mask.sum() * d_om)
    assert np.max(np.abs(got - ref) / tol) <= 1.0
    unmasked = rad.rad_angular_spectrum(b, np.array([90]), *dev_grid(wl), d_om, 0.0, model=model,
                                        hbarc_over_E=lam if model else None, kernel=kernel).cpu().numpy()
    ref_all = ref_cube.sum((1, 2)) * d_om
    assert np.max(np.abs(unmasked - ref_all) / np.maximum(RTOL * ref_all, FLOOR * ref_cube.max() * mask.size * d_om)) <= 1.0
    assert np.all(unmasked >= got)


def test_angular_spectrum_three_thousand_squared_sampled_per_omega(rad, oracle_mod):
    """"more than 3000 points in both spatial dimension ... approach the limit" of memory.  3000 x 3000
    angles x 24 omegas = 2.2e8 integrals: the 1.7 GB cube is never written; two omegas are checked against the oracle's
    sum over all 9e6 angles (collimator cut active), the rest against the ensemble identity sum_p = p-fold."""
    wl = workloads.make("cfg2", n=48, n_omega=24, n_th=3000, seed=37)
    d_om = (wl.thx[1] - wl.thx[0]) * (wl.thy[1] - wl.thy[0])
    cut = 0.8 * wl.thx.max()
    need = rad.load_library().rad_angular_spectrum_workspace_bytes(1, 48, 24, 3000, 3000)
    assert need < 24 * 3000 * 3000 * 8 / 4                              # far below the cube
    b = {k: v[None, :].contiguous() for k, v in dev_dict(wl.traj).items()}
    got = rad.rad_angular_spectrum(b, np.array([48]), *dev_grid(wl), d_om, cut).cpu().numpy()
    X, Y = np.meshgrid(wl.thx, wl.thy)
    mask = (X * X + Y * Y <= cut * cut).ravel()
    for iw in (3, 20):
        vals = oracle_mod.points(wl.traj, np.full(mask.sum(), wl.omega[iw]), X.ravel()[mask], Y.ravel()[mask])
        ref = vals.sum() * d_om
        assert abs(got[iw] - ref) <= max(RTOL * ref, FLOOR * vals.max() * mask.sum() * d_om)
    twice = rad.rad_angular_spectrum({k: v.repeat(2, 1) for k, v in b.items()}, np.array([48, 48]), *dev_grid(wl), d_om,
                                     cut).cpu().numpy()
    np.testing.assert_allclose(twice, 2 * got, rtol=1e-13)


def test_angular_spectrum_small_grid_with_cut(rad, oracle_mod):
    """Grids too small to give every SM its tiles take the cube path inside the workspace (the cube is then < 40 MB);
    same contract: real solid-angle element, active cut, against the oracle; workspace exactly as the library asks."""
    import torch
    ws = workloads.make("cfg3", n=800, n_omega=9, n_th=21, seed=23)
    assert rad.rad_plan_describe(1, 800, 9, 21, 21, SH)["mode"] != 0
    d_om = (ws.thx[1] - ws.thx[0]) * (ws.thy[1] - ws.thy[0])
    cut = 0.7 * ws.thx.max()
    b = {k: v[None, :].contiguous() for k, v in dev_dict(ws.traj).items()}
    need = rad.load_library().rad_angular_spectrum_workspace_bytes(1, 800, 9, 21, 21)
    wsp = torch.empty(need, dtype=torch.uint8, device="cuda")
    got = rad.rad_angular_spectrum(b, np.array([800]), *dev_grid(ws), d_om, cut, model=SH, hbarc_over_E=ws.hbarc_over_E,
                                   workspace=wsp).cpu().numpy()
    X, Y = np.meshgrid(ws.thx, ws.thy)
    mask = X * X + Y * Y <= cut * cut
    assert 0.2 < mask.mean() < 0.6
    cube = oracle_mod.grid(ws.traj, ws.omega, ws.thx, ws.thy, SH, ws.hbarc_over_E)
    ref = (cube * mask).sum((1, 2)) * d_om
    assert np.max(np.abs(got - ref) / np.maximum(RTOL * ref, FLOOR * cube.max() * mask.sum() * d_om)) <= 1.0


def test_number_spectrum(rad):
    import torch
    spec = torch.tensor([1.0, 4.0, 9.0], dtype=torch.float64, device="cuda")
    om = torch.tensor([2.0, 4.0, 0.5], dtype=torch.float64, device="cuda")
    got = rad.rad_number_spectrum(spec, om, 0.25).cpu().numpy()
    assert np.array_equal(got, np.array([1.0 / 0.5, 4.0 / 1.0, 9.0 / 0.125]))
    with pytest.raises(rad.RadError):
        rad.rad_number_spectrum(spec, om, 0.0)


def test_profile_object_times_one_call(rad):
    """rad_options.profile: per-call events; two profiles used by two calls do not disturb each other."""
    wl = workloads.make("cfg2", n=3000, n_omega=32, n_th=16)
    tr, g = dev_dict(wl.traj), dev_grid(wl)
    p1, p2 = rad.RadProfile(), rad.RadProfile()
    rad.rad_classical(tr, *g, profile=p1, kernel=2)
    rad.rad_classical(tr, *g, profile=p2, kernel=3 if rad.rad_plan_kernel(32, 16, 16, CL, kernel=0, n_max=3000) == 3 else 1)
    a, b_ = p1.read(), p2.read()
    assert a[1] > 0 and b_[1] > 0 and a[0] >= 0 and a[2] > 0
    p1.close(); p2.close()
