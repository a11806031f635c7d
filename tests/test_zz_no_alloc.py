"""rad_eval_static: the entry point that allocates nothing (include/rad.h) against the existing path.

Collected last on purpose (file name): the suite runs with pytest -x, and a failure here must not hide other tests.
The scratch of rad_eval_static is ONE static device array of rad_static_scratch_bytes() = 16 MiB shared by every call,
which keeps the previous call's contents: the checks below run two (three) calls in a row with different shapes,
kernels and models, so that a stale byte read from the previous call would show.  Reference = rad_classical /
rad_semiclassical with the library's usual scratch; tolerance = the one of the parity tests (BASELINE.json:
|a - b| <= max(1e-9 |b|, 1e-12 max b)), although the two paths run the same kernels and agree bit for bit.
Passes alone in a fresh process and after the other tests (it keeps no state but the array itself).
"""
import numpy as np
import pytest

import workloads

pytestmark = pytest.mark.gpu

CL, S0, SH = 0, 1, 2
RAD_ETOOBIG = -5


@pytest.fixture(scope="module")
def rad():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the CUDA path has no CPU fallback")
    import paper_1910_10391_b200 as rad
    rad.build_library()
    rad.load_library()
    return rad


def _dev(d):
    import torch
    return {k: torch.from_numpy(np.ascontiguousarray(v)).cuda() for k, v in d.items()}


def _grid(wl):
    import torch
    return [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (wl.omega, wl.thx, wl.thy)]


def _close(a, b):
    a, b = a.cpu().numpy(), b.cpu().numpy()
    assert np.all(np.isfinite(a))
    tol = np.maximum(1e-9 * np.abs(b), 1e-12 * b.max())
    assert np.max(np.abs(a - b) / tol) <= 1.0


def test_static_scratch_entry_point_matches_the_existing_path_on_calls_in_a_row(rad):
    import torch
    assert rad.rad_static_scratch_bytes() == 16 << 20
    # (1) BASELINE config 1 at full size, classical: the fused single-launch kernel, 9.7 MB of partial amplitudes
    w1 = workloads.make("cfg1")
    t1, g1 = _dev(w1.traj), _grid(w1)
    assert rad.rad_plan_describe(1, 4000, 64, 8, 8, CL)["kernel"] == 3
    ref1 = rad.rad_classical(t1, *g1)
    # (2) a grid that fills the separable kernel's tiles, spin-1/2, time split: packed records + partial amplitudes
    w2 = workloads.make("cfg2", n=1100, n_omega=32, n_th=16, seed=7)
    t2, g2 = _dev(w2.traj), _grid(w2)
    lam2 = 0.5 / w2.omega.max()
    assert rad.rad_plan_describe(1, 1100, 32, 16, 16, SH)["kernel"] == 2
    ref2 = rad.rad_semiclassical(t2, *g2, 1, lam2)
    # (3) a ragged shape through the direct kernel, spin-0
    w3 = workloads.make("cfg3", n=777, n_omega=19, n_th=5, model=S0)
    t3, g3 = _dev(w3.traj), _grid(w3)
    ref3 = rad.rad_semiclassical(t3, *g3, 0, w3.hbarc_over_E, kernel=1)

    out1, out2, out3 = torch.empty_like(ref1), torch.empty_like(ref2), torch.empty_like(ref3)
    for rep in range(2):                                   # calls in a row, each finding the previous one's scratch
        out1.fill_(-1.0); out2.fill_(-1.0); out3.fill_(-1.0)
        rad.rad_eval_static(t1, *g1, CL, 0.0, out=out1)
        rad.rad_eval_static(t2, *g2, SH, lam2, out=out2)
        rad.rad_eval_static(t3, *g3, S0, w3.hbarc_over_E, out=out3, kernel=1)
        rad.rad_eval_static(t1, *g1, CL, 0.0, out=out1)    # and the first again, over the others' leftovers
        torch.cuda.synchronize()
        _close(out1, ref1)
        _close(out2, ref2)
        _close(out3, ref3)
        assert torch.equal(out1, ref1) and torch.equal(out2, ref2) and torch.equal(out3, ref3)   # same kernels: same bits


def test_static_scratch_entry_point_allocates_nothing_and_rejects_what_does_not_fit(rad):
    import torch
    w1 = workloads.make("cfg1")
    t1, g1 = _dev(w1.traj), _grid(w1)
    out = torch.empty((64, 8, 8), dtype=torch.float64, device="cuda")
    rad.rad_eval_static(t1, *g1, CL, 0.0, out=out)          # first call: kernels loaded, symbol address asked
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(5):
        rad.rad_eval_static(t1, *g1, CL, 0.0, out=out)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0                                    # no device memory taken or given back by the calls

    # BASELINE config 2's plan (16-way time split: 75 MB of partial amplitudes) is beyond the 16 MiB: a clear error,
    # nothing enqueued, `out` untouched
    w2 = workloads.make("cfg2")
    big = torch.full((256, 32, 32), -3.0, dtype=torch.float64, device="cuda")
    with pytest.raises(rad.RadError) as err:
        rad.rad_eval_static(_dev(w2.traj), *_grid(w2), CL, 0.0, out=big)
    assert err.value.code == RAD_ETOOBIG and "static scratch" in str(err.value)
    torch.cuda.synchronize()
    assert torch.all(big == -3.0)
    with pytest.raises(rad.RadError):                        # argument checks as elsewhere
        rad.rad_eval_static(t1, *g1, 7, 0.0, out=out)
