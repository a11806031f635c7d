"""SURVEY.md 8(e) on real GPUs: one process per GPU, `nccl` backend, world size 2.

Runs only where two CUDA devices are visible (marker `multigpu`); on a one-GPU box it is skipped with that reason
spelled out -- the same control flow is covered on CPU by tests/test_sharding_gloo.py (gloo, world 2 and 3) and the
CUDA calls it makes by the single-GPU parity tests.  Ensemble sharding: trajectories dealt out, rad_ensemble_sum per
rank, ONE exchange (all-gather of partial cubes + rad_sum_cubes in rank order); grid sharding: omega slabs, gather.
Checks: the sharded cubes match the CPU oracle at the BASELINE.json tolerance and are bit-identical on both ranks.
"""
import os
import socket
import sys
from pathlib import Path

import numpy as np
import pytest

ROOT = Path(__file__).resolve().parent.parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

pytestmark = [pytest.mark.gpu, pytest.mark.multigpu]


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, ret):
    import torch
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    torch.cuda.set_device(rank)
    dev = torch.device("cuda", rank)
    dist.init_process_group("nccl", rank=rank, world_size=world, device_id=dev)
    try:
        import paper_1910_10391_b200 as rad
        import workloads
        from paper_1910_10391_b200.sharding import shard_range
        rad.load_library()

        def to_dev(a):
            return torch.from_numpy(np.ascontiguousarray(a)).to(dev)

        # ---- ensemble sharding: 5 trajectories over 2 ranks (3 + 2), spin-1/2 with per-trajectory energies
        we = workloads.make("cfg4", count=5, n=600, n_omega=12, n_th=6, seed0=300)
        lam = np.linspace(0.2, 0.6, 5) / we.omega.max()
        lo, hi = shard_range(5, rank, world)
        g = [to_dev(a) for a in (we.omega, we.thx, we.thy)]
        local = {k: to_dev(v[lo:hi]) for k, v in we.batch.items()}
        total = rad.rad_ensemble_sum_sharded(local, we.n[lo:hi], *g, model=2, local_hbarc_over_E=lam[lo:hi])
        ret[f"ens{rank}"] = total.cpu().numpy()

        # ---- grid sharding: 11 omegas over 2 ranks (6 + 5), gathered
        wl = workloads.make("cfg2", n=900, n_omega=11, n_th=6, seed=14)
        tr = {k: to_dev(v) for k, v in wl.traj.items()}
        g2 = [to_dev(a) for a in (wl.omega, wl.thx, wl.thy)]
        cube = rad.rad_eval_grid_sharded(tr, *g2, gather=True)
        ret[f"grid{rank}"] = cube.cpu().numpy()
        ret[f"ok{rank}"] = True
    finally:
        dist.destroy_process_group()


def test_sharded_paths_on_two_gpus(oracle_mod):
    import torch
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the CUDA path has no CPU fallback")
    if torch.cuda.device_count() < 2:
        pytest.skip("multigpu: needs >= 2 CUDA devices (this box has %d); the N > 1 control flow runs on CPU in "
                    "tests/test_sharding_gloo.py" % torch.cuda.device_count())
    import torch.multiprocessing as mp
    import paper_1910_10391_b200 as rad
    import workloads
    rad.build_library()
    mgr = mp.Manager()
    ret = mgr.dict()
    mp.spawn(_worker, args=(2, _free_port(), ret), nprocs=2, join=True)
    assert ret.get("ok0") and ret.get("ok1")
    assert np.array_equal(ret["ens0"], ret["ens1"]) and np.array_equal(ret["grid0"], ret["grid1"])   # identical bits

    def check(gpu, ref):
        tol = np.maximum(1e-9 * np.abs(ref), 1e-12 * gpu.max())
        assert np.max(np.abs(gpu - ref) / tol) <= 1.0

    we = workloads.make("cfg4", count=5, n=600, n_omega=12, n_th=6, seed0=300)
    lam = np.linspace(0.2, 0.6, 5) / we.omega.max()
    w, nx, ny = oracle_mod.grid_points(we.omega, we.thx, we.thy)
    check(ret["ens0"], oracle_mod.ensemble_points(we.batch, we.n, w, nx, ny, 2, lam).reshape(ret["ens0"].shape))
    wl = workloads.make("cfg2", n=900, n_omega=11, n_th=6, seed=14)
    check(ret["grid0"], oracle_mod.grid(wl.traj, wl.omega, wl.thx, wl.thy))
