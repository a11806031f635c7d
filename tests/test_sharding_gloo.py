"""Multi-process (gloo, world_size 2 and 3, CPU) tests of the N > 1 path: the sharding host logic
of paper_1910_10391_b200/sharding.py -- ranges, padding of ragged slabs, the all-gather and the
rank-ordered sum -- driven with test doubles for the two CUDA calls (the CPU oracle evaluates,
numpy sums in order).  The product defaults are the CUDA calls; nothing here is a CPU fallback
of the library (tests may call the oracle; the product path may not)."""
import os
import socket
import sys
from pathlib import Path

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = Path(__file__).resolve().parent.parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _oracle_single(traj, omega, thx, thy, model, lam):
    import oracle
    tr = {k: v.numpy() for k, v in traj.items()}
    return torch.from_numpy(oracle.grid(tr, omega.numpy(), thx.numpy(), thy.numpy(), model, lam))


def _oracle_ensemble(batch, n, omega, thx, thy, model, lam):
    import oracle
    b = {k: v.numpy() for k, v in batch.items()}
    w, nx, ny = oracle.grid_points(omega.numpy(), thx.numpy(), thy.numpy())
    out = oracle.ensemble_points(b, n, w, nx, ny, model, lam)
    return torch.from_numpy(out.reshape(omega.numel(), thy.numel(), thx.numel()))


def _ordered_sum(parts):
    acc = parts[0].clone()
    for r in range(1, parts.shape[0]):
        acc += parts[r]
    return acc


def _worker(rank: int, world: int, port: int, ret):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), OMP_NUM_THREADS="2")
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import workloads
        from paper_1910_10391_b200 import sharding

        # ---- grid sharding: 7 omegas over `world` ranks (ragged slabs), spin-1/2
        wl = workloads.make("cfg2", n=300, n_omega=7, n_th=3, seed=31)
        lam = 0.5 / wl.omega.max()
        tr = {k: torch.from_numpy(v) for k, v in wl.traj.items()}
        g = [torch.from_numpy(a) for a in (wl.omega, wl.thx, wl.thy)]
        cube = sharding.rad_eval_grid_sharded(tr, *g, model=2, hbarc_over_E=lam, evaluate=_oracle_single)
        slab = sharding.rad_eval_grid_sharded(tr, *g, model=2, hbarc_over_E=lam, gather=False,
                                              evaluate=_oracle_single)
        lo, hi = sharding.shard_range(7, rank, world)
        # ---- ensemble sharding: 5 ragged trajectories dealt out in contiguous blocks
        we = workloads.make("cfg4", count=5, n=200, n_omega=4, n_th=3, seed0=77)
        nvec = np.array([200, 150, 2, 97, 200], dtype=np.int64)
        plo, phi = sharding.shard_range(5, rank, world)
        local = {k: torch.from_numpy(np.ascontiguousarray(v[plo:phi])) for k, v in we.batch.items()}
        ge = [torch.from_numpy(a) for a in (we.omega, we.thx, we.thy)]
        total = sharding.rad_ensemble_sum_sharded(local, nvec[plo:phi], *ge, evaluate=_oracle_ensemble,
                                                  reduce=_ordered_sum)
        # a rank with nothing to do contributes zeros
        empty_total = sharding.rad_ensemble_sum_sharded(
            local if rank == 0 else None, nvec[plo:phi] if rank == 0 else [], *ge,
            evaluate=_oracle_ensemble, reduce=_ordered_sum)
        ret[rank] = dict(cube=cube.numpy(), slab=slab.numpy(), lo=lo, hi=hi, total=total.numpy(),
                         empty_total=empty_total.numpy(), plo=plo, phi=phi)
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_sharded_paths_match_unsharded(world, oracle_mod):
    import workloads
    mgr = mp.Manager()
    ret = mgr.dict()
    mp.spawn(_worker, args=(world, _free_port(), ret), nprocs=world, join=True)
    assert sorted(ret.keys()) == list(range(world))

    wl = workloads.make("cfg2", n=300, n_omega=7, n_th=3, seed=31)
    lam = 0.5 / wl.omega.max()
    ref = oracle_mod.grid(wl.traj, wl.omega, wl.thx, wl.thy, 2, lam)
    covered = []
    for r in range(world):
        np.testing.assert_array_equal(ret[r]["cube"], ref)                    # same oracle, same bits
        np.testing.assert_array_equal(ret[r]["slab"], ref[ret[r]["lo"]:ret[r]["hi"]])
        covered += list(range(ret[r]["lo"], ret[r]["hi"]))
    assert covered == list(range(7))                                          # a partition, in order

    we = workloads.make("cfg4", count=5, n=200, n_omega=4, n_th=3, seed0=77)
    nvec = np.array([200, 150, 2, 97, 200], dtype=np.int64)
    w, nx, ny = oracle_mod.grid_points(we.omega, we.thx, we.thy)
    ref_e = oracle_mod.ensemble_points(we.batch, nvec, w, nx, ny).reshape(4, 3, 3)
    p0 = ret[0]["phi"]
    ref_first = oracle_mod.ensemble_points({k: v[:p0] for k, v in we.batch.items()}, nvec[:p0],
                                           w, nx, ny).reshape(4, 3, 3)
    for r in range(world):
        np.testing.assert_allclose(ret[r]["total"], ref_e, rtol=1e-14)        # summation order differs
        np.testing.assert_array_equal(ret[r]["total"], ret[0]["total"])       # identical on all ranks
        np.testing.assert_allclose(ret[r]["empty_total"], ref_first, rtol=1e-14)


def test_shard_range_properties():
    from paper_1910_10391_b200.sharding import shard_range, shard_sizes
    for total in (0, 1, 5, 128, 1000):
        for world in (1, 2, 3, 8):
            ranges = [shard_range(total, r, world) for r in range(world)]
            assert ranges[0][0] == 0 and ranges[-1][1] == total
            assert all(a[1] == b[0] for a, b in zip(ranges, ranges[1:]))
            sizes = shard_sizes(total, world)
            assert max(sizes) - min(sizes) <= 1 and sum(sizes) == total
    with pytest.raises(ValueError):
        shard_range(4, 2, 2)


def test_bench_generates_each_ranks_block_of_the_ensemble():
    """bench.py under torchrun: a rank generates only its own block of cfg4's trajectories (seed of trajectory p =
    4000 + p wherever it is generated); the blocks tile the global ensemble and the job's eval count stays the whole
    job's.  (Small n: the full-size ensemble is 8.8 GB.)"""
    import bench
    import workloads
    from paper_1910_10391_b200.sharding import shard_range
    whole = workloads.make("cfg4", count=7, n=50, n_omega=3, n_th=2)
    for world in (2, 3):
        for rank in range(world):
            lo, hi = shard_range(7, rank, world)
            blk = workloads.make("cfg4", count=hi - lo, n=50, n_omega=3, n_th=2, seed0=4000 + lo)
            for k in whole.batch:
                assert np.array_equal(blk.batch[k], whole.batch[k][lo:hi])
    wl = workloads.make("cfg4", count=2, n=50, n_omega=3, n_th=2, seed0=4003)
    wl.meta.update(global_count=7, block=(3, 5))
    assert bench.job_evals(wl) == whole.evals and bench.job_evals(whole) == whole.evals
