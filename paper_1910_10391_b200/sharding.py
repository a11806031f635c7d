"""Multi-GPU use of the radiation-integral library: one process per GPU, ``torch.distributed``.

The method shards two ways:

* **grid sharding** -- every grid point is an independent integral ("each thread ... evaluates
  one integral"), so the omega axis is cut into ``world`` contiguous slabs; every
  rank holds the whole trajectory and writes its own slab.  There is no exchange step in the
  computation; an all-gather assembles the cube for callers that want it everywhere.
* **ensemble sharding** -- the spectrum of a beam is the sum of the spectra of its particles /
  crystal sections, so the trajectories are dealt out in contiguous blocks,
  each rank sums its block on the full grid (``rad_ensemble_sum``), and ONE exchange -- an
  all-gather of the ``world`` partial cubes followed by a sum in rank order (``rad_sum_cubes``,
  fixed order => run-to-run deterministic, Q13) -- produces the total.

Only the host logic lives here (ranges, padding, the collective call).  The arithmetic is the
CUDA library's; ``evaluate`` / ``reduce`` hooks exist so that the CPU ``gloo`` tests can drive
the same control flow without a GPU (they inject test doubles; the defaults are the CUDA calls
and there is no CPU fallback).
"""
from __future__ import annotations

from typing import Callable, Optional, Sequence

import numpy as np
import torch
import torch.distributed as dist

from . import binding as _b


def shard_range(total: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous, balanced block [lo, hi) of ``total`` units for ``rank`` of ``world``:
    the first ``total % world`` ranks get one extra unit; empty blocks are allowed."""
    if world < 1 or not 0 <= rank < world or total < 0:
        raise ValueError("shard_range: need 0 <= rank < world and total >= 0")
    base, extra = divmod(total, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def shard_sizes(total: int, world: int) -> list[int]:
    return [hi - lo for lo, hi in (shard_range(total, r, world) for r in range(world))]


def _world(group) -> tuple[int, int]:
    if not dist.is_available() or not dist.is_initialized():
        return 0, 1
    return dist.get_rank(group), dist.get_world_size(group)


# ----------------------------------------------------------------------------- grid sharding
def rad_eval_grid_sharded(traj: dict, omega: torch.Tensor, thx: torch.Tensor, thy: torch.Tensor,
                          model: int = _b.CLASSICAL, hbarc_over_E: float = 0.0, gather: bool = True,
                          group=None, evaluate: Optional[Callable] = None) -> torch.Tensor:
    """Cube of one trajectory with the omega axis split across the ranks of ``group``.

    Every rank passes the same trajectory and the same full grid.  Returns the full cube
    (n_omega, n_thy, n_thx) on every rank if ``gather`` (one all-gather of equal-size padded
    slabs), else this rank's slab (n_local, n_thy, n_thx).
    """
    rank, world = _world(group)
    lo, hi = shard_range(omega.numel(), rank, world)
    if evaluate is None:
        evaluate = _evaluate_single_cuda
    A = (thy.numel(), thx.numel())
    if hi > lo:
        slab = evaluate(traj, omega[lo:hi].contiguous(), thx, thy, model, hbarc_over_E)
    else:
        slab = torch.empty((0, *A), dtype=torch.float64, device=omega.device)
    if not gather or world == 1:
        return slab
    sizes = shard_sizes(omega.numel(), world)
    pad = max(sizes)
    mine = torch.zeros((pad, *A), dtype=torch.float64, device=omega.device)
    mine[: hi - lo] = slab
    parts = torch.empty((world, pad, *A), dtype=torch.float64, device=omega.device)
    dist.all_gather_into_tensor(parts.view(-1), mine.view(-1), group=group)
    return torch.cat([parts[r, : sizes[r]] for r in range(world)], dim=0)


def _evaluate_single_cuda(traj, omega, thx, thy, model, lam):
    if model == _b.CLASSICAL:
        return _b.rad_classical(traj, omega, thx, thy)
    return _b.rad_semiclassical(traj, omega, thx, thy, 0 if model == _b.SPIN0 else 1, lam)


# ----------------------------------------------------------------------------- ensemble sharding
def rad_ensemble_sum_sharded(local_batch: Optional[dict], local_n: Sequence[int], omega: torch.Tensor,
                             thx: torch.Tensor, thy: torch.Tensor, model: int = _b.CLASSICAL,
                             local_hbarc_over_E=None, group=None, evaluate: Optional[Callable] = None,
                             reduce: Optional[Callable] = None) -> torch.Tensor:
    """Sum of the spectra of ALL ranks' trajectories, identical on every rank.

    ``local_batch`` / ``local_n`` / ``local_hbarc_over_E`` describe THIS rank's block (use
    ``shard_range(count, rank, world)`` to cut a global ensemble); a rank with no trajectory
    passes ``local_n = []`` (``local_batch`` is then ignored) and contributes zeros.
    Exchange: all-gather of the ``world`` partial cubes (M doubles each), then their sum in
    rank order on every rank -- the same bits everywhere and from run to run.
    """
    rank, world = _world(group)
    shape = (omega.numel(), thy.numel(), thx.numel())
    local_n = np.ascontiguousarray(local_n, dtype=np.int64)
    if evaluate is None:
        evaluate = _evaluate_ensemble_cuda
    if reduce is None:
        reduce = _b.rad_sum_cubes
    if local_n.size:
        part = evaluate(local_batch, local_n, omega, thx, thy, model, local_hbarc_over_E)
    else:
        part = torch.zeros(shape, dtype=torch.float64, device=omega.device)
    if world == 1:
        return part
    parts = torch.empty((world, *shape), dtype=torch.float64, device=omega.device)
    dist.all_gather_into_tensor(parts.view(-1), part.contiguous().view(-1), group=group)
    return reduce(parts)


def _evaluate_ensemble_cuda(batch, n, omega, thx, thy, model, lam):
    return _b.rad_ensemble_sum(batch, n, omega, thx, thy, model=model, hbarc_over_E=lam)
