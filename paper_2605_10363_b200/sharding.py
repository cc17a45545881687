"""Multi-GPU form of one EXC evaluation: shard the quadrature grid, reduce V and E.

The paper distributes filtered grid batches over GPUs and reduces the partial EXC contributions
at the end (§III-E).  Here each rank owns a contiguous range of the caller's
grid points (whole atomic grids where possible, so a rank's points are spatially compact), builds
its own kldi plan on that range, and the only exchange step is one all-reduce(sum) of V
([n_ao][n_ao] FP64; or of the [n_atoms][3] nuclear gradient) and of the scalar E_xc.  rho stays sharded.  D is replicated.

This module holds host logic only (index arithmetic and the torch.distributed calls); it is
exercised on CPU with the gloo backend in tests/test_sharding.py.
"""
from __future__ import annotations

import dataclasses

import numpy as np


def shard_bounds(n_pts: int, world_size: int, align: int = 1) -> list:
    """Contiguous, near-equal ranges [lo, hi) of the grid, boundaries rounded to a multiple of `align`
    (e.g. the number of points of one atomic grid).  Every point belongs to exactly one rank."""
    if world_size < 1 or n_pts < 0 or align < 1:
        raise ValueError("bad arguments")
    units = (n_pts + align - 1) // align
    out = []
    for r in range(world_size + 1):
        out.append(min(n_pts, ((units * r) // world_size) * align))
    return [(out[r], out[r + 1]) for r in range(world_size)]


def shard_workload(wl, rank: int, world_size: int, align: int = 5500):
    """The rank's view of a workload: same atoms, basis and D; its own slice of the grid."""
    lo, hi = shard_bounds(wl.n_pts, world_size, align)[rank]
    return dataclasses.replace(wl, grid_xyz=np.ascontiguousarray(wl.grid_xyz[lo:hi]),
                               grid_w=np.ascontiguousarray(wl.grid_w[lo:hi])), (lo, hi)


def allreduce_exc(E_local: float, V_local, group=None):
    """Sum the per-rank partial energy and potential matrix over all ranks (in place on V_local).
    V_local: torch tensor on the backend's device (cuda for nccl, cpu for gloo).  The nuclear gradient of
    kldi_exc_grad is a sum over grid points too: pass the rank's [n_atoms][3] partial instead of V."""
    import torch
    import torch.distributed as dist

    e = torch.tensor([E_local], dtype=torch.float64, device=V_local.device)
    dist.all_reduce(V_local, op=dist.ReduceOp.SUM, group=group)
    dist.all_reduce(e, op=dist.ReduceOp.SUM, group=group)
    return float(e.item()), V_local
