"""Multi-GPU form of one EXC evaluation: shard the quadrature grid, reduce V and E.

The paper distributes filtered grid batches over GPUs and reduces the partial EXC contributions
at the end (§III-E; heterogeneous task costs).  Here each rank owns a
CONTIGUOUS RANGE OF THE PLAN'S CURVE ORDER (the Hilbert order the plan sorts the grid by, kldi_grid_key), so its
points are spatially compact and its grid blocks are the ones a single-GPU plan would form; the ranges are balanced
by the cost model of the contractions, sum over 128-point blocks of K(K+1) with K the number of AOs whose cutoff
sphere reaches the block, not by point counts.  Each rank builds its own kldi plan on its points,
D is replicated, rho stays sharded, and the only exchange step is one all-reduce(sum) of V (packed lower triangle:
V is symmetric) or of the [n_atoms][3] nuclear gradient, and of the scalar E_xc.

This module holds host logic only (index arithmetic, a cost estimate from geometry, and the torch.distributed
calls); it is exercised on CPU with the gloo backend in tests/test_sharding.py.
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

GB = 128  # points per grid block (include/kldi.h)


def shard_bounds(n_pts: int, world_size: int, align: int = 1) -> list:
    """Contiguous, near-equal ranges [lo, hi) of n_pts items, boundaries rounded to a multiple of `align`.
    Every item belongs to exactly one rank."""
    if world_size < 1 or n_pts < 0 or align < 1:
        raise ValueError("bad arguments")
    units = (n_pts + align - 1) // align
    out = []
    for r in range(world_size + 1):
        out.append(min(n_pts, ((units * r) // world_size) * align))
    return [(out[r], out[r + 1]) for r in range(world_size)]


def shell_cutoff_radii(wl, eps: float) -> np.ndarray:
    """Radius beyond which every primitive of a shell is below eps: N r^l exp(-a r^2) < eps, solved by a few fixed-point
    steps per primitive (an estimate for load balancing only; the plan's filter evaluates the functions themselves)."""
    eps = max(float(eps), 1e-300)
    out = np.zeros(len(wl.shell_l))
    for s, l in enumerate(wl.shell_l):
        l = int(l)
        for p in range(int(wl.shell_prim_off[s]), int(wl.shell_prim_off[s + 1])):
            a, c = float(wl.prim_alpha[p]), abs(float(wl.prim_coef[p]))
            n = c * (2.0 * a / math.pi) ** 0.75 * (4.0 * a) ** (0.5 * l)
            r = 1.0
            for _ in range(30):
                arg = math.log(max(n, 1e-300) / eps) + l * math.log(max(r, 1e-12))
                r = math.sqrt(max(arg, 0.0) / a)
            out[s] = max(out[s], r)
    return out


def curve_order(grid_xyz: np.ndarray) -> np.ndarray:
    """Indices of the grid points in the plan's order: stable sort by kldi_grid_key (host function, no GPU)."""
    from . import binding

    keys = binding.grid_keys(grid_xyz, grid_xyz.min(axis=0))
    return np.argsort(keys, kind="stable")


def block_costs(wl, order: np.ndarray, eps: float, samples_per_block: int = 8) -> np.ndarray:
    """Estimated cost K(K+1) of every 128-point block of the curve order, K = AOs of the shells whose cutoff sphere
    contains at least one of `samples_per_block` evenly spaced points of the block (a block far from the molecule is large
    and sparse: a bounding-sphere test would count every atom there, the plan's filter retains almost nothing)."""
    from scipy.spatial import cKDTree

    pts = wl.grid_xyz[order]
    nb = (len(pts) + GB - 1) // GB
    step = GB // samples_per_block
    sidx = np.arange(0, len(pts), step)
    sblock = sidx // GB
    tree = cKDTree(pts[sidx])
    rc = shell_cutoff_radii(wl, eps)
    ncart = np.array([(int(l) + 1) * (int(l) + 2) // 2 for l in wl.shell_l])
    k = np.zeros(nb)
    # group the shells by (atom, cutoff): one ball query per distinct sphere
    by_sphere = {}
    for s in range(len(rc)):
        by_sphere.setdefault((int(wl.shell_atom[s]), round(float(rc[s]), 6)), []).append(s)
    for (atom, r), shells in by_sphere.items():
        hit = tree.query_ball_point(wl.atom_xyz[atom], r)
        if hit:
            k[np.unique(sblock[np.asarray(hit, dtype=np.int64)])] += float(ncart[shells].sum())
    return k * (k + 1.0)


def balanced_ranges(cost: np.ndarray, world_size: int) -> list:
    """Contiguous block ranges [b0, b1) with near-equal summed cost (prefix-sum split)."""
    if world_size < 1:
        raise ValueError("bad arguments")
    c = np.concatenate([[0.0], np.cumsum(cost + 1e-9)])  # the epsilon keeps empty regions splittable
    cuts = [int(np.searchsorted(c, c[-1] * r / world_size, side="left")) for r in range(world_size + 1)]
    cuts[0], cuts[-1] = 0, len(cost)
    for r in range(1, world_size + 1):
        cuts[r] = max(cuts[r], cuts[r - 1])
    return [(cuts[r], cuts[r + 1]) for r in range(world_size)]


def shard_workload(wl, rank: int, world_size: int, eps=None):
    """The rank's view of a workload: same atoms, basis and D; the grid points of its range of the curve order.
    Returns (workload, idx) with idx the caller indices of the rank's points (rho of the rank maps back through it)."""
    order = curve_order(wl.grid_xyz)
    cost = block_costs(wl, order, wl.eps if eps is None else eps)
    b0, b1 = balanced_ranges(cost, world_size)[rank]
    idx = order[b0 * GB:min(len(order), b1 * GB)]
    part = dataclasses.replace(wl, grid_xyz=np.ascontiguousarray(wl.grid_xyz[idx]),
                               grid_w=np.ascontiguousarray(wl.grid_w[idx]))
    return part, idx


_BANDS = 32


def _band_slices(n: int):
    nb = 1 if n < 1024 else _BANDS
    return [(n * b // nb, n * (b + 1) // nb) for b in range(nb) if n * (b + 1) // nb > n * b // nb]


def pack_lower(V):
    """Lower triangle of a square matrix in row bands (band [r0, r1) keeps the columns [0, r1)): ~52 % of the matrix
    as one flat buffer of contiguous row segments."""
    import torch

    n = V.shape[0]
    return torch.cat([V[r0:r1, :r1].reshape(-1) for r0, r1 in _band_slices(n)])


def unpack_lower_symmetric(buf, V):
    """Inverse of pack_lower into V, then the strict upper part by symmetry (V[i, j] = V[j, i])."""
    n, o = V.shape[0], 0
    for r0, r1 in _band_slices(n):
        m = (r1 - r0) * r1
        V[r0:r1, :r1] = buf[o:o + m].view(r1 - r0, r1)
        o += m
    for r0, r1 in _band_slices(n):
        if r1 < n:
            V[r0:r1, r1:] = V[r1:, r0:r1].T
    return V


def allreduce_exc(E_local: float, V_local, group=None, triangle: bool = True):
    """Sum the per-rank partial energy and potential matrix over all ranks (in place on V_local).
    V_local: torch tensor on the backend's device (cuda for nccl, cpu for gloo).  A square V is symmetric, so with
    `triangle` only its packed lower triangle crosses the links (52 % of the bytes) and the other half is mirrored
    afterwards.  The nuclear gradient of kldi_exc_grad is a sum over grid points too: pass the rank's [n_atoms][3]
    partial instead of V (reduced whole)."""
    import torch
    import torch.distributed as dist

    e = torch.tensor([E_local], dtype=torch.float64, device=V_local.device)
    if triangle and V_local.dim() == 2 and V_local.shape[0] == V_local.shape[1] and V_local.shape[0] > 1:
        buf = pack_lower(V_local)
        dist.all_reduce(buf, op=dist.ReduceOp.SUM, group=group)
        unpack_lower_symmetric(buf, V_local)
    else:
        dist.all_reduce(V_local, op=dist.ReduceOp.SUM, group=group)
    dist.all_reduce(e, op=dist.ReduceOp.SUM, group=group)
    return float(e.item()), V_local
