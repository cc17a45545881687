"""Host logic of the multi-GPU form: cost-balanced sharding of the grid along the plan's curve order +
the one all-reduce of V (packed lower triangle) and E, run on CPU with 2 gloo ranks.  The per-rank compute is the CPU
oracle here (test infrastructure); on GPUs it is kldi_exc on the rank's shard (bench.py --gpus N, and
tests/test_gpu_parity.py::test_sharded_plans_sum_to_whole on one GPU)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2605_10363_b200 import sharding


def test_shard_bounds_partition():
    for n, w, a in [(16500, 2, 5500), (528000, 8, 5500), (1000, 3, 1), (5, 8, 1), (0, 2, 7), (16500, 4, 5500)]:
        b = sharding.shard_bounds(n, w, a)
        assert len(b) == w and b[0][0] == 0 and b[-1][1] == n
        for (lo, hi), (lo2, _) in zip(b, b[1:]):
            assert lo <= hi == lo2
        assert all(lo % a == 0 for lo, _ in b)
    with pytest.raises(ValueError):
        sharding.shard_bounds(10, 0)


def test_cost_balanced_curve_ranges():
    """contiguous ranges of the curve order balanced by sum K(K+1), not by point counts."""
    from paper_2605_10363_b200 import workloads as W

    wl = W.named_config("cfg1", becke_backend="none")       # weights play no role in the partition
    order = sharding.curve_order(wl.grid_xyz)
    assert np.array_equal(np.sort(order), np.arange(wl.n_pts))
    cost = sharding.block_costs(wl, order, wl.eps)
    assert cost.shape[0] == (wl.n_pts + 127) // 128 and cost.min() >= 0.0 and cost.max() > 0.0
    for world in (2, 4, 8):
        rng = sharding.balanced_ranges(cost, world)
        assert rng[0][0] == 0 and rng[-1][1] == len(cost) and all(a[1] == b[0] for a, b in zip(rng, rng[1:]))
        per = np.array([cost[a:b].sum() for a, b in rng])
        assert per.max() / per.mean() <= 1.05, (world, per)
        npts = np.array([(b - a) for a, b in rng], dtype=float)
        assert npts.max() / npts.mean() > 1.05              # equal cost is NOT equal point counts on a cluster
    parts = [sharding.shard_workload(wl, r, 4)[1] for r in range(4)]
    assert np.array_equal(np.sort(np.concatenate(parts)), np.arange(wl.n_pts))   # every point on exactly one rank
    # a rank's points are spatially compact: its bounding box is well inside the molecule's
    ext_all = np.prod(np.ptp(wl.grid_xyz[np.abs(wl.grid_xyz).max(axis=1) < 60.0], axis=0))
    inner = [p for p in parts if np.abs(wl.grid_xyz[p]).max() < 60.0]
    assert all(np.prod(np.ptp(wl.grid_xyz[p], axis=0)) < ext_all for p in inner)


def test_triangle_pack_roundtrip():
    for n in (1, 5, 1023, 1500):
        a = torch.randn(n, n, dtype=torch.float64)
        v = a + a.T
        buf = sharding.pack_lower(v)
        assert buf.numel() <= (0.53 if n >= 1024 else 1.0) * n * n + n
        out = torch.full_like(v, float("nan"))
        sharding.unpack_lower_symmetric(buf, out)
        assert torch.equal(out, v)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from oracle import exc_oracle as O
    from paper_2605_10363_b200 import workloads as W

    wl = W.named_config("cfg0")
    part, idx = sharding.shard_workload(wl, rank, world)
    basis = (wl.atom_xyz, wl.shell_atom, wl.shell_l, wl.shell_prim_off, wl.prim_alpha, wl.prim_coef)
    loc = O.exc(basis, part.grid_xyz, part.grid_w, part.D, "lda")
    E, V = sharding.allreduce_exc(loc["E"], torch.as_tensor(loc["V"].copy()))
    g_loc = O.exc_nuclear_gradient_lda(basis, part.grid_xyz, part.grid_w, part.D)
    _, g = sharding.allreduce_exc(loc["E"], torch.as_tensor(g_loc.copy()))
    np.savez(os.path.join(out_dir, f"r{rank}.npz"), E=E, V=V.numpy(), idx=idx, rho=loc["rho"], grad=g.numpy())
    dist.destroy_process_group()


def test_two_rank_gloo_matches_single(tmp_path):
    from oracle import exc_oracle as O
    from paper_2605_10363_b200 import workloads as W

    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    wl = W.named_config("cfg0")
    basis = (wl.atom_xyz, wl.shell_atom, wl.shell_l, wl.shell_prim_off, wl.prim_alpha, wl.prim_coef)
    ref = O.exc(basis, wl.grid_xyz, wl.grid_w, wl.D, "lda")
    parts = [np.load(os.path.join(str(tmp_path), f"r{r}.npz")) for r in range(world)]
    allidx = np.concatenate([p["idx"] for p in parts])
    assert np.array_equal(np.sort(allidx), np.arange(wl.n_pts))
    for p in parts:   # every rank holds the reduced result
        assert abs(float(p["E"]) - ref["E"]) < 1e-12
        assert np.max(np.abs(p["V"] - ref["V"])) < 1e-12
    rho = np.empty(wl.n_pts)
    rho[allidx] = np.concatenate([p["rho"] for p in parts])     # rho stays sharded: each rank's values map back through idx
    assert np.max(np.abs(rho - ref["rho"])) < 1e-13
    for p in parts:
        assert np.max(np.abs(p["V"] - p["V"].T)) < 1e-13        # (one band below 1024 AOs: the oracle's own rounding)
    gref = O.exc_nuclear_gradient_lda(basis, wl.grid_xyz, wl.grid_w, wl.D)
    for p in parts:   # the nuclear gradient is a sum over grid shards as well
        assert np.max(np.abs(p["grad"] - gref)) < 1e-12
