"""Host logic of the multi-GPU form: grid sharding + the one all-reduce of V and E,
run on CPU with 2 gloo ranks.  The per-rank compute is the CPU oracle here (test infrastructure);
on GPUs it is kldi_exc on the rank's shard (bench.py --gpus N)."""
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
    part, (lo, hi) = sharding.shard_workload(wl, rank, world)
    basis = (wl.atom_xyz, wl.shell_atom, wl.shell_l, wl.shell_prim_off, wl.prim_alpha, wl.prim_coef)
    loc = O.exc(basis, part.grid_xyz, part.grid_w, part.D, "lda")
    E, V = sharding.allreduce_exc(loc["E"], torch.as_tensor(loc["V"].copy()))
    g_loc = O.exc_nuclear_gradient_lda(basis, part.grid_xyz, part.grid_w, part.D)
    _, g = sharding.allreduce_exc(loc["E"], torch.as_tensor(g_loc.copy()))
    np.savez(os.path.join(out_dir, f"r{rank}.npz"), E=E, V=V.numpy(), lo=lo, hi=hi, rho=loc["rho"], grad=g.numpy())
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
    assert parts[0]["lo"] == 0 and parts[0]["hi"] == parts[1]["lo"] and parts[1]["hi"] == wl.n_pts
    for p in parts:   # every rank holds the reduced result
        assert abs(float(p["E"]) - ref["E"]) < 1e-12
        assert np.max(np.abs(p["V"] - ref["V"])) < 1e-12
    assert np.max(np.abs(np.concatenate([p["rho"] for p in parts]) - ref["rho"])) < 1e-13
    gref = O.exc_nuclear_gradient_lda(basis, wl.grid_xyz, wl.grid_w, wl.D)
    for p in parts:   # the nuclear gradient is a sum over grid shards as well
        assert np.max(np.abs(p["grad"] - gref)) < 1e-12
