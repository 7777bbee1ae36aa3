"""N > 1 path of bench.py on CPU (gloo, world_size 2): trajectories are independent
(PAPER.md:64), so ranks own disjoint row blocks of one grid, there is no data-path collective,
and the only exchange is the max-over-ranks of the timed duration."""
import os
import sys
import types

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out_dir):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    args = types.SimpleNamespace(workload="C2", side=24, n_steps=10)
    wl = bench.workload_inputs(args, rank, world)
    # the max-over-ranks reduction bench.py applies to its device-timed duration
    t = torch.tensor([0.5 + rank], dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    gathered = [torch.empty_like(torch.from_numpy(wl["y0"])) for _ in range(world)]
    dist.all_gather(gathered, torch.from_numpy(wl["y0"]))
    if rank == 0:
        np.save(os.path.join(out_dir, "gathered.npy"), torch.cat(gathered, dim=1).numpy())
        np.save(os.path.join(out_dir, "tmax.npy"), t.numpy())
        np.save(os.path.join(out_dir, "rk.npy"), np.array([wl["rk_steps"]]))
    dist.destroy_process_group()


def test_row_sharding_world2(tmp_path):
    world, port = 2, 29500 + os.getpid() % 2000
    mp.spawn(_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    from paper_2507_00622_b200 import workloads as W
    full = W.hh_grid(0.125, 24 * world, 24)
    got = np.load(tmp_path / "gathered.npy")
    assert got.shape == full.shape and (got == full).all()     # disjoint blocks, in rank order
    assert np.load(tmp_path / "tmax.npy")[0] == 0.5 + (world - 1)
    assert np.load(tmp_path / "rk.npy")[0] == 2.0 * 24 * 24 * 10   # per-rank work is fixed (weak scaling)


def test_reference_arm_runs_only_on_rank0(monkeypatch, capsys):
    sys.path.insert(0, ROOT)
    import bench
    monkeypatch.setenv("RANK", "1")
    args = types.SimpleNamespace(side=32, n_steps=5, steps=1, warmup=0, gpus=2)
    assert bench.run_reference(args) is None
    assert capsys.readouterr().out == ""
