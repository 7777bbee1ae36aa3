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
    # the rank layout main() takes from the torchrun environment
    plan = bench.launch_plan(world, os.environ, ["--gpus", str(world)])
    assert plan == ("run", rank, int(os.environ.get("LOCAL_RANK", "0")), world)
    assert bench.launch_plan(world + 1, os.environ, [])[0] == "error"    # --gpus contradicts WORLD_SIZE
    wl = bench.workload_inputs(args, rank, world)
    # the max-over-ranks reduction bench.py applies to its device-timed duration, and its aggregate
    tmax = bench.rank_max(0.5 + rank, world)
    t = torch.tensor([tmax], dtype=torch.float64)
    agg = bench.aggregate(wl["rk_steps"], world, 3, tmax)
    assert agg == wl["rk_steps"] * world * 3 / (0.5 + world - 1)
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


def test_gpus_flag_never_silently_ignored(monkeypatch):
    """--gpus N outside torchrun re-launches under torch.distributed.run with N ranks; inside torchrun it
    must equal WORLD_SIZE; bench.py never times one GPU and reports another count."""
    sys.path.insert(0, ROOT)
    import bench
    assert bench.launch_plan(1, {}, []) == ("run", 0, 0, 1)
    kind, cmd = bench.launch_plan(8, {}, ["--gpus", "8", "--steps", "2"])
    assert kind == "spawn" and "--nproc-per-node=8" in cmd and cmd[-4:] == ["--gpus", "8", "--steps", "2"]
    assert "torch.distributed.run" in cmd and "127.0.0.1" in cmd
    assert bench.launch_plan(8, {"WORLD_SIZE": "1"}, [])[0] == "error"
    assert bench.launch_plan(0, {}, [])[0] == "error"
    assert bench.launch_plan(2, {"WORLD_SIZE": "2", "RANK": "1", "LOCAL_RANK": "1"}, []) == ("run", 1, 1, 2)
    # no CUDA device here: the spawned ranks must fail loudly, not print a line
    import subprocess
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "1", "--warmup", "0",
                        "--configs", ""], capture_output=True, text=True, timeout=600)
    import torch
    if not torch.cuda.is_available():
        assert r.returncode != 0 and '"n_gpus"' not in r.stdout


def test_kernel_traffic_comes_from_the_tracked_profile():
    sys.path.insert(0, ROOT)
    import bench
    assert os.path.exists(bench.TRAFFIC_CSV)
    t = bench.kernel_traffic("C2")
    assert t is not None and 1e7 < t < 1e8
    assert bench.kernel_traffic("no-such-workload") is None
