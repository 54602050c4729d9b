"""N > 1 path of bench.py on CPU (gloo, world_size 2): the path does not shard a mesh, every rank runs an
independent replica (replicas only), so the only cross-rank logic is the reporting
rule -- device time = MAX over ranks, value = whole-job aggregate.  No GPU, no collective on the data path."""
import os
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _worker(rank: int, world: int, port: int, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    ms_local = 10.0 + 5.0 * rank  # rank 1 is the slow one
    ms = bench.reduce_max(ms_local, world, "cpu")
    val = bench.whole_job_value(2_000_000, 100, world, ms / 1e3)
    dist.barrier()
    out[rank] = (ms, val)
    dist.destroy_process_group()


def test_max_over_ranks_and_whole_job_value():
    world = 2
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, 29611, out), nprocs=world, join=True)
    assert out[0] == out[1]
    ms, val = out[0]
    assert ms == 15.0
    assert abs(val - 2 * 2_000_000 * 100 / 0.015) < 1e-3


def test_single_rank_is_identity():
    import bench
    assert bench.reduce_max(3.5, 1, "cpu") == 3.5
    assert bench.whole_job_value(10, 2, 1, 0.5) == 40.0


def test_reference_arm_runs_on_rank_zero_only(monkeypatch, capsys):
    """bench.py --impl reference under torchrun: only rank 0 runs and prints."""
    import bench
    monkeypatch.setenv("RANK", "1")
    monkeypatch.setenv("WORLD_SIZE", "2")
    monkeypatch.setattr(sys, "argv", ["bench.py", "--impl", "reference", "--steps", "1", "--warmup", "1"])
    bench.main()
    assert capsys.readouterr().out == ""
