"""The N>1 path of bench.py is "replicas only": no data-path collective, the whole-job time
is the slowest rank's, the value the sum of all ranks' work.  Covered here on CPU with world_size 2 (gloo)."""
import os
import socket
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    t = bench.max_over_ranks(1.0 + rank, dist, torch.device("cpu"))       # rank 1 is the slow one
    dist.barrier()
    out[rank] = t
    dist.destroy_process_group()


def test_replicas_time_is_max_over_ranks_and_value_is_whole_job():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
    assert out[0] == out[1] == 2.0
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.5, None, None) == 3.5
    # two replicas, 10 steps of 1.5e9 updates in 2 s
    assert abs(bench.whole_job_value(2, 1.5e9, 10, out[0]) - 15.0) < 1e-12


def test_reference_arm_only_rank0_works(monkeypatch, capsys):
    sys.path.insert(0, ROOT)
    import bench
    monkeypatch.setenv("RANK", "1")
    monkeypatch.setenv("WORLD_SIZE", "2")
    bench.run_reference(type("A", (), {"steps": 1, "warmup": 0})())
    assert capsys.readouterr().out == ""
