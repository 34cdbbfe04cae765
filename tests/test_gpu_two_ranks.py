"""NEXT-4 on hardware with two PROCESSES: cbct_fbs_reconstruct_sharded with a real torch.distributed all-reduce between
two ranks, each holding every second view, on a side stream.

Only one GPU is visible to the tests and NCCL refuses two ranks on one device ("Duplicate GPU detected", NCCL 2.28.9,
measured on this pool), so the ranks share cuda:0 and the exchange is torch.distributed's gloo backend on CUDA tensors (it
stages the buffer through the host): the stated stand-in of DESIGN.md section 8.  Everything else is the multi-GPU path as
it would run under NCCL: one handle per rank over that rank's angles, the library's cascade, the exchange callback on the
library's stream.  The ranks do not wait on one another inside kernels, only in the collective between launches.
"""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
pytestmark = pytest.mark.gpu

N_LEVELS, N_OUTER = 2, [3, 2]


def _rank(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import paper_1002_3675_b200 as cb
    from cbct_synth import make_config
    from paper_1002_3675_b200.sharded import fbs_reconstruct_sharded, shard_angles
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dev = torch.device("cuda:0")
    torch.cuda.set_device(dev)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        cfg = make_config("c3", shrink=4)                       # 128 x 128 x 16, 40 noisy views of 128 x 96
        g = cfg.geom
        mine = shard_angles(g.n_angles, rank, world)
        G = cb.Geometry.from_synth(g.with_angles(g.angles[mine]))
        d_Y = torch.from_numpy(np.ascontiguousarray(cfg.projections()[mine], dtype=np.float32)).to(dev)
        side = torch.cuda.Stream()
        f = fbs_reconstruct_sharded(G, d_Y, None, N_LEVELS, N_OUTER, cfg.n_inner, cfg.step, cfg.mu, cfg.eps, cfg.omega,
                                    g.n_angles, dist, stream=side)
        side.synchronize()
        out[rank] = f.cpu().numpy()
        G.close()
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_two_processes_reconstruct_the_full_scan(cuda_lib):
    cb = cuda_lib
    sys.path.insert(0, ROOT)
    from cbct_synth import make_config
    from oracle import fbs
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    out = mp.get_context("spawn").Manager().dict()     # no fork() of a process that has initialised CUDA
    mp.spawn(_rank, args=(2, port, out), nprocs=2, join=True)
    cfg = make_config("c3", shrink=4)
    g = cfg.geom
    # every rank applied the same prox step to the same summed gradient
    assert np.array_equal(out[0], out[1])
    # the single-rank library result: equal up to the order in which the partial gradients are added (fp32)
    dev = torch.device("cuda:0")
    G = cb.Geometry.from_synth(g)
    d_Y = torch.from_numpy(np.ascontiguousarray(cfg.projections(), dtype=np.float32)).to(dev)
    f_one = torch.empty(G.vol_shape, device=dev)
    cb.fbs_reconstruct(G, d_Y, None, N_LEVELS, N_OUTER, cfg.n_inner, cfg.step, cfg.mu, cfg.eps, cfg.omega, f_one)
    torch.cuda.synchronize()
    one = f_one.cpu().numpy().astype(np.float64)
    G.close()
    rel = lambda a, b: float(np.linalg.norm(a.astype(np.float64) - b) / np.linalg.norm(b))
    assert rel(out[0], one) <= 1e-5
    # and the oracle's reconstruction of the full scan, at the reconstruction tolerance of north_star
    ref = fbs.fbs_reconstruct(g, cfg.projections(), None, N_LEVELS, N_OUTER, cfg.n_inner, cfg.step, cfg.mu, cfg.eps, cfg.omega)
    assert rel(out[0], ref) <= 1e-4
