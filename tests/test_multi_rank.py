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


# ---- NEXT-4: angle-sharded A1 (paper_1002_3675_b200/sharded.py) over gloo, world_size 2 ---------------------
class _OracleOps:
    """The driver's `ops` interface on top of the fp64 oracle (tests only): lets the host-side logic of the
    sharded driver (partition, constants, level order, the exchange) run on CPU."""

    def __init__(self, g, n_levels):
        from oracle import fbs
        self.fbs = fbs
        self.geoms, self.axes, self.binned = fbs.level_geometries(g, n_levels)

    def n_vox(self, l): return self.geoms[l].n_vox
    def n_pix(self, l): return self.geoms[l].nu * self.geoms[l].nv
    def zeros(self, l):
        import numpy as np
        return np.zeros(self.geoms[l].vol_shape)
    def bin(self, l, Y): return self.fbs.bin2x2(Y) if self.binned[l] else Y
    def restrict(self, l, f): return self.fbs.restrict_volume(f, self.axes[l])
    def prolong(self, l, fc): return self.fbs.prolong(fc, self.axes[l])
    def data_gradient(self, l, f, Y):
        import oracle as o
        return o.backproject(self.geoms[l], o.forward(self.geoms[l], f) - Y)
    def all_reduce(self, G, dist_):
        if dist_ is not None:
            t = torch.from_numpy(G)
            dist_.all_reduce(t, op=dist_.ReduceOp.SUM)          # in place: t shares G's memory
    def prox_step(self, l, f, G, c, beta, eps, omega, n_inner):
        import numpy as np
        import oracle as o
        gv = f - c * G
        return np.maximum(o.tv_prox(self.geoms[l], gv, gv, beta, eps, omega, n_inner), 0.0)


def _sharded_worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import numpy as np
    from cbct_synth import make_config
    from paper_1002_3675_b200.sharded import fbs_reconstruct_sharded, shard_angles
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      OMP_NUM_THREADS="2")
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cfg = make_config("c1", shrink=2)
    g, Y = cfg.geom, cfg.projections()
    mine = shard_angles(g.n_angles, rank, world)
    ops = _OracleOps(g.with_angles(g.angles[mine]), 2)
    f = fbs_reconstruct_sharded(ops, np.ascontiguousarray(Y[mine]), None, 2, [3, 2], cfg.n_inner, cfg.step, cfg.mu,
                                cfg.eps, cfg.omega, g.n_angles, dist)
    out[rank] = f
    dist.barrier()
    dist.destroy_process_group()


def test_angle_sharded_driver_equals_the_single_rank_reconstruction():
    """Two ranks, each with every second angle and its share of Y: after the per-iteration all-reduce of the
    gradient volume both hold the reconstruction of the full scan (P^T over a subset is an exact partial sum)."""
    import numpy as np
    sys.path.insert(0, ROOT)
    from cbct_synth import make_config
    from oracle import fbs
    from paper_1002_3675_b200.sharded import shard_angles
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    out = mp.Manager().dict()
    mp.spawn(_sharded_worker, args=(2, port, out), nprocs=2, join=True)
    cfg = make_config("c1", shrink=2)
    ref = fbs.fbs_reconstruct(cfg.geom, cfg.projections(), None, 2, [3, 2], cfg.n_inner, cfg.step, cfg.mu, cfg.eps, cfg.omega)
    assert np.array_equal(out[0], out[1])                       # every rank applies the same prox step to the same sum
    assert np.linalg.norm(out[0] - ref) <= 1e-12 * np.linalg.norm(ref)
    # the partition covers every angle exactly once
    idx = np.sort(np.concatenate([shard_angles(17, r, 3) for r in range(3)]))
    assert np.array_equal(idx, np.arange(17))


def test_bench_gpus_n_starts_n_ranks_by_itself():
    """`python bench.py --gpus 2` with no RANK in the environment re-runs itself as 2 ranks under torch.distributed.run
    (replicas and --shard-angles alike); --rank-probe makes every rank print its environment instead of touching a GPU."""
    import json
    import subprocess
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "LOCAL_RANK", "WORLD_SIZE", "MASTER_ADDR", "MASTER_PORT")}
    for extra, mode in (([], "replicas"), (["--shard-angles"], "shard-angles")):
        r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--rank-probe"] + extra,
                           capture_output=True, text=True, env=env, timeout=300)
        assert r.returncode == 0, r.stderr[-2000:]
        rows = [json.loads(l) for l in r.stdout.splitlines() if l.startswith("{")]
        assert sorted(x["RANK"] for x in rows) == ["0", "1"]
        assert sorted(x["LOCAL_RANK"] for x in rows) == ["0", "1"]
        assert all(x["WORLD_SIZE"] == "2" and x["MASTER_ADDR"] == "127.0.0.1" and x["mode"] == mode for x in rows)
    # under a launcher (RANK set) the command does not spawn again
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--rank-probe"], capture_output=True,
                       text=True, env=dict(env, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2"), timeout=120)
    rows = [json.loads(l) for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(rows) == 1 and rows[0]["RANK"] == "1"
