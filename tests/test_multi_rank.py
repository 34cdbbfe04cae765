"""The N>1 path of bench.py is "replicas only": no data-path collective, the whole-job time
is the slowest rank's, the value the sum of all ranks' work.  Covered here on CPU with world_size 2 (gloo)."""
import ctypes as C
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


# ---- NEXT-4: the angle-sharded cascade of the C ABI (cbct_cascade_run, csrc/cascade.cu) over gloo, world_size 2 -------
def _oracle_cascade_ops(g, n_levels, Y_local, f0, n_inner, eps, omega, dist_):
    """The callback table of cbct_cascade_run filled with the fp64 oracle's operators (tests only).  The level order, c and
    beta come from the LIBRARY; this side only keeps the per-level state and applies the operators it is asked for."""
    import numpy as np
    import oracle as o
    from oracle import fbs
    from paper_1002_3675_b200.binding import CascadeOps
    geoms, axes, binned = fbs.level_geometries(g, n_levels)
    st = {"Y": [np.asarray(Y_local, dtype=np.float64)] + [None] * (n_levels - 1), "f": [None] * n_levels, "G": [None] * n_levels,
          "calls": []}

    def level_sizes(user, l, p_nvox, p_npix):
        p_nvox[0], p_npix[0] = geoms[l].n_vox, geoms[l].nu * geoms[l].nv
        return 0

    def bin_(user, l):
        st["Y"][l + 1] = fbs.bin2x2(st["Y"][l]) if binned[l] else st["Y"][l]
        return 0

    def start(user, L, have_f0):
        if not have_f0:
            st["f"][L] = np.zeros(geoms[L].vol_shape)
        else:
            f = np.asarray(f0, dtype=np.float64)
            for l in range(L):
                f = fbs.restrict_volume(f, axes[l])
            st["f"][L] = f
        return 0

    def data_gradient(user, l):
        st["G"][l] = o.backproject(geoms[l], o.forward(geoms[l], st["f"][l]) - st["Y"][l])
        st["calls"].append(("grad", l))
        return 0

    def all_reduce(user, l):
        t = torch.from_numpy(st["G"][l])
        dist_.all_reduce(t, op=dist_.ReduceOp.SUM)              # in place: t shares G's memory
        st["calls"].append(("allreduce", l))
        return 0

    def prox_step(user, l, c, beta):
        gv = st["f"][l] - c * st["G"][l]
        st["f"][l] = np.maximum(o.tv_prox(geoms[l], gv, gv, beta, eps, omega, n_inner), 0.0)
        st["calls"].append(("prox", l, c, beta))
        return 0

    def prolong(user, l):
        st["f"][l - 1] = fbs.prolong(st["f"][l], axes[l - 1])
        return 0

    F = dict(CascadeOps._fields_)
    ops = CascadeOps(None, F["level_sizes"](level_sizes), F["bin"](bin_), F["start"](start), F["data_gradient"](data_gradient),
                     F["all_reduce"](all_reduce) if dist_ is not None else C.cast(None, F["all_reduce"]),
                     F["prox_step"](prox_step), F["prolong"](prolong))
    return ops, st


def _run_cascade(ops, n_outer, step, mu, n_angles_total, have_f0=0):
    import paper_1002_3675_b200 as cb
    L = cb.load()                                               # loads on a CPU-only box; cbct_cascade_run makes no CUDA call
    arr = (C.c_int * len(n_outer))(*n_outer)
    return L.cbct_cascade_run(C.byref(ops), len(n_outer), arr, float(step), float(mu), int(n_angles_total), int(have_f0))


def _sharded_worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import numpy as np
    from cbct_synth import make_config
    from paper_1002_3675_b200.sharded import shard_angles
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      OMP_NUM_THREADS="2")
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cfg = make_config("c3", shrink=16)                          # noisy data: the shards must partition ONE noisy scan
    g, Y = cfg.geom, cfg.projections()
    mine = shard_angles(g.n_angles, rank, world)
    assert np.array_equal(cfg.projections(mine), Y[mine])
    ops, st = _oracle_cascade_ops(g.with_angles(g.angles[mine]), 2, np.ascontiguousarray(Y[mine]), None, cfg.n_inner, cfg.eps,
                                  cfg.omega, dist)
    rc = _run_cascade(ops, [3, 2], cfg.step, cfg.mu, g.n_angles)
    out[rank] = (rc, st["f"][0], st["calls"])
    dist.barrier()
    dist.destroy_process_group()


def test_angle_sharded_cascade_of_the_library_equals_the_single_rank_reconstruction():
    """Two ranks, each with every second angle and its share of Y, driven by the LIBRARY's cbct_cascade_run: after the
    per-iteration all-reduce of the gradient volume both hold the reconstruction of the full scan (P^T over a subset is an
    exact partial sum).  Also checks the constants the library hands to the prox step and the order of its calls."""
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
    cfg = make_config("c3", shrink=16)
    g = cfg.geom
    ref = fbs.fbs_reconstruct(g, cfg.projections(), None, 2, [3, 2], cfg.n_inner, cfg.step, cfg.mu, cfg.eps, cfg.omega)
    assert out[0][0] == 0 and out[1][0] == 0
    assert np.array_equal(out[0][1], out[1][1])                 # every rank applies the same prox step to the same sum
    assert np.linalg.norm(out[0][1] - ref) <= 1e-12 * np.linalg.norm(ref)
    calls = out[0][2]
    assert [c[0] for c in calls] == ["grad", "allreduce", "prox"] * 5 and [c[1] for c in calls] == [1] * 9 + [0] * 6
    gc = fbs.coarsen_geometry(g)[0]
    for (_, l, c, beta), gl in zip([c for c in calls if c[0] == "prox"], [gc] * 3 + [g] * 2):
        assert c == 2.0 * cfg.step * gl.n_vox / (g.n_angles * gl.n_pix) and beta == cfg.mu / cfg.step
    # the partition covers every angle exactly once
    idx = np.sort(np.concatenate([shard_angles(17, r, 3) for r in range(3)]))
    assert np.array_equal(idx, np.arange(17))


def test_cascade_run_single_rank_and_errors():
    """One rank, no exchange callback: cbct_cascade_run with the oracle's operators IS the oracle's cascade (with a caller's
    f0 restricted down); bad arguments and failing callbacks come back as status codes."""
    import numpy as np
    sys.path.insert(0, ROOT)
    import paper_1002_3675_b200 as cb
    from cbct_synth import make_config
    from oracle import fbs
    cfg = make_config("c1", shrink=2)
    g, Y = cfg.geom, cfg.projections()
    f0 = np.abs(np.random.default_rng(0).normal(size=g.vol_shape)) * 0.01
    ops, st = _oracle_cascade_ops(g, 2, Y, f0, cfg.n_inner, cfg.eps, cfg.omega, None)
    assert _run_cascade(ops, [2, 3], cfg.step, cfg.mu, g.n_angles, have_f0=1) == 0
    ref = fbs.fbs_reconstruct(g, Y, f0, 2, [2, 3], cfg.n_inner, cfg.step, cfg.mu, cfg.eps, cfg.omega)
    assert np.array_equal(st["f"][0], ref)
    assert all(c[0] != "allreduce" for c in st["calls"])
    assert _run_cascade(ops, [2, -1], cfg.step, cfg.mu, g.n_angles) == 1          # negative count
    assert _run_cascade(ops, [1, 1], 0.0, cfg.mu, g.n_angles) == 1                 # step <= 0
    F = dict(cb.CascadeOps._fields_)
    ops.prox_step = F["prox_step"](lambda u, l, c, b: 3)                           # a callback's status is passed through
    assert _run_cascade(ops, [1, 1], cfg.step, cfg.mu, g.n_angles) == 3


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
