#!/usr/bin/env python
"""bench.py — measurement contract of the CBCT TV-FBS hot path.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]

Workload (N=1): BASELINE.json configs[1] ("c2"): 256^3 volume @ 1 mm, 40 views of 512x384 @ 0.78 mm.
One STEP = one pass of the whole hot path: a 2-level coarse-to-fine
cascade with one outer FBS iteration per level — bin Y 2x2, [P, residual, P^T, gradient step,
10 TV-prox sweeps, clamp] on the 128^3 level, prolong, the same on the 256^3 level — through the C ABI
call cbct_fbs_reconstruct.  Each step continues from the previous step's volume.
metric  = projector+backprojector GUPS = voxel-projection updates of P and of P^T on all levels / step time
value   = device-resident inputs (CUDA events around each step, L2 flushed between steps)
e2e     = same through cbct_fbs_reconstruct_host: pinned HOST buffers, H2D of Y and f, D2H of f every step
Extra keys: per-operator GUPS, TV GB/s, seconds per full c3 reconstruction, roofline of the dominant
kernel (live CUDA-event timing of each kernel class), the oracle timed on the host cores.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "projector+backprojector GUPS (voxel-projection updates/s of P and P^T through one full FBS cascade step)"
UNIT = "GUPS"
N_INNER = 10
LEVELS = 2
TRAFFIC_COVERS = ("dram__bytes_read.sum + dram__bytes_write.sum of ONE fine-level launch of the dominant kernel "
                  "(profiles/traffic.csv, from the committed ncu --set full capture)")
LANE_OPS_PER_CHORD = 16          # issue-bound model of the exact-chord march/gather
NNZ = {"c2": 2.45e9, "c3": 3.85e9}   # chords per application of P; refined by frozen_params.json


def peaks():
    p = {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "which": "fallback"}
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            m = json.load(fh)
        p.update(hbm_gbs=float(m["hbm_gbs"]), sm_max_mhz=float(m.get("sm_max_mhz", 1965.0)), which="measured")
    except Exception:
        pass
    return p


def frozen(key, name, default):
    try:
        with open(os.path.join(ROOT, "cbct_synth", "frozen_params.json")) as fh:
            return json.load(fh).get(f"{name}/1", {}).get(key, default)
    except Exception:
        return default


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def __exit__(self, *a):
        if self.proc:
            time.sleep(0.25)
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except Exception:
                self.proc.kill()

    def summary(self):
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except Exception:
                continue
            for n, v in zip(names, r[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "reasons": sorted(reasons), "samples": len(sm)}


def level_dims(G, levels):
    """(n_vox, n_rays) per level, asked of the library's own coarse-level handles (cbct_geometry_coarsen)."""
    out, cur = [], G
    for l in range(levels):
        out.append((cur.n_vox, cur.n_proj))
        if l + 1 < levels:
            cur = cur.coarsen()[0]
    return out


def max_over_ranks(seconds: float, dist, device) -> float:
    """Whole-job time of a replicas-only run: the slowest rank's device-timed seconds (all-reduce MAX)."""
    if dist is None:
        return float(seconds)
    import torch
    t = torch.tensor([seconds], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(world: int, updates_per_step: float, steps: int, seconds: float) -> float:
    """Aggregate GUPS over all ranks: every rank processed `updates_per_step` per step (weak scaling)."""
    return world * updates_per_step * steps / seconds / 1e9


def run_gpu(args):
    import torch
    import paper_1002_3675_b200 as cb
    from cbct_synth import make_config

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    cb.load()

    cfg = make_config("c2")
    g = cfg.geom
    # replicas only: every rank runs its own copy of the same seeded scan; no data-path collective
    Y = np.ascontiguousarray(cfg.projections(), dtype=np.float32)
    G = cb.Geometry.from_synth(g)
    if args.staged_projector:
        G.set_projector_staging(True)
    if args.plain_kernels:
        G.set_mirror_symmetry(False)
    n_outer = [1] * LEVELS
    lv = level_dims(G, LEVELS)
    updates = 2.0 * sum(nvox * g.n_angles for nvox, _ in lv)

    st = torch.cuda.Stream(device=dev)
    d_Y = torch.from_numpy(Y).to(dev)
    d_f = torch.zeros(g.vol_shape, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)       # > 126 MB L2
    h_Y = torch.from_numpy(Y).pin_memory()
    h_f = torch.zeros(g.vol_shape, dtype=torch.float32).pin_memory()

    def step_dev():
        cb.fbs_reconstruct(G, d_Y, d_f, LEVELS, n_outer, N_INNER, cfg.step, cfg.mu, cfg.eps, cfg.omega, d_f, stream=st)

    def step_host():
        cb.fbs_reconstruct_host(G, h_Y, h_f, LEVELS, n_outer, N_INNER, cfg.step, cfg.mu, cfg.eps, cfg.omega, h_f, stream=st)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    with torch.cuda.stream(st):
        for _ in range(args.warmup):
            step_dev()
    barrier()

    # ---- timed region: K steps, device-resident, per-step events, L2 flushed between steps ----
    cb.profile_enable(True)
    cb.profile_read(reset=True)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    n0 = cb.launch_count()
    with ClockSampler(local) as clk:
        with torch.cuda.stream(st):
            for a, b in ev:
                flush.fill_(1)
                a.record(st)
                step_dev()
                b.record(st)
        barrier()
    launches = cb.launch_count() - n0
    prof = cb.profile_read(reset=True)
    cb.profile_enable(False)
    ms = [a.elapsed_time(b) for a, b in ev]
    t_total = max_over_ranks(sum(ms) / 1e3, dist, dev)

    # ---- end-to-end: host buffers through the C ABI, copies inside the timed region ----
    h_f.copy_(d_f.cpu())
    with torch.cuda.stream(st):
        step_host()                                                       # warm the staging buffers
    barrier()
    ev2 = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    with torch.cuda.stream(st):
        for a, b in ev2:
            flush.fill_(1)
            a.record(st)
            step_host()
            b.record(st)
    barrier()
    t_e2e = max_over_ranks(sum(a.elapsed_time(b) for a, b in ev2) / 1e3, dist, dev)

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    pk = peaks()
    K = args.steps
    value = whole_job_value(world, updates, K, t_total)
    e2e_value = whole_job_value(world, updates, K, t_e2e)

    # per-operator numbers from the live per-class event timing (fine + coarse level launches summed)
    def per_step_ms(tag):
        return prof[tag][0] / K
    upd_one = sum(nvox * g.n_angles for nvox, _ in lv)
    gups_p = upd_one / (per_step_ms("forward") / 1e3) / 1e9
    gups_bp = upd_one / (per_step_ms("backproject") / 1e3) / 1e9
    tv_bytes = 12.0 * sum(nvox for nvox, _ in lv) * N_INNER
    tv_gbs = tv_bytes / (per_step_ms("tv_sweep") / 1e3) / 1e9

    # roofline of the dominant kernel class
    dom = max(("forward", "backproject", "tv_sweep"), key=lambda t: prof[t][0])
    nnz_fine = float(frozen("nnz", "c2", NNZ["c2"]))
    nnz_step = nnz_fine * (1.0 + frozen("nnz_coarse_ratio", "c2", 0.125))
    sm_count = torch.cuda.get_device_properties(dev).multi_processor_count
    traffic, traffic_stale = committed_traffic(dom)
    if dom == "tv_sweep":
        roof = {"kernel": "tv_sweep_kernel", "bound": "hbm", "achieved": tv_gbs, "peak": pk["hbm_gbs"], "unit": "GB/s",
                "frac": tv_gbs / pk["hbm_gbs"], "traffic": traffic, "traffic_stale": traffic_stale, "traffic_covers": TRAFFIC_COVERS,
                "peak_source": "MEASURED_PEAKS.json copy bandwidth" if pk["which"] == "measured" else "fallback (B200_PROFILING.md)"}
    else:
        peak = sm_count * 128 * pk["sm_max_mhz"] * 1e6 / 1e12            # T lane-op/s (fp32 issue: SMs x 128 lanes x clock)
        ach = LANE_OPS_PER_CHORD * nnz_step / (per_step_ms(dom) / 1e3) / 1e12
        roof = {"kernel": dom + "_kernel", "bound": "alu", "achieved": ach, "peak": peak, "unit": "Tlane-op/s",
                "frac": ach / peak, "traffic": traffic, "traffic_stale": traffic_stale, "traffic_covers": TRAFFIC_COVERS,
                "peak_source": f"nominal lanes ({sm_count} SMs x 128 fp32 lanes) x max SM clock ({pk['sm_max_mhz']:.0f} MHz, {pk['which']})",
                "model": f"{LANE_OPS_PER_CHORD} fp32 lane-ops per chord x {nnz_step:.3e} chords per step (SURVEY.md 8(d))",
                "chords_per_s": nnz_step / (per_step_ms(dom) / 1e3)}

    extra = {"gups_forward": gups_p, "gups_backproject": gups_bp, "tv_GBps": tv_gbs,
             "tv_frac_of_hbm": tv_gbs / pk["hbm_gbs"],
             "tv_note": "tv_GBps is the c2 step's figure (256^3 + 128^3 volumes of 67 + 8 MB: partly L2-resident between sweeps, so "
                        "not an HBM fraction); tv_GBps_512cube is the same kernel on 512^3 volumes (537 MB each, nothing resident)",
             "ms_per_step_by_kernel": {k: v[0] / K for k, v in prof.items()}}
    if not args.no_recon and world == 1:
        tvb = time_tv_512(cb, dev, st, flush)
        extra.update(tv_GBps_512cube=tvb, tv_512cube_frac_of_hbm=tvb / pk["hbm_gbs"])
    if not args.no_recon and world == 1:
        extra["sec_per_fbs_recon_c3"] = time_c3_recon(cb, dev, st)
        # NEXT-1 (not part of `value`): the paper's eq. 2 backprojector, alone at c2 and inside the c3 reconstruction
        extra["sec_per_fbs_recon_c3_eq2"] = time_c3_recon(cb, dev, st, eq2=True)
        q = torch.empty(g.proj_shape, device=dev)
        b = torch.empty(g.vol_shape, device=dev)
        ea, eb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        with torch.cuda.stream(st):
            cb.forward(G, d_f, q, stream=st)
            cb.backproject_eq2(G, q, b, stream=st)
            ea.record(st)
            for _ in range(5):
                cb.backproject_eq2(G, q, b, stream=st)
            eb.record(st)
        torch.cuda.synchronize()
        extra["gups_backproject_eq2"] = g.n_vox * g.n_angles / (ea.elapsed_time(eb) / 5e3) / 1e9
        # NEXT-4 (not part of `value`): the FDK baseline on c3's data, beside the FBS reconstruction of the same scan
        extra["sec_fdk_c3"] = time_c3_fdk(cb, dev, st)
        # metric (3) of BASELINE.json on the other configs, and the c3 reconstruction end to end from host buffers
        extra["sec_per_fbs_recon_c1"] = time_recon(cb, dev, st, "c1")
        extra["sec_per_fbs_recon_c4"] = time_recon(cb, dev, st, "c4")
        sec_h, h2d, d2h = time_c3_recon_host(cb, dev, st)
        extra["sec_per_fbs_recon_c3_e2e_host"] = {"value": sec_h, "h2d_bytes": h2d, "d2h_bytes": d2h,
                                                  "through": "cbct_fbs_reconstruct_host, pinned host buffers, host clock"}
        if not args.no_c5:
            sec5, (gp5, gb5) = time_recon(cb, dev, st, "c5", synthetic_noise_only=True, operators=True)
            extra.update(sec_per_fbs_recon_c5=sec5, gups_forward_c5=gp5, gups_backproject_c5=gb5,
                         c5_note="512^3 volume, 363 views of 1024 x 768, 3 levels x 50 outer x 10 TV sweeps; projections are "
                                 "device-made uniform noise (fixed iteration counts: the work does not depend on the values)")
    cpu = cpu_baseline_sample(cfg, n_angles=args.cpu_angles) if world == 1 and not args.no_cpu else None

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": args.warmup,
        "ms_per_step": 1e3 * t_total / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": "c2: 256^3 fp32 volume @1mm, 40 views x 384x512 @0.78mm, SAD 1000/SDD 1500; "
                               "step = 2-level FBS cascade, 1 outer iteration per level, 10 TV sweeps",
                   "levels": LEVELS, "n_tv_inner": N_INNER, "updates_per_step": updates,
                   "l2": "flushed between steps (256 MiB write); per-step working set ~0.9 GB > 126 MB L2",
                   "parallelism": "replicas only (one independent reconstruction per GPU)" if world > 1 else "1 GPU",
                   "kernels": ("TMA-staged projector" if args.staged_projector else "cached march") +
                              (", plain (unmirrored) march and gather" if args.plain_kernels else ", z-mirrored march and gather")},
        "clocks": clk.summary(),
        "e2e": {"value": e2e_value, "unit": UNIT, "ms_per_step": 1e3 * t_e2e / K,
                "h2d_bytes_per_step": int(h_Y.numel() * 4 + h_f.numel() * 4), "d2h_bytes_per_step": int(h_f.numel() * 4)},
        "gpu_launches": int(launches),
        "roofline": roof,
        "cpu_baseline": cpu,
        "extra": extra,
    }
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


def run_sharded(args):
    """--shard-angles (NEXT-4, not the default): ONE reconstruction step of c2 with the 40 views partitioned over
    the ranks and one NCCL all-reduce of the gradient volume per outer iteration; strong scaling."""
    import torch
    import paper_1002_3675_b200 as cb
    from paper_1002_3675_b200.sharded import fbs_reconstruct_sharded, shard_angles
    from cbct_synth import make_config
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    cb.load()
    cfg = make_config("c2")
    g = cfg.geom
    mine = shard_angles(g.n_angles, rank, world)
    G = cb.Geometry.from_synth(g.with_angles(g.angles[mine]))
    d_Y = torch.from_numpy(np.ascontiguousarray(cfg.projections(mine), dtype=np.float32)).to(dev)
    state = {"f": torch.zeros(g.vol_shape, device=dev)}
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)

    def step():
        state["f"] = fbs_reconstruct_sharded(G, d_Y, state["f"], LEVELS, [1] * LEVELS, N_INNER, cfg.step, cfg.mu, cfg.eps,
                                             cfg.omega, g.n_angles, dist)

    for _ in range(args.warmup):
        step()
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    with ClockSampler(local) as clk:
        for a, b in ev:
            flush.fill_(1)
            a.record()
            step()
            b.record()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()
    t = max_over_ranks(sum(a.elapsed_time(b) for a, b in ev) / 1e3, dist, dev)
    if rank == 0:
        updates = 2.0 * sum(nvox * g.n_angles for nvox, _ in level_dims(G, LEVELS))
        print(json.dumps({"metric": METRIC, "value": whole_job_value(1, updates, args.steps, t), "unit": UNIT, "n_gpus": world,
                          "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t / args.steps,
                          "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                          "config": {"workload": "c2, one reconstruction step with its 40 views sharded over the ranks",
                                     "parallelism": f"angles sharded over {world} rank(s), one all-reduce of the gradient "
                                                    "volume per outer iteration (NEXT-4)", "l2": "flushed between steps"},
                          "clocks": clk.summary()}))
    if dist is not None:
        dist.destroy_process_group()


def kernel_source_sha(rel_path):
    """First 16 hex digits of the SHA-256 of a kernel source file (the stamp profiles/traffic.csv carries per row)."""
    import hashlib
    with open(os.path.join(ROOT, rel_path), "rb") as fh:
        return hashlib.sha256(fh.read()).hexdigest()[:16]


def committed_traffic(kernel_class):
    """(DRAM bytes per launch of that kernel class from the committed ncu capture, None) - or (None, reason) when
    profiles/traffic.csv has no row for the class or its row was captured from ANOTHER version of the kernel's source file:
    a traffic figure that no longer belongs to the kernel being timed is reported as missing, loudly, not carried along.
    Rows: kernel_class,dram_bytes_per_launch,source_file,source_sha256_16,capture."""
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.csv")) as fh:
            rows = [line.split(",", 4) for line in fh.read().splitlines()[1:] if line.strip()]
    except OSError as e:
        return None, f"profiles/traffic.csv: {e}"
    for r in rows:
        if r[0] == kernel_class:
            if len(r) < 4:
                return None, "profiles/traffic.csv row carries no source stamp"
            now = kernel_source_sha(r[2])
            if now != r[3]:
                return None, (f"{r[2]} has changed since the ncu capture in profiles/traffic.csv (stamp {r[3]}, now {now}): "
                              "re-capture with ncu --set full and update the row")
            return float(r[1]), None
    return None, f"profiles/traffic.csv has no row for {kernel_class}"


def time_recon(cb, dev, st, name, eq2=False, synthetic_noise_only=False, operators=False):
    """Seconds per full reconstruction of config `name` at its own level and iteration counts (c1: 1 x 20 outer x 5 inner;
    c3 / c4: 2 / 3 levels x 100 x 10; c5: 3 levels x 50 x 10), device-resident data, CUDA events on the launching stream, after
    a short warm-up cascade that makes every allocation.  synthetic_noise_only (c5): the 363 projections of 1024 x 768 are
    uniform noise made on the device instead of line integrals of the phantom (a minute of host time saved; with fixed
    iteration counts the kernels' work does not depend on the values).  operators: also returns projector / backprojector GUPS
    at that size (mean of 2 applications each)."""
    import torch
    from cbct_synth import make_config
    cfg = make_config(name)
    g = cfg.geom
    if synthetic_noise_only:
        Y = torch.rand(g.proj_shape, device=dev) * 20.0
    else:
        Y = torch.from_numpy(np.ascontiguousarray(cfg.projections(), dtype=np.float32)).to(dev)
    G = cb.Geometry.from_synth(g)
    if eq2:
        cb.set_backprojector(G, cb.BACKPROJECTOR_EQ2)
    f = torch.empty(g.vol_shape, device=dev)
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with torch.cuda.stream(st):
        cb.fbs_reconstruct(G, Y, None, cfg.n_levels, [2] * cfg.n_levels, cfg.n_inner, cfg.step, cfg.mu, cfg.eps, cfg.omega, f, stream=st)
        a.record(st)
        cb.fbs_reconstruct(G, Y, None, cfg.n_levels, cfg.n_outer, cfg.n_inner, cfg.step, cfg.mu, cfg.eps, cfg.omega, f, stream=st)
        b.record(st)
    torch.cuda.synchronize()
    sec = a.elapsed_time(b) / 1e3
    ops = None
    if operators:
        q = torch.empty(g.proj_shape, device=dev)
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
        with torch.cuda.stream(st):
            cb.forward(G, f, q, stream=st)
            cb.backproject(G, q, f, stream=st)
            ev[0].record(st)
            for _ in range(2):
                cb.forward(G, f, q, stream=st)
            ev[1].record(st)
            for _ in range(2):
                cb.backproject(G, q, f, stream=st)
            ev[2].record(st)
        torch.cuda.synchronize()
        upd = float(g.n_vox) * g.n_angles
        ops = (upd / (ev[0].elapsed_time(ev[1]) / 2e3) / 1e9, upd / (ev[1].elapsed_time(ev[2]) / 2e3) / 1e9)
    G.close()
    return (sec, ops) if operators else sec


def time_c3_recon(cb, dev, st, eq2=False):
    """seconds per full c3 reconstruction (2 levels x 100 outer x 10 inner; noisy 40-view data)."""
    return time_recon(cb, dev, st, "c3", eq2=eq2)


def time_c3_recon_host(cb, dev, st):
    """Seconds per full c3 reconstruction END TO END through cbct_fbs_reconstruct_host, the call a user with host data makes:
    pinned host buffers, the upload of Y (31.5 MB) and the download of f (67 MB) inside the timed region, host clock around the
    call (it returns after synchronising its stream); second of two calls (the first makes the allocations)."""
    import torch
    from cbct_synth import make_config
    cfg = make_config("c3")
    g = cfg.geom
    h_Y = torch.from_numpy(np.ascontiguousarray(cfg.projections(), dtype=np.float32)).pin_memory()
    h_f = torch.empty(g.vol_shape, dtype=torch.float32).pin_memory()
    G = cb.Geometry.from_synth(g)
    args = (cfg.n_inner, cfg.step, cfg.mu, cfg.eps, cfg.omega)
    cb.fbs_reconstruct_host(G, h_Y, None, cfg.n_levels, [2] * cfg.n_levels, *args, h_f, stream=st)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    cb.fbs_reconstruct_host(G, h_Y, None, cfg.n_levels, cfg.n_outer, *args, h_f, stream=st)
    sec = time.perf_counter() - t0
    G.close()
    return sec, int(h_Y.numel() * 4), int(h_f.numel() * 4)


def time_tv_512(cb, dev, st, flush):
    """GB/s (12 B per voxel and sweep) of 10 TV-prox sweeps on a 512^3 volume of 0.5 mm voxels (c5's shape), L2 flushed first."""
    import torch
    G = cb.Geometry(1000.0, 1500.0, np.array([0.0]), 8, 8, 1.0, 1.0, 512, 512, 512, 0.5, 0.5, 0.5)
    gv = torch.rand((512, 512, 512), device=dev) * 0.02
    u = gv.clone()
    best = None
    with torch.cuda.stream(st):
        for _ in range(4):
            flush.fill_(1)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(st)
            cb.tv_prox(G, gv, u, 4.0e4, 1e-4, 1.0, 10, stream=st)
            b.record(st)
            st.synchronize()
            t = a.elapsed_time(b)
            best = t if best is None else min(best, t)
    G.close()
    return 12.0 * 512 ** 3 * 10 / best / 1e6


def time_c3_fdk(cb, dev, st):
    import torch
    from cbct_synth import make_config
    cfg = make_config("c3")
    g = cfg.geom
    Y = torch.from_numpy(np.ascontiguousarray(cfg.projections(), dtype=np.float32)).to(dev)
    G = cb.Geometry.from_synth(g)
    f = torch.empty(g.vol_shape, device=dev)
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with torch.cuda.stream(st):
        cb.fdk_reconstruct(G, Y, f, stream=st)
        a.record(st)
        cb.fdk_reconstruct(G, Y, f, stream=st)
        b.record(st)
    torch.cuda.synchronize()
    G.close()
    return a.elapsed_time(b) / 1e3


def oracle_step(cfg, g, Y, f):
    """One fine-level FBS outer iteration with the oracle as it stands."""
    import oracle as o
    return o.fbs_reconstruct(g, Y, f, 1, [1], N_INNER, cfg.step, cfg.mu, cfg.eps, cfg.omega)


def cpu_baseline_sample(cfg, n_angles=8, steps=1, warmup=0):
    """The oracle timed on this box's host cores on a bounded sample of the workload: one fine-level
    outer iteration (P, P^T, 10 TV sweeps, clamp) of c2 restricted to `n_angles` of its 40 views."""
    import oracle as o
    g = cfg.geom
    idx = np.linspace(0, g.n_angles, n_angles, endpoint=False).astype(int)
    gs = g.with_angles(g.angles[idx])
    Y = cfg.clean_projections(idx)
    f = np.zeros(gs.vol_shape)
    for _ in range(warmup):
        f = oracle_step(cfg, gs, Y, f)
    t0 = time.perf_counter()
    for _ in range(steps):
        f = oracle_step(cfg, gs, Y, f)
    dt = (time.perf_counter() - t0) / steps
    updates = 2.0 * gs.n_vox * gs.n_angles
    return {"value": updates / dt / 1e9, "unit": UNIT, "cores": o.num_threads(), "kind": "oracle",
            "seconds_per_sample_step": dt,
            "sample": f"one fine-level FBS outer iteration (P, P^T, {N_INNER} TV sweeps, clamp) on {n_angles} of the 40 "
                      f"views of c2 at full 256^3 volume size, fp64, OpenMP"}


def run_ops_only(args):
    """--ops-only NAME: one projection, one exact backprojection and one TV sweep at the size of config NAME (plus one TV sweep
    on a 512^3 volume for c5), after one untimed application of each, and nothing else.  Not a bench line: this is the
    command the ncu captures at sizes that leave L2 are taken from (profiles/r03_*); it prints the three event times."""
    import torch
    import paper_1002_3675_b200 as cb
    from cbct_synth import make_config
    dev = torch.device("cuda:0")
    torch.cuda.set_device(dev)
    g = make_config(args.ops_only).geom
    G = cb.Geometry.from_synth(g)
    f = torch.rand(g.vol_shape, device=dev) * 0.02
    u = f.clone()
    q = torch.empty(g.proj_shape, device=dev)
    b = torch.empty(g.vol_shape, device=dev)
    st = torch.cuda.Stream()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
    with torch.cuda.stream(st):
        for timed in (False, True):
            if timed:
                ev[0].record(st)
            cb.forward(G, f, q, stream=st)
            if timed:
                ev[1].record(st)
            cb.backproject(G, q, b, stream=st)
            if timed:
                ev[2].record(st)
            cb.tv_prox(G, f, u, 4.0e4, 1e-4, 1.0, 1, stream=st)
            if timed:
                ev[3].record(st)
    torch.cuda.synchronize()
    ms = [ev[k].elapsed_time(ev[k + 1]) for k in range(3)]
    upd = float(g.n_vox) * g.n_angles
    print(json.dumps({"ops_only": args.ops_only, "dims": [g.nx, g.ny, g.nz, g.n_angles, g.nu, g.nv],
                      "ms_forward": ms[0], "ms_backproject": ms[1], "ms_tv_sweep": ms[2],
                      "gups_forward": upd / ms[0] / 1e6, "gups_backproject": upd / ms[1] / 1e6,
                      "tv_GBps": 12.0 * g.n_vox / ms[2] / 1e6}))
    G.close()


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores; each step a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from cbct_synth import make_config
    cfg = make_config("c2")
    total = max(args.steps + args.warmup, 1)
    n_angles = int(max(1, min(40, round(40 * 150.0 / (total * 45.0)))))      # ~45 s per full 40-view step on 8 cores
    cpu = cpu_baseline_sample(cfg, n_angles=n_angles, steps=args.steps, warmup=args.warmup)
    line = {
        "impl": "reference", "metric": METRIC, "value": cpu["value"], "unit": UNIT, "n_gpus": int(os.environ.get("WORLD_SIZE", "1")),
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * cpu["seconds_per_sample_step"],
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "c2 (bounded sample): " + cpu["sample"]},
        "cpu_baseline": cpu,
        "e2e": {"value": cpu["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def launch_ranks(n: int) -> int:
    """`bench.py --gpus N` started by hand (no RANK in the environment): re-run this command as N ranks, one per GPU, under
    torch.distributed.run on this node (rendezvous on 127.0.0.1, a free port), exactly as the driver launches it."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "INFO")                       # the communicator log shows the ranks (and NVLS, if used)
    env.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd, env=env)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--no-cpu", action="store_true", help="skip the oracle cpu_baseline leg")
    ap.add_argument("--no-recon", action="store_true", help="skip the full c3 reconstruction timing")
    ap.add_argument("--no-c5", action="store_true", help="skip the c5 (512^3, 363 views) reconstruction and operator timing (~30 s)")
    ap.add_argument("--ops-only", default="", metavar="CONFIG",
                    help="one projection, backprojection and TV sweep at the size of a config (c2..c5) and exit: the ncu target of profiles/r03_*")
    ap.add_argument("--cpu-angles", type=int, default=8)
    ap.add_argument("--shard-angles", action="store_true",
                    help="NEXT-4: shard the views of ONE reconstruction over the ranks (strong scaling) instead of replicas")
    ap.add_argument("--staged-projector", action="store_true",
                    help="measured variant: the TMA-staged projector (cbct_set_projector_staging) instead of the cached march")
    ap.add_argument("--plain-kernels", action="store_true",
                    help="measured variant: the plain march and gather (cbct_set_mirror_symmetry off) instead of the mirrored ones")
    ap.add_argument("--rank-probe", action="store_true",
                    help="every rank prints its RANK/LOCAL_RANK/WORLD_SIZE and exits (checks the launcher without a GPU)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "cuda" else args.warmup
    if args.gpus > 1 and "RANK" not in os.environ and args.impl == "cuda":
        raise SystemExit(launch_ranks(args.gpus))              # one process per GPU; rank 0 prints the JSON line
    if args.rank_probe:
        print(json.dumps({k: os.environ.get(k) for k in ("RANK", "LOCAL_RANK", "WORLD_SIZE", "MASTER_ADDR", "MASTER_PORT")}
                         | {"mode": "shard-angles" if args.shard_angles else "replicas"}), flush=True)
        return
    if args.impl == "reference":
        run_reference(args)
    elif args.shard_angles:
        run_sharded(args)
    elif args.ops_only:
        run_ops_only(args)
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()
