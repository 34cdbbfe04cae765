"""Parity at BASELINE.json's full sizes (c2..c5), in the launch configuration bench.py times, on
sampled outputs the oracle computes one by one (single rays by traversal, single voxels by brute-force
clipping), plus properties that hold at any size and one full-size loop iteration for c3."""
import numpy as np
import pytest

import oracle as o
from cbct_synth import make_config, gaussian_field

pytestmark = pytest.mark.gpu


def f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def rel(a, b):
    a = np.asarray(a, dtype=np.float64)
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))


def sampled_operator_parity(cb, cfg, n_rays=4000, n_vox=600, angle_subset=None, adjoint=True, vol=None):
    import torch
    dev = torch.device("cuda:0")
    g = cfg.geom if angle_subset is None else cfg.geom.with_angles(cfg.geom.angles[angle_subset])
    G = cb.Geometry.from_synth(g)
    vol = f32(cfg.volume()) if vol is None else vol
    d_vol = torch.from_numpy(vol).to(dev)
    d_q = torch.empty(g.proj_shape, device=dev)
    cb.forward(G, d_vol, d_q)
    rng = np.random.default_rng(cfg.seed + 99)
    ia, iv, iu = rng.integers(g.n_angles, size=n_rays), rng.integers(g.nv, size=n_rays), rng.integers(g.nu, size=n_rays)
    # include detector corners / edges and tile boundaries
    iv[:8] = [0, 0, g.nv - 1, g.nv - 1, g.nv // 2, g.nv // 2 - 1, 31, 32]
    iu[:8] = [0, g.nu - 1, 0, g.nu - 1, g.nu // 2, g.nu // 2 - 1, 31, 32]
    q = d_q.cpu().numpy()
    ref = o.forward_rays(g, vol.astype(np.float64), ia, iv, iu)
    e_fwd = rel(q[ia, iv, iu], ref)
    # backproject P(phantom); sampled voxels by brute-force clipping
    d_b = torch.empty(g.vol_shape, device=dev)
    cb.backproject(G, d_q, d_b)
    ix, iy, iz = rng.integers(g.nx, size=n_vox), rng.integers(g.ny, size=n_vox), rng.integers(g.nz, size=n_vox)
    ix[:6] = [0, g.nx - 1, 0, g.nx // 2, 31, 32]
    iy[:6] = [0, g.ny - 1, g.ny - 1, g.ny // 2, 32, 31]
    iz[:6] = [0, g.nz - 1, g.nz // 2, 0, 15, 16]
    b = d_b.cpu().numpy()
    bref = o.backproject_voxels(g, q.astype(np.float64), ix, iy, iz)
    e_bp = rel(b[iz, iy, ix], bref)
    e_adj = None
    if adjoint:
        x = torch.from_numpy(f32(gaussian_field(g.vol_shape, 11))).to(dev)
        y = torch.from_numpy(f32(gaussian_field(g.proj_shape, 12))).to(dev)
        Px = torch.empty(g.proj_shape, device=dev)
        Pty = torch.empty(g.vol_shape, device=dev)
        cb.forward(G, x, Px)
        cb.backproject(G, y, Pty)
        lhs = float((Px.double() * y.double()).sum())
        rhs = float((x.double() * Pty.double()).sum())
        e_adj = abs(lhs - rhs) / (float(Px.double().norm()) * float(y.double().norm()))
    G.close()
    return e_fwd, e_bp, e_adj


def test_c2_operator_bench_config(cuda_lib):
    """configs[1]: 256^3 volume, 40 views of 512x384 — the workload bench.py times."""
    e_fwd, e_bp, e_adj = sampled_operator_parity(cuda_lib, make_config("c2"))
    assert e_fwd <= 1e-5 and e_bp <= 1e-5 and e_adj <= 1e-5, (e_fwd, e_bp, e_adj)


def maxerr(a, b):
    a = np.asarray(a, dtype=np.float64)
    return float(np.abs(a - b).max() / max(np.abs(b).max(), 1e-300))


def test_c2_every_ray_and_every_voxel(cuda_lib):
    """The benchmarked config in full, not a sample: all 7.86 M rays of P(phantom) and all 16.8 M voxels of P^T(P(phantom))
    against the oracle (about 20 s of oracle time on 16 cores), rel-L2 <= 1e-5 and every element within 1e-4 of the largest
    (K_MAX * TOL_OP of tests/test_gpu_parity.py), in the launch configuration bench.py times (default kernels)."""
    import torch
    cb = cuda_lib
    dev = torch.device("cuda:0")
    cfg = make_config("c2")
    g = cfg.geom
    G = cb.Geometry.from_synth(g)
    vol = f32(cfg.volume())
    d_q = torch.empty(g.proj_shape, device=dev)
    d_b = torch.empty(g.vol_shape, device=dev)
    cb.forward(G, torch.from_numpy(vol).to(dev), d_q)
    cb.backproject(G, d_q, d_b)
    q, b = d_q.cpu().numpy(), d_b.cpu().numpy()
    G.close()
    q_ref = o.forward(g, vol.astype(np.float64))
    b_ref = o.backproject(g, q.astype(np.float64))
    print(f"PARITY c2 whole arrays: P {rel(q, q_ref):.2e} / max {maxerr(q, q_ref):.2e}   Pt {rel(b, b_ref):.2e} / max {maxerr(b, b_ref):.2e}")
    assert np.linalg.norm(q_ref) > 0 and np.linalg.norm(b_ref) > 0
    assert rel(q, q_ref) <= 1e-5 and maxerr(q, q_ref) <= 1e-4
    assert rel(b, b_ref) <= 1e-5 and maxerr(b, b_ref) <= 1e-4
    # rays that miss the volume: exactly where the oracle has zeros, up to grazing rays (a few 1e-7 of a voxel)
    assert np.all(np.abs(q[q_ref == 0.0]) <= 1e-6 * np.abs(q_ref).max())


@pytest.mark.parametrize("name", ["c3", "c4"])
def test_c3_c4_operators_full_size(cuda_lib, name):
    e_fwd, e_bp, e_adj = sampled_operator_parity(cuda_lib, make_config(name))
    assert e_fwd <= 1e-5 and e_bp <= 1e-5 and e_adj <= 1e-5, (e_fwd, e_bp, e_adj)


def test_c3_one_full_size_outer_iteration(cuda_lib):
    """One outer FBS iteration at the full c3 size (finest level, warm start) against the oracle."""
    import torch
    cb = cuda_lib
    dev = torch.device("cuda:0")
    cfg = make_config("c3")
    g = cfg.geom
    G = cb.Geometry.from_synth(g)
    Y = f32(cfg.projections())
    f0 = f32(0.7 * cfg.volume())
    f = torch.empty(g.vol_shape, device=dev)
    cb.fbs_reconstruct(G, torch.from_numpy(Y).to(dev), torch.from_numpy(f0).to(dev), 1, [1], cfg.n_inner,
                       cfg.step, cfg.mu, cfg.eps, cfg.omega, f)
    ref = o.fbs_reconstruct(g, Y.astype(np.float64), f0.astype(np.float64), 1, [1], cfg.n_inner, cfg.step, cfg.mu,
                            cfg.eps, cfg.omega)
    out = f.cpu().numpy()
    assert rel(out, ref) <= 1e-4
    # the update itself (not just f0 carried over) matches
    assert rel(out - f0, ref - f0.astype(np.float64)) <= 2e-4
    assert out.min() >= 0.0
    G.close()


@pytest.mark.parametrize("name,n_outer", [("c3", [15, 15]), ("c4", [25, 25, 25])])
def test_full_size_cascade_many_iterations(cuda_lib, name, n_outer):
    """The c3 / c4 cascades at their FULL sizes (512x512x64, 40 / 20 noisy views of 512x384, all multigrid levels), with
    enough outer iterations per level to see the fp32 error accumulate (the full 100 per level run once under
    CBCT_FULL_COUNT=1, tests/test_gpu_fullcount.py; its growth table is in DESIGN.md)."""
    import torch
    cb = cuda_lib
    dev = torch.device("cuda:0")
    cfg = make_config(name)
    g = cfg.geom
    G = cb.Geometry.from_synth(g)
    Y = f32(cfg.projections())
    f = torch.empty(g.vol_shape, device=dev)
    cb.fbs_reconstruct(G, torch.from_numpy(Y).to(dev), None, cfg.n_levels, n_outer, cfg.n_inner, cfg.step, cfg.mu, cfg.eps,
                       cfg.omega, f)
    ref = o.fbs_reconstruct(g, Y.astype(np.float64), None, cfg.n_levels, n_outer, cfg.n_inner, cfg.step, cfg.mu, cfg.eps,
                            cfg.omega)
    out = f.cpu().numpy()
    assert np.linalg.norm(ref) > 0 and rel(out, ref) <= 1e-4
    assert out.min() >= 0.0
    G.close()


_C5 = {}


def c5_config():
    if "cfg" not in _C5:
        _C5["cfg"] = make_config("c5")
        _C5["vol"] = f32(_C5["cfg"].volume())
    return _C5["cfg"]


@pytest.mark.parametrize("first", [3, 0, 17, 31])
def test_c5_operator_subsets(cuda_lib, first):
    """c5 (512^3, 360 views of 1024x768): operator parity on 8-angle subsets {first + 45 m} (row blocks of P and partial
    sums of P^T are exact sub-problems).  first = 0 holds the axis-aligned views and the 45-degree views where the ray class
    changes inside a projection."""
    cfg = c5_config()
    subset = np.arange(0, 360, 45) + first
    e_fwd, e_bp, e_adj = sampled_operator_parity(cuda_lib, cfg, n_rays=3000, n_vox=400, angle_subset=subset, vol=_C5["vol"])
    print(f"c5 subset {first}: forward {e_fwd:.2e} backproject {e_bp:.2e} adjoint {e_adj:.2e}")
    assert e_fwd <= 1e-5 and e_bp <= 1e-5 and e_adj <= 1e-5, (e_fwd, e_bp, e_adj)


def test_c5_tv_full_volume(cuda_lib):
    """TV parity on the full 512^3 volume."""
    import torch
    cb = cuda_lib
    dev = torch.device("cuda:0")
    cfg = c5_config()
    g = cfg.geom.with_angles(cfg.geom.angles[:1])
    G = cb.Geometry.from_synth(g)
    rng = np.random.default_rng(77)
    gv = f32(_C5["vol"] + 0.002 * rng.standard_normal(g.vol_shape, dtype=np.float32))
    d_g = torch.from_numpy(gv).to(dev)
    u = d_g.clone()
    cb.tv_prox(G, d_g, u, cfg.beta, cfg.eps, 1.0, 2)
    ref = o.tv_prox(g, gv.astype(np.float64), gv.astype(np.float64), cfg.beta, cfg.eps, 1.0, 2)
    assert rel(u.cpu().numpy(), ref) <= 1e-5
    G.close()


def test_c3_eq2_backprojector_full_size(cuda_lib):
    """NEXT-1 at the full c3 size (512x512x64, 40 views of 512x384): the paper's eq. 2 backprojection of P(phantom)
    against the oracle, every voxel."""
    import torch
    cb = cuda_lib
    dev = torch.device("cuda:0")
    cfg = make_config("c3")
    g = cfg.geom
    G = cb.Geometry.from_synth(g)
    d_q = torch.empty(g.proj_shape, device=dev)
    cb.forward(G, torch.from_numpy(f32(cfg.volume())).to(dev), d_q)
    d_b = torch.empty(g.vol_shape, device=dev)
    cb.backproject_eq2(G, d_q, d_b)
    ref = o.backproject_eq2(g, d_q.cpu().numpy().astype(np.float64))
    assert rel(d_b.cpu().numpy(), ref) <= 1e-5
    G.close()


def test_c5_coarsest_level_two_outer_iterations(cuda_lib):
    """c5's loop: the full-size oracle is infeasible, so the first 2 outer iterations at the size
    of its coarsest level (128^3 voxels of 2 mm, 360 views of 256x192, the same scene) against the oracle."""
    import torch
    cb = cuda_lib
    dev = torch.device("cuda:0")
    cfg = make_config("c5", shrink=4)
    g = cfg.geom
    assert (g.nx, g.ny, g.nz, g.n_angles, g.nu, g.nv) == (128, 128, 128, 360, 256, 192)
    G = cb.Geometry.from_synth(g)
    Y = f32(cfg.projections())
    f = torch.empty(g.vol_shape, device=dev)
    cb.fbs_reconstruct(G, torch.from_numpy(Y).to(dev), None, 1, [2], cfg.n_inner, cfg.step, cfg.mu, cfg.eps, cfg.omega, f)
    ref = o.fbs_reconstruct(g, Y.astype(np.float64), None, 1, [2], cfg.n_inner, cfg.step, cfg.mu, cfg.eps, cfg.omega)
    assert np.linalg.norm(ref) > 0 and rel(f.cpu().numpy(), ref) <= 1e-4
    G.close()
