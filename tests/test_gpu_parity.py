"""Parity of the CUDA path (through the C ABI) against the fp64 oracle, element by element on the
same seeded inputs.  Tolerances are the north_star's: rel-L2 <= 1e-5 per operator (forward on a
voxelised phantom, backproject on P(phantom), tv_prox on a seeded noisy phantom), <= 1e-4 on the
reconstruction after the fixed iteration count, adjoint identity <= 1e-5 on Gaussian x, y.
All inputs are rounded to fp32 first so that both sides see identical numbers."""
import numpy as np
import pytest

import oracle as o
from cbct_synth import Geometry, make_config, gaussian_field
from cbct_synth.geometry import equispaced_angles

pytestmark = pytest.mark.gpu

TOL_OP = 1e-5
TOL_RECON = 1e-4
TOL_ADJ = 1e-5


def f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def rel(a, b):
    a = np.asarray(a, dtype=np.float64)
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))


def maxerr(a, b):
    """Largest element error over the largest element of the oracle's array (the per-element companion of rel)."""
    a = np.asarray(a, dtype=np.float64)
    return float(np.abs(a - b).max() / max(np.abs(b).max(), 1e-300))


# Per-element bound beside every operator rel-L2: max|gpu - oracle| <= K_MAX * TOL_OP * max|oracle|.  rel-L2 at 1e-5 sees one
# element that is 10 % off among 1e7 but not one that is 1 % off; this bound does (K_MAX * TOL_OP = 1e-4 of the largest
# element).  K_MAX = 10: fp32 sums of a few hundred chord * value products carry element errors of a few 1e-7 of the largest
# element on smooth inputs and up to ~5e-6 on Gaussian ones (printed by the tests, recorded in DESIGN.md "Tolerances").
K_MAX = 10.0


@pytest.fixture(scope="module")
def dev(cuda_lib):
    import torch
    return torch.device("cuda:0")


def to_dev(a, dev):
    import torch
    return torch.from_numpy(f32(a)).to(dev)


def run_forward(cb, G, vol, dev):
    import torch
    q = torch.empty(G.proj_shape, device=dev)
    cb.forward(G, to_dev(vol, dev), q)
    torch.cuda.synchronize()
    return q.cpu().numpy()


def run_backproject(cb, G, y, dev):
    import torch
    b = torch.empty(G.vol_shape, device=dev)
    cb.backproject(G, to_dev(y, dev), b)
    torch.cuda.synchronize()
    return b.cpu().numpy()


GEOMS = {
    # spans several 32-wide u tiles, 32-row v groups and 16-deep k chunks, with ragged tails
    "c1": lambda: make_config("c1").geom,
    "aniso_ragged": lambda: Geometry(1000., 1500., equispaced_angles(7) + 0.123, 50, 38, 1.3, 1.7, 40, 36, 20, 1.0, 1.25, 2.5),
    "odd_dims_axis_angles": lambda: Geometry(1000., 1500., np.array([0.0, np.pi / 4, np.pi / 2, 3.0, -2.2]), 33, 21, 2.0, 2.0, 31, 29, 17, 2.0, 2.0, 2.0),
    "wide_detector_misses": lambda: Geometry(1000., 1500., equispaced_angles(5) + 0.4, 70, 45, 4.0, 6.0, 24, 24, 12, 2.0, 2.0, 2.0),
    "short_arc_200deg": lambda: Geometry(1000., 1500., np.deg2rad(np.linspace(-10.0, 190.0, 9)), 48, 40, 2.0, 2.0, 36, 36, 40, 1.5, 1.5, 1.5),
    # detector rows 100x finer than the slices: several rays of a column cross one z plane inside a slab (the gather's loop)
    "fine_rows_multicross": lambda: Geometry(1000., 1500., np.array([0.2, 1.9, 4.0]), 20, 2400, 3.0, 0.02, 16, 16, 16, 2.0, 2.0, 2.0),
    # 25 detector columns per voxel row (long candidate loops), and a detector so coarse that rays skip voxel rows
    "fine_columns": lambda: Geometry(1000., 1500., np.array([0.5, 2.4]), 600, 12, 0.12, 4.0, 16, 16, 8, 2.0, 2.0, 3.0),
    "coarse_detector": lambda: Geometry(1000., 1500., equispaced_angles(6) + 0.1, 9, 7, 9.0, 11.0, 24, 24, 16, 1.5, 1.5, 2.0),
    # degenerate sizes: a single slice, a single detector row, one voxel column
    "one_slice_one_row": lambda: Geometry(1000., 1500., np.array([0.3, 2.0]), 24, 1, 2.0, 2.0, 12, 10, 1, 2.0, 2.0, 2.0),
    "one_column": lambda: Geometry(1000., 1500., np.array([0.0, 1.0, 2.5]), 6, 30, 1.0, 1.0, 1, 1, 24, 2.0, 2.0, 1.0),
    "single_angle": lambda: Geometry(1000., 1500., np.array([0.77]), 40, 40, 2.0, 2.0, 32, 32, 32, 1.5, 1.5, 1.5),
    # odd nv with even nz: the central detector row lies exactly in the voxel plane k = nz/2 (reading Q15: it belongs to the
    # row above); 40 detector rows per slice, so the run bounds of that plane sit in a higher binade than the row index
    "odd_rows_even_slices": lambda: Geometry(1000., 1500., np.array([0.1, 0.9, 2.3, 4.4]), 24, 401, 2.5, 0.05, 20, 20, 16, 2.0, 2.0, 2.0),
    # angle lists closed under + 180 degrees (the march takes half-turn twins along): ragged and odd in-plane sizes, a detector
    # wider than the volume's shadow (twins read the zero pads on the other side), detector offset in u (allowed: the half turn
    # maps pixel u onto itself)
    "twin_ragged": lambda: Geometry(1000., 1500., equispaced_angles(8) + 0.3, 50, 38, 1.3, 1.7, 40, 36, 20, 1.0, 1.25, 2.5),
    "twin_odd_xy": lambda: Geometry(1000., 1500., equispaced_angles(10) + 0.05, 45, 30, 2.0, 2.0, 31, 29, 18, 2.0, 2.0, 2.0),
    "twin_wide": lambda: Geometry(1000., 1500., equispaced_angles(6) + 0.2, 70, 44, 4.0, 6.0, 24, 24, 12, 2.0, 2.0, 2.0),
    "odd_rows_even_slices_coarse": lambda: Geometry(1000., 1500., equispaced_angles(5) + 0.05, 40, 33, 2.0, 2.0, 24, 24, 12, 2.0, 2.0, 2.0),
}


def smooth_phantom(g, seed):
    """A phantom-like volume for any geometry: a few seeded ellipsoids, voxelised."""
    from cbct_synth import random_ellipsoids, voxelize
    ext = (g.nx * g.hx, g.ny * g.hy, g.nz * g.hz)
    ells = random_ellipsoids(np.random.default_rng(seed), 6, ext, (0.1 * min(ext), 0.3 * min(ext)))
    return voxelize(ells, g)


@pytest.mark.parametrize("name", list(GEOMS))
def test_forward_backproject_adjoint(cuda_lib, dev, name):
    cb = cuda_lib
    g = GEOMS[name]()
    G = cb.Geometry.from_synth(g)
    vol = f32(smooth_phantom(g, 3) if name != "c1" else make_config("c1").volume())
    q = run_forward(cb, G, vol, dev)
    q_ref = o.forward(g, vol.astype(np.float64))
    assert rel(q, q_ref) <= TOL_OP and maxerr(q, q_ref) <= K_MAX * TOL_OP
    # rays that miss the volume give 0 (a ray grazing an edge within fp32 rounding may leave ~1e-7 of a voxel)
    assert np.all(np.abs(q[q_ref == 0.0]) <= 1e-6 * np.abs(q_ref).max())
    assert np.count_nonzero(q[q_ref == 0.0]) <= 0.01 * max(1, np.count_nonzero(q_ref == 0.0))
    b = run_backproject(cb, G, q, dev)                         # backproject on P(phantom)
    b_ref = o.backproject(g, q.astype(np.float64))
    assert rel(b, b_ref) <= TOL_OP and maxerr(b, b_ref) <= K_MAX * TOL_OP
    # adjoint identity on seeded Gaussian x, y (dot products in fp64)
    x = f32(gaussian_field(g.vol_shape, 11))
    y = f32(gaussian_field(g.proj_shape, 12))
    Px = run_forward(cb, G, x, dev).astype(np.float64)
    Pty = run_backproject(cb, G, y, dev).astype(np.float64)
    lhs, rhs = np.vdot(Px, y.astype(np.float64)), np.vdot(x.astype(np.float64), Pty)
    assert abs(lhs - rhs) / (np.linalg.norm(Px) * np.linalg.norm(y)) <= TOL_ADJ
    # Gaussian inputs are the worst case for fp32 chord boundaries (no smoothness to average the boundary errors out)
    Px_ref, Pty_ref = o.forward(g, x.astype(np.float64)), o.backproject(g, y.astype(np.float64))
    print(f"PARITY {name}: P phantom {rel(q, q_ref):.1e}/{maxerr(q, q_ref):.1e}  Pt {rel(b, b_ref):.1e}/{maxerr(b, b_ref):.1e}  "
          f"P gauss {rel(Px, Px_ref):.1e}/{maxerr(Px, Px_ref):.1e}  Pt gauss {rel(Pty, Pty_ref):.1e}/{maxerr(Pty, Pty_ref):.1e}")
    # The gather places its crossings with two-float positions and holds the operator bound on white noise as well (measured
    # 6e-8 .. 5e-7).  The march reads fp32 ray tables: a chord boundary sits up to ~3e-5 voxel off, which smooth volumes
    # average out (1e-7 .. 2.5e-6 above) and white noise does not: measured 5e-7 .. 8e-6, 2.8e-5 on the one-column detector
    # (no neighbouring columns to share a boundary error with).  Stated bound for the march on white noise: 5e-5 (DESIGN.md
    # "Tolerances"; SURVEY.md section 7 anticipated it).
    TOL_MARCH_NOISE = 5e-5
    assert rel(Px, Px_ref) <= TOL_MARCH_NOISE and maxerr(Px, Px_ref) <= K_MAX * TOL_MARCH_NOISE
    assert rel(Pty, Pty_ref) <= TOL_OP and maxerr(Pty, Pty_ref) <= K_MAX * TOL_OP
    G.close()


@pytest.mark.parametrize("name", ["c1", "aniso_ragged", "odd_dims_axis_angles", "wide_detector_misses", "short_arc_200deg", "fine_rows_multicross",
                                  "fine_columns", "coarse_detector", "one_slice_one_row", "one_column", "odd_rows_even_slices"])
def test_tma_staged_projector_equals_the_cached_march(cuda_lib, dev, name):
    """The TMA-staged projector (cbct_set_projector_staging, csrc/projector_tma.cu) marches the same rays with the same
    arithmetic in the same order: bit-identical to the default kernel, in all three output modes (through the loop)."""
    import torch
    cb = cuda_lib
    g = GEOMS[name]()
    vol = f32(smooth_phantom(g, 3) if name != "c1" else make_config("c1").volume())
    G0, G1 = cb.Geometry.from_synth(g), cb.Geometry.from_synth(g)
    G0.set_mirror_symmetry(False)                  # the plain march (the symmetric marches use one ray's table entries for its images)
    G1.set_mirror_symmetry(False)
    G1.set_projector_staging(True)
    q0, q1 = torch.empty(G0.proj_shape, device=dev), torch.empty(G0.proj_shape, device=dev)
    cb.forward(G0, to_dev(vol, dev), q0)
    cb.forward(G1, to_dev(vol, dev), q1)
    assert torch.equal(q0, q1)
    assert rel(q1.cpu().numpy(), o.forward(g, vol.astype(np.float64))) <= TOL_OP
    Y = to_dev(0.9 * q0.cpu().numpy() + 0.01, dev)
    d0, d1 = torch.empty(G0.vol_shape, device=dev), torch.empty(G0.vol_shape, device=dev)
    for mode in (cb.BACKPROJECTOR_EXACT, cb.BACKPROJECTOR_EQ2):
        cb.set_backprojector(G0, mode); cb.set_backprojector(G1, mode)
        cb.data_gradient(G0, to_dev(vol, dev), Y, d0)
        cb.data_gradient(G1, to_dev(vol, dev), Y, d1)
        assert torch.equal(d0, d1)
    G0.close(); G1.close()


@pytest.mark.parametrize("name", ["c1", "aniso_ragged", "wide_detector_misses", "short_arc_200deg", "fine_rows_multicross", "fine_columns",
                                  "coarse_detector", "one_column", "odd_rows_even_slices", "odd_rows_even_slices_coarse",
                                  "twin_ragged", "twin_odd_xy", "twin_wide"])
def test_plain_kernels_equal_the_mirrored_kernels(cuda_lib, dev, name):
    """Scans that are their own mirror image about z = 0 (nz even, detector centred in v) are marched two rays and gathered
    two voxel rows at a time, and on angle lists closed under + 180 degrees the march also takes a ray's half-turn twin along
    (cbct_set_mirror_symmetry, the default); the plain kernels (forced here, and the only ones for odd nz or shifted panels)
    must give the same matrix: within the operator tolerance of the oracle and equal to each other to fp32 rounding, on
    phantom-like inputs and on Gaussian ones."""
    import torch
    cb = cuda_lib
    g = GEOMS[name]()
    assert g.nz % 2 == 0
    G = cb.Geometry.from_synth(g)
    vol = f32(smooth_phantom(g, 5) if name != "c1" else make_config("c1").volume())
    G.set_mirror_symmetry(False)
    q_p = run_forward(cb, G, vol, dev)
    G.set_mirror_symmetry(True)
    q_m = run_forward(cb, G, vol, dev)
    # the z-mirrored march repeats the plain arithmetic per ray (bit-identical); where the angle list is closed under + 180
    # degrees the march also takes the rays of angle a + 180 from the table entries of angle a (an equally good fp32 rounding
    # of the same ray): equal to a few 1e-7
    assert rel(q_m, q_p.astype(np.float64)) <= 0.5 * TOL_OP
    assert rel(q_m, o.forward(g, vol.astype(np.float64))) <= TOL_OP
    for y, tol in ((q_m, TOL_OP), (f32(gaussian_field(g.proj_shape, 21)), TOL_OP)):
        ref = o.backproject(g, y.astype(np.float64))
        G.set_mirror_symmetry(True)
        b_m = run_backproject(cb, G, y, dev)
        G.set_mirror_symmetry(False)
        b_p = run_backproject(cb, G, y, dev)
        assert rel(b_m, ref) <= tol and rel(b_p, ref) <= tol
        assert maxerr(b_m, ref) <= K_MAX * tol and maxerr(b_p, ref) <= K_MAX * tol
        assert rel(b_m, b_p.astype(np.float64)) <= 0.2 * tol          # both are one matrix: far closer to each other than to the bound
    # the loop (residual modes of the march, gradient step) agrees too
    Y = to_dev(0.9 * q_m + 0.01, dev)
    d = {}
    for sym in (True, False):
        G.set_mirror_symmetry(sym)
        d[sym] = torch.empty(G.vol_shape, device=dev)
        cb.data_gradient(G, to_dev(vol, dev), Y, d[sym])
    # (the residual P f - Y is a tenth of P f here, so a 1e-6 difference of the marches is a 1e-5 difference of the gradient)
    assert rel(d[True].cpu().numpy(), d[False].cpu().numpy().astype(np.float64)) <= 2e-5
    G.close()


def test_backproject_of_unit_projections_matches_brute_force_clip(cuda_lib, dev):
    """Exact adjoint, entry by entry: P^T applied to single-pixel images equals the matrix column
    the oracle gets by clipping that ray against each voxel box."""
    cb = cuda_lib
    g = GEOMS["aniso_ragged"]()
    G = cb.Geometry.from_synth(g)
    rng = np.random.default_rng(5)
    for _ in range(6):
        ia, iv, iu = rng.integers(g.n_angles), rng.integers(g.nv), rng.integers(g.nu)
        y = np.zeros(g.proj_shape, dtype=np.float32)
        y[ia, iv, iu] = 1.0
        b = run_backproject(cb, G, y, dev)
        kk, jj, ii = np.nonzero(b)
        ref = o.backproject(g, y.astype(np.float64))
        assert rel(b, ref) <= TOL_OP
        assert (ref > 0).sum() > 0 and np.count_nonzero(b[ref == 0.0] > 1e-5) == 0
    G.close()


@pytest.mark.parametrize("shape,h", [((64, 48, 40), (0.5, 0.5, 2.5)), ((33, 21, 10), (1.0, 2.0, 0.7)), ((8, 8, 8), (1.0, 1.0, 1.0)),
                                     # every instantiation of the row kernel: scalar rows (nx % 4 != 0) of 4, 8 and 16 voxels
                                     # per lane, vector rows of 4, 8, 16; and the tile kernel for nx > 512 (ragged and full tiles)
                                     ((102, 9, 7), (1.0, 1.0, 2.0)), ((130, 7, 6), (0.5, 0.5, 2.5)), ((258, 6, 5), (1.0, 1.0, 1.0)),
                                     ((100, 13, 9), (1.0, 1.0, 1.0)), ((200, 11, 5), (1.0, 1.0, 1.0)), ((512, 12, 6), (0.5, 0.5, 2.5)),
                                     ((320, 9, 7), (1.0, 1.0, 1.0)), ((36, 5, 3), (1.0, 1.0, 1.0)), ((256, 40, 21), (1.0, 1.0, 1.0)), ((448, 23, 9), (0.5, 0.5, 2.5)),
                                     ((516, 10, 9), (1.0, 1.0, 1.0)), ((1024, 9, 10), (0.5, 0.5, 0.5))])
def test_tv_prox(cuda_lib, dev, shape, h):
    import torch
    cb = cuda_lib
    nx, ny, nz = shape
    g = Geometry(1000., 1500., np.array([0.0]), 8, 8, 1.0, 1.0, nx, ny, nz, *h)
    G = cb.Geometry.from_synth(g)
    rng = np.random.default_rng(21)
    gv = f32(smooth_phantom(g, 8) + 0.002 * rng.normal(size=g.vol_shape))          # seeded noisy phantom
    for beta, eps, omega, n in [(3.0e4, 1e-4, 1.0, 5), (40.0, 1e-3, 1.0, 4), (40.0, 1e-3, 0.5, 1), (7.0, 1e-2, 1.0, 0)]:
        u = to_dev(gv, dev).clone()
        cb.tv_prox(G, to_dev(gv, dev), u, beta, eps, omega, n)
        torch.cuda.synchronize()
        ref = o.tv_prox(g, gv.astype(np.float64), gv.astype(np.float64), beta, eps, omega, n)
        assert rel(u.cpu().numpy(), ref) <= TOL_OP
        if n == 0:
            assert np.array_equal(u.cpu().numpy(), gv)
    # a different start u0 != g, and constants stay constant bit for bit (I7)
    u0 = f32(gv[::-1].copy())
    u = to_dev(u0, dev)
    cb.tv_prox(G, to_dev(gv, dev), u, 40.0, 1e-3, 1.0, 3)
    assert rel(u.cpu().numpy(), o.tv_prox(g, gv.astype(np.float64), u0.astype(np.float64), 40.0, 1e-3, 1.0, 3)) <= TOL_OP
    c = torch.full(g.vol_shape, 0.37, device=dev)
    u = c.clone()
    cb.tv_prox(G, c, u, 123.0, 1e-4, 1.0, 7)
    assert torch.equal(u, c)
    G.close()


def test_transfers_and_energy(cuda_lib, dev):
    import torch
    cb = cuda_lib
    for g in (make_config("c3", shrink=8).geom, make_config("c5", shrink=16).geom):
        G = cb.Geometry.from_synth(g)
        Gc, flags = G.coarsen()
        gc, ax, binned = o.coarsen_geometry(g)
        assert flags == tuple(ax) + (binned,)
        assert (Gc.nx, Gc.ny, Gc.nz, Gc.nu, Gc.nv) == (gc.nx, gc.ny, gc.nz, gc.nu, gc.nv)
        rng = np.random.default_rng(4)
        c = f32(rng.random(gc.vol_shape))
        f = torch.empty(g.vol_shape, device=dev)
        cb.prolong(G, to_dev(c, dev), f)
        assert rel(f.cpu().numpy(), o.prolong(c.astype(np.float64), ax)) <= 1e-6
        fine = f32(rng.random(g.vol_shape))
        cc = torch.empty(gc.vol_shape, device=dev)
        cb.restrict(G, to_dev(fine, dev), cc)
        assert rel(cc.cpu().numpy(), o.restrict_volume(fine.astype(np.float64), ax)) <= 1e-6
        Y = f32(rng.random(g.proj_shape))
        yc = torch.empty(gc.proj_shape, device=dev)
        cb.bin2x2(G, to_dev(Y, dev), yc)
        assert rel(yc.cpu().numpy(), o.bin2x2(Y.astype(np.float64))) <= 1e-6
        # energy
        vol = f32(smooth_phantom(g, 2))
        e = cb.energy(G, to_dev(vol, dev), to_dev(Y, dev), 3.5, 1e-3)
        e_ref = o.energy(g, vol.astype(np.float64), Y.astype(np.float64), 3.5, 1e-3)
        assert e["E_eps"] == pytest.approx(e_ref["E_eps"], rel=1e-5)
        assert e["E1_eps"] == pytest.approx(e_ref["E1_eps"], rel=1e-5)
        assert e["E2"] == pytest.approx(e_ref["E2"], rel=1e-5)
        G.close()
    with pytest.raises(cb.CbctError) as ei:                                       # odd dim on a coarsening axis
        cb.Geometry(1000., 1500., np.zeros(2), 8, 8, 1., 1., 9, 8, 8, 1., 1., 1.).coarsen()
    assert ei.value.status == 2


def test_fbs_c1_full_loop_with_energy_trace(cuda_lib, dev):
    """Config 1 end to end: 20 outer x 5 inner, 1 level; every recorded energy matches the oracle's."""
    import torch
    cb = cuda_lib
    cfg = make_config("c1")
    g = cfg.geom
    G = cb.Geometry.from_synth(g)
    Y = f32(cfg.projections())
    f = torch.empty(g.vol_shape, device=dev)
    tr = cb.fbs_reconstruct(G, to_dev(Y, dev), None, 1, cfg.n_outer, cfg.n_inner, cfg.step, cfg.mu, cfg.eps, cfg.omega, f, trace=True)
    tr_ref = []
    f_ref = o.fbs_reconstruct(g, Y.astype(np.float64), None, 1, cfg.n_outer, cfg.n_inner, cfg.step, cfg.mu, cfg.eps, cfg.omega, trace=tr_ref)
    out = f.cpu().numpy()
    assert rel(out, f_ref) <= TOL_RECON
    assert out.min() >= 0.0
    E_ref = np.array([t["E_eps"] for t in tr_ref])
    assert np.allclose(np.array(tr), E_ref, rtol=2e-5, atol=0)
    assert np.all(np.diff(np.array(tr)) < 0)                                      # monotone on this config (I9)
    # same call without the trace and through the host-buffer entry point give the same volume
    f2 = torch.empty_like(f)
    cb.fbs_reconstruct(G, to_dev(Y, dev), None, 1, cfg.n_outer, cfg.n_inner, cfg.step, cfg.mu, cfg.eps, cfg.omega, f2)
    assert torch.equal(f, f2)
    h_out = np.empty(g.vol_shape, dtype=np.float32)
    cb.fbs_reconstruct_host(G, Y, None, 1, cfg.n_outer, cfg.n_inner, cfg.step, cfg.mu, cfg.eps, cfg.omega, h_out)
    assert np.array_equal(h_out, out)
    G.close()


@pytest.mark.parametrize("name,shrink,n_levels,n_outer", [("c3", 4, 2, [30, 30]), ("c4", 4, 3, [12, 12, 12]), ("c5", 8, 3, [6, 6, 6])])
def test_fbs_multilevel_cascade(cuda_lib, dev, name, shrink, n_levels, n_outer):
    """The c3/c4/c5 loops (noisy data, 2-3 multigrid levels, 10 inner sweeps) at sizes the oracle runs in
    seconds: same scene, grid dims divided by `shrink`."""
    import torch
    cb = cuda_lib
    cfg = make_config(name, shrink=shrink)
    g = cfg.geom
    G = cb.Geometry.from_synth(g)
    Y = f32(cfg.projections())
    f = torch.empty(g.vol_shape, device=dev)
    cb.fbs_reconstruct(G, to_dev(Y, dev), None, n_levels, n_outer, cfg.n_inner, cfg.step, cfg.mu, cfg.eps, cfg.omega, f)
    f_ref = o.fbs_reconstruct(g, Y.astype(np.float64), None, n_levels, n_outer, cfg.n_inner, cfg.step, cfg.mu, cfg.eps, cfg.omega)
    out = f.cpu().numpy()
    assert rel(out, f_ref) <= TOL_RECON
    assert out.min() >= 0.0
    G.close()


def test_fbs_degenerate_cases(cuda_lib, dev):
    import torch
    cb = cuda_lib
    cfg = make_config("c1")
    g = cfg.geom
    G = cb.Geometry.from_synth(g)
    Y = f32(cfg.projections())
    dY = to_dev(Y, dev)
    f0 = f32(np.abs(gaussian_field(g.vol_shape, 3)) * 0.01)
    f = torch.empty(g.vol_shape, device=dev)
    # zero outer iterations: result is f0 (or zeros)
    cb.fbs_reconstruct(G, dY, to_dev(f0, dev), 1, [0], 3, cfg.step, cfg.mu, cfg.eps, 1.0, f)
    assert np.array_equal(f.cpu().numpy(), f0)
    cb.fbs_reconstruct(G, dY, None, 1, [0], 3, cfg.step, cfg.mu, cfg.eps, 1.0, f)
    assert float(f.abs().max()) == 0.0
    # n_inner = 0: projected Landweber (I11 form), warm start, in-place output
    buf = to_dev(f0, dev)
    cb.fbs_reconstruct(G, dY, buf, 1, [4], 0, cfg.step, cfg.mu, cfg.eps, 1.0, buf)
    ref = o.fbs_reconstruct(g, Y.astype(np.float64), f0.astype(np.float64), 1, [4], 0, cfg.step, cfg.mu, cfg.eps, 1.0)
    assert rel(buf.cpu().numpy(), ref) <= TOL_RECON
    # two levels with a caller-supplied fine f0 (restricted down), odd inner count
    cb.fbs_reconstruct(G, dY, to_dev(f0, dev), 2, [3, 2], 3, cfg.step, cfg.mu, cfg.eps, 0.8, f)
    ref = o.fbs_reconstruct(g, Y.astype(np.float64), f0.astype(np.float64), 2, [3, 2], 3, cfg.step, cfg.mu, cfg.eps, 0.8)
    assert rel(f.cpu().numpy(), ref) <= TOL_RECON
    # bad arguments
    for kw in (dict(step=0.0), dict(mu=-1.0), dict(eps=0.0), dict(n_levels=0)):
        a = dict(n_levels=1, step=cfg.step, mu=cfg.mu, eps=cfg.eps)
        a.update(kw)
        with pytest.raises(cb.CbctError) as ei:
            cb.fbs_reconstruct(G, dY, None, a["n_levels"], [1] * max(a["n_levels"], 1), 1, a["step"], a["mu"], a["eps"], 1.0, f)
        assert ei.value.status == 1
    with pytest.raises(TypeError):
        cb.forward(G, torch.zeros(g.vol_shape), f)                                 # host tensor where a device one is required
    G.close()


@pytest.mark.parametrize("name", ["aniso_ragged", "twin_ragged"])
def test_host_entry_points(cuda_lib, dev, name):
    cb = cuda_lib
    g = GEOMS[name]()
    G = cb.Geometry.from_synth(g)
    vol = f32(smooth_phantom(g, 3))
    q = np.empty(g.proj_shape, dtype=np.float32)
    cb.forward_host(G, vol, q)
    assert np.array_equal(q, run_forward(cb, G, vol, dev))
    b = np.empty(g.vol_shape, dtype=np.float32)
    cb.backproject_host(G, q, b)
    assert np.array_equal(b, run_backproject(cb, G, q, dev))
    u = vol.copy()
    cb.tv_prox_host(G, vol, u, 40.0, 1e-3, 1.0, 3)
    assert rel(u, o.tv_prox(g, vol.astype(np.float64), vol.astype(np.float64), 40.0, 1e-3, 1.0, 3)) <= TOL_OP
    # the host-buffer cascade uploads Y beside its first kernels (projection without the fused residual, then a2 on its own):
    # bit for bit the device-resident cascade, with and without a start volume, with either backprojector, also on a side stream
    import torch
    Y = f32(0.9 * q + 0.01)
    st = torch.cuda.Stream(device=dev)
    for mode in (cb.BACKPROJECTOR_EXACT, cb.BACKPROJECTOR_EQ2):
        cb.set_backprojector(G, mode)
        for f0 in (None, f32(0.5 * vol)):
            for stream in (None, st):
                d_f = torch.empty(G.vol_shape, device=dev)
                cb.fbs_reconstruct(G, to_dev(Y, dev), None if f0 is None else to_dev(f0, dev), 2, [2, 3], 3, 1e-4, 1.0, 1e-4, 1.0, d_f)
                torch.cuda.synchronize()
                h_f = np.empty(g.vol_shape, dtype=np.float32)
                cb.fbs_reconstruct_host(G, Y, f0, 2, [2, 3], 3, 1e-4, 1.0, 1e-4, 1.0, h_f, stream=stream)
                assert np.array_equal(h_f, d_f.cpu().numpy())
    G.close()


# ---- NEXT-1: the paper's eq. 2 backprojector ---------------------------------------------
@pytest.mark.parametrize("name", ["c1", "aniso_ragged", "odd_dims_axis_angles", "wide_detector_misses"])
def test_backproject_eq2_matches_oracle(cuda_lib, dev, name):
    import torch
    cb = cuda_lib
    g = GEOMS[name]()
    G = cb.Geometry.from_synth(g)
    vol = f32(smooth_phantom(g, 3) if name != "c1" else make_config("c1").volume())
    q = f32(o.forward(g, vol.astype(np.float64)))              # phantom-like projections
    b = torch.empty(G.vol_shape, device=dev)
    cb.backproject_eq2(G, to_dev(q, dev), b)
    torch.cuda.synchronize()
    assert rel(b.cpu().numpy(), o.backproject_eq2(g, q.astype(np.float64))) <= TOL_OP
    # Gaussian images: every interpolation weight matters (fp32 position of (u*,v*) ~ 3e-5 pixel): stated bound 5e-5
    y = f32(gaussian_field(g.proj_shape, 12))
    cb.backproject_eq2(G, to_dev(y, dev), b)
    torch.cuda.synchronize()
    assert rel(b.cpu().numpy(), o.backproject_eq2(g, y.astype(np.float64))) <= 5e-5
    G.close()


def test_fbs_with_eq2_backprojector_matches_oracle(cuda_lib, dev):
    """Algorithm A1 as the paper ran it (eq. 2 in step 1) on c1, 2 levels x 6 iterations, against the oracle."""
    import torch
    from oracle import fbs
    cb = cuda_lib
    cfg = make_config("c1")
    g = cfg.geom
    G = cb.Geometry.from_synth(g)
    Y = f32(cfg.projections())
    cb.set_backprojector(G, cb.BACKPROJECTOR_EQ2)
    f = torch.empty(G.vol_shape, device=dev)
    cb.fbs_reconstruct(G, to_dev(Y, dev), None, 2, [6, 6], cfg.n_inner, cfg.step, cfg.mu, cfg.eps, cfg.omega, f)
    torch.cuda.synchronize()
    ref = fbs.fbs_reconstruct(g, Y.astype(np.float64), None, 2, [6, 6], cfg.n_inner, cfg.step, cfg.mu, cfg.eps, cfg.omega,
                              backprojector="eq2")
    assert rel(f.cpu().numpy(), ref) <= TOL_RECON
    # and the default is untouched by the option of another handle
    G2 = cb.Geometry.from_synth(g)
    f2 = torch.empty(G.vol_shape, device=dev)
    cb.fbs_reconstruct(G2, to_dev(Y, dev), None, 1, [3], cfg.n_inner, cfg.step, cfg.mu, cfg.eps, cfg.omega, f2)
    ref2 = fbs.fbs_reconstruct(g, Y.astype(np.float64), None, 1, [3], cfg.n_inner, cfg.step, cfg.mu, cfg.eps, cfg.omega)
    assert rel(f2.cpu().numpy(), ref2) <= TOL_RECON
    with pytest.raises(cb.CbctError):
        cb.set_backprojector(G, 7)
    G.close(); G2.close()


def test_fbs_until_stops_where_the_oracle_stops(cuda_lib, dev):
    """NEXT-2: the stopping rule ||f_new - f_old|| <= rel_tol ||f_new|| ("until convergence").  The tolerance
    sits half-way between two consecutive relative updates of the oracle's trajectory, so the fp32 path and the
    fp64 oracle take the same decision; iteration counts and volumes must then match."""
    import torch
    from oracle import fbs
    cb = cuda_lib
    cfg = make_config("c1")
    g = cfg.geom
    G = cb.Geometry.from_synth(g)
    Y = f32(cfg.projections())
    args = (cfg.n_inner, cfg.step, cfg.mu, cfg.eps, cfg.omega)
    Y64 = Y.astype(np.float64)
    prev, change = np.zeros(g.vol_shape), []
    for n in range(1, 9):
        cur = fbs.fbs_reconstruct(g, Y64, None, 1, [n], *args)
        change.append(np.linalg.norm(cur - prev) / np.linalg.norm(cur))
        prev = cur
    tol = 0.5 * (change[4] + change[5])
    done = []
    ref = fbs.fbs_reconstruct(g, Y64, None, 1, [8], *args, rel_tol=tol, iters_done=done)
    f = torch.empty(G.vol_shape, device=dev)
    iters = cb.fbs_reconstruct_until(G, to_dev(Y, dev), None, 1, [8], *args, tol, f)
    assert iters == done and 1 < iters[0] < 8
    assert rel(f.cpu().numpy(), ref) <= TOL_RECON
    # rel_tol = 0 is the fixed-count loop; a huge tolerance stops every level after one iteration
    iters = cb.fbs_reconstruct_until(G, to_dev(Y, dev), None, 2, [3, 2], *args, 0.0, f)
    assert iters == [3, 2]
    ref2 = fbs.fbs_reconstruct(g, Y64, None, 2, [3, 2], *args)
    assert rel(f.cpu().numpy(), ref2) <= TOL_RECON
    assert cb.fbs_reconstruct_until(G, to_dev(Y, dev), None, 2, [3, 2], *args, 1e9, f) == [1, 1]
    G.close()


def test_short_scan_subset_reconstruction_matches_oracle(cuda_lib, dev):
    """The shape of the paper's CatPhan experiment (379 views over 200 degrees, a subset of 40 used), shrunk:
    every 9th-10th of 379 angles over 200 degrees, noisy data, 2-level cascade, against the oracle."""
    import torch
    from oracle import fbs
    from cbct_synth import line_integrals, random_ellipsoids, poisson_log
    cb = cuda_lib
    all_angles = np.deg2rad(np.linspace(0.0, 200.0, 379, endpoint=False))
    angles = all_angles[np.linspace(0, 378, 40).round().astype(int)]
    g = Geometry(1000., 1500., angles, 64, 48, 3.0, 3.0, 32, 32, 16, 3.0, 3.0, 5.0)
    rng = np.random.default_rng(600)
    ells = random_ellipsoids(rng, 8, (g.nx * g.hx, g.ny * g.hy, g.nz * g.hz), (6.0, 25.0))
    Y = f32(poisson_log(line_integrals(ells, g), 1e5, rng))
    cfg = make_config("c1")
    step = 0.5 * (g.nu * g.nv * g.du * g.dv) / (g.n_vox * g.hx * g.hy * g.hz * 140.0 * 1.6 ** 2)
    mu = step * 4.0 * (2 / 3.0 ** 2 + 1 / 5.0 ** 2) / cfg.eps
    G = cb.Geometry.from_synth(g)
    f = torch.empty(G.vol_shape, device=dev)
    cb.fbs_reconstruct(G, to_dev(Y, dev), None, 2, [8, 8], 5, step, mu, cfg.eps, 1.0, f)
    torch.cuda.synchronize()
    ref = fbs.fbs_reconstruct(g, Y.astype(np.float64), None, 2, [8, 8], 5, step, mu, cfg.eps, 1.0)
    assert np.linalg.norm(ref) > 0 and rel(f.cpu().numpy(), ref) <= TOL_RECON
    G.close()


def test_eq2_loop_writes_the_residual_of_rays_that_miss(cuda_lib, dev):
    """Step 1 with eq. 2 on a detector much wider than the volume's shadow, with data that is NOT zero outside
    the shadow: the residual of a ray that misses the volume is -Y, and eq. 2's bilinear fetch reads such pixels for voxels at
    the lateral edge.  The handle first runs a backprojection, so its residual scratch holds other values beforehand."""
    import torch
    from oracle import fbs
    from cbct_synth.configs import s_max_estimate
    cb = cuda_lib
    cases = {"wide_detector_misses": (GEOMS["wide_detector_misses"](), 1, [4]),
             "wide_even_2_levels": (Geometry(1000., 1500., equispaced_angles(5) + 0.4, 72, 44, 4.0, 6.0, 24, 24, 12, 2.0, 2.0, 2.0), 2, [2, 3]),
             "coarse_detector": (GEOMS["coarse_detector"](), 1, [4])}
    for name, (g, nl, n_outer) in cases.items():
        G = cb.Geometry.from_synth(g)
        rng = np.random.default_rng(31)
        vol = f32(smooth_phantom(g, 3))
        Y = f32(o.forward(g, vol.astype(np.float64)) + 0.3 + 0.1 * rng.random(g.proj_shape))
        step = 0.5 * s_max_estimate(g)
        eps = 1e-3
        mu = step * 4.0 * (1 / g.hx ** 2 + 1 / g.hy ** 2 + 1 / g.hz ** 2) / eps
        junk = torch.empty(G.vol_shape, device=dev)
        cb.backproject(G, to_dev(7.0 + rng.random(g.proj_shape), dev), junk)         # leaves l*y in the scratch projections
        for mode, bp in ((cb.BACKPROJECTOR_EQ2, "eq2"), (cb.BACKPROJECTOR_EXACT, "exact")):
            cb.set_backprojector(G, mode)
            f = torch.empty(G.vol_shape, device=dev)
            cb.fbs_reconstruct(G, to_dev(Y, dev), to_dev(vol, dev), nl, n_outer, 3, step, mu, eps, 1.0, f)
            ref = fbs.fbs_reconstruct(g, Y.astype(np.float64), vol.astype(np.float64), nl, n_outer, 3, step, mu, eps, 1.0, backprojector=bp)
            assert np.linalg.norm(ref) > 0 and rel(f.cpu().numpy(), ref) <= TOL_RECON, (name, bp)
            # the data gradient alone (no prox in between): every residual pixel counts
            Gd = torch.empty(G.vol_shape, device=dev)
            cb.data_gradient(G, to_dev(vol, dev), to_dev(Y, dev), Gd)
            r = o.forward(g, vol.astype(np.float64)) - Y.astype(np.float64)
            gref = o.backproject(g, r) if bp == "exact" else (g.hx * g.hy * g.hz / (g.du * g.dv)) * o.backproject_eq2(g, r)
            assert rel(Gd.cpu().numpy(), gref) <= TOL_OP, (name, bp)
        G.close()


def test_first_call_on_a_side_stream(cuda_lib, dev):
    """The handle allocates and zero-fills its scratch (padded volume copies, scratch projections) on first use: that must be
    ordered on the CALLER'S stream.  Every first call here runs on a fresh non-blocking torch stream while the legacy default
    stream is kept busy."""
    import torch
    cb = cuda_lib
    cfg = make_config("c2", shrink=2)
    g = cfg.geom
    vol = f32(cfg.volume())
    q_ref = o.forward(g, vol.astype(np.float64))
    busy = torch.empty(64 << 20, device=dev)
    for first in ("forward", "fbs", "backproject"):
        G = cb.Geometry.from_synth(g)
        st = torch.cuda.Stream(device=dev)
        d_vol = to_dev(vol, dev)
        q = torch.empty(G.proj_shape, device=dev)
        b = torch.empty(G.vol_shape, device=dev)
        torch.cuda.synchronize()
        for _ in range(4):
            busy.add_(1.0)                                   # work on the default stream around the first call
        with torch.cuda.stream(st):
            if first == "forward":
                cb.forward(G, d_vol, q, stream=st)
                st.synchronize()
                assert rel(q.cpu().numpy(), q_ref) <= TOL_OP
            elif first == "backproject":
                cb.backproject(G, to_dev(q_ref, dev), b, stream=st)
                st.synchronize()
                assert rel(b.cpu().numpy(), o.backproject(g, f32(q_ref).astype(np.float64))) <= TOL_OP
            else:
                Y = f32(cfg.projections())
                cb.fbs_reconstruct(G, to_dev(Y, dev), None, 2, [1, 1], 4, cfg.step, cfg.mu, cfg.eps, 1.0, b, stream=st)
                st.synchronize()
                ref = o.fbs_reconstruct(g, Y.astype(np.float64), None, 2, [1, 1], 4, cfg.step, cfg.mu, cfg.eps, 1.0)
                assert rel(b.cpu().numpy(), ref) <= TOL_RECON
        torch.cuda.synchronize()
        G.close()


# ---- NEXT-4: the two halves of an outer iteration and the angle-sharded driver on the CUDA path ---------------
def test_sharded_halves_and_driver(cuda_lib, dev):
    """(1) partial data gradients over two angle shards add up to the full one; (2) the driver with one rank
    reproduces cbct_fbs_reconstruct bit for bit; (3) two shards emulated in one process (their partial gradients
    summed where the all-reduce would be) match the oracle's reconstruction of the full scan."""
    import torch
    from oracle import fbs
    from paper_1002_3675_b200.sharded import fbs_reconstruct_sharded, shard_angles
    cb = cuda_lib
    cfg = make_config("c1")
    g = cfg.geom
    Y = f32(cfg.projections())
    f0 = to_dev(f32(0.5 * cfg.volume()), dev)
    G_all = cb.Geometry.from_synth(g)
    d_Y = to_dev(Y, dev)
    grad = torch.empty(G_all.vol_shape, device=dev)
    cb.data_gradient(G_all, f0, d_Y, grad)
    ref = o.backproject(g, o.forward(g, f0.cpu().numpy().astype(np.float64)) - Y.astype(np.float64))
    assert rel(grad.cpu().numpy(), ref) <= TOL_OP
    shards, part = [], torch.zeros_like(grad)
    for r in range(2):
        idx = shard_angles(g.n_angles, r, 2)
        Gr = cb.Geometry.from_synth(g.with_angles(g.angles[idx]))
        Yr = to_dev(Y[idx], dev)
        tmp = torch.empty_like(grad)
        cb.data_gradient(Gr, f0, Yr, tmp)
        part += tmp
        shards.append((Gr, Yr))
    assert rel(part.cpu().numpy(), grad.cpu().numpy().astype(np.float64)) <= 1e-6
    # (2) one rank through cbct_fbs_reconstruct_sharded: the library's own cascade, bit for bit
    args = (cfg.n_inner, cfg.step, cfg.mu, cfg.eps, cfg.omega)
    f_ref = torch.empty(G_all.vol_shape, device=dev)
    cb.fbs_reconstruct(G_all, d_Y, None, 2, [3, 2], *args, f_ref)
    f_one = fbs_reconstruct_sharded(G_all, d_Y, None, 2, [3, 2], *args, g.n_angles, None)
    torch.cuda.synchronize()
    assert torch.equal(f_one, f_ref)
    # ... and with an exchange callback that counts its calls (a one-rank "sum" leaves the buffer as it is)
    Gs = torch.empty(G_all.vol_shape, device=dev)
    f_cb = torch.empty(G_all.vol_shape, device=dev)
    counts = []
    cb.fbs_reconstruct_sharded(G_all, d_Y, None, 2, [3, 2], *args, g.n_angles, counts.append, Gs, f_cb)
    torch.cuda.synchronize()
    gcoarse = G_all.coarsen()[0]
    assert counts == [gcoarse.n_vox] * 3 + [G_all.n_vox] * 2 and torch.equal(f_cb, f_ref)
    with pytest.raises(ZeroDivisionError):                                         # an exception in the callback surfaces in Python
        cb.fbs_reconstruct_sharded(G_all, d_Y, None, 1, [1], *args, g.n_angles, lambda n: 1 / 0, Gs, f_cb)

    # (3) two shards in one process, driven by the library's cbct_cascade_run: each shard's halves run in the CUDA kernels,
    # their partial gradients are added where the all-reduce would be
    import ctypes as C
    lv = [[G_, G_.coarsen()[0]] for G_, _ in shards]
    Ys = [[Y_, torch.empty(l[1].proj_shape, device=dev)] for (_, Y_), l in zip(shards, lv)]
    f = [None, None]
    Gl = [None, None]
    beta_seen = []

    def level_sizes(u, l, pv, pp):
        pv[0], pp[0] = lv[0][l].n_vox, lv[0][l].nu * lv[0][l].nv
        return 0

    def bin_(u, l):
        for r in range(2):
            cb.bin2x2(lv[r][l], Ys[r][l], Ys[r][l + 1])
        return 0

    def start(u, L, have):
        f[L] = torch.zeros(lv[0][L].vol_shape, device=dev)
        return 0

    def grad_cb(u, l):
        parts = []
        for r in range(2):
            t = torch.empty(lv[r][l].vol_shape, device=dev)
            cb.data_gradient(lv[r][l], f[l], Ys[r][l], t)
            parts.append(t)
        Gl[l] = parts[0] + parts[1]
        return 0

    def prox(u, l, c, beta):
        beta_seen.append(beta)
        out = torch.empty_like(f[l])
        cb.prox_step(lv[0][l], f[l], Gl[l], c, beta, cfg.eps, cfg.omega, cfg.n_inner, out)
        f[l] = out
        return 0

    def prolong(u, l):
        f[l - 1] = torch.empty(lv[0][l - 1].vol_shape, device=dev)
        cb.prolong(lv[0][l - 1], f[l], f[l - 1])
        return 0

    F = dict(cb.CascadeOps._fields_)
    ops = cb.CascadeOps(None, F["level_sizes"](level_sizes), F["bin"](bin_), F["start"](start), F["data_gradient"](grad_cb),
                        C.cast(None, F["all_reduce"]), F["prox_step"](prox), F["prolong"](prolong))
    rc = cb.load().cbct_cascade_run(C.byref(ops), 2, (C.c_int * 2)(3, 2), float(cfg.step), float(cfg.mu), g.n_angles, 0)
    assert rc == 0 and len(beta_seen) == 5
    ref2 = fbs.fbs_reconstruct(g, Y.astype(np.float64), None, 2, [3, 2], *args)
    assert rel(f[0].cpu().numpy(), ref2) <= TOL_RECON
    # argument errors of the new entry points
    with pytest.raises(cb.CbctError) as ei:
        cb.prox_step(G_all, f0, grad, 1e-3, 10.0, 1e-4, 1.0, 2, grad)              # output aliases the gradient
    assert ei.value.status == 1
    with pytest.raises(cb.CbctError) as ei:
        cb.fbs_reconstruct_until(G_all, d_Y, None, 1, [2], *args, -1.0, f_ref)    # negative tolerance
    assert ei.value.status == 1
    for G_, _ in shards:
        G_.close()
    G_all.close()


def test_graph_replay_equals_eager_launches(cuda_lib, dev):
    """Small volumes replay one captured outer iteration as a CUDA graph (n_outer >= 6, <= 2^20 voxels, no trace, no stopping
    rule, profiling off); per-kernel profiling forces the same iterations to be launched eagerly.  Same kernels, same
    arguments, same order: the volumes must be equal bit for bit, with either backprojector and with / without TV sweeps."""
    import torch
    cb = cuda_lib
    cfg = make_config("c1")
    g = cfg.geom
    d_Y = to_dev(f32(cfg.projections()), dev)
    for mode, n_inner, n_levels, n_outer in ((cb.BACKPROJECTOR_EXACT, cfg.n_inner, 1, [9]), (cb.BACKPROJECTOR_EXACT, 0, 1, [7]),
                                             (cb.BACKPROJECTOR_EQ2, cfg.n_inner, 1, [8]), (cb.BACKPROJECTOR_EXACT, 2, 2, [6, 7])):
        res = []
        for eager in (False, True):
            G = cb.Geometry.from_synth(g)                 # a fresh handle each time: the first iteration allocates in both runs
            cb.set_backprojector(G, mode)
            f = torch.empty(G.vol_shape, device=dev)
            cb.profile_enable(eager)
            try:
                n0 = cb.launch_count()
                cb.fbs_reconstruct(G, d_Y, None, n_levels, n_outer, n_inner, cfg.step, cfg.mu, cfg.eps, cfg.omega, f)
                torch.cuda.synchronize()
                res.append((f.clone(), cb.launch_count() - n0))
            finally:
                cb.profile_enable(False)
                cb.profile_read(reset=True)
            G.close()
        assert torch.equal(res[0][0], res[1][0]), (mode, n_inner, n_levels)
        assert res[0][1] == res[1][1]                      # the launch counter counts replayed kernels like launched ones
        assert float(res[0][0].abs().sum()) > 0


def test_sharded_driver_exchange_is_ordered_on_a_side_stream(cuda_lib, dev):
    """The exchange callback must run on the stream the library hands it, not on torch's current stream.  Stand-in for two
    ranks that hold the same views: the "sum over ranks" doubles the gradient volume in place and n_angles_total doubles,
    so c G is unchanged bit for bit (factors of two) and the result must equal cbct_fbs_reconstruct's.  The whole cascade
    runs on a side stream while torch's current stream stays the default one: an exchange issued on the current stream would
    be unordered against the kernels on either side of it."""
    import torch
    from paper_1002_3675_b200.sharded import fbs_reconstruct_sharded
    cb = cuda_lib
    cfg = make_config("c3", shrink=4)          # 128 x 128 x 16: kernels long enough for a misplaced exchange to overtake them
    g = cfg.geom
    G = cb.Geometry.from_synth(g)
    d_Y = to_dev(f32(cfg.projections()), dev)
    args = (cfg.n_inner, cfg.step, cfg.mu, cfg.eps, cfg.omega)
    f_ref = torch.empty(G.vol_shape, device=dev)
    cb.fbs_reconstruct(G, d_Y, None, 2, [4, 3], *args, f_ref)
    torch.cuda.synchronize()
    side = torch.cuda.Stream()
    Gs = torch.empty(G.vol_shape, device=dev)
    f_side = torch.empty(G.vol_shape, device=dev)
    seen = []

    def twice(count):
        seen.append(torch.cuda.current_stream().cuda_stream)
        Gs.view(-1)[:count].mul_(2.0)

    cb.fbs_reconstruct_sharded(G, d_Y, None, 2, [4, 3], *args, 2 * g.n_angles, twice, Gs, f_side, stream=side)
    side.synchronize()
    assert seen == [side.cuda_stream] * 7
    assert torch.equal(f_side, f_ref)

    class OneRankDist:                         # the wiring of sharded.py with a one-rank stand-in for torch.distributed
        class ReduceOp:
            SUM = 0

        @staticmethod
        def all_reduce(t, op=None):
            seen.append(torch.cuda.current_stream().cuda_stream)

    del seen[:]
    f_one = fbs_reconstruct_sharded(G, d_Y, None, 2, [4, 3], *args, g.n_angles, OneRankDist, stream=side)
    side.synchronize()
    assert seen == [side.cuda_stream] * 7 and torch.equal(f_one, f_ref)
    G.close()


@pytest.mark.parametrize("name", ["c1", "aniso_ragged", "odd_dims_axis_angles", "wide_detector_misses", "fine_rows_multicross", "coarse_detector",
                                  "one_slice_one_row", "one_column", "odd_rows_even_slices_coarse", "twin_ragged", "twin_odd_xy", "twin_wide"])
def test_no_kernel_writes_outside_its_buffers(cuda_lib, dev, name):
    """compute-sanitizer is closed on this pool, so the library brings its own check: in guard mode every device buffer a handle
    owns (tables, padded copies, prefix sums, per-class gather outputs, ping-pong volumes, coarse-level data, FDK / V-cycle
    scratch) sits between two pattern-filled regions, and the caller's outputs get pattern-filled margins here.  Every
    entry point runs on ragged and degenerate shapes, on both kernel families and with the staged projector; afterwards no
    pattern byte may have changed."""
    import torch
    cb = cuda_lib
    g = GEOMS[name]()
    cb.set_guard_mode(True)
    try:
        G = cb.Geometry.from_synth(g)
        MARGIN, PAT = 1024, -123.25

        def guarded(shape):
            n = int(np.prod(shape))
            buf = torch.full((n + 2 * MARGIN,), PAT, device=dev)
            return buf, buf[MARGIN:MARGIN + n].view(*shape)

        def intact(buf, n):
            return bool((buf[:MARGIN] == PAT).all()) and bool((buf[MARGIN + n:] == PAT).all())

        vol = to_dev(smooth_phantom(g, 5) if name != "c1" else make_config("c1").volume(), dev)
        qb, q = guarded(G.proj_shape)
        bb, b = guarded(G.vol_shape)
        fb, f = guarded(G.vol_shape)
        n_levels = 1
        try:
            G.coarsen()
            n_levels = 2
        except cb.CbctError:
            pass
        for sym in (True, False):
            for staged in (False, True):
                G.set_mirror_symmetry(sym)
                G.set_projector_staging(staged)
                cb.forward(G, vol, q)
                cb.backproject(G, q, b)
                cb.backproject_eq2(G, q, b)
                cb.fbs_reconstruct(G, q, None, n_levels, [2] * n_levels, 3, 1e-4, 1.0, 1e-4, 1.0, f)
        cb.set_backprojector(G, cb.BACKPROJECTOR_EQ2)
        cb.fbs_reconstruct(G, q, vol, n_levels, [2] * n_levels, 2, 1e-4, 1.0, 1e-4, 1.0, f)
        cb.set_backprojector(G, cb.BACKPROJECTOR_EXACT)
        cb.fbs_reconstruct_until(G, q, None, n_levels, [3] * n_levels, 2, 1e-4, 1.0, 1e-4, 1.0, 1e-3, f)
        cb.fbs_vcycle(G, q, None, n_levels, 1, 1, 1, 2, 2, 1e-4, 1.0, 1e-4, 1.0, f)
        try:
            cb.fdk_reconstruct(G, q, b)
        except cb.CbctError as e:                      # angle lists that are not a full turn in equal steps are refused
            assert e.status == 2 and "equally spaced" in str(e)
        cb.energy(G, f, q, 1.0, 1e-4)
        cb.tv_prox(G, vol, f, 10.0, 1e-4, 1.0, 3)
        torch.cuda.synchronize()
        assert G.check_guards() == 0
        assert intact(qb, q.numel()) and intact(bb, b.numel()) and intact(fb, f.numel())
        G.close()
    finally:
        cb.set_guard_mode(False)
