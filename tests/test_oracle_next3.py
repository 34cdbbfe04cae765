"""Pins for the NEXT-3 rows: detector offsets, full-resolution detector on coarse levels, FAS V-cycles.
The paper gives none of this ("we employed the well developed multi-grid method", ref. 20 at P:170); the readings are in
DESIGN.md §2 (Q19-Q21).  CPU only; nothing here calls the CUDA path."""
from dataclasses import replace

import numpy as np
import pytest

import oracle as o
from oracle import fbs
from cbct_synth import Geometry, make_config
from cbct_synth.geometry import equispaced_angles

import bruteforce as bf


def geom(off_u=0.0, off_v=0.0, nu=12, nv=10, dims=(8, 8, 8), h=(2.0, 2.0, 2.0), na=4):
    return Geometry(1000.0, 1500.0, equispaced_angles(na) + 0.3, nu, nv, 2.5, 2.5, *dims, *h, off_u=off_u, off_v=off_v)


# ---- Q19: detector offsets -------------------------------------------------------------------------------------------
def test_zero_offset_is_the_centred_geometry_bit_for_bit():
    g0 = Geometry(1000.0, 1500.0, equispaced_angles(4) + 0.3, 12, 10, 2.5, 2.5, 8, 8, 8, 2.0, 2.0, 2.0)
    g1 = geom(0.0, 0.0)
    rng = np.random.default_rng(0)
    f, y = rng.normal(size=g0.vol_shape), rng.normal(size=g0.proj_shape)
    assert np.array_equal(o.forward(g0, f), o.forward(g1, f))
    assert np.array_equal(o.backproject(g0, y), o.backproject(g1, y))
    assert np.array_equal(o.backproject_eq2(g0, y), o.backproject_eq2(g1, y))


@pytest.mark.parametrize("off", [(1.25, 0.0), (0.0, -0.9), (-7.3, 4.1)])
def test_offset_detector_equals_brute_force_clipping(off):
    """A shifted panel (half a pixel in u; a fraction in v; several pixels in both): the traversal equals the dense matrix
    built by clipping every ray of the shifted detector against every voxel box (tests/bruteforce.py has its own endpoint
    formula); the transpose and the per-voxel clip path follow."""
    g = geom(*off, dims=(6, 8, 4), h=(1.0, 1.5, 3.0))
    A = bf.dense_matrix(g)
    rng = np.random.default_rng(5)
    f, y = rng.normal(size=g.vol_shape), rng.normal(size=g.proj_shape)
    assert np.max(np.abs(o.forward(g, f).ravel() - A @ f.ravel())) <= 1e-12 * np.abs(A @ f.ravel()).max()
    b = o.backproject(g, y)
    assert np.max(np.abs(b.ravel() - A.T @ y.ravel())) <= 1e-12 * np.abs(A.T @ y.ravel()).max()
    kk, jj, ii = np.unravel_index(np.arange(g.n_vox), g.vol_shape)
    assert np.max(np.abs(o.backproject_voxels(g, y, ii, jj, kk) - b.ravel())) <= 1e-12 * np.abs(b).max()
    # and the shift changes the operator (the pin is not vacuous)
    assert np.abs(o.forward(g, f) - o.forward(geom(0.0, 0.0, dims=(6, 8, 4), h=(1.0, 1.5, 3.0)), f)).max() > 1e-3


def test_offset_by_whole_pixels_is_a_window_of_a_wider_centred_detector():
    """Closed form: a panel of nu x nv pixels shifted by (+2 du, -1 dv) is the window [4, nu+4) x [0, nv) of the centred
    panel with nu+4 columns and nv+2 rows (worked out below)."""
    nu, nv = 10, 8
    g_shift = geom(2 * 2.5, -1 * 2.5, nu=nu, nv=nv)
    # centred panel with nu+4 columns: centre of column iu' is (iu' - (nu+3)/2) du; shifted column iu is (iu - (nu-1)/2 + 2) du
    # = (iu + 4 - (nu+3)/2) du, so iu' = iu + 4.  Rows: nv+2 rows, (iv' - (nv+1)/2) dv = (iv - (nv-1)/2 - 1) dv gives iv' = iv.
    g_wide = geom(0.0, 0.0, nu=nu + 4, nv=nv + 2)
    rng = np.random.default_rng(9)
    f = rng.normal(size=g_shift.vol_shape)
    q_s, q_w = o.forward(g_shift, f), o.forward(g_wide, f)
    assert np.max(np.abs(q_s - q_w[:, 0:nv, 4:4 + nu])) <= 1e-12 * np.abs(q_w).max()
    y = rng.normal(size=g_shift.proj_shape)
    y_w = np.zeros(g_wide.proj_shape)
    y_w[:, 0:nv, 4:4 + nu] = y
    assert np.max(np.abs(o.backproject(g_shift, y) - o.backproject(g_wide, y_w))) <= 1e-12 * np.abs(y).max() * 100
    # eq. 2 interpolates between pixel centres: compare where all four neighbours lie inside both panels
    r_w = rng.normal(size=g_wide.proj_shape)
    b_s = o.backproject_eq2(g_shift, np.ascontiguousarray(r_w[:, 0:nv, 4:4 + nu]))
    b_ref = bf.eq2_backproject(g_shift, np.ascontiguousarray(r_w[:, 0:nv, 4:4 + nu]))
    assert np.max(np.abs(b_s - b_ref)) <= 1e-11 * np.abs(b_ref).max()


def test_offset_half_fan_coverage_and_adjoint_identity():
    """A half-fan panel (shifted by 40 % of its width) sees one side of the volume only: rays left of the shadow are zero,
    and <P x, y> = <x, P^T y> holds as for any matrix."""
    g = Geometry(1000.0, 1500.0, equispaced_angles(6), 16, 12, 3.0, 3.0, 12, 12, 8, 2.0, 2.0, 2.0, off_u=0.4 * 16 * 3.0)
    x = np.random.default_rng(1).normal(size=g.vol_shape)
    y = np.random.default_rng(2).normal(size=g.proj_shape)
    a, b = np.vdot(o.forward(g, x), y), np.vdot(x, o.backproject(g, y))
    assert abs(a - b) <= 1e-12 * abs(a)
    q1 = o.forward(g, np.ones(g.vol_shape))
    assert np.all(q1[:, :, -3:] == 0.0) and np.all(q1[:, 4:8, 0] > 0.0)
    assert np.max(np.abs(q1 - bf.box_chords(g))) <= 1e-12 * q1.max()


def test_offsets_survive_coarsening_unchanged():
    """2x2 binning of a shifted panel: the mean position of a pixel pair is the centre of the binned pixel with the SAME
    shift, so the coarse geometry keeps (off_u, off_v) (checked against the pixel centres themselves)."""
    g = Geometry(1000.0, 1500.0, equispaced_angles(3), 16, 12, 3.0, 2.0, 8, 8, 8, 2.0, 2.0, 2.0, off_u=4.7, off_v=-1.3)
    gc, ax, binned = o.coarsen_geometry(g)
    assert binned and (gc.off_u, gc.off_v) == (g.off_u, g.off_v)
    fine, coarse = g.pixel_centres(1), gc.pixel_centres(1)
    mean = fine.reshape(6, 2, 8, 2, 3).mean(axis=(1, 3))
    assert np.max(np.abs(mean - coarse)) <= 1e-12 * np.abs(coarse).max()


# ---- Q20: full-resolution detector on the coarse levels ----------------------------------------------------------------
def test_full_resolution_detector_on_coarse_levels():
    cfg = make_config("c1", shrink=2)
    g, Y = cfg.geom, cfg.projections()
    geoms, axes, binned = o.level_geometries(g, 3, bin_detector=False)
    assert binned == [False, False]
    assert [(q.nx, q.nu, q.nv, q.du) for q in geoms] == [(16, 32, 32, 3.0), (8, 32, 32, 3.0), (4, 32, 32, 3.0)]
    assert o.level_geometries(g, 2)[2] == [True]                                   # the default still bins
    args = (cfg.n_inner, cfg.step, cfg.mu, cfg.eps, cfg.omega)
    # two levels by hand: coarse solve on the halved volume with the SAME detector and data, prolong, fine solve
    gc = replace(g, nx=g.nx // 2, ny=g.ny // 2, nz=g.nz // 2, hx=2 * g.hx, hy=2 * g.hy, hz=2 * g.hz)
    fc = fbs.fbs_level(gc, Y, np.zeros(gc.vol_shape), 3, *args)
    ff = fbs.fbs_level(g, Y, fbs.prolong(fc, (True, True, True)), 2, *args)
    got = fbs.fbs_reconstruct(g, Y, None, 2, [3, 2], *args, bin_detector=False)
    assert np.array_equal(got, ff)
    assert np.abs(got - fbs.fbs_reconstruct(g, Y, None, 2, [3, 2], *args)).max() > 0          # and it is a different cascade


# ---- Q21: FAS V-cycles ---------------------------------------------------------------------------------------------------
def _levels_by_hand(g, dims_h):
    """Level geometries written out by hand (not through the oracle's coarsening rule): dims_h = [(nx,ny,nz,hx,hy,hz,nu,nv,du,dv)]."""
    return [replace(g, nx=a, ny=b, nz=c, hx=d, hy=e, hz=f, nu=p, nv=q, du=r, dv=s) for (a, b, c, d, e, f, p, q, r, s) in dims_h]


@pytest.mark.parametrize("case", ["iso_2_levels", "aniso_3_levels", "iso_full_res_detector"])
def test_vcycle_equals_explicit_matrix_algebra(case):
    rng = np.random.default_rng(3)
    if case == "iso_2_levels":
        g = Geometry(1000.0, 1500.0, equispaced_angles(5) + 0.2, 12, 10, 3.0, 3.0, 8, 8, 8, 2.0, 2.0, 2.0)
        geoms = _levels_by_hand(g, [(8, 8, 8, 2., 2., 2., 12, 10, 3., 3.), (4, 4, 4, 4., 4., 4., 6, 5, 6., 6.)])
        binflag = True
    elif case == "iso_full_res_detector":
        g = Geometry(1000.0, 1500.0, equispaced_angles(4) + 0.2, 12, 10, 3.0, 3.0, 8, 8, 8, 2.0, 2.0, 2.0, off_u=1.0)
        geoms = _levels_by_hand(g, [(8, 8, 8, 2., 2., 2., 12, 10, 3., 3.), (4, 4, 4, 4., 4., 4., 12, 10, 3., 3.)])
        binflag = False
    else:   # x,y coarsen first (0.5 x 0.5 x 1.25 voxels as in c3), then all three axes
        g = Geometry(1000.0, 1500.0, equispaced_angles(4) + 0.1, 16, 8, 2.0, 2.0, 8, 8, 4, 1.0, 1.0, 2.5)
        geoms = _levels_by_hand(g, [(8, 8, 4, 1., 1., 2.5, 16, 8, 2., 2.), (4, 4, 4, 2., 2., 2.5, 8, 4, 4., 4.),
                                    (2, 2, 2, 4., 4., 5., 4, 2, 8., 8.)])
        binflag = True
    vol = np.abs(rng.normal(size=g.vol_shape)) * 0.02
    Y = o.forward(g, vol) * (1.0 + 0.05 * rng.normal(size=g.proj_shape))
    Ys = [Y]
    for l in range(1, len(geoms)):
        Yp = Ys[-1]
        Ys.append(Yp.reshape(Yp.shape[0], Yp.shape[1] // 2, 2, Yp.shape[2] // 2, 2).mean(axis=(2, 4)) if binflag else Yp)
    levels = [dict(g=q, A=bf.dense_matrix(q), Y=y) for q, y in zip(geoms, Ys)]
    from cbct_synth.configs import s_max_estimate
    step = 0.5 * s_max_estimate(g)
    eps = 1e-3
    mu = step * 4.0 * (1 / g.hx ** 2 + 1 / g.hy ** 2 + 1 / g.hz ** 2) / eps
    f0 = 0.5 * vol
    for (ncyc, n1, n2, nc) in ((1, 1, 1, 2), (2, 2, 1, 3)):
        ref = bf.dense_vcycle(levels, f0, ncyc, n1, n2, nc, 3, step, mu, eps, 0.9)
        got = o.fbs_vcycle(g, Y, f0, len(geoms), ncyc, n1, n2, nc, 3, step, mu, eps, 0.9, bin_detector=binflag)
        assert np.linalg.norm(ref) > 0
        assert np.max(np.abs(got - ref)) <= 1e-10 * np.abs(ref).max(), case
        # the coarse-grid correction does something: the result differs from plain smoothing alone
        plain = fbs.fbs_level(g, Y, f0, ncyc * (n1 + n2), 3, step, mu, eps, 0.9)
        assert np.max(np.abs(got - plain)) > 1e-6 * np.abs(ref).max()


def test_vcycle_special_cases_reduce_to_algorithm_A1():
    cfg = make_config("c1", shrink=2)
    g, Y = cfg.geom, cfg.projections()
    args = (cfg.n_inner, cfg.step, cfg.mu, cfg.eps, cfg.omega)
    # one level: n_cycles x nu_coarse iterations of A1
    a = o.fbs_vcycle(g, Y, None, 1, 2, 5, 7, 3, *args)
    assert np.array_equal(a, fbs.fbs_level(g, Y, np.zeros(g.vol_shape), 6, *args))
    # no coarse iterations: the correction is zero, the cycle is nu_pre + nu_post iterations of A1
    b = o.fbs_vcycle(g, Y, None, 2, 2, 2, 1, 0, *args)
    assert np.max(np.abs(b - fbs.fbs_level(g, Y, np.zeros(g.vol_shape), 6, *args))) <= 1e-13 * np.abs(b).max()


def test_linear_term_equals_a_shift_of_the_data():
    """The FAS term enters step 1 as +tau/beta.  For tau = 2 mu' P^T D the smooth part's gradient is
    2 mu' P^T (P f - (Y + D)), so smoothing with tau must equal Algorithm A1 on the data Y + D (sign and scale of tau)."""
    cfg = make_config("c1", shrink=2)
    g, Y = cfg.geom, cfg.projections()
    D = 0.1 * np.random.default_rng(8).normal(size=g.proj_shape)
    mu_p = cfg.mu * g.n_vox / (g.n_angles * g.n_pix)
    tau = 2.0 * mu_p * o.backproject(g, D)
    args = (4, cfg.n_inner, cfg.step, cfg.mu, cfg.eps, cfg.omega)
    a = fbs.fbs_level(g, Y, np.zeros(g.vol_shape), *args, tau=tau)
    b = fbs.fbs_level(g, Y + D, np.zeros(g.vol_shape), *args)
    assert np.max(np.abs(a - b)) <= 1e-11 * np.abs(b).max()
    # grad_objective is N_vox times the gradient of the recorded energy (finite differences along a random direction)
    f = np.abs(np.random.default_rng(9).normal(size=g.vol_shape)) * 0.01
    d = np.random.default_rng(10).normal(size=g.vol_shape)
    h = 1e-6
    Ep = fbs.energy(g, f + h * d, Y, cfg.mu, cfg.eps)["E_eps"]
    Em = fbs.energy(g, f - h * d, Y, cfg.mu, cfg.eps)["E_eps"]
    lhs = g.n_vox * (Ep - Em) / (2 * h)
    rhs = float(np.vdot(o.grad_objective(g, f, Y, cfg.mu, cfg.eps), d))
    assert abs(lhs - rhs) <= 1e-5 * abs(rhs)


def test_vcycles_lower_the_energy_faster_than_plain_iterations_on_c1():
    """Empirical (like I13): on c1, two V(2,2) cycles over 2 levels end at a lower energy than the same number of fine-level
    iterations of plain A1, and every cycle lowers the energy."""
    cfg = make_config("c1")
    g, Y = cfg.geom, cfg.projections()
    args = (cfg.n_inner, cfg.step, cfg.mu, cfg.eps, cfg.omega)
    tr = []
    o.fbs_vcycle(g, Y, None, 2, 2, 2, 2, 8, *args, trace=tr)
    E = [t["E_eps"] for t in tr]
    plain = fbs.fbs_level(g, Y, np.zeros(g.vol_shape), 8, *args)
    Ep = fbs.energy(g, plain, Y, cfg.mu, cfg.eps)["E_eps"]
    assert E[1] < E[0] and E[1] < Ep, (E, Ep)
