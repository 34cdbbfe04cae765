"""Pins for the oracle's FBS loop and multigrid cascade (O5/O6). CPU only."""
import numpy as np
import pytest
from scipy.optimize import nnls

import oracle as o
from oracle import fbs
from cbct_synth import Geometry, make_config
from cbct_synth.geometry import equispaced_angles

import bruteforce as bf


def toy(n=8, na=6, nd=14, pitch=2.4, h=2.0):
    return Geometry(1000.0, 1500.0, equispaced_angles(na) + 0.2, nd, nd, pitch, pitch, n, n, n, h, h, h)


def toy_data(g, seed=0):
    rng = np.random.default_rng(seed)
    f_true = np.zeros(g.vol_shape)
    f_true[2:6, 2:6, 2:6] = 0.02
    f_true[3:5, 3:5, 3:5] = 0.035
    A = bf.dense_matrix(g)
    Y = (A @ f_true.ravel()).reshape(g.proj_shape) + 0.01 * rng.normal(size=g.proj_shape)
    return A, f_true, Y


def s_max(A, g):
    lam = np.linalg.eigvalsh(A.T @ A).max()
    return g.n_angles * g.n_pix / (g.n_vox * lam), lam


def test_lambda_max_power_iteration():
    g = toy()
    A, _, _ = toy_data(g)
    _, lam = s_max(A, g)
    assert o.lambda_max(g, iters=60) == pytest.approx(lam, rel=1e-3)


def test_step1_is_the_papers_update_with_its_constant():
    """P:87 verbatim: g = f - (mu V / beta) dE2/df.  On the grid V = N_vox dV and the functional derivative is (1/dV) times
    the partial derivative with respect to a voxel value, so the update is g = f - (mu N_vox / beta) grad E2(f).  One outer
    iteration without TV steps and without the clamp returns g itself; grad E2 comes from central differences of the
    separately evaluated energy term (E2 is quadratic in f, so they are exact up to rounding) at EVERY voxel.  This pins the
    constant c = 2 step N_vox / (N_theta N_pix) of fbs_level, factor 2 included, against eq. 1's E2."""
    g = toy()
    _, f_true, Y = toy_data(g, seed=3)
    rng = np.random.default_rng(5)
    f0 = f_true + 0.01 * rng.random(g.vol_shape)
    mu, step, eps = 3.0, 0.37, 1e-3
    beta = mu / step
    f1 = fbs.fbs_level(g, Y, f0, 1, 0, step, mu, eps, clamp=False)
    E2 = lambda f: fbs.energy(g, f, Y, mu, eps)["E2"]
    grad = np.zeros(g.vol_shape)
    d = 1e-2
    for idx in np.ndindex(*g.vol_shape):
        fp, fm = f0.copy(), f0.copy()
        fp[idx] += d
        fm[idx] -= d
        grad[idx] = (E2(fp) - E2(fm)) / (2 * d)
    lhs, rhs = (f0 - f1) * beta, g.n_vox * mu * grad
    assert np.abs(rhs).max() > 0
    assert np.abs(lhs - rhs).max() <= 1e-9 * np.abs(rhs).max()
    # a dropped factor 2, N_vox or 1/(N_theta N_pix) would be off by far more than this
    assert np.abs(lhs - 0.5 * rhs).max() > 0.1 * np.abs(rhs).max()


@pytest.mark.parametrize("u0_mode,clamp", [("g", True), ("f", False)])
def test_I10_dense_matrix_fbs(u0_mode, clamp):
    """O5 = Algorithm A1 with explicit numpy matrix algebra, per iteration."""
    g = toy()
    A, _, Y = toy_data(g)
    s, _ = s_max(A, g)
    step, mu, eps = 0.5 * s, 50.0, 1e-3
    f0 = np.zeros(g.vol_shape)
    ref = bf.dense_fbs(A, g, Y, f0, 6, 4, step, mu, eps, 1.0, u0_mode, clamp)
    for n in (1, 3, 6):
        f = o.fbs_level(g, Y, f0, n, 4, step, mu, eps, 1.0, u0_mode=u0_mode, clamp=clamp)
        assert np.max(np.abs(f - ref[n - 1])) <= 1e-12 * np.abs(ref[n - 1]).max()
        if clamp:
            assert f.min() >= 0.0                                      # I12


def test_I9_monotone_energy_u0_f_clamp_off():
    """With u0 = f, gamma <= 1, omega <= 1 and no clamp, N_vox*E_eps is non-increasing (MM theorem)."""
    g = toy()
    A, _, Y = toy_data(g, 3)
    s, _ = s_max(A, g)
    for mu in (1.0, 100.0):        # TV-dominated and data-dominated
        tr = []
        o.fbs_level(g, Y, np.zeros(g.vol_shape), 40, 3, 0.5 * s, mu, 1e-3, 1.0, u0_mode="f", clamp=False, trace=tr)
        E = np.array([t["E_eps"] for t in tr])
        assert np.all(np.diff(E) <= 1e-13 * np.abs(E[:-1])), np.diff(E).max()
        # the energy record is what an independent evaluation gives
        f = o.fbs_level(g, Y, np.zeros(g.vol_shape), 40, 3, 0.5 * s, mu, 1e-3, 1.0, u0_mode="f", clamp=False)
        e_ref = bf.tv_value(f, g, 1e-3) / g.n_vox + mu * np.sum((A @ f.ravel() - Y.ravel()) ** 2) / (g.n_angles * g.n_pix)
        assert tr[-1]["E_eps"] == pytest.approx(e_ref, rel=1e-12)
        assert tr[-1]["E_0"] <= tr[-1]["E_eps"]


def test_I11_projected_landweber_reaches_nnls():
    """n_inner = 0: O5 is projected Landweber; with full column rank it converges to the NNLS solution."""
    g = Geometry(1000.0, 1500.0, equispaced_angles(8) + 0.1, 10, 10, 1.6, 1.6, 4, 4, 4, 2.0, 2.0, 2.0)
    A = bf.dense_matrix(g)
    assert np.linalg.matrix_rank(A) == g.n_vox
    rng = np.random.default_rng(8)
    f_true = np.maximum(rng.normal(size=g.vol_shape), 0.0) * 0.02
    Y = (A @ f_true.ravel()).reshape(g.proj_shape) + 0.02 * rng.normal(size=g.proj_shape)
    x_ref, _ = nnls(A, Y.ravel(), maxiter=10000)
    s, _ = s_max(A, g)
    f = o.fbs_level(g, Y, np.zeros(g.vol_shape), 6000, 0, 0.9 * s, 1.0, 1e-3, 1.0)
    r_ref = np.linalg.norm(A @ x_ref - Y.ravel())
    r = np.linalg.norm(A @ f.ravel() - Y.ravel())
    assert r <= r_ref * (1 + 1e-6)
    assert np.max(np.abs(f.ravel() - x_ref)) <= 2e-3 * np.abs(x_ref).max()


def test_I12_transfer_identities():
    rng = np.random.default_rng(2)
    c = np.full((4, 6, 8), 1.25)
    for ax in [(True, True, True), (True, True, False), (False, False, True)]:
        p = o.prolong(c, ax)
        assert p.shape == tuple(n * (2 if a else 1) for n, a in zip(c.shape, ax[::-1]))
        assert np.all(p == 1.25)
    # linear field: exact at interior voxels (cell-centred coordinates)
    k, j, i = np.meshgrid(np.arange(4), np.arange(6), np.arange(8), indexing="ij")
    lin = 2.0 * (i + 0.5) * 2 - 1.0 * (j + 0.5) * 2 + 0.5 * (k + 0.5) * 2
    p = o.prolong(lin, (True, True, True))
    K, J, I = np.meshgrid(np.arange(8), np.arange(12), np.arange(16), indexing="ij")
    fine = 2.0 * (I + 0.5) - 1.0 * (J + 0.5) + 0.5 * (K + 0.5)
    assert np.max(np.abs(p[1:-1, 1:-1, 1:-1] - fine[1:-1, 1:-1, 1:-1])) < 1e-12
    # explicit 1-D weights (3/4, 1/4), clamped ends
    c1 = rng.normal(size=(1, 1, 5))
    p1 = o.prolong(c1, (True, False, False))[0, 0]
    v = c1[0, 0]
    want = [0.75 * v[0] + 0.25 * v[0], 0.75 * v[0] + 0.25 * v[1], 0.75 * v[1] + 0.25 * v[0], 0.75 * v[1] + 0.25 * v[2]]
    assert np.allclose(p1[:4], want, rtol=0, atol=1e-15)
    assert p1[-1] == pytest.approx(v[-1])
    # prolongation preserves >= 0; binning / restriction of constants
    assert o.prolong(np.abs(rng.normal(size=(3, 4, 5))), (True, True, True)).min() >= 0.0
    Y = np.full((3, 6, 8), 2.5)
    assert np.all(o.bin2x2(Y) == 2.5) and o.bin2x2(Y).shape == (3, 3, 4)
    Yr = rng.normal(size=(2, 4, 4))
    assert o.bin2x2(Yr)[1, 1, 0] == pytest.approx(Yr[1, 2:4, 0:2].mean())
    f = rng.normal(size=(4, 6, 8))
    r = o.restrict_volume(f, (True, True, False))
    assert r.shape == (4, 3, 4) and r[2, 1, 3] == pytest.approx(f[2, 2:4, 6:8].mean())


def test_level_geometries_follow_the_coarsening_rule():
    g3 = make_config("c3").geom
    geoms, axes, binned = o.level_geometries(g3, 3)
    assert [(q.nx, q.ny, q.nz) for q in geoms] == [(512, 512, 64), (256, 256, 64), (128, 128, 64)]
    assert [(q.nu, q.nv) for q in geoms] == [(512, 384), (256, 192), (128, 96)]
    assert axes == [(True, True, False), (True, True, False)] and binned == [True, True]
    assert geoms[2].hx == 2.0 and geoms[2].hz == 2.5 and geoms[2].du == pytest.approx(3.12)
    g5 = make_config("c5").geom
    geoms, axes, _ = o.level_geometries(g5, 3)
    assert [(q.nx, q.ny, q.nz) for q in geoms] == [(512,) * 3, (256,) * 3, (128,) * 3]
    with pytest.raises(ValueError):
        o.coarsen_geometry(Geometry(1000.0, 1500.0, np.array([0.0]), 4, 4, 1.0, 1.0, 5, 4, 4, 1.0, 1.0, 1.0))


def test_I12_one_level_cascade_is_O5_and_multilevel_runs():
    g = toy()
    A, _, Y = toy_data(g, 1)
    s, _ = s_max(A, g)
    a = o.fbs_reconstruct(g, Y, None, 1, [5], 3, 0.5 * s, 50.0, 1e-3)
    b = o.fbs_level(g, Y, np.zeros(g.vol_shape), 5, 3, 0.5 * s, 50.0, 1e-3)
    assert np.array_equal(a, b)
    # two levels: coarse solve, prolong, fine solve == doing the same by hand
    gc, ax, binned = o.coarsen_geometry(g)
    fc = o.fbs_level(gc, o.bin2x2(Y), np.zeros(gc.vol_shape), 4, 3, 0.5 * s, 50.0, 1e-3)
    want = o.fbs_level(g, Y, o.prolong(fc, ax), 5, 3, 0.5 * s, 50.0, 1e-3)
    got = o.fbs_reconstruct(g, Y, None, 2, [4, 5], 3, 0.5 * s, 50.0, 1e-3)
    assert np.array_equal(got, want) and binned and got.min() >= 0.0


def test_I13_c1_quality_sanity():
    """Config 1 (noiseless analytic data): RMSE against the phantom decreases and beats f = 0;
    f >= 0 after every iteration; energy (default mode) decreases on this beta-dominated config."""
    cfg = make_config("c1")
    g = cfg.geom
    Y = cfg.projections()
    truth = cfg.volume()
    tr = []
    errs = [np.linalg.norm(truth)]
    f = np.zeros(g.vol_shape)
    for _ in range(4):
        f = o.fbs_level(g, Y, f, 5, cfg.n_inner, cfg.step, cfg.mu, cfg.eps, cfg.omega, trace=tr)
        assert f.min() >= 0.0
        errs.append(np.linalg.norm(f - truth))
    assert all(b < a for a, b in zip(errs, errs[1:])), errs
    assert errs[-1] < 0.6 * errs[0]
    E = np.array([t["E_eps"] for t in tr])
    assert np.all(np.diff(E) < 0)


def test_stopping_rule_is_the_first_iteration_below_the_tolerance():
    """NEXT-2 ("Repeat ... until convergence"): with rel_tol the loop stops after the first iteration
    whose relative update is <= rel_tol; the count is checked against fixed-count runs, rel_tol = 0 is the
    fixed-count loop, a huge rel_tol stops after one iteration."""
    cfg = make_config("c1", shrink=2)
    g, Y = cfg.geom, cfg.projections()
    args = (cfg.n_inner, cfg.step, cfg.mu, cfg.eps, cfg.omega)
    traj = [np.zeros(g.vol_shape)]
    for n in range(1, 13):
        traj.append(fbs.fbs_reconstruct(g, Y, None, 1, [n], *args))
    change = [np.linalg.norm(traj[n] - traj[n - 1]) / np.linalg.norm(traj[n]) for n in range(1, 13)]
    assert all(b < a for a, b in zip(change[2:], change[3:]))          # the update shrinks on this problem
    tol = 0.5 * (change[6] + change[7])                                # clear margin: stops at iteration 8
    done = []
    f = fbs.fbs_reconstruct(g, Y, None, 1, [12], *args, rel_tol=tol, iters_done=done)
    first = next(n for n in range(1, 13) if change[n - 1] <= tol)
    assert done == [first] and first == 8
    assert np.array_equal(f, traj[first])
    done = []
    assert np.array_equal(fbs.fbs_reconstruct(g, Y, None, 1, [5], *args, rel_tol=0.0, iters_done=done), traj[5]) and done == [5]
    done = []
    assert np.array_equal(fbs.fbs_reconstruct(g, Y, None, 1, [5], *args, rel_tol=1e9, iters_done=done), traj[1]) and done == [1]
