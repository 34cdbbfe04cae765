"""Pins for the oracle's smoothed TV (O3/O4).  CPU only."""
import numpy as np
import pytest

import oracle as o
from cbct_synth import Geometry

import bruteforce as bf


def vg(nx, ny, nz, h=(1.0, 1.0, 1.0)):
    return Geometry(1000.0, 1500.0, np.array([0.0]), 4, 4, 1.0, 1.0, nx, ny, nz, *h)


def test_I7_constant_volume_zero_gradient_and_prox_invariance():
    g = vg(9, 7, 5, (0.5, 0.75, 2.5))
    f = np.full(g.vol_shape, 0.37)
    assert np.all(o.tv_grad(g, f, 1e-4) == 0.0)
    u = o.tv_prox(g, f, f, beta=123.0, eps=1e-4, omega=1.0, n_inner=7)
    assert np.array_equal(u, f)                     # bit for bit
    assert o.tv_value(g, f, 0.0) == 0.0
    assert o.tv_value(g, f, 1e-3) == pytest.approx(1e-3 * g.n_vox, rel=1e-14)


def test_I7_linear_ramp_zero_gradient_at_interior():
    g = vg(8, 8, 8, (0.5, 1.0, 2.0))
    k, j, i = np.meshgrid(np.arange(8), np.arange(8), np.arange(8), indexing="ij")
    f = 0.3 * i * g.hx - 0.2 * j * g.hy + 0.1 * k * g.hz
    gr = o.tv_grad(g, f, 1e-3)
    assert np.max(np.abs(gr[1:-1, 1:-1, 1:-1])) < 1e-12
    # closed form: |grad| = sqrt(.09+.04+.01) at interior, TV_0 counts the Neumann zeros at far faces
    dx = np.full(g.vol_shape, 0.3); dx[:, :, -1] = 0
    dy = np.full(g.vol_shape, -0.2); dy[:, -1, :] = 0
    dz = np.full(g.vol_shape, 0.1); dz[-1, :, :] = 0
    assert o.tv_value(g, f, 0.0) == pytest.approx(np.sqrt(dx**2 + dy**2 + dz**2).sum(), rel=1e-13)


@pytest.mark.parametrize("h", [(1.0, 1.0, 1.0), (0.5, 0.7, 2.5)])
def test_I7_gradient_vs_finite_differences(h):
    """grad TV_eps against central differences of an independent numpy TV_eps, on 8^3."""
    g = vg(8, 8, 8, h)
    rng = np.random.default_rng(9)
    f = rng.normal(size=g.vol_shape)
    eps = 0.05
    assert o.tv_value(g, f, eps) == pytest.approx(bf.tv_value(f, g, eps), rel=1e-13)
    gr = o.tv_grad(g, f, eps)
    assert np.max(np.abs(gr - bf.tv_grad(f, g, eps))) < 1e-12
    d = 1e-6
    idx = [tuple(rng.integers(0, 8, 3)) for _ in range(40)] + [(0, 0, 0), (7, 7, 7), (0, 7, 3), (7, 0, 0)]
    for q in idx:
        fp = f.astype(np.longdouble); fp[q] += d     # extended precision: the difference of two ~1e3 sums
        fm = f.astype(np.longdouble); fm[q] -= d
        fd = float((bf.tv_value(fp, g, eps) - bf.tv_value(fm, g, eps)) / (2 * d))
        assert abs(fd - gr[q]) <= 1e-7 * max(1.0, abs(fd))


def test_I8_inner_objective_non_increasing_and_matches_numpy():
    g = vg(10, 9, 8, (0.5, 0.5, 2.5))
    rng = np.random.default_rng(4)
    gv = np.abs(rng.normal(size=g.vol_shape)) * 0.02
    eps, beta = 1e-3, 40.0

    def obj(u):
        return bf.tv_value(u, g, eps) + 0.5 * beta * np.sum((u - gv) ** 2)

    for omega in (1.0, 0.5):
        prev = obj(gv)
        u_np = gv.copy()
        dt = omega / (beta + 4.0 * (1 / g.hx**2 + 1 / g.hy**2 + 1 / g.hz**2) / eps)
        for m in range(1, 9):
            u = o.tv_prox(g, gv, gv, beta, eps, omega, m)
            u_np = u_np - dt * (beta * (u_np - gv) + bf.tv_grad(u_np, g, eps))
            assert np.max(np.abs(u - u_np)) <= 1e-13 * np.abs(u_np).max()
            cur = obj(u)
            assert cur <= prev + 1e-12 * abs(prev)
            prev = cur
    # zero sweeps = identity on the start
    assert np.array_equal(o.tv_prox(g, gv, gv * 2, beta, eps, 1.0, 0), gv * 2)
