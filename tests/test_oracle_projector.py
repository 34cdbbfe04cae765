"""Pins for the oracle's projector O1 and backprojector O2.
CPU only; none of these call the CUDA path."""
import os

import numpy as np
import pytest

import oracle as o
from cbct_synth import Geometry, make_config
from cbct_synth.geometry import equispaced_angles
from cbct_synth import phantom as ph

import bruteforce as bf

HERE = os.path.dirname(os.path.abspath(__file__))


def small_geom(nx=8, ny=8, nz=8, h=(2.0, 2.0, 2.0), na=3, nu=12, nv=12, du=3.0, dv=3.0, offset=0.3):
    ang = equispaced_angles(na) + offset
    return Geometry(1000.0, 1500.0, ang, nu, nv, du, dv, nx, ny, nz, *h)


def test_golden_hand_chords():
    """tests/golden/hand_chords.txt: closed forms worked by hand from the definition (O1)."""
    n = 0
    for line in open(os.path.join(HERE, "golden", "hand_chords.txt")):
        if line.startswith("#") or not line.strip():
            continue
        t = line.split()
        sad, sdd, th = float(t[1]), float(t[2]), float(t[3])
        nu, nv, du, dv = int(t[4]), int(t[5]), float(t[6]), float(t[7])
        nx, ny, nz = int(t[8]), int(t[9]), int(t[10])
        hx, hy, hz = float(t[11]), float(t[12]), float(t[13])
        rule, iu, iv, want = t[14], int(t[15]), int(t[16]), float(t[17])
        g = Geometry(sad, sdd, np.array([np.deg2rad(th)]), nu, nv, du, dv, nx, ny, nz, hx, hy, hz)
        lin = np.arange(nx * ny * nz, dtype=np.float64).reshape(nz, ny, nx)
        f = lin ** 2 if rule == "sq" else lin + 1.0
        got = o.forward(g, f)[0, iv, iu]
        assert got == pytest.approx(want, rel=1e-12, abs=1e-12), (t[0], got, want)
        n += 1
    assert n == 7


def test_I1_ones_volume_is_box_chord():
    """P·1 = length of each ray inside the volume's bounding box, to 1e-12."""
    for g in (make_config("c1").geom, small_geom(6, 8, 4, (1.0, 2.0, 3.0), na=5, nu=16, nv=10)):
        q = o.forward(g, np.ones(g.vol_shape))
        ref = bf.box_chords(g)
        assert np.max(np.abs(q - ref)) <= 1e-12 * max(1.0, ref.max())
        assert (ref > 0).any()


@pytest.mark.parametrize("dims,h", [((8, 8, 8), (2.0, 2.0, 2.0)), ((6, 8, 4), (1.0, 1.5, 3.0))])
def test_I2_dense_matrix_bruteforce(dims, h):
    """Traversal = dense matrix built by clipping every ray against every voxel box; its
    transpose = the backprojector."""
    g = small_geom(*dims, h=h, na=4, nu=12, nv=10, du=2.5, dv=2.5)
    A = bf.dense_matrix(g)
    rng = np.random.default_rng(5)
    f = rng.normal(size=g.vol_shape)
    y = rng.normal(size=g.proj_shape)
    q = o.forward(g, f)
    assert np.max(np.abs(q.ravel() - A @ f.ravel())) <= 1e-12 * np.abs(A @ f.ravel()).max()
    b = o.backproject(g, y)
    assert np.max(np.abs(b.ravel() - A.T @ y.ravel())) <= 1e-12 * np.abs(A.T @ y.ravel()).max()
    # every unit vector reproduces its column (a wrong voxel index would show up here)
    for j in rng.choice(g.n_vox, 12, replace=False):
        e = np.zeros(g.n_vox); e[j] = 1.0
        assert np.max(np.abs(o.forward(g, e.reshape(g.vol_shape)).ravel() - A[:, j])) <= 1e-12
    # the per-voxel brute-force clip path agrees with the scatter
    kk, jj, ii = np.unravel_index(np.arange(g.n_vox), g.vol_shape)
    bv = o.backproject_voxels(g, y, ii, jj, kk)
    assert np.max(np.abs(bv - b.ravel())) <= 1e-12 * np.abs(b).max()
    # sampled-ray path agrees with the full operator
    ia, iv, iu = np.unravel_index(np.arange(g.n_rays), g.proj_shape)
    assert np.array_equal(o.forward_rays(g, f, ia, iv, iu), q.ravel())
    assert o.count_chords(g) == int((A > 0).sum())


def test_I3_converges_to_analytic_ellipsoid_chords():
    """P(voxelised ellipsoids) -> analytic chord integrals at first order in h."""
    ells = np.zeros((2, 16))
    ells[0, 0:3] = (10.0, -20.0, 5.0); ells[0, 3:6] = (60.0, 40.0, 30.0)
    ells[1, 0:3] = (-30.0, 25.0, -10.0); ells[1, 3:6] = (25.0, 45.0, 20.0)
    rng = np.random.default_rng(11)
    ells[:, 6:15] = ph._random_rotations(rng, 2).reshape(2, 9)
    ells[:, 15] = (0.02, 0.015)
    errs = []
    for n in (32, 64, 128):
        g = Geometry(1000.0, 1500.0, equispaced_angles(7) + 0.1, 48, 40, 8.0, 8.0, n, n, n,
                     256.0 / n, 256.0 / n, 256.0 / n)
        ref = ph.line_integrals(ells, g)
        q = o.forward(g, ph.voxelize(ells, g))
        errs.append(np.linalg.norm(q - ref) / np.linalg.norm(ref))
    assert errs[2] < 0.05, errs   # absolute level depends on the ellipsoids; the rate is the pin
    assert 0.3 < errs[1] / errs[0] < 0.75 and 0.3 < errs[2] / errs[1] < 0.75, errs


def test_I4_dot_product_identity():
    for g in (make_config("c1").geom, small_geom(6, 8, 4, (1.0, 1.5, 3.0), na=5)):
        x = np.random.default_rng(1).normal(size=g.vol_shape)
        y = np.random.default_rng(2).normal(size=g.proj_shape)
        a = np.vdot(o.forward(g, x), y)
        b = np.vdot(x, o.backproject(g, y))
        assert abs(a - b) <= 1e-12 * abs(a)


def test_I5_eq2_weight():
    """PAPER.md:97-99 eq. 2: the continuous adjoint's weight L^3(u*,v*)/(L0 l^2(x)) equals
    (du dv / dV) (P^T 1)_j for a voxel whose shadow lies on the detector (within the
    discretisation scatter)."""
    g = Geometry(1000.0, 1500.0, np.array([0.4]), 96, 96, 0.375, 0.375, 8, 8, 8, 2.0, 2.0, 2.0)
    w = o.backproject(g, np.ones(g.proj_shape)) * (g.du * g.dv / (g.hx * g.hy * g.hz))
    x, y, z = g.voxel_centres_1d()
    X, Y, Z = np.meshgrid(x, y, z, indexing="ij")
    X, Y, Z = (a.transpose(2, 1, 0) for a in (X, Y, Z))
    S = g.source(0)
    c, s = np.cos(0.4), np.sin(0.4)
    l = np.sqrt((X - S[0]) ** 2 + (Y - S[1]) ** 2 + (Z - S[2]) ** 2)
    depth = g.sad - (X * c + Y * s)
    L = l * g.sdd / depth                      # source -> (u*,v*) along the same ray
    ref = L ** 3 / (g.sdd * l ** 2)
    ratio = w / ref
    assert abs(ratio.mean() - 1.0) < 2e-3
    assert ratio.min() > 0.97 and ratio.max() < 1.03


def test_I6_rot90_and_zflip_symmetry():
    """Equally spaced angles over 360 deg: rotating the source by 90 deg about z is
    the same as rotating the volume by -90 deg; flipping z flips v."""
    g = Geometry(1000.0, 1500.0, np.array([0.35, 0.35 + np.pi / 2]), 14, 10, 2.5, 2.5, 8, 8, 6, 2.0, 2.0, 3.0)
    f = np.random.default_rng(3).normal(size=g.vol_shape)
    q = o.forward(g, f)
    fR = f.transpose(0, 2, 1)[:, ::-1, :]       # (f∘R)[k][j][i] = f[k][i][ny-1-j]
    qR = o.forward(g, fR)
    assert np.max(np.abs(q[1] - qR[0])) <= 1e-12 * np.abs(q).max()
    qz = o.forward(g, f[::-1])
    assert np.max(np.abs(qz - q[:, ::-1, :])) <= 1e-12 * np.abs(q).max()


def test_rays_missing_the_volume_give_zero():
    g = Geometry(1000.0, 1500.0, np.array([0.2]), 8, 8, 200.0, 200.0, 4, 4, 4, 1.0, 1.0, 1.0)
    q = o.forward(g, np.ones(g.vol_shape))
    assert np.all(q == 0.0)
    b = o.backproject(g, np.ones(g.proj_shape))
    assert np.all(b == 0.0)
