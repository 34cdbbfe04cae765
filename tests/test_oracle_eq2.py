"""Pins for the oracle's eq. 2 backprojector.  CPU only."""
import os

import numpy as np
import pytest

import oracle as o
from oracle import fbs
from cbct_synth import Geometry, make_config, gaussian_field
from cbct_synth.geometry import equispaced_angles

import bruteforce as bf

HERE = os.path.dirname(os.path.abspath(__file__))


def test_golden_hand_eq2():
    """tests/golden/hand_eq2.txt: weights L^3/(L0 l^2) and interpolated values worked by hand."""
    n = 0
    for line in open(os.path.join(HERE, "golden", "hand_eq2.txt")):
        if line.startswith("#") or not line.strip():
            continue
        t = line.split()
        sad, sdd, th = float(t[1]), float(t[2]), float(t[3])
        nu, nv, du, dv = int(t[4]), int(t[5]), float(t[6]), float(t[7])
        nx, ny, nz = int(t[8]), int(t[9]), int(t[10])
        hx, hy, hz = float(t[11]), float(t[12]), float(t[13])
        rule, i, j, k, want = t[14], int(t[15]), int(t[16]), int(t[17]), float(t[18])
        g = Geometry(sad, sdd, np.array([np.deg2rad(th)]), nu, nv, du, dv, nx, ny, nz, hx, hy, hz)
        iv, iu = np.meshgrid(np.arange(nv), np.arange(nu), indexing="ij")
        r = np.ones((1, nv, nu)) if rule == "one" else (iu + 100.0 * iv)[None].astype(np.float64)
        got = o.backproject_eq2(g, r)[k, j, i]
        assert got == pytest.approx(want, rel=1e-12, abs=1e-12), (t[0], got, want)
        n += 1
    assert n == 7


@pytest.mark.parametrize("shape", [(6, 8, 4, 1.0, 2.0, 3.0, 14, 9, 1.7, 2.9), (9, 7, 5, 2.0, 2.0, 2.0, 10, 12, 4.0, 3.0)])
def test_eq2_equals_library_interpolation(shape):
    """The oracle (3-D distances, hand-written bilinear) against similar triangles + scipy's
    map_coordinates on seeded images, including voxels whose shadow leaves the detector."""
    nx, ny, nz, hx, hy, hz, nu, nv, du, dv = shape
    g = Geometry(1000.0, 1500.0, equispaced_angles(5) + 0.37, nu, nv, du, dv, nx, ny, nz, hx, hy, hz)
    r = gaussian_field(g.proj_shape, 21)
    a, b = o.backproject_eq2(g, r), bf.eq2_backproject(g, r)
    assert np.max(np.abs(a - b)) <= 1e-11 * np.max(np.abs(b))
    assert np.count_nonzero(b) > 0


def smooth_images(g):
    """A smooth, strictly positive projection stack (a wide Gaussian bump per angle)."""
    uu = (np.arange(g.nu) - (g.nu - 1) / 2.0) * g.du
    vv = (np.arange(g.nv) - (g.nv - 1) / 2.0) * g.dv
    V, U = np.meshgrid(vv, uu, indexing="ij")
    return np.stack([np.exp(-((U - 5.0 * np.cos(t)) ** 2 + (V + 3.0 * np.sin(t)) ** 2) / (2 * 25.0 ** 2)) for t in g.angles])


def test_eq2_converges_to_the_scaled_transpose():
    """eq. 2 replaces sum_theta P^T(...) "apart from some constants": (du dv/dV) (P^T r)_j is the mean
    of the continuous backprojection over voxel j sampled by the rays that cross it, so it tends to the
    centre value (B r)_j when the voxels shrink AND the rays per voxel grow (pitch ~ h^2): a fixed 64 mm
    cube, a fixed 180 mm detector that sees all of it, smooth positive images."""
    errs = []
    for n, nd in ((4, 32), (8, 128), (16, 512)):
        h = 64.0 / n
        g = Geometry(1000.0, 1500.0, equispaced_angles(4) + 0.2, nd, nd, 180.0 / nd, 180.0 / nd, n, n, n, h, h, h)
        r = smooth_images(g)
        exact = (g.du * g.dv / (h ** 3)) * o.backproject(g, r)
        eq2 = o.backproject_eq2(g, r)
        errs.append(np.linalg.norm(exact - eq2) / np.linalg.norm(eq2))
    assert errs[0] < 0.15 and errs[1] < 0.5 * errs[0] and errs[2] < 0.7 * errs[1] and errs[2] < 0.02, errs


def test_eq2_of_ones_is_the_weight_sum():
    """r = 1 on a detector that sees every voxel: B 1 = sum_theta L^3/(L0 l^2) (closed form per voxel)."""
    g = Geometry(1000.0, 1500.0, equispaced_angles(6), 64, 64, 3.0, 3.0, 8, 8, 8, 4.0, 4.0, 4.0)
    b = o.backproject_eq2(g, np.ones(g.proj_shape))
    xs = (np.arange(8) - 3.5) * 4.0
    Z, Y, X = np.meshgrid(xs, xs, xs, indexing="ij")
    ref = np.zeros_like(b)
    for th in g.angles:
        S = np.array([1000.0 * np.cos(th), 1000.0 * np.sin(th), 0.0])
        l2 = (X - S[0]) ** 2 + (Y - S[1]) ** 2 + Z ** 2
        depth = 1000.0 - (X * np.cos(th) + Y * np.sin(th))
        L = np.sqrt(l2) * 1500.0 / depth
        ref += L ** 3 / (1500.0 * l2)
    assert np.max(np.abs(b - ref)) <= 1e-12 * ref.max()


def test_eq2_symmetries():
    """90-degree rotation of the source == -90-degree rotation of the volume; z flip == v flip."""
    g = Geometry(1000.0, 1500.0, np.array([0.3, 0.3 + np.pi / 2]), 20, 16, 3.0, 3.5, 10, 10, 6, 2.0, 2.0, 3.0)
    r = gaussian_field((1,) + g.proj_shape[1:], 5)
    g0, g1 = g.with_angles(g.angles[:1]), g.with_angles(g.angles[1:])
    b0, b1 = o.backproject_eq2(g0, r), o.backproject_eq2(g1, r)
    # P^{theta+90} f = P^theta (f o R) with (f o R)[k][j][i] = f[k][i][ny-1-j] (pin I6), so B^{theta+90} r = (B^theta r) o R^-1
    assert np.max(np.abs(b1.transpose(0, 2, 1)[:, ::-1, :] - b0)) <= 1e-12 * np.abs(b0).max()
    bz = o.backproject_eq2(g0, r[:, ::-1, :])
    assert np.max(np.abs(bz - b0[::-1])) <= 1e-12 * np.abs(b0).max()


def test_fbs_with_eq2_reconstructs_c1_like_the_exact_adjoint():
    """Algorithm A1 with eq. 2 in step 1 (what the paper ran): on a shrunken c1 the reconstruction error
    against the phantom falls and ends close to the exact-adjoint loop's."""
    cfg = make_config("c1", shrink=2)
    g, Y, vol = cfg.geom, cfg.projections(), cfg.volume()
    args = (g, Y, None, 1, [12], cfg.n_inner, cfg.step, cfg.mu, cfg.eps, cfg.omega)
    fa = fbs.fbs_reconstruct(*args)
    fb = fbs.fbs_reconstruct(*args, backprojector="eq2")
    ea, eb = np.linalg.norm(fa - vol), np.linalg.norm(fb - vol)
    assert eb < np.linalg.norm(vol) and abs(eb - ea) < 0.1 * ea, (ea, eb)
    assert fb.min() >= 0.0
