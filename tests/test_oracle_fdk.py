"""Pins for the FDK oracle (NEXT-4; Feldkamp-Davis-Kress = ref. 1 of the paper; comparison images at P:105,
P:125).  CPU only; nothing here calls the CUDA path."""
import math

import numpy as np
import pytest

import oracle as o
from cbct_synth import Geometry
from cbct_synth.geometry import equispaced_angles
from cbct_synth import phantom as ph

import bruteforce as bf


def test_preweight_hand_values():
    """3x3 detector, 300 mm pitch, SDD 1500: centre 1; edge 1500/sqrt(1500^2+300^2) = 0.98058067569092...;
    corner 1500/sqrt(1500^2+2*300^2) = 0.96225044864937... (worked by hand)."""
    g = Geometry(1000.0, 1500.0, np.array([0.0, 1.0]), 3, 3, 300.0, 300.0, 4, 4, 4, 1.0, 1.0, 1.0)
    w = o.fdk_preweight(g, np.ones(g.proj_shape))
    edge, corner = 0.980580675690920, 0.962250448649376
    want = np.array([[corner, edge, corner], [edge, 1.0, edge], [corner, edge, corner]])
    assert np.max(np.abs(w[0] - want)) <= 1e-14 and np.array_equal(w[0], w[1])
    # a panel shifted by one pixel in u: the old edge column is now the centre column
    gs = Geometry(1000.0, 1500.0, np.array([0.0]), 3, 3, 300.0, 300.0, 4, 4, 4, 1.0, 1.0, 1.0, off_u=-300.0)
    ws = o.fdk_preweight(gs, np.ones(gs.proj_shape))
    assert np.max(np.abs(ws[0][:, 2] - want[:, 1])) <= 1e-14


def test_ramp_kernel_closed_forms():
    g = Geometry(1000.0, 1500.0, np.array([0.0]), 2048, 1, 0.75, 1.0, 4, 4, 4, 1.0, 1.0, 1.0)
    D = 0.75 * 1000.0 / 1500.0
    h = o.fdk_ramp_kernel(g)
    k0 = g.nu - 1
    assert h[k0] == pytest.approx(1.0 / (4 * D * D), rel=1e-15)
    assert h[k0 + 1] == pytest.approx(-1.0 / (math.pi ** 2 * D * D), rel=1e-15) and h[k0 - 3] == pytest.approx(-1.0 / (9 * math.pi ** 2 * D * D), rel=1e-15)
    assert np.all(h[k0 + 2::2] == 0.0) and np.array_equal(h, h[::-1])
    # zero DC gain: sum_k h[k] = 1/(4 D^2) - (2/(pi^2 D^2)) (pi^2/8) = 0; the truncated sum leaves the tail ~ 1/(pi^2 D^2 nu)
    assert abs(h.sum() * D * D) <= 1.0 / (math.pi ** 2 * (g.nu - 1)) * 1.01


def test_filter_is_the_ramp_response_and_equals_fft_convolution():
    """D sum_m h[n-m] cos(2 pi nu m D) = |nu| cos(2 pi nu n D) for |nu| < 1/(2D) (the band-limited ramp), up to the
    truncation of the row; and the Toeplitz product equals the zero-padded circular convolution by numpy.fft."""
    g = Geometry(1000.0, 1500.0, np.array([0.0]), 1024, 2, 0.6, 1.0, 4, 4, 4, 1.0, 1.0, 1.0)
    D = 0.6 * 1000.0 / 1500.0
    n = np.arange(g.nu)
    for cyc in (8, 50, 200):                                    # whole cycles over the row
        nu_f = cyc / (g.nu * D)
        p = np.cos(2 * math.pi * nu_f * n * D)
        q = o.fdk_filter(g, np.stack([p, 2 * p])[None])[0]
        mid = slice(g.nu // 2 - 100, g.nu // 2 + 100)
        assert np.max(np.abs(q[0][mid] - nu_f * p[mid])) <= 2e-3 * nu_f + 2e-4
        assert np.allclose(q[1], 2 * q[0], rtol=1e-13, atol=1e-16)
    rng = np.random.default_rng(4)
    p = rng.normal(size=(1, 2, g.nu))
    h = o.fdk_ramp_kernel(g)
    L = 4 * g.nu
    hp = np.zeros(L); hp[:g.nu] = h[g.nu - 1:]; hp[-(g.nu - 1):] = h[:g.nu - 1]
    pp = np.zeros((2, L)); pp[:, :g.nu] = p[0]
    ref = D * np.fft.irfft(np.fft.rfft(pp, axis=-1) * np.fft.rfft(hp), n=L, axis=-1)[:, :g.nu]
    assert np.max(np.abs(o.fdk_filter(g, p)[0] - ref)) <= 1e-11 * np.abs(ref).max()


def test_backprojection_of_ones_is_the_closed_form_weight_integral():
    """q = 1 on a detector that covers everything: f(x) = (pi/N) sum_a SAD^2/(SAD - r cos(a - phi))^2, and for equally
    spaced views this trapezoid sum equals (1/2) int_0^2pi SAD^2/(SAD - r cos t)^2 dt = pi SAD^3/(SAD^2 - r^2)^(3/2)."""
    g = Geometry(1000.0, 1500.0, equispaced_angles(64), 64, 64, 20.0, 20.0, 8, 6, 4, 30.0, 40.0, 25.0)
    f = o.fdk_backproject(g, np.ones(g.proj_shape), math.pi / g.n_angles)
    x, y, z = g.voxel_centres_1d()
    r2 = x[None, None, :] ** 2 + y[None, :, None] ** 2 + 0 * z[:, None, None]
    ref = math.pi * g.sad ** 3 / (g.sad ** 2 - r2) ** 1.5
    assert np.max(np.abs(f - ref)) <= 1e-12 * ref.max()


def test_backprojection_equals_library_interpolation_restatement():
    g = Geometry(1000.0, 1500.0, np.array([0.3, 1.7, 4.0]), 14, 11, 3.0, 2.5, 9, 8, 6, 2.0, 2.5, 3.0, off_u=1.3, off_v=-0.7)
    q = np.random.default_rng(2).normal(size=g.proj_shape)
    a, b = o.fdk_backproject(g, q, 0.37), bf.fdk_backproject(g, q, 0.37)
    assert np.max(np.abs(a - b)) <= 1e-11 * np.abs(b).max()
    # a detector too small for the volume: voxels whose shadow falls outside get nothing from there (zero outside, Q4)
    gs = Geometry(1000.0, 1500.0, np.array([0.0]), 4, 4, 1.0, 1.0, 8, 8, 8, 0.5, 0.5, 0.5)
    fs = o.fdk_backproject(gs, np.ones(gs.proj_shape), 1.0)
    assert fs[0, 0, 0] == 0.0 and fs[4, 4, 4] > 0.0


def test_uniform_ball_reconstructs_to_its_density():
    """A centred uniform ball (radius 30 mm, density 0.02/mm) from analytic line integrals, 180 views: FDK is exact in the
    mid-plane up to discretisation (measured 0.04 %; bound 0.5 %), the cone-beam error off the mid-plane stays small, and
    the air around it is ~0.  This fixes the overall constant (dtheta/2, the pitch D in the filter, SAD^2/U^2)."""
    g = Geometry(1000.0, 1500.0, equispaced_angles(180), 128, 96, 1.5, 1.5, 48, 48, 32, 2.0, 2.0, 2.0)
    ells = np.zeros((1, 16))
    ells[0, 3:6] = 30.0
    ells[0, 6:15] = np.eye(3).ravel()
    ells[0, 15] = 0.02
    f = o.fdk_reconstruct(g, ph.line_integrals(ells, g))
    mid = f[15:17, 20:28, 20:28]
    assert abs(mid.mean() / 0.02 - 1.0) < 5e-3 and np.abs(mid / 0.02 - 1.0).max() < 1e-2
    assert abs(f[24, 24, 24] / 0.02 - 1.0) < 2e-2                      # 17 mm above the mid-plane, still inside the ball
    assert np.abs(f[16, 2:6, 2:6]).max() < 0.03 * 0.02                 # air (view-aliasing streaks of 180 views: 2 % measured)
    # symmetries of the scan: z-flip and (64 views -> 45 x 4) rotation by 90 degrees about z
    assert np.max(np.abs(f - f[::-1])) <= 1e-9 * 0.02
    assert np.max(np.abs(f - f.transpose(0, 2, 1)[:, ::-1, :])) <= 1e-9 * 0.02


def test_rot90_symmetry_on_a_random_scan():
    """Shifting the view index by a quarter turn rotates the reconstruction by 90 degrees about z (equally spaced
    views over 360 degrees)."""
    g = Geometry(1000.0, 1500.0, equispaced_angles(8), 20, 12, 3.0, 3.0, 10, 10, 6, 2.5, 2.5, 3.0)
    Y = np.random.default_rng(6).normal(size=g.proj_shape)
    f = o.fdk_reconstruct(g, Y)
    fr = o.fdk_reconstruct(g, np.roll(Y, 2, axis=0))         # view a now holds what view a - 90 deg saw: the object turned by +90 deg
    # rotation by +90 deg about z: f_rot(x, y) = f(y, -x)  ->  array [k][j][i] = f[k][nx-1-i][j]
    want = f.transpose(0, 2, 1)[:, :, ::-1]
    assert np.max(np.abs(fr - want)) <= 1e-12 * np.abs(f).max()
