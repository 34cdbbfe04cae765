"""Seeded ellipsoid phantoms: voxelised volumes, analytic line integrals, noise.

An ellipsoid is a row of 16 float64: centre (3, mm), semi-axes (3, mm), rotation
matrix R row-major (9; columns are the ellipsoid's principal axes in world
coordinates) and the attenuation increment (1, 1/mm).  Phantoms are ADDITIVE:
the attenuation at a point is the sum of the increments of all ellipsoids that
contain it.  Recipe and the workloads it stands in for: SURVEY.md §8(d),
DESIGN.md "Input recipe".
"""
from __future__ import annotations

import numpy as np

from .geometry import Geometry

ATT_SCALE = 0.02  # 1/mm per unit density, so that line integrals stay <~ 5


def _random_rotations(rng: np.random.Generator, n: int) -> np.ndarray:
    """Uniform random rotations from uniform unit quaternions."""
    q = rng.normal(size=(n, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    w, x, y, z = q[:, 0], q[:, 1], q[:, 2], q[:, 3]
    R = np.empty((n, 3, 3))
    R[:, 0, 0] = 1 - 2 * (y * y + z * z)
    R[:, 0, 1] = 2 * (x * y - z * w)
    R[:, 0, 2] = 2 * (x * z + y * w)
    R[:, 1, 0] = 2 * (x * y + z * w)
    R[:, 1, 1] = 1 - 2 * (x * x + z * z)
    R[:, 1, 2] = 2 * (y * z - x * w)
    R[:, 2, 0] = 2 * (x * z - y * w)
    R[:, 2, 1] = 2 * (y * z + x * w)
    R[:, 2, 2] = 1 - 2 * (x * x + y * y)
    return R


def _pack(centres, semis, R, dens) -> np.ndarray:
    n = centres.shape[0]
    out = np.empty((n, 16))
    out[:, 0:3] = centres
    out[:, 3:6] = semis
    out[:, 6:15] = R.reshape(n, 9)
    out[:, 15] = dens
    return out


def random_ellipsoids(rng, n, extent_mm, semi_range_mm, dens_range=(0.1, 1.0),
                      centre_frac=(0.7, 0.7, 0.7)) -> np.ndarray:
    """n ellipsoids: centres uniform in the inner `centre_frac` of the volume extent,
    semi-axes U[semi_range], densities U[dens_range] (x ATT_SCALE), random rotations."""
    ext = np.asarray(extent_mm, dtype=np.float64)
    frac = np.asarray(centre_frac, dtype=np.float64)
    centres = (rng.random((n, 3)) - 0.5) * ext * frac
    semis = rng.uniform(semi_range_mm[0], semi_range_mm[1], size=(n, 3))
    R = _random_rotations(rng, n)
    dens = rng.uniform(dens_range[0], dens_range[1], size=n) * ATT_SCALE
    return _pack(centres, semis, R, dens)


def head_ellipsoids(rng, n_small=28) -> np.ndarray:
    """'Head-like' phantom of SURVEY.md §8(d) c3: outer ellipsoid (88,110,72) mm density +1.0,
    inner (82,104,66) mm density -0.8 (shell 1.0, interior 0.2), then n_small small ellipsoids
    inside with increments U[0,0.2] (interior stays 0.2..0.6 where at most two overlap)."""
    eye = np.eye(3)[None]
    big = _pack(np.zeros((2, 3)), np.array([[88.0, 110.0, 72.0], [82.0, 104.0, 66.0]]),
                np.repeat(eye, 2, 0), np.array([1.0, -0.8]) * ATT_SCALE)
    # small ones: centres inside the inner ellipsoid scaled by 0.6 so they stay interior
    c = rng.normal(size=(n_small, 3))
    c /= np.linalg.norm(c, axis=1, keepdims=True)
    c *= rng.random((n_small, 1)) ** (1.0 / 3.0)
    centres = c * np.array([82.0, 104.0, 66.0]) * 0.6
    semis = rng.uniform(6.0, 24.0, size=(n_small, 3))
    R = _random_rotations(rng, n_small)
    dens = rng.uniform(0.0, 0.2, size=n_small) * ATT_SCALE
    return np.concatenate([big, _pack(centres, semis, R, dens)], axis=0)


def voxelize(ells: np.ndarray, geom: Geometry, dtype=np.float64) -> np.ndarray:
    """Volume f[k][j][i] sampled at voxel centres (additive ellipsoids)."""
    x, y, z = geom.voxel_centres_1d()
    vol = np.zeros(geom.vol_shape, dtype=np.float64)
    for e in ells:
        c, a, R, rho = e[0:3], e[3:6], e[6:15].reshape(3, 3), e[15]
        rad = float(np.max(a))
        ix = np.nonzero(np.abs(x - c[0]) <= rad)[0]
        iy = np.nonzero(np.abs(y - c[1]) <= rad)[0]
        iz = np.nonzero(np.abs(z - c[2]) <= rad)[0]
        if ix.size == 0 or iy.size == 0 or iz.size == 0:
            continue
        sx, sy, sz = slice(ix[0], ix[-1] + 1), slice(iy[0], iy[-1] + 1), slice(iz[0], iz[-1] + 1)
        dx = (x[sx] - c[0])[None, None, :]
        dy = (y[sy] - c[1])[None, :, None]
        dz = (z[sz] - c[2])[:, None, None]
        # local coordinates p = R^T (x - c), scaled by 1/a
        q = np.zeros((iz.size, iy.size, ix.size))
        for m in range(3):
            pm = (R[0, m] * dx + R[1, m] * dy + R[2, m] * dz) / a[m]
            q += pm * pm
        vol[sz, sy, sx] += rho * (q <= 1.0)
    return vol.astype(dtype, copy=False)


def line_integrals(ells: np.ndarray, geom: Geometry, angle_indices=None) -> np.ndarray:
    """Analytic line integrals through the additive ellipsoids for every detector pixel
    (closed-form chord of a line through an ellipsoid; SURVEY.md §8(c) pin I3):
    o' = diag(a)^-1 R^T (o-c), d' = diag(a)^-1 R^T d^, chord = 2 sqrt(B^2 - A C)/A."""
    if angle_indices is None:
        angle_indices = range(geom.n_angles)
    angle_indices = list(angle_indices)
    out = np.zeros((len(angle_indices), geom.nv, geom.nu))
    for n, ia in enumerate(angle_indices):
        S = geom.source(ia)
        D = geom.pixel_centres(ia)               # (nv,nu,3)
        d = D - S
        d /= np.linalg.norm(d, axis=-1, keepdims=True)
        acc = out[n]
        for e in ells:
            c, a, R, rho = e[0:3], e[3:6], e[6:15].reshape(3, 3), e[15]
            o_l = (R.T @ (S - c)) / a            # (3,)
            d_l = (d @ R) / a                    # (nv,nu,3): rows are R^T d
            A = np.einsum("...k,...k->...", d_l, d_l)
            B = d_l @ o_l
            C = float(o_l @ o_l) - 1.0
            disc = B * B - A * C
            np.maximum(disc, 0.0, out=disc)
            acc += rho * 2.0 * np.sqrt(disc) / A
    return out


def poisson_log(p: np.ndarray, I0: float, rng: np.random.Generator) -> np.ndarray:
    """Noisy log-transformed data: N ~ Poisson(I0 exp(-p)), Y = -ln(max(N,1)/I0)."""
    N = rng.poisson(I0 * np.exp(-p)).astype(np.float64)
    return -np.log(np.maximum(N, 1.0) / I0)


def gaussian_field(shape, seed: int) -> np.ndarray:
    """Seeded N(0,1) field (adjoint dot-product tests)."""
    return np.random.default_rng(seed).normal(size=shape)
