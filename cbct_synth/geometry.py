"""Scan geometry record shared by the input generators, the oracle binding and the
CUDA binding (a plain data holder; SURVEY.md §8(c) O0 / DESIGN.md "Geometry").

Lengths are mm.  Rotation axis is z.  For projection angle theta:
  source          S = (SAD cos t, SAD sin t, 0)
  detector centre C = -(SDD - SAD) (cos t, sin t, 0)
  detector axes   u^ = (-sin t, cos t, 0),  v^ = (0, 0, 1)
  pixel (iu, iv) centre  D = C + ((iu-(nu-1)/2) du + off_u) u^ + ((iv-(nv-1)/2) dv + off_v) v^
  (off_u, off_v: in-plane shift of the detector panel in mm, 0 for the centred full-fan scans of the
  configs; a half-fan scan shifts the panel along u)
The volume is centred at the origin; voxel (i,j,k) is the box
  [ (i-nx/2) hx, (i+1-nx/2) hx ] x [ (j-ny/2) hy, ... ] x [ (k-nz/2) hz, ... ].
Array layouts: volume f[k][j][i] (x fastest), projections Y[theta][iv][iu] (u fastest).
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace

import numpy as np


@dataclass(frozen=True)
class Geometry:
    sad: float
    sdd: float
    angles: np.ndarray = field(repr=False)  # radians, float64, any list
    nu: int = 0
    nv: int = 0
    du: float = 1.0
    dv: float = 1.0
    nx: int = 0
    ny: int = 0
    nz: int = 0
    hx: float = 1.0
    hy: float = 1.0
    hz: float = 1.0
    off_u: float = 0.0
    off_v: float = 0.0

    def __post_init__(self):
        object.__setattr__(self, "angles", np.ascontiguousarray(self.angles, dtype=np.float64))

    @property
    def n_angles(self) -> int:
        return int(self.angles.shape[0])

    @property
    def vol_shape(self):
        return (self.nz, self.ny, self.nx)

    @property
    def proj_shape(self):
        return (self.n_angles, self.nv, self.nu)

    @property
    def n_vox(self) -> int:
        return self.nx * self.ny * self.nz

    @property
    def n_pix(self) -> int:
        return self.nu * self.nv

    @property
    def n_rays(self) -> int:
        return self.n_angles * self.n_pix

    def with_angles(self, angles) -> "Geometry":
        return replace(self, angles=np.asarray(angles, dtype=np.float64))

    # --- positions used by the analytic-projection generator ------------------
    def source(self, ia: int) -> np.ndarray:
        t = self.angles[ia]
        return np.array([self.sad * np.cos(t), self.sad * np.sin(t), 0.0])

    def pixel_centres(self, ia: int) -> np.ndarray:
        """(nv, nu, 3) array of detector pixel centres for angle index ia."""
        t = self.angles[ia]
        c, s = np.cos(t), np.sin(t)
        uu = (np.arange(self.nu) - (self.nu - 1) / 2.0) * self.du + self.off_u
        vv = (np.arange(self.nv) - (self.nv - 1) / 2.0) * self.dv + self.off_v
        cen = -(self.sdd - self.sad) * np.array([c, s, 0.0])
        out = np.empty((self.nv, self.nu, 3))
        out[..., 0] = cen[0] + uu[None, :] * (-s)
        out[..., 1] = cen[1] + uu[None, :] * c
        out[..., 2] = vv[:, None]
        return out

    def voxel_centres_1d(self):
        x = (np.arange(self.nx) - (self.nx - 1) / 2.0) * self.hx
        y = (np.arange(self.ny) - (self.ny - 1) / 2.0) * self.hy
        z = (np.arange(self.nz) - (self.nz - 1) / 2.0) * self.hz
        return x, y, z


def equispaced_angles(n: int) -> np.ndarray:
    """n angles equally spaced over a full 360 degree rotation."""
    return 2.0 * np.pi * np.arange(n, dtype=np.float64) / n
