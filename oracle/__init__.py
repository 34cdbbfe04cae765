"""fp64 CPU oracle for the CBCT TV-FBS hot path — TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / `--impl reference` leg may
import this package.  It shares no code with `paper_1002_3675_b200` and never imports it.

Layout:
  cbct_oracle.c   O1 projector (Siddon merge), O2 literal-scatter transpose, brute-force
                  per-voxel clipping, O3/O4 smoothed TV value / gradient / inner descent  (C, OpenMP)
  fbs.py          O3 energy, O5 outer FBS loop, O6 multigrid cascade and its transfers      (numpy)
  fdk.py          NEXT-4: the FDK baseline (cosine pre-weight, ramp filter, weighted backprojection)    (numpy + C)
  build.py        gcc build of liboracle.so (also run by __graft_entry__.build())
See each function's docstring for the PAPER.md passage it follows.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

_lib = None


class _Geom(C.Structure):
    _fields_ = [("sad", C.c_double), ("sdd", C.c_double), ("n_angles", C.c_int),
                ("angles", C.POINTER(C.c_double)), ("nu", C.c_int), ("nv", C.c_int),
                ("du", C.c_double), ("dv", C.c_double), ("nx", C.c_int), ("ny", C.c_int),
                ("nz", C.c_int), ("hx", C.c_double), ("hy", C.c_double), ("hz", C.c_double),
                ("off_u", C.c_double), ("off_v", C.c_double)]


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        dp, ip = C.POINTER(C.c_double), C.POINTER(C.c_int)
        gp = C.POINTER(_Geom)
        L.oracle_num_threads.restype = C.c_int
        L.oracle_forward.argtypes = [gp, dp, dp]
        L.oracle_forward_rays.argtypes = [gp, dp, C.c_long, ip, ip, ip, dp]
        L.oracle_count_chords.argtypes = [gp]
        L.oracle_count_chords.restype = C.c_long
        L.oracle_backproject.argtypes = [gp, dp, dp]
        L.oracle_backproject.restype = C.c_int
        L.oracle_backproject_voxels.argtypes = [gp, dp, C.c_long, ip, ip, ip, dp]
        L.oracle_backproject_eq2.argtypes = [gp, dp, dp]
        L.oracle_backproject_eq2.restype = None
        L.oracle_fdk_backproject.argtypes = [gp, dp, C.c_double, dp]
        L.oracle_fdk_backproject.restype = None
        d, i = C.c_double, C.c_int
        L.oracle_tv_value.argtypes = [dp, i, i, i, d, d, d, d]
        L.oracle_tv_value.restype = d
        L.oracle_tv_grad.argtypes = [dp, i, i, i, d, d, d, d, dp]
        L.oracle_tv_prox.argtypes = [dp, dp, i, i, i, d, d, d, d, d, d, i]
        _lib = L
    return _lib


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def _dptr(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _iptr(a):
    return a.ctypes.data_as(C.POINTER(C.c_int))


def _geom(g):
    ang = np.ascontiguousarray(g.angles, dtype=np.float64)
    s = _Geom(float(g.sad), float(g.sdd), int(ang.shape[0]), _dptr(ang), int(g.nu), int(g.nv),
              float(g.du), float(g.dv), int(g.nx), int(g.ny), int(g.nz),
              float(g.hx), float(g.hy), float(g.hz), float(getattr(g, "off_u", 0.0)), float(getattr(g, "off_v", 0.0)))
    s._keep = ang
    return s


def _vol(g, a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    assert a.shape == tuple(g.vol_shape), (a.shape, g.vol_shape)
    return a


def _proj(g, a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    assert a.shape == tuple(g.proj_shape), (a.shape, g.proj_shape)
    return a


def forward(g, vol) -> np.ndarray:
    """O1: (P f)[theta,iv,iu] = sum_voxels (chord length) * f."""
    vol = _vol(g, vol)
    out = np.empty(g.proj_shape)
    gs = _geom(g)
    lib().oracle_forward(C.byref(gs), _dptr(vol), _dptr(out))
    return out


def forward_rays(g, vol, ia, iv, iu) -> np.ndarray:
    """O1 for a list of rays (sampled outputs at sizes where the full operator is too slow)."""
    vol = _vol(g, vol)
    ia, iv, iu = (np.ascontiguousarray(x, dtype=np.int32) for x in (ia, iv, iu))
    out = np.empty(ia.shape[0])
    gs = _geom(g)
    lib().oracle_forward_rays(C.byref(gs), _dptr(vol), ia.shape[0], _iptr(ia), _iptr(iv), _iptr(iu), _dptr(out))
    return out


def count_chords(g) -> int:
    gs = _geom(g)
    return int(lib().oracle_count_chords(C.byref(gs)))


def backproject(g, proj) -> np.ndarray:
    """O2: (P^T y)[k,j,i] = sum_rays (chord length) * y — the transpose of O1's matrix."""
    proj = _proj(g, proj)
    out = np.empty(g.vol_shape)
    gs = _geom(g)
    if lib().oracle_backproject(C.byref(gs), _dptr(proj), _dptr(out)):
        raise MemoryError("oracle_backproject: private volumes")
    return out


def backproject_voxels(g, proj, ix, iy, iz) -> np.ndarray:
    """O2 for a list of voxels by brute-force clipping of candidate rays against the voxel box."""
    proj = _proj(g, proj)
    ix, iy, iz = (np.ascontiguousarray(x, dtype=np.int32) for x in (ix, iy, iz))
    out = np.empty(ix.shape[0])
    gs = _geom(g)
    lib().oracle_backproject_voxels(C.byref(gs), _dptr(proj), ix.shape[0], _iptr(ix), _iptr(iy), _iptr(iz), _dptr(out))
    return out


def backproject_eq2(g, proj) -> np.ndarray:
    """Eq. 2 without its prefactor 2/(N_theta A):
    (B r)(x) = sum_theta L^3(u*,v*) / (L0 l^2(x)) r(u*,v*), bilinear r, zero outside the detector (Q4)."""
    proj = _proj(g, proj)
    out = np.empty(g.vol_shape)
    gs = _geom(g)
    lib().oracle_backproject_eq2(C.byref(gs), _dptr(proj), _dptr(out))
    return out


def fdk_backproject(g, q, scale: float) -> np.ndarray:
    """FDK backprojection step: scale * sum_theta SAD^2/U^2 q(u*,v*) (see oracle/fdk.py for the whole algorithm)."""
    q = _proj(g, q)
    out = np.empty(g.vol_shape)
    gs = _geom(g)
    lib().oracle_fdk_backproject(C.byref(gs), _dptr(q), float(scale), _dptr(out))
    return out


def tv_value(g, f, eps: float) -> float:
    """O3: TV_eps(f) = sum_ijk sqrt(dx^2+dy^2+dz^2+eps^2)  (PAPER.md:69 E1 times N_vox; eps=0 is the paper's)."""
    f = _vol(g, f)
    return float(lib().oracle_tv_value(_dptr(f), g.nx, g.ny, g.nz, g.hx, g.hy, g.hz, float(eps)))


def tv_grad(g, f, eps: float) -> np.ndarray:
    """O4: exact gradient of TV_eps."""
    f = _vol(g, f)
    out = np.empty(g.vol_shape)
    lib().oracle_tv_grad(_dptr(f), g.nx, g.ny, g.nz, g.hx, g.hy, g.hz, float(eps), _dptr(out))
    return out


def tv_prox(g, gvol, u0, beta: float, eps: float, omega: float, n_inner: int) -> np.ndarray:
    """O4 inner loop: n_inner Jacobi gradient-descent steps on
    TV_eps(u) + (beta/2)||u-g||^2 starting from u0."""
    gvol = _vol(g, gvol)
    u = np.array(_vol(g, u0), dtype=np.float64, copy=True)
    lib().oracle_tv_prox(_dptr(gvol), _dptr(u), g.nx, g.ny, g.nz, g.hx, g.hy, g.hz,
                         float(beta), float(eps), float(omega), int(n_inner))
    return u


from .fbs import (  # noqa: E402  (needs the primitives above)
    energy, fbs_level, fbs_reconstruct, coarsen_geometry, level_geometries,
    prolong, bin2x2, restrict_volume, lambda_max, grad_objective, fbs_vcycle,
)
from .fdk import fdk_reconstruct, fdk_preweight, fdk_ramp_kernel, fdk_filter  # noqa: E402
