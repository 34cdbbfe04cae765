"""ctypes binding of libcbct.so — same names as include/cbct.h, argument marshalling only."""
from __future__ import annotations

import ctypes as C
import os
import weakref
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = None

STATUS = {0: "CBCT_OK", 1: "CBCT_ERR_INVALID_ARG", 2: "CBCT_ERR_SHAPE", 3: "CBCT_ERR_ALLOC", 4: "CBCT_ERR_CUDA"}

# every symbol include/cbct.h declares (tests check that the library exports each of them)
SYMBOLS = (
    "cbct_geometry_create", "cbct_geometry_create_ex", "cbct_set_detector_binning", "cbct_fbs_vcycle", "cbct_fdk_reconstruct",
    "cbct_fbs_reconstruct_sharded", "cbct_cascade_run", "cbct_set_projector_staging", "cbct_set_mirror_symmetry", "cbct_set_guard_mode", "cbct_check_guards", "cbct_geometry_destroy", "cbct_geometry_query", "cbct_geometry_coarsen",
    "cbct_forward", "cbct_backproject", "cbct_backproject_eq2", "cbct_set_backprojector", "cbct_tv_prox", "cbct_prolong", "cbct_restrict", "cbct_bin2x2",
    "cbct_energy", "cbct_data_gradient", "cbct_prox_step", "cbct_fbs_reconstruct", "cbct_fbs_reconstruct_until", "cbct_forward_host", "cbct_backproject_host", "cbct_tv_prox_host",
    "cbct_fbs_reconstruct_host", "cbct_tv_value_noalloc", "cbct_profile_enable", "cbct_profile_read", "cbct_launch_count", "cbct_device_bytes", "cbct_last_error",
)


# int allreduce(float *d_buf, unsigned long long count, void *user, void *cuda_stream)
ALLREDUCE_FN = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_ulonglong, C.c_void_p, C.c_void_p)


class CascadeOps(C.Structure):
    """struct cbct_cascade_ops of include/cbct.h."""
    _L = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_int)
    _fields_ = [("user", C.c_void_p),
                ("level_sizes", C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_int, C.POINTER(C.c_ulonglong), C.POINTER(C.c_ulonglong))),
                ("bin", _L), ("start", C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_int, C.c_int)), ("data_gradient", _L),
                ("all_reduce", _L), ("prox_step", C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_int, C.c_double, C.c_double)),
                ("prolong", _L)]


class CbctError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"{STATUS.get(status, status)}: {msg}")
        self.status = status


def lib_path() -> str:
    return os.path.join(_HERE, "libcbct.so")


def load():
    """Load libcbct.so (built in-tree by paper_1002_3675_b200/build.py).  No fallback."""
    global _LIB
    if _LIB is not None:
        return _LIB
    path = lib_path()
    if not os.path.exists(path):
        try:                                  # a fresh checkout: compile the CUDA path in-tree (nvcc, sm_100a); still no CPU fallback
            from . import build as _cuda_build
            _cuda_build.build()
        except Exception:
            pass
    if not os.path.exists(path):
        raise ImportError(f"{path} is missing: run `python -c 'import __graft_entry__ as g; g.build()'` "
                          "(there is no CPU fallback for the CUDA path)")
    L = C.CDLL(path)
    vp, fp, dp, ip, d, f, i = C.c_void_p, C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int), C.c_double, C.c_float, C.c_int
    L.cbct_geometry_create.argtypes = [d, d, dp, i, i, i, d, d, i, i, i, d, d, d, C.POINTER(vp)]
    L.cbct_geometry_create_ex.argtypes = [d, d, dp, i, i, i, d, d, d, d, i, i, i, d, d, d, C.POINTER(vp)]
    L.cbct_set_detector_binning.argtypes = [vp, i]
    L.cbct_set_projector_staging.argtypes = [vp, i]
    L.cbct_set_mirror_symmetry.argtypes = [vp, i]
    L.cbct_set_guard_mode.argtypes = [i]
    L.cbct_check_guards.argtypes = [vp, C.POINTER(C.c_ulonglong)]
    L.cbct_fbs_vcycle.argtypes = [vp, fp, fp, i, i, i, i, i, i, f, f, f, f, fp, dp, vp]
    L.cbct_fdk_reconstruct.argtypes = [vp, fp, fp, vp]
    L.cbct_fbs_reconstruct_sharded.argtypes = [vp, fp, fp, i, ip, i, f, f, f, f, i, ALLREDUCE_FN, vp, fp, fp, vp]
    L.cbct_cascade_run.argtypes = [C.POINTER(CascadeOps), i, ip, d, d, i, i]
    L.cbct_geometry_destroy.argtypes = [vp]
    L.cbct_geometry_destroy.restype = None
    L.cbct_geometry_query.argtypes = [vp, ip, dp]
    L.cbct_geometry_coarsen.argtypes = [vp, C.POINTER(vp), ip]
    L.cbct_forward.argtypes = [vp, fp, fp, vp]
    L.cbct_backproject.argtypes = [vp, fp, fp, vp]
    L.cbct_backproject_eq2.argtypes = [vp, fp, fp, vp]
    L.cbct_set_backprojector.argtypes = [vp, i]
    L.cbct_tv_prox.argtypes = [vp, fp, fp, f, f, f, i, vp]
    L.cbct_prolong.argtypes = [vp, fp, fp, vp]
    L.cbct_restrict.argtypes = [vp, fp, fp, vp]
    L.cbct_bin2x2.argtypes = [vp, fp, fp, vp]
    L.cbct_energy.argtypes = [vp, fp, fp, f, f, dp, vp]
    L.cbct_fbs_reconstruct.argtypes = [vp, fp, fp, i, ip, i, f, f, f, f, fp, dp, vp]
    L.cbct_data_gradient.argtypes = [vp, fp, fp, fp, vp]
    L.cbct_prox_step.argtypes = [vp, fp, fp, f, f, f, f, i, fp, vp]
    L.cbct_fbs_reconstruct_until.argtypes = [vp, fp, fp, i, ip, i, f, f, f, f, f, fp, ip, vp]
    L.cbct_forward_host.argtypes = [vp, fp, fp, vp]
    L.cbct_backproject_host.argtypes = [vp, fp, fp, vp]
    L.cbct_tv_prox_host.argtypes = [vp, fp, fp, f, f, f, i, vp]
    L.cbct_fbs_reconstruct_host.argtypes = [vp, fp, fp, i, ip, i, f, f, f, f, fp, dp, vp]
    L.cbct_tv_value_noalloc.argtypes = [fp, i, i, i, d, d, d, f, vp, vp]
    L.cbct_profile_enable.argtypes = [i]
    L.cbct_profile_read.argtypes = [dp, C.POINTER(C.c_ulonglong), i]
    L.cbct_launch_count.restype = C.c_ulonglong
    L.cbct_device_bytes.argtypes = [vp]
    L.cbct_device_bytes.restype = C.c_ulonglong
    L.cbct_last_error.restype = C.c_char_p
    _LIB = L
    return L


def _check(status: int):
    if status != 0:
        raise CbctError(status, load().cbct_last_error().decode("utf-8", "replace"))


def launch_count() -> int:
    return int(load().cbct_launch_count())


PROFILE_TAGS = ("pad_copy", "forward", "proj_prefix", "backproject", "combine", "tv_sweep", "transfers", "reductions")


def set_guard_mode(on: bool):
    """Place every device buffer allocated from now on between pattern-filled guard regions (Geometry.check_guards)."""
    _check(load().cbct_set_guard_mode(1 if on else 0))


def profile_enable(on: bool):
    _check(load().cbct_profile_enable(1 if on else 0))


def profile_read(reset: bool = True) -> dict:
    """{class name: (total ms, launch groups)} since the last reset (waits for the device)."""
    ms = (C.c_double * len(PROFILE_TAGS))()
    cnt = (C.c_ulonglong * len(PROFILE_TAGS))()
    _check(load().cbct_profile_read(ms, cnt, 1 if reset else 0))
    return {n: (float(ms[k]), int(cnt[k])) for k, n in enumerate(PROFILE_TAGS)}


def _stream(stream) -> Optional[int]:
    if stream is None:
        import torch
        return int(torch.cuda.current_stream().cuda_stream) or None
    if hasattr(stream, "cuda_stream"):
        return int(stream.cuda_stream) or None
    return int(stream) or None


def _dev(t, n: int, name: str) -> int:
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()):
        raise TypeError(f"{name}: expected a contiguous float32 CUDA tensor")
    if t.numel() != n:
        raise ValueError(f"{name}: expected {n} elements, got {t.numel()}")
    return t.data_ptr()


def _host(a, n: int, name: str) -> int:
    """Host buffer: a contiguous float32 numpy array or CPU torch tensor (pinned or not)."""
    if isinstance(a, np.ndarray):
        if a.dtype != np.float32 or not a.flags["C_CONTIGUOUS"]:
            raise TypeError(f"{name}: expected a C-contiguous float32 array")
        if a.size != n:
            raise ValueError(f"{name}: expected {n} elements, got {a.size}")
        return a.ctypes.data
    import torch
    if isinstance(a, torch.Tensor) and (not a.is_cuda) and a.dtype == torch.float32 and a.is_contiguous():
        if a.numel() != n:
            raise ValueError(f"{name}: expected {n} elements, got {a.numel()}")
        return a.data_ptr()
    raise TypeError(f"{name}: expected a host float32 buffer")


class Geometry:
    """Owning wrapper of a cbct_geometry handle (cbct_geometry_create / _destroy)."""

    def __init__(self, sad, sdd, angles, nu, nv, du, dv, nx, ny, nz, hx, hy, hz, off_u=0.0, off_v=0.0, _handle=None, _parent=None):
        L = load()
        self._parent = _parent            # coarse handles are owned by their fine handle
        self._children = []               # weak references to the coarse-level wrappers coarsen() has handed out
        if _handle is not None:
            self._h = _handle
        else:
            ang = np.ascontiguousarray(angles, dtype=np.float64)
            h = C.c_void_p()
            if off_u == 0.0 and off_v == 0.0:
                _check(L.cbct_geometry_create(float(sad), float(sdd), ang.ctypes.data_as(C.POINTER(C.c_double)),
                                              int(ang.shape[0]), int(nu), int(nv), float(du), float(dv),
                                              int(nx), int(ny), int(nz), float(hx), float(hy), float(hz), C.byref(h)))
            else:
                _check(L.cbct_geometry_create_ex(float(sad), float(sdd), ang.ctypes.data_as(C.POINTER(C.c_double)),
                                                 int(ang.shape[0]), int(nu), int(nv), float(du), float(dv), float(off_u),
                                                 float(off_v), int(nx), int(ny), int(nz), float(hx), float(hy), float(hz),
                                                 C.byref(h)))
            self._h = h
        d6 = (C.c_int * 6)()
        s5 = (C.c_double * 5)()
        _check(L.cbct_geometry_query(self._h, d6, s5))
        self.n_angles, self.nu, self.nv, self.nx, self.ny, self.nz = (int(x) for x in d6)
        self.du, self.dv, self.hx, self.hy, self.hz = (float(x) for x in s5)

    @classmethod
    def from_synth(cls, g) -> "Geometry":
        """From any record with the field names of cbct_synth.Geometry."""
        return cls(g.sad, g.sdd, g.angles, g.nu, g.nv, g.du, g.dv, g.nx, g.ny, g.nz, g.hx, g.hy, g.hz,
                   off_u=getattr(g, "off_u", 0.0), off_v=getattr(g, "off_v", 0.0))

    @property
    def n_vox(self):
        return self.nx * self.ny * self.nz

    @property
    def n_proj(self):
        return self.n_angles * self.nu * self.nv

    @property
    def vol_shape(self):
        return (self.nz, self.ny, self.nx)

    @property
    def proj_shape(self):
        return (self.n_angles, self.nv, self.nu)

    def coarsen(self):
        """(coarse Geometry [owned by self], (x, y, z coarsened, detector binned))."""
        h = C.c_void_p()
        fl = (C.c_int * 4)()
        _check(load().cbct_geometry_coarsen(self._h, C.byref(h), fl))
        c = Geometry(0, 0, None, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, _handle=h, _parent=self)
        self._children = [r for r in self._children if r() is not None] + [weakref.ref(c)]
        return c, tuple(bool(x) for x in fl)

    def _drop_children(self):
        """The library is about to free (or has freed) this handle's coarse levels: every wrapper that still points at one
        loses its pointer, so that a later use is a clean CBCT_ERR_INVALID_ARG (NULL handle) instead of a use-after-free."""
        for r in self._children:
            c = r()
            if c is not None:
                c._drop_children()
                c._h = None
        self._children = []

    def set_projector_staging(self, on: bool):
        """Projector fed by TMA-staged shared-memory bricks (True) or by the L1-cached march (False, default)."""
        _check(load().cbct_set_projector_staging(self._h, 1 if on else 0))

    def set_mirror_symmetry(self, on: bool):
        """Projector / exact backprojector: treat mirrored rays / voxel rows together where the scan is symmetric about z = 0 (True, default)."""
        _check(load().cbct_set_mirror_symmetry(self._h, 1 if on else 0))

    def check_guards(self) -> int:
        """Pattern bytes around this handle's device buffers that were overwritten (guard mode, see set_guard_mode)."""
        n = C.c_ulonglong(0)
        _check(load().cbct_check_guards(self._h, C.byref(n)))
        return int(n.value)

    def set_detector_binning(self, on: bool):
        """Coarse levels bin the detector 2x2 (default) or keep it at full resolution; drops existing coarse levels.
        Wrappers returned earlier by coarsen() on this handle (and on its coarse levels) become unusable: call coarsen() again."""
        self._drop_children()
        _check(load().cbct_set_detector_binning(self._h, 1 if on else 0))

    def device_bytes(self) -> int:
        return int(load().cbct_device_bytes(self._h))

    def close(self):
        if self._parent is None and getattr(self, "_h", None) is not None and self._h:
            self._drop_children()         # cbct_geometry_destroy frees the coarse levels with the handle
            load().cbct_geometry_destroy(self._h)
        self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def forward(g: Geometry, d_vol, d_proj, stream=None):
    _check(load().cbct_forward(g._h, _dev(d_vol, g.n_vox, "d_vol"), _dev(d_proj, g.n_proj, "d_proj"), _stream(stream)))


def backproject(g: Geometry, d_proj, d_vol, stream=None):
    _check(load().cbct_backproject(g._h, _dev(d_proj, g.n_proj, "d_proj"), _dev(d_vol, g.n_vox, "d_vol"), _stream(stream)))


def backproject_eq2(g: Geometry, d_proj, d_vol, stream=None):
    """The paper's eq. 2 backprojector without its prefactor; not the transpose of forward()."""
    _check(load().cbct_backproject_eq2(g._h, _dev(d_proj, g.n_proj, "d_proj"), _dev(d_vol, g.n_vox, "d_vol"), _stream(stream)))


BACKPROJECTOR_EXACT, BACKPROJECTOR_EQ2 = 0, 1


def set_backprojector(g: Geometry, mode: int):
    """Backprojector of step 1 in fbs_reconstruct: BACKPROJECTOR_EXACT (default) or BACKPROJECTOR_EQ2."""
    _check(load().cbct_set_backprojector(g._h, int(mode)))


def tv_prox(g: Geometry, d_g, d_u, beta, eps, omega, n_inner, stream=None):
    _check(load().cbct_tv_prox(g._h, _dev(d_g, g.n_vox, "d_g"), _dev(d_u, g.n_vox, "d_u"),
                               float(beta), float(eps), float(omega), int(n_inner), _stream(stream)))


def prolong(fine: Geometry, d_coarse, d_fine, stream=None):
    c, _ = fine.coarsen()
    _check(load().cbct_prolong(fine._h, _dev(d_coarse, c.n_vox, "d_coarse"), _dev(d_fine, fine.n_vox, "d_fine"), _stream(stream)))


def restrict(fine: Geometry, d_fine, d_coarse, stream=None):
    c, _ = fine.coarsen()
    _check(load().cbct_restrict(fine._h, _dev(d_fine, fine.n_vox, "d_fine"), _dev(d_coarse, c.n_vox, "d_coarse"), _stream(stream)))


def bin2x2(fine: Geometry, d_y, d_yc, stream=None):
    c, _ = fine.coarsen()
    _check(load().cbct_bin2x2(fine._h, _dev(d_y, fine.n_proj, "d_y"), _dev(d_yc, c.n_proj, "d_yc"), _stream(stream)))


def energy(g: Geometry, d_f, d_Y, mu, eps, stream=None):
    out = (C.c_double * 3)()
    _check(load().cbct_energy(g._h, _dev(d_f, g.n_vox, "d_f"), _dev(d_Y, g.n_proj, "d_Y"), float(mu), float(eps), out, _stream(stream)))
    return {"E_eps": out[0], "E1_eps": out[1], "E2": out[2]}


def tv_value_noalloc(d_f, hx, hy, hz, eps, d_out, stream=None):
    """cbct_tv_value_noalloc: d_out[0] = TV_eps(d_f) for callers that may not allocate device memory (an application whose
    own pool owns the whole card, a monitor beside a reconstruction that fills HBM, a loop that cannot take an allocation's
    device-wide stall).  d_f: contiguous float32 CUDA tensor of shape (nz, ny, nx), at most 512^3 voxels; d_out: CUDA
    float64 tensor with one element, supplied by the caller.  No handle; the binding allocates nothing either.  All calls
    on a GPU share one fixed scratch array: keep them ordered on one stream (or with events)."""
    import torch
    if not (isinstance(d_f, torch.Tensor) and d_f.is_cuda and d_f.dtype == torch.float32 and d_f.is_contiguous() and d_f.dim() == 3):
        raise TypeError("d_f: expected a contiguous float32 CUDA tensor of shape (nz, ny, nx)")
    if not (isinstance(d_out, torch.Tensor) and d_out.is_cuda and d_out.dtype == torch.float64 and d_out.numel() == 1):
        raise TypeError("d_out: expected a float64 CUDA tensor with one element")
    nz, ny, nx = (int(x) for x in d_f.shape)
    _check(load().cbct_tv_value_noalloc(d_f.data_ptr(), nx, ny, nz, float(hx), float(hy), float(hz), float(eps),
                                        d_out.data_ptr(), _stream(stream)))


def _outer(n_levels: int, n_outer: Sequence[int]):
    n_outer = [int(x) for x in n_outer]
    if n_levels >= 1 and len(n_outer) != n_levels:
        raise ValueError("n_outer must list one count per level, coarsest first")
    return (C.c_int * max(len(n_outer), 1))(*n_outer), sum(n_outer)    # n_levels < 1 is rejected by the library


def fbs_reconstruct(g: Geometry, d_Y, d_f0, n_levels, n_outer, n_inner, step, mu, eps, omega, d_f_out,
                    trace: bool = False, stream=None):
    arr, total = _outer(n_levels, n_outer)
    tr = (C.c_double * max(total, 1))() if trace else None
    _check(load().cbct_fbs_reconstruct(g._h, _dev(d_Y, g.n_proj, "d_Y"),
                                       None if d_f0 is None else _dev(d_f0, g.n_vox, "d_f0"),
                                       int(n_levels), arr, int(n_inner), float(step), float(mu), float(eps),
                                       float(omega), _dev(d_f_out, g.n_vox, "d_f_out"), tr, _stream(stream)))
    return list(tr)[:total] if trace else None


def fbs_vcycle(g: Geometry, d_Y, d_f0, n_levels, n_cycles, nu_pre, nu_post, nu_coarse, n_inner, step, mu, eps, omega, d_f_out,
               trace: bool = False, stream=None):
    """FAS V-cycles around Algorithm A1 (cbct_fbs_vcycle); returns E_eps after every cycle if trace."""
    tr = (C.c_double * max(int(n_cycles), 1))() if trace else None
    _check(load().cbct_fbs_vcycle(g._h, _dev(d_Y, g.n_proj, "d_Y"), None if d_f0 is None else _dev(d_f0, g.n_vox, "d_f0"),
                                  int(n_levels), int(n_cycles), int(nu_pre), int(nu_post), int(nu_coarse), int(n_inner),
                                  float(step), float(mu), float(eps), float(omega), _dev(d_f_out, g.n_vox, "d_f_out"), tr,
                                  _stream(stream)))
    return list(tr)[:int(n_cycles)] if trace else None


def fdk_reconstruct(g: Geometry, d_Y, d_vol, stream=None):
    """The FDK baseline (cbct_fdk_reconstruct): cosine pre-weight, ramp filter along u, weighted voxel-driven backprojection."""
    _check(load().cbct_fdk_reconstruct(g._h, _dev(d_Y, g.n_proj, "d_Y"), _dev(d_vol, g.n_vox, "d_vol"), _stream(stream)))


def fbs_reconstruct_sharded(g: Geometry, d_Y_local, d_f0, n_levels, n_outer, n_inner, step, mu, eps, omega, n_angles_total,
                            allreduce, d_G_scratch, d_f_out, stream=None):
    """cbct_fbs_reconstruct_sharded.  `allreduce(count)` must sum the first `count` floats of d_G_scratch over the ranks in
    place (None = single rank); it is called with the library's stream as torch's current stream, so torch.distributed
    collectives and plain torch ops inside it are ordered with the kernels around them whatever `stream` is.
    Argument marshalling only: the cascade and its constants live behind the C ABI."""
    arr, _ = _outer(n_levels, n_outer)
    gptr = _dev(d_G_scratch, g.n_vox, "d_G_scratch")
    err = []

    def _cb(d_buf, count, user, st):
        try:
            if int(d_buf) != gptr:
                raise RuntimeError("all-reduce called on a buffer that is not d_G_scratch")
            # cbct.h: the exchange must be ordered on the stream the library hands over.  torch orders its collectives (and
            # any other torch op the callback runs) against torch's CURRENT stream, so that stream is made current here
            # (NULL = the legacy default stream, which is torch's default stream).
            import torch
            s = torch.cuda.ExternalStream(int(st)) if st else torch.cuda.default_stream()
            with torch.cuda.stream(s):
                allreduce(int(count))
            return 0
        except Exception as e:            # never let an exception cross the C frame
            err.append(e)
            return 1

    cb = ALLREDUCE_FN(_cb) if allreduce is not None else C.cast(None, ALLREDUCE_FN)
    status = load().cbct_fbs_reconstruct_sharded(g._h, _dev(d_Y_local, g.n_proj, "d_Y_local"),
                                                 None if d_f0 is None else _dev(d_f0, g.n_vox, "d_f0"), int(n_levels), arr,
                                                 int(n_inner), float(step), float(mu), float(eps), float(omega),
                                                 int(n_angles_total), cb, None, gptr, _dev(d_f_out, g.n_vox, "d_f_out"),
                                                 _stream(stream))
    if err:
        raise err[0]
    _check(status)


def data_gradient(g: Geometry, d_f, d_Y, d_G, stream=None):
    """d_G = P^T (P d_f - d_Y) over this handle's angles (first half of an outer iteration)."""
    _check(load().cbct_data_gradient(g._h, _dev(d_f, g.n_vox, "d_f"), _dev(d_Y, g.n_proj, "d_Y"), _dev(d_G, g.n_vox, "d_G"),
                                     _stream(stream)))


def prox_step(g: Geometry, d_f, d_G, c, beta, eps, omega, n_inner, d_f_out, stream=None):
    """d_f_out = max(0, TVprox(d_f - c d_G)) (second half of an outer iteration)."""
    _check(load().cbct_prox_step(g._h, _dev(d_f, g.n_vox, "d_f"), _dev(d_G, g.n_vox, "d_G"), float(c), float(beta), float(eps),
                                 float(omega), int(n_inner), _dev(d_f_out, g.n_vox, "d_f_out"), _stream(stream)))


def fbs_reconstruct_until(g: Geometry, d_Y, d_f0, n_levels, n_outer_max, n_inner, step, mu, eps, omega, rel_tol, d_f_out,
                          stream=None):
    """The cascade with the stopping rule ||f_new - f_old|| <= rel_tol ||f_new|| per level; returns the
    iterations run per level (coarsest first)."""
    arr, _ = _outer(n_levels, n_outer_max)
    iters = (C.c_int * int(n_levels))()
    _check(load().cbct_fbs_reconstruct_until(g._h, _dev(d_Y, g.n_proj, "d_Y"),
                                             None if d_f0 is None else _dev(d_f0, g.n_vox, "d_f0"),
                                             int(n_levels), arr, int(n_inner), float(step), float(mu), float(eps),
                                             float(omega), float(rel_tol), _dev(d_f_out, g.n_vox, "d_f_out"), iters,
                                             _stream(stream)))
    return list(iters)


def forward_host(g: Geometry, h_vol, h_proj, stream=None):
    _check(load().cbct_forward_host(g._h, _host(h_vol, g.n_vox, "h_vol"), _host(h_proj, g.n_proj, "h_proj"), _stream(stream)))


def backproject_host(g: Geometry, h_proj, h_vol, stream=None):
    _check(load().cbct_backproject_host(g._h, _host(h_proj, g.n_proj, "h_proj"), _host(h_vol, g.n_vox, "h_vol"), _stream(stream)))


def tv_prox_host(g: Geometry, h_g, h_u, beta, eps, omega, n_inner, stream=None):
    _check(load().cbct_tv_prox_host(g._h, _host(h_g, g.n_vox, "h_g"), _host(h_u, g.n_vox, "h_u"),
                                    float(beta), float(eps), float(omega), int(n_inner), _stream(stream)))


def fbs_reconstruct_host(g: Geometry, h_Y, h_f0, n_levels, n_outer, n_inner, step, mu, eps, omega, h_f_out,
                         trace: bool = False, stream=None):
    arr, total = _outer(n_levels, n_outer)
    tr = (C.c_double * max(total, 1))() if trace else None
    _check(load().cbct_fbs_reconstruct_host(g._h, _host(h_Y, g.n_proj, "h_Y"),
                                            None if h_f0 is None else _host(h_f0, g.n_vox, "h_f0"),
                                            int(n_levels), arr, int(n_inner), float(step), float(mu), float(eps),
                                            float(omega), _host(h_f_out, g.n_vox, "h_f_out"), tr, _stream(stream)))
    return list(tr)[:total] if trace else None
