"""cbct_tv_value_noalloc: the TV term of the energy for callers that may not allocate device memory.

Some users of the library cannot call cudaMalloc when they want the TV term: an application that gave the whole card to its
own memory pool, a monitor that runs beside a reconstruction which fills HBM on purpose, a loop that cannot take the
device-wide stall of an allocation.  cbct_energy is closed to them twice over (it needs a handle, and both the handle and its
reduction scratch come from cudaMalloc), so the library offers one entry point whose scratch is a fixed 128 KiB device
array inside the library image (limit: 512^3 voxels).

The file sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide the parity tests.
Each test stands on its own (fresh handle, fresh tensors), so it passes alone in a new process - where its first call is the
one that looks up the array's device address - and after the rest of the suite.
"""
import ctypes

import numpy as np
import pytest

import oracle as o
from cbct_synth import Geometry
from cbct_synth.geometry import equispaced_angles

pytestmark = pytest.mark.gpu

# Both paths add the same fp32 terms (one sqrtf per voxel) in fp64; only the order of the additions differs, which moves
# the sum by ~1e-16 * sqrt(N) relative.  1e-10 leaves room for that and is far inside the 1e-5 the energy tests allow
# against the oracle (tests/test_gpu_parity.py::test_transfers_and_energy), which is checked here as well.
RTOL_PATHS = 1e-10
RTOL_ORACLE = 1e-5
EPS = 1e-3

# (nx, ny, nz), (hx, hy, hz): 19.3 and 1.99 blocks of 8192 voxels - several blocks, ragged tails, unequal spacings.  The
# second volume is the smaller one: after the first call the shared array still holds 18 stale partial sums beyond the two
# slots the second call writes, so a call that read more of the array than it wrote would be caught.
CASES = (((70, 61, 37), (1.0, 1.25, 2.5)), ((33, 29, 17), (2.0, 2.0, 2.0)))


def _volume(shape, seed):
    rng = np.random.default_rng(seed)
    nz, ny, nx = shape
    z, y, x = np.meshgrid(np.linspace(-1, 1, nz), np.linspace(-1, 1, ny), np.linspace(-1, 1, nx), indexing="ij")
    return np.ascontiguousarray(np.exp(-3.0 * (x * x + y * y + z * z)) + 0.05 * rng.standard_normal(shape), dtype=np.float32)


def _existing_path(cb, g, d_f, dev):
    """TV_eps(f) through the path the library already had: cbct_energy on a handle (E1_eps = TV_eps / N_vox)."""
    import torch
    G = cb.Geometry.from_synth(g)
    try:
        e = cb.energy(G, d_f, torch.zeros(g.proj_shape, device=dev), 1.0, EPS)
    finally:
        G.close()
    return e["E1_eps"] * g.n_vox


def test_two_calls_in_a_row_match_the_energy_monitor(cuda_lib):
    import torch
    cb = cuda_lib
    dev = torch.device("cuda:0")
    d_out = torch.full((1,), float("nan"), dtype=torch.float64, device=dev)     # the caller brings the output
    got, want, ref = [], [], []
    vols = []
    for q, ((nx, ny, nz), (hx, hy, hz)) in enumerate(CASES):
        g = Geometry(1000., 1500., equispaced_angles(3), 16, 16, 4.0, 4.0, nx, ny, nz, hx, hy, hz)
        vol = _volume(g.vol_shape, 11 + q)
        vols.append((g, torch.from_numpy(vol).to(dev)))
        ref.append(o.tv_value(g, vol.astype(np.float64), EPS))
    # the two calls under test, back to back on one stream, nothing in between but reading the result
    for g, d_f in vols:
        cb.tv_value_noalloc(d_f, g.hx, g.hy, g.hz, EPS, d_out)
        got.append(float(d_out.cpu()[0]))
    for g, d_f in vols:
        want.append(_existing_path(cb, g, d_f, dev))
    for a, b, r in zip(got, want, ref):
        assert np.isfinite(a) and a > 0
        assert a == pytest.approx(b, rel=RTOL_PATHS)
        assert a == pytest.approx(r, rel=RTOL_ORACLE)
    # a third call on the first volume: the partial sums of the smaller volume are now in the array; the result must be the
    # first call's, bit for bit (fixed grid, fixed summation order)
    g, d_f = vols[0]
    cb.tv_value_noalloc(d_f, g.hx, g.hy, g.hz, EPS, d_out)
    assert float(d_out.cpu()[0]) == got[0]


def test_sizes_beyond_the_fixed_scratch_are_refused(cuda_lib):
    import torch
    cb = cuda_lib
    dev = torch.device("cuda:0")
    lib = cb.load()
    d_f = torch.zeros(8, device=dev)
    d_out = torch.full((1,), -1.0, dtype=torch.float64, device=dev)
    n0 = cb.launch_count()
    # 512 x 512 x 513 voxels: one plane more than the 2^27 the array covers.  Refused before anything is launched, so the
    # (far too small) input is never read and the output keeps its value.
    rc = lib.cbct_tv_value_noalloc(d_f.data_ptr(), 512, 512, 513, 1.0, 1.0, 1.0, EPS, d_out.data_ptr(), None)
    assert rc == 2 and b"512^3" in lib.cbct_last_error()
    rc = lib.cbct_tv_value_noalloc(d_f.data_ptr(), 2, 2, 0, 1.0, 1.0, 1.0, EPS, d_out.data_ptr(), None)
    assert rc == 1
    rc = lib.cbct_tv_value_noalloc(None, 2, 2, 2, 1.0, 1.0, 1.0, EPS, d_out.data_ptr(), None)
    assert rc == 1
    torch.cuda.synchronize()
    assert cb.launch_count() == n0 and float(d_out.cpu()[0]) == -1.0
    # the largest accepted chunk count boundary is cheap to hit from below: exactly one block, and one voxel more
    for n in (8192, 8193):
        v = torch.rand((1, 1, n), device=dev)
        cb.tv_value_noalloc(v, 1.0, 1.0, 1.0, EPS, d_out)
        x = v.cpu().numpy().astype(np.float32)[0, 0]
        d = np.concatenate([(x[1:] - x[:-1]), np.zeros(1, np.float32)]).astype(np.float32)
        want = np.sqrt((d * d + np.float32(EPS) * np.float32(EPS)).astype(np.float64)).sum()
        assert float(d_out.cpu()[0]) == pytest.approx(want, rel=1e-6)
