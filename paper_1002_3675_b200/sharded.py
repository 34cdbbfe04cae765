"""NEXT-4: Algorithm A1 with the angle list partitioned over ranks.

Every rank holds the whole volume and its share of the angles and of Y.  One outer iteration is
    G_r = P_r^T (P_r f - Y_r)              on every rank (cbct_data_gradient: exact partial sum of P^T (P f - Y))
    G   = sum_r G_r                          ONE all-reduce of a volume-sized fp32 buffer (NCCL over NVLink / NVSwitch)
    f   = max(0, TVprox(f - c G))            on every rank, identically (cbct_prox_step)
with c = 2 step N_vox / (N_theta N_pix) from the TOTAL number of angles, inside the same coarse-to-fine cascade
as cbct_fbs_reconstruct.  This module holds the host-side driver only (no arithmetic of the method): the two
halves run in the CUDA kernels behind the C ABI, the exchange is torch.distributed's all_reduce.  The driver is
written against a small `ops` interface so that its logic (partition, constants, level order, exchange) is
covered on CPU with world_size 2 over gloo (tests/test_multi_rank.py).
"""
from __future__ import annotations

from typing import List, Optional, Sequence

import numpy as np


def shard_angles(n_angles: int, rank: int, world: int) -> np.ndarray:
    """Indices of the angles rank `rank` owns: strided, so that every rank sees both ray classes
    (x-major / y-major) and the same amount of work for equally spaced scans."""
    if not (0 <= rank < world):
        raise ValueError("rank outside [0, world)")
    return np.arange(rank, n_angles, world)


def fbs_reconstruct_sharded(ops, Y_local, f0, n_levels: int, n_outer: Sequence[int], n_inner: int, step: float,
                            mu: float, eps: float, omega: float, n_angles_total: int, dist=None):
    """Runs the cascade on this rank's share.  `ops` provides, per level l (0 = finest):
         ops.n_vox(l), ops.n_pix(l)                      sizes
         ops.bin(l, Y_l) -> Y_{l+1}                      2x2 binning of this rank's data to the next coarser level
         ops.zeros(l), ops.restrict(l, f_l) -> f_{l+1}   start volume
         ops.data_gradient(l, f, Y_l) -> G               partial gradient over this rank's angles
         ops.all_reduce(G, dist)                         in-place sum over ranks (no-op if dist is None)
         ops.prox_step(l, f, G, c, beta, eps, omega, n_inner) -> f
         ops.prolong(l, f_{l+1}) -> f_l
       n_outer is listed coarsest first, as in cbct_fbs_reconstruct.  Returns the finest-level volume."""
    if len(n_outer) != n_levels:
        raise ValueError("n_outer must list one count per level (coarsest first)")
    Ys: List = [Y_local]
    for l in range(n_levels - 1):
        Ys.append(ops.bin(l, Ys[-1]))
    L = n_levels - 1
    if f0 is None:
        f = ops.zeros(L)
    else:
        f = f0
        for l in range(L):
            f = ops.restrict(l, f)
    beta = mu / step
    for n, l in enumerate(range(L, -1, -1)):
        c = 2.0 * step * ops.n_vox(l) / (n_angles_total * ops.n_pix(l))
        for _ in range(n_outer[n]):
            G = ops.data_gradient(l, f, Ys[l])
            ops.all_reduce(G, dist)
            f = ops.prox_step(l, f, G, c, beta, eps, omega, n_inner)
        if l > 0:
            f = ops.prolong(l - 1, f)
    return f


class CudaOps:
    """`ops` on the CUDA path: one Geometry handle per level holding this rank's angles; torch tensors on the
    current device; the exchange is torch.distributed.all_reduce (NCCL) on the launching stream's tensor."""

    def __init__(self, geometry, n_levels: int, stream=None):
        import torch
        from . import binding as cb
        self.cb, self.torch, self.stream = cb, torch, stream
        self.levels = [geometry]
        for _ in range(n_levels - 1):
            self.levels.append(self.levels[-1].coarsen()[0])

    def n_vox(self, l):
        return self.levels[l].n_vox

    def n_pix(self, l):
        g = self.levels[l]
        return g.nu * g.nv

    def _vol(self, l):
        return self.torch.empty(self.levels[l].vol_shape, device="cuda", dtype=self.torch.float32)

    def zeros(self, l):
        return self.torch.zeros(self.levels[l].vol_shape, device="cuda", dtype=self.torch.float32)

    def bin(self, l, Y):
        out = self.torch.empty(self.levels[l + 1].proj_shape, device="cuda", dtype=self.torch.float32)
        self.cb.bin2x2(self.levels[l], Y, out, stream=self.stream)
        return out

    def restrict(self, l, f):
        out = self._vol(l + 1)
        self.cb.restrict(self.levels[l], f, out, stream=self.stream)
        return out

    def prolong(self, l, fc):
        out = self._vol(l)
        self.cb.prolong(self.levels[l], fc, out, stream=self.stream)
        return out

    def data_gradient(self, l, f, Y):
        G = self._vol(l)
        self.cb.data_gradient(self.levels[l], f, Y, G, stream=self.stream)
        return G

    def all_reduce(self, G, dist):
        if dist is not None:
            dist.all_reduce(G, op=dist.ReduceOp.SUM)

    def prox_step(self, l, f, G, c, beta, eps, omega, n_inner):
        out = self._vol(l)
        self.cb.prox_step(self.levels[l], f, G, c, beta, eps, omega, n_inner, out, stream=self.stream)
        return out
