"""NEXT-4: Algorithm A1 with the angle list partitioned over ranks.

Every rank holds the whole volume and its share of the angles and of Y.  One outer iteration is
    G_r = P_r^T (P_r f - Y_r)              on every rank (exact partial sum of P^T (P f - Y))
    G   = sum_r G_r                          ONE all-reduce of a volume-sized fp32 buffer (NCCL over NVLink / NVSwitch)
    f   = max(0, TVprox(f - c G))            on every rank, identically
with c = 2 step N_vox / (N_theta N_pix) from the TOTAL number of angles, inside the same coarse-to-fine cascade as
cbct_fbs_reconstruct.  The cascade, its constants and the two halves all live behind the C ABI
(cbct_fbs_reconstruct_sharded / cbct_cascade_run, csrc/cascade.cu); this module only partitions the angle list and wires
torch.distributed's all_reduce to the library's exchange callback.
"""
from __future__ import annotations

import numpy as np


def shard_angles(n_angles: int, rank: int, world: int) -> np.ndarray:
    """Indices of the angles rank `rank` owns: strided, so that every rank sees both ray classes
    (x-major / y-major) and the same amount of work for equally spaced scans."""
    if not (0 <= rank < world):
        raise ValueError("rank outside [0, world)")
    return np.arange(rank, n_angles, world)


def fbs_reconstruct_sharded(geometry, d_Y_local, d_f0, n_levels, n_outer, n_inner, step, mu, eps, omega, n_angles_total,
                            dist=None, stream=None):
    """Runs the sharded cascade on this rank (geometry = a handle over this rank's angles, d_Y_local their data) and returns
    the finest-level volume.  dist = torch.distributed (initialised) or None for a single rank."""
    import torch
    from . import binding as cb
    G = torch.empty(geometry.vol_shape, device=d_Y_local.device, dtype=torch.float32)     # the exchanged gradient volume
    out = torch.empty(geometry.vol_shape, device=d_Y_local.device, dtype=torch.float32)
    flat = G.view(-1)
    allreduce = None
    if dist is not None:
        def allreduce(count):
            dist.all_reduce(flat[:count], op=dist.ReduceOp.SUM)
    cb.fbs_reconstruct_sharded(geometry, d_Y_local, d_f0, n_levels, n_outer, n_inner, step, mu, eps, omega, n_angles_total,
                               allreduce, G, out, stream=stream)
    return out
