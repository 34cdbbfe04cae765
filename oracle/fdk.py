"""Oracle for NEXT-4: the FDK reconstruction the paper compares against (Feldkamp, Davis, Kress 1984 = ref. 1 at
PAPER.md:147; "the image reconstructed by the conventional FDK algorithm", Fig. 1(d) at P:105 and Fig. 2 at P:125).
TEST INFRASTRUCTURE — see oracle/__init__.py.  Plain fp64, step by step:

  1. cosine pre-weight     p1[a,v,u] = Y[a,v,u] * SDD / sqrt(SDD^2 + us^2 + vs^2),   (us, vs) = pixel centre on the imager
  2. ramp filter along u   q[a,v,n]  = D * sum_m h[n-m] p1[a,v,m],   D = du * SAD/SDD (pixel pitch scaled to the axis),
                           h[0] = 1/(4 D^2),  h[k] = 0 (k even),  h[k] = -1/(pi^2 k^2 D^2) (k odd)     (band-limited ramp)
  3. backprojection        f(x) = (dtheta/2) sum_a SAD^2/U^2 q[a](u*, v*),   U = SAD - (x cos a + y sin a),
                           (u*, v*) = SDD (lat, z)/U, bilinear, zero outside the detector;  dtheta = 2 pi / N_theta.

Reading (Q22; the paper only names the algorithm): equally spaced views over a full rotation (the factor 1/2
is the 360-degree redundancy), no short-scan (Parker) or half-fan redundancy weights, no apodisation window.
"""
from __future__ import annotations

import math

import numpy as np


def fdk_preweight(g, Y: np.ndarray) -> np.ndarray:
    """Step 1: Y * cos(angle between the ray and the central ray)."""
    us = (np.arange(g.nu) - (g.nu - 1) / 2.0) * g.du + getattr(g, "off_u", 0.0)
    vs = (np.arange(g.nv) - (g.nv - 1) / 2.0) * g.dv + getattr(g, "off_v", 0.0)
    w = g.sdd / np.sqrt(g.sdd ** 2 + us[None, :] ** 2 + vs[:, None] ** 2)
    return np.asarray(Y, dtype=np.float64) * w[None]


def fdk_ramp_kernel(g) -> np.ndarray:
    """h[k] for k = -(nu-1) .. nu-1 (index k + nu - 1), pitch D = du SAD/SDD."""
    D = g.du * g.sad / g.sdd
    k = np.arange(-(g.nu - 1), g.nu)
    h = np.zeros(k.shape)
    h[k == 0] = 1.0 / (4.0 * D * D)
    odd = (k % 2) != 0
    h[odd] = -1.0 / (math.pi ** 2 * k[odd].astype(np.float64) ** 2 * D * D)
    return h


def fdk_filter(g, p1: np.ndarray) -> np.ndarray:
    """Step 2: q[...,n] = D sum_m h[n-m] p1[...,m] — the convolution sum written as a product with the Toeplitz matrix
    T[n,m] = h[n-m]."""
    D = g.du * g.sad / g.sdd
    h = fdk_ramp_kernel(g)
    n = np.arange(g.nu)
    T = h[(n[:, None] - n[None, :]) + g.nu - 1]
    return D * (np.asarray(p1, dtype=np.float64) @ T.T)


def fdk_reconstruct(g, Y: np.ndarray) -> np.ndarray:
    import oracle as o
    q = fdk_filter(g, fdk_preweight(g, Y))
    return o.fdk_backproject(g, q, math.pi / g.n_angles)
