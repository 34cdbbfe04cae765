"""The five BASELINE.json workloads (c1..c5) as seeded synthetic configurations.

Shapes follow BASELINE.json:configs / SURVEY.md §8(d); everything the configs leave
open (eps, omega, mu, step) is fixed here once and handed unchanged to BOTH the oracle and
the CUDA path.  `shrink=k` divides every grid dimension by k and multiplies voxel and pixel
sizes by k (same physical scene, same ellipsoids): the sizes the fp64 oracle can run the
full loop on in seconds.
"""
from __future__ import annotations

import json
import os
from dataclasses import dataclass, field
from typing import List, Optional

import numpy as np

from .geometry import Geometry, equispaced_angles
from . import phantom as ph

SEED_BASE = 10023675          # + config index
CONFIG_NAMES = ("c1", "c2", "c3", "c4", "c5")
_FROZEN = os.path.join(os.path.dirname(__file__), "frozen_params.json")


@dataclass
class Config:
    name: str
    seed: int
    geom: Geometry
    ells: np.ndarray = field(repr=False)
    n_levels: int = 1
    n_outer: List[int] = field(default_factory=lambda: [1])   # coarsest level first
    n_inner: int = 10
    eps: float = 1e-4        # TV smoothing, units of f/mm
    omega: float = 1.0       # inner step relaxation
    mu: float = 1.0          # data weight of eq. 1
    step: float = 1e-5       # s = mu/beta, mm^-2
    I0: Optional[float] = None   # photons / pixel; None = noiseless

    @property
    def beta(self) -> float:
        return self.mu / self.step

    def volume(self, dtype=np.float64) -> np.ndarray:
        return ph.voxelize(self.ells, self.geom, dtype=dtype)

    def clean_projections(self, angle_indices=None) -> np.ndarray:
        return ph.line_integrals(self.ells, self.geom, angle_indices)

    def projections(self, angle_indices=None) -> np.ndarray:
        """The observed data Y: analytic line integrals, Poisson/log noise if I0 is set.  Every view draws its
        noise from its own stream seeded by (config seed, view index), so a subset of the views (an angle shard of
        a multi-GPU run, a sampled sub-problem) is exactly that part of the one full noisy scan."""
        p = self.clean_projections(angle_indices)
        if self.I0 is None:
            return p
        idx = range(self.geom.n_angles) if angle_indices is None else list(angle_indices)
        out = np.empty_like(p)
        for n, ia in enumerate(idx):
            out[n] = ph.poisson_log(p[n], self.I0, np.random.default_rng([self.seed + 7919, int(ia)]))
        return out


def s_max_estimate(g: Geometry) -> float:
    """A / (V * D_max * M_max^2): a (safe, ~2x low) estimate of the FBS step bound
    s_max = N_theta N_pix / (N_vox lambda_max(P^T P))."""
    A = g.nu * g.du * g.nv * g.dv
    ex, ey, ez = g.nx * g.hx, g.ny * g.hy, g.nz * g.hz
    V = ex * ey * ez
    D = float(np.sqrt(ex * ex + ey * ey + ez * ez))
    r = 0.5 * float(np.hypot(ex, ey))
    M = g.sdd / max(g.sad - r, 1e-9)
    return A / (V * D * M * M)


def _frozen(name: str, shrink: int) -> dict:
    try:
        with open(_FROZEN) as fh:
            return json.load(fh).get(f"{name}/{shrink}", {})
    except FileNotFoundError:
        return {}


def make_config(name: str, shrink: int = 1, n_angles: Optional[int] = None) -> Config:
    idx = CONFIG_NAMES.index(name)
    seed = SEED_BASE + idx + 1
    rng = np.random.default_rng(seed)
    k = int(shrink)
    sad, sdd = 1000.0, 1500.0

    def geom(nx, ny, nz, hx, hy, hz, na, nu, nv, du, dv):
        assert nx % k == 0 and ny % k == 0 and nz % k == 0 and nu % k == 0 and nv % k == 0
        return Geometry(sad, sdd, equispaced_angles(n_angles or na), nu // k, nv // k, du * k, dv * k,
                        nx // k, ny // k, nz // k, hx * k, hy * k, hz * k)

    if name == "c1":
        g = geom(32, 32, 32, 2.0, 2.0, 2.0, 16, 64, 64, 1.5, 1.5)
        ells = ph.random_ellipsoids(rng, 10, (64.0, 64.0, 64.0), (2.0, 12.0))
        cfg = Config(name, seed, g, ells, n_levels=1, n_outer=[20], n_inner=5, I0=None)
    elif name == "c2":
        g = geom(256, 256, 256, 1.0, 1.0, 1.0, 40, 512, 384, 0.78, 0.78)
        ells = ph.random_ellipsoids(rng, 20, (256.0, 256.0, 256.0), (0.0625 * 128, 0.375 * 128))
        cfg = Config(name, seed, g, ells, n_levels=1, n_outer=[1], n_inner=10, I0=None)
    elif name in ("c3", "c4"):
        na = 40 if name == "c3" else 20
        g = geom(512, 512, 64, 0.5, 0.5, 2.5, na, 512, 384, 0.78, 0.78)
        # c4 uses "the same phantom" as c3 (BASELINE.json): same seed stream for the ellipsoids
        ells = ph.head_ellipsoids(np.random.default_rng(SEED_BASE + 3), 28)
        if name == "c3":
            cfg = Config(name, seed, g, ells, n_levels=2, n_outer=[100, 100], n_inner=10, I0=1e5)
        else:
            cfg = Config(name, seed, g, ells, n_levels=3, n_outer=[100, 100, 100], n_inner=10, I0=2.5e4)
    elif name == "c5":
        g = geom(512, 512, 512, 0.5, 0.5, 0.5, 360, 1024, 768, 0.4, 0.4)
        ells = ph.random_ellipsoids(rng, 50, (256.0, 256.0, 256.0), (0.0625 * 128, 0.375 * 128),
                                    centre_frac=(0.7, 0.7, 0.5))
        cfg = Config(name, seed, g, ells, n_levels=3, n_outer=[50, 50, 50], n_inner=10, I0=1e5)
    else:
        raise ValueError(name)

    # parameters the configs leave open ("mu fixed"): see DESIGN.md "Input recipe".
    cfg.eps = 1e-4
    cfg.omega = 1.0
    cfg.step = 0.5 * s_max_estimate(cfg.geom)         # gamma ~ 0.5 with the safe estimate
    K = 4.0 * (1 / g.hx ** 2 + 1 / g.hy ** 2 + 1 / g.hz ** 2)
    cfg.mu = cfg.step * K / cfg.eps                   # dt*beta = 0.5 (quadratic-dominated inner step)
    fz = _frozen(name, k)                             # oracle-tuned overrides (oracle/tune_params.py)
    for key in ("step", "mu", "eps", "omega"):
        if key in fz:
            setattr(cfg, key, float(fz[key]))
    return cfg
