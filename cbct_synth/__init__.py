"""Seeded synthetic inputs for the CBCT TV-FBS hot path.

This module holds ONLY input generation: the scan geometry record, seeded
ellipsoid phantoms (voxelised and as analytic line integrals), Poisson/log
noise and Gaussian test fields.  It contains none of the method's arithmetic
(no projector, no adjoint, no TV, no FBS loop) and imports neither the oracle
(`oracle/`) nor the CUDA path (`paper_1002_3675_b200/`); both are fed the same
arrays produced here.

The phantoms stand in for the paper's NCAT thorax phantom and CatPhan 600 scans
(PAPER.md:101), which are not available; see DESIGN.md "Input recipe".
"""
from .geometry import Geometry
from .phantom import (
    random_ellipsoids,
    head_ellipsoids,
    voxelize,
    line_integrals,
    poisson_log,
    gaussian_field,
)
from .configs import make_config, CONFIG_NAMES, SEED_BASE

__all__ = [
    "Geometry", "random_ellipsoids", "head_ellipsoids", "voxelize", "line_integrals",
    "poisson_log", "gaussian_field", "make_config", "CONFIG_NAMES", "SEED_BASE",
]
