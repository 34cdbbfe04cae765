"""Committed script that writes cbct_synth/frozen_params.json from the ORACLE ONLY (never the CUDA path):
exact chord counts of the system matrix per config (work units for the roofline arithmetic) and the
power-iteration estimate of lambda_max(P^T P) on a shrunk copy of each scene (the FBS step bound
s_max = N_theta N_pix / (N_vox lambda_max) is level-independent).

  python -m oracle.tune_params            # a few minutes on 8 cores
"""
from __future__ import annotations

import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import oracle as o
from cbct_synth import make_config
from cbct_synth.configs import s_max_estimate

OUT = os.path.join(ROOT, "cbct_synth", "frozen_params.json")


def main():
    out = {}
    for name, shrink_lam in (("c1", 1), ("c2", 4), ("c3", 4), ("c4", 4), ("c5", 8)):
        cfg = make_config(name)
        g = cfg.geom
        rec = {}
        if name in ("c1", "c2", "c3", "c4"):
            rec["nnz"] = o.count_chords(g)
            gc, _, _ = o.coarsen_geometry(g)
            rec["nnz_coarse_ratio"] = o.count_chords(gc) / rec["nnz"]
        gs = make_config(name, shrink=shrink_lam).geom
        lam = o.lambda_max(gs, iters=30, seed=1)
        rec["s_max_power_iteration"] = gs.n_angles * gs.n_pix / (gs.n_vox * lam)
        rec["s_max_estimate"] = s_max_estimate(g)
        out[f"{name}/1"] = rec
        print(name, rec, flush=True)
    with open(OUT, "w") as fh:
        json.dump(out, fh, indent=1, sort_keys=True)


if __name__ == "__main__":
    main()
