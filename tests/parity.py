"""Parity metrics of BASELINE.json's north_star, shared by the GPU tests, smoke() and bench.py's report.

Pure comparison arithmetic on two arrays; nothing of the method lives here.
  relative L2 norm        ||gpu - oracle||_2 / ||oracle||_2                     <= 1e-4
  per-voxel relative err  max |gpu - oracle| / oracle over {oracle > 1e-6 max}  <= 1e-3
evaluated per snapshot (time step), all bins together.
"""
from __future__ import annotations

import json
import os

import numpy as np

REL_L2_TOL = 1e-4
PER_VOXEL_TOL = 1e-3
MASK_FRACTION = 1e-6


def compare(gpu: np.ndarray, ref: np.ndarray) -> list[dict]:
    """gpu float32/64, ref float64, both [n_steps, nx, ny, nz, nb].  One dict per snapshot."""
    if gpu.shape != ref.shape:
        raise ValueError(f"shape mismatch {gpu.shape} vs {ref.shape}")
    rows = []
    for m in range(ref.shape[0]):
        r = ref[m].ravel()
        g = gpu[m].ravel().astype(np.float64)
        d = g - r
        nr = float(np.sqrt(np.dot(r, r)))
        rel_l2 = float(np.sqrt(np.dot(d, d))) / nr if nr > 0 else float(np.abs(d).max())
        mx = float(r.max())
        mask = r > MASK_FRACTION * mx
        rel = np.abs(d[mask]) / r[mask]
        dark = ~(r > 0)
        rows.append({
            "snapshot": m, "rel_l2": rel_l2, "max_voxel_rel": float(rel.max()) if rel.size else 0.0,
            "mask_voxels": int(mask.sum()), "over_tol": int((rel > PER_VOXEL_TOL).sum()), "field_max": mx,
            "nonfinite": int((~np.isfinite(g)).sum()),
            "lit_where_dark": int(np.count_nonzero(g[dark])),   # the horizon must stay exactly dark
        })
    return rows


def assert_parity(gpu, ref, what=""):
    rows = compare(gpu, ref)
    report = os.environ.get("RT_PARITY_REPORT")       # optional: append every comparison to a JSON-lines file
    if report:
        with open(report, "a") as f:
            for row in rows:
                f.write(json.dumps(dict(row, what=str(what))) + "\n")
    for row in rows:
        assert row["nonfinite"] == 0, (what, row)
        assert row["mask_voxels"] > 0, (what, row)
        assert row["rel_l2"] <= REL_L2_TOL, (what, row)
        assert row["max_voxel_rel"] <= PER_VOXEL_TOL, (what, row)
        assert row["lit_where_dark"] == 0, (what, row)
    return rows
