"""Writes tests/golden/cfg0_H_rows.npz: rows H[node, :, :] of the ORACLE's H table for config 0
(BASELINE.json configs[0]: 32^3 grid, nt = 128, dt = 10 ps, 40 Euler substeps per output step) at a
fixed set of sampled nodes.  Calls only oracle/ and wtide_inputs/ (about two minutes of CPU).

    python tests/golden/make_cfg0_golden.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import wtide_oracle as wo  # noqa: E402
from wtide_inputs import geometry_desc  # noqa: E402


def sample_nodes(shape, n=64, seed=0):
    rng = np.random.default_rng(seed)
    nodes = np.stack([rng.integers(0, s, n) for s in shape], axis=1)
    # plus a few structured ones: on the readout column axis, next to it, on the bias column, mid-cell
    nx, ny, nz = shape
    extra = [(nx // 2, ny // 2, 0), (nx // 2, ny // 2, nz // 2), (nx // 2 + 3, ny // 2, nz // 2), (0, 0, nz - 1),
             (nx // 4, ny // 4, nz // 2), (nx // 2 + 4, ny // 2 + 1, 1), (1, 0, nz // 3), (nx - 1, ny - 1, 5)]
    return np.concatenate([nodes, np.array(extra)], axis=0)


if __name__ == "__main__":
    d = geometry_desc(0)
    H = wo.solve_H_from_desc(d)
    nodes = sample_nodes((d["nx"], d["ny"], d["nz"]))
    rows = H[nodes[:, 0], nodes[:, 1], nodes[:, 2]]            # [n, nt, 3] float64
    norms = np.sqrt((H.astype(np.float64) ** 2).sum(axis=(0, 1, 2, 4)))   # per-time-sample L2 norm of the table
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "cfg0_H_rows.npz")
    np.savez_compressed(out, nodes=nodes, rows=rows, slice_norms=norms, total_norm=np.linalg.norm(H))
    print("wrote", out, rows.shape, "total norm", np.linalg.norm(H))
