"""GPU parity of wt_solve_H (steps a1-a8) against the oracle through the C ABI.

Tolerance (north_star / R27): relative L2 error of the fp32 H table <= 1e-4 against the double
precision oracle, over the whole table (or the compared window)."""
import os

import numpy as np
import pytest
import torch

import paper_2605_13987_b200 as wt
from oracle import wtide_oracle as wo
from wtide_inputs import geometry_desc, reduced_desc
from wtide_inputs.configs import square_cell

pytestmark = pytest.mark.gpu
TOL = 1e-4
DEV = "cuda:0"
GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "cfg0_H_rows.npz")


def _solve(descs):
    geoms = [wt.wt_make_geometry(d) for d in descs]
    H = wt.wt_solve_H(geoms)
    torch.cuda.synchronize()
    return geoms, [h.cpu().numpy() for h in H]


def _slice_report(h, ref):
    num = np.sqrt(((h.astype(np.float64) - ref) ** 2).sum(axis=(0, 1, 2, 4)))
    den = np.sqrt((ref ** 2).sum(axis=(0, 1, 2, 4)))
    return num / np.maximum(den, 1e-300)


@pytest.mark.parametrize("grid,nt,env", [
    ((32, 32, 32), 8, {}),                        # register-FFT plane + z-line kernels
    ((32, 32, 32), 8, {"WTIDE_GENERIC": "1"}),    # the size-generic kernels on the same grid
    ((32, 32, 32), 8, {"WTIDE_NO_GRAPH": "1"}),   # direct launches instead of the replayed CUDA graph
    ((12, 24, 18), 4, {}), ((16, 8, 6), 12, {}),  # ragged grids with radix-3 factors (generic kernels)
    ((32, 32, 6), 4, {}),                         # register-FFT plane kernel + generic z-line kernel
    ((16, 16, 256), 4, {}),                       # generic plane kernel + register-FFT z-line kernel (nz = 256)
    ((64, 64, 4), 4, {}), ((128, 128, 4), 4, {}), # the 64^2 and 128^2 plane kernels
    ((16, 32, 128), 4, {}),                       # nz = 128 z-line kernel
])
def test_small_tables_match_the_oracle(grid, nt, env, monkeypatch):
    """Config 0 geometry on its own grid (window of 8 output steps = 280 Euler substeps), on ragged
    grids with radix-3 factors and nx != ny != nz, and on grids that select each size-specialised
    kernel of solve_fast.cuh."""
    for k, v in env.items():
        monkeypatch.setenv(k, v)
    d = reduced_desc(geometry_desc(0), grid=grid, nt=nt)
    _, (h,) = _solve([d])
    ref = wo.solve_H_from_desc(d)
    err = wo.h_rel_l2(h, ref)
    per_slice = _slice_report(h, ref)
    assert np.isfinite(h).all()
    assert err <= TOL, (err, per_slice)
    assert per_slice.max() <= 20 * TOL, per_slice      # late, small samples too (not required by R27)


def test_cfg0_full_length_rows_match_the_golden_oracle_rows():
    """BASELINE.json configs[0] at full length (nt = 128, 5080 substeps): the oracle's rows at 72
    sampled nodes (tests/golden/make_cfg0_golden.py), normalised by the oracle's table norm."""
    if not os.path.exists(GOLD):
        pytest.skip("golden file missing")
    z = np.load(GOLD)
    d = geometry_desc(0)
    _, (h,) = _solve([d])
    nodes, rows = z["nodes"], z["rows"]
    got = h[nodes[:, 0], nodes[:, 1], nodes[:, 2]].astype(np.float64)
    assert np.linalg.norm(got - rows) / np.linalg.norm(rows) <= TOL
    # diagnostic beyond R27: per time sample, worst sampled node against that sample's RMS over the
    # whole table (late samples are 1e3 times smaller than H[0] and carry the fp32 rounding of
    # 5080 substeps)
    n_nodes = 32 ** 3
    rms = z["slice_norms"] / np.sqrt(n_nodes * 3)
    dev = np.abs(got - rows).max(axis=(0, 2)) / rms
    assert dev.max() <= 2e-2, dev
    assert abs(np.linalg.norm(h.astype(np.float64)) / float(z["total_norm"]) - 1) <= TOL


def test_lock_step_batch_with_different_substeps():
    """Two geometries of one grid solved in one call (resistivities 0.5 and 2 ohm cm -> n_sub 40 and 10)
    equal their single solves and the oracle."""
    da = square_cell(55.0, 50.0, (16, 16, 8), 8, 0.01, 5.0, 0.5, 5.0, 0.5)
    db = square_cell(40.0, 50.0, (16, 16, 8), 8, 0.01, 4.0, 2.0, 6.0, 2.0)
    geoms, (ha, hb) = _solve([da, db])
    assert wt.wt_query(geoms[0], wt.WT_Q_SUBSTEPS) != wt.wt_query(geoms[1], wt.WT_Q_SUBSTEPS)
    _, (ha1,) = _solve([da])
    _, (hb1,) = _solve([db])
    assert np.array_equal(ha, ha1) and np.array_equal(hb, hb1)
    for h, d in ((ha, da), (hb, db)):
        assert wo.h_rel_l2(h, wo.solve_H_from_desc(d)) <= TOL


def test_properties_that_hold_at_any_size():
    """Config 1 grid (64x64x256, 100 substeps per step) for a window of 4 output steps, in the launch
    configuration bench.py times: (i) telescoping, sum_n H[n] dt equals the field of W[nt-1], which the
    oracle evaluates from ONE potential solve of the charge the oracle itself would hold -- too slow at
    this size, so instead (ii) check 2 of north_star: driving every pad gives H == 0 to rounding, and
    (iii) D4 symmetry of the centred square cell."""
    d = reduced_desc(geometry_desc(1), nt=4)
    (g,), (h,) = _solve([d])
    assert np.isfinite(h).all()
    scale = np.abs(h).max()
    # (iii) swap symmetry H_x(x,y) = H_y(y,x) (the cell and both columns are symmetric under x <-> y)
    assert np.abs(np.swapaxes(h, 0, 1)[..., 0] - h[..., 1]).max() <= 2e-4 * scale
    refl = (64 - np.arange(64)) % 64
    assert np.abs(h[refl][..., 0] + h[..., 0]).max() <= 2e-4 * scale
    # (ii) all pads driven
    dd = reduced_desc(d)
    for c in dd["columns"]:
        c["role"] = wt.WT_READOUT
    _, (h1,) = _solve([dd])
    assert np.abs(h1).max() <= 1e-5 * scale
    # the prompt (capacitive) response H[0] is of the order of the static field / dt
    assert np.linalg.norm(h[..., 0, :]) > 0.1 * np.linalg.norm(h)


def test_cfg1_window_matches_the_oracle_at_sampled_rows():
    """Config 1 geometry on a reduced grid 32x32x64 for 3 output steps (n_sub as at full size)."""
    d = reduced_desc(geometry_desc(1), grid=(32, 32, 64), nt=4)
    _, (h,) = _solve([d])
    ref = wo.solve_H_from_desc(d)
    assert wo.h_rel_l2(h, ref) <= TOL


def test_every_config_geometry_on_a_reduced_grid():
    """The geometries of BASELINE.json configs 2, 3 and 4 (hexagonal stand-in with 7 columns; two cells of the
    what-if sweep solved in lock step; the radix-3 grid of the high-statistics config) on grids the oracle
    finishes in seconds, 3 output steps each, n_sub as the geometry demands."""
    from wtide_inputs.configs import sweep_descs
    d2 = reduced_desc(geometry_desc(2), grid=(32, 32, 16), nt=4)
    d4 = reduced_desc(geometry_desc(4), grid=(24, 24, 48), nt=4)
    sw = sweep_descs(grid=(16, 16, 32), nt=4)
    d3a, d3b = sw[10], sw[11]                    # pitch 55 um, bias radius 5 um, resistivity 0.1 and 1 ohm cm
    for d in (d2, d4):
        _, (h,) = _solve([d])
        assert wo.h_rel_l2(h, wo.solve_H_from_desc(d)) <= TOL
    geoms, (ha, hb) = _solve([d3a, d3b])
    assert wt.wt_query(geoms[0], wt.WT_Q_SUBSTEPS) == 10 * wt.wt_query(geoms[1], wt.WT_Q_SUBSTEPS)
    for h, d in ((ha, d3a), (hb, d3b)):
        assert wo.h_rel_l2(h, wo.solve_H_from_desc(d)) <= TOL


def test_cfg1_full_grid_window_matches_the_oracle():
    """BASELINE.json configs[1] at its full grid (64x64x256, 370 pad nodes, n_sub = 50) in the launch configuration
    bench.py times (k_plane_fast<64>, k_pencil2<256>, k_boundary_fast<6,5>, replayed graph): the first 4 time samples
    (150 Euler substeps) against the oracle, whole table.  The oracle needs about two minutes of one host core."""
    d = reduced_desc(geometry_desc(1), nt=4)
    _, (h,) = _solve([d])
    ref = wo.solve_H_from_desc(d)
    err = wo.h_rel_l2(h, ref)
    per_slice = _slice_report(h, ref)
    assert err <= TOL, (err, per_slice)
    assert per_slice.max() <= 20 * TOL, per_slice
