"""Host-side checks of libwtide that need no GPU: the shared library loads and exports every symbol
include/wtide.h declares, wt_make_geometry (step a0, host fp64) agrees bit for bit with the oracle's
voxeliser, and the documented error behaviour holds.  No compute call is made."""
import ctypes
import os
import re

import numpy as np
import pytest

import paper_2605_13987_b200 as wt
from oracle import wtide_oracle as wo
from wtide_inputs import geometry_desc, reduced_desc, sweep_descs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "wtide.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(wt_[a-z_A-Z0-9]+)\s*\(", hdr))
    assert declared == set(wt.EXPORTS)
    lib = ctypes.CDLL(wt.LIBRARY_PATH)
    for name in declared:
        assert hasattr(lib, name), name


@pytest.mark.parametrize("cfg,grid", [(0, None), (1, (32, 32, 16)), (2, (48, 48, 12)), (4, (24, 24, 12))])
def test_voxeliser_matches_the_oracle_bit_for_bit(cfg, grid):
    d = geometry_desc(cfg)
    if grid is not None:
        d = reduced_desc(d, grid=grid, nt=8)
    g = wt.wt_make_geometry(d)
    col_id, sigma, pads, vpad, pcol = wo.voxelize(d)
    np.testing.assert_array_equal(wt.wt_get_array(g, wt.WT_A_COLUMN_ID), col_id.astype(np.int8))
    np.testing.assert_array_equal(wt.wt_get_array(g, wt.WT_A_PAD_NODES), pads.astype(np.int32))
    np.testing.assert_array_equal(wt.wt_get_array(g, wt.WT_A_PAD_POTENTIAL), vpad)
    assert wt.wt_query(g, wt.WT_Q_SUBSTEPS) == wo.substeps_from_desc(d)
    assert wt.wt_query(g, wt.WT_Q_N_PADS) == len(pads)
    assert wt.wt_query(g, wt.WT_Q_N_CONDUCTING) == int((col_id >= 0).sum())
    assert wt.wt_query(g, wt.WT_Q_H_BYTES) == d["nx"] * d["ny"] * d["nz"] * d["nt"] * 12
    assert wt.wt_query(g, wt.WT_Q_N_PAD_LAYERS) == len(set(pads[:, 2].tolist()))
    assert wt.wt_query(g, wt.WT_Q_SOLVE_WORKSPACE_BYTES) > 0
    wt.wt_free(g)
    wt.wt_free(g)      # double free through the binding is a no-op


def test_sweep_geometries_are_all_valid():
    """R29: with the swept radius on the bias column all 32 geometries voxelise without overlap errors."""
    for d in sweep_descs(grid=(32, 32, 8), nt=4):
        g = wt.wt_make_geometry(d)
        assert wt.wt_query(g, wt.WT_Q_N_PADS) > 0


def test_error_codes():
    d = reduced_desc(geometry_desc(0), grid=(16, 16, 8), nt=8)
    bad = dict(d, nt=6)
    with pytest.raises(wt.WtideError) as e:
        wt.wt_make_geometry(bad)
    assert e.value.code == wt.WT_EINVAL
    with pytest.raises(wt.WtideError) as e:
        wt.wt_make_geometry(dict(d, nx=20))            # 20 = 2^2 * 5
    assert e.value.code == wt.WT_EINVAL
    no_readout = dict(d, columns=[dict(c, role=wt.WT_BIAS) for c in d["columns"]])
    with pytest.raises(wt.WtideError) as e:
        wt.wt_make_geometry(no_readout)
    assert e.value.code == wt.WT_EGEOM
    thin = dict(d, columns=[dict(d["columns"][0]), dict(d["columns"][1], radius=0.01, cx=1.0, cy=1.0)])
    with pytest.raises(wt.WtideError) as e:
        wt.wt_make_geometry(thin)                      # a column that contains no node
    assert e.value.code == wt.WT_EGEOM
    with pytest.raises(wt.WtideError) as e:
        wt.wt_make_geometry(dict(d, substeps=10))      # dt/10 = 1 ps >= 2 tau = 0.5 ps
    assert e.value.code == wt.WT_EUNSTABLE
    assert "unstable" in str(e.value)
    g = wt.wt_make_geometry(dict(d, substeps=25))      # 0.4 ps < 0.5 ps: allowed
    assert wt.wt_query(g, wt.WT_Q_SUBSTEPS) == 25
    with pytest.raises(wt.WtideError):
        wt.wt_query(g, 999)


def test_segments_give_a_depth_dependent_profile_and_match_the_oracle_voxeliser():
    """WT_SEGMENT (PAPER.md:143 'depth-dependent conductivity profile'): a readout column whose lower
    part is a stack of two segments of other resistivities.  Same node sets and pads as the oracle's voxeliser, bit-exact;
    a stack of segments with the SAME resistivity equals the single full-depth column."""
    from wtide_inputs.configs import square_cell
    base = square_cell(40.0, 60.0, (16, 16, 24), 8, 0.01, 5.0, 0.5, 5.0, 0.5)
    ro = base["columns"][0]
    seg = dict(base)
    seg["columns"] = [dict(ro, z1=20.0), dict(ro, z0=20.0, z1=40.0, resistivity=2.0, role=wt.WT_SEGMENT), dict(ro, z0=40.0, resistivity=8.0, role=wt.WT_SEGMENT),
                      base["columns"][1]]
    g = wt.wt_make_geometry(seg)
    col_id, sigma, pads, pot, pcol = wo.voxelize(seg)
    assert np.array_equal(wt.wt_get_array(g, wt.WT_A_COLUMN_ID), col_id.astype(np.int8))
    assert np.array_equal(wt.wt_get_array(g, wt.WT_A_PAD_NODES), pads.astype(np.int32))
    assert set(pcol) == {0, 3} and (col_id == 1).any() and (col_id == 2).any()
    assert wt.wt_query(g, wt.WT_Q_SUBSTEPS) == wo.substeps_from_desc(seg)
    same = dict(base)
    same["columns"] = [dict(ro, z1=20.0), dict(ro, z0=20.0, role=wt.WT_SEGMENT), base["columns"][1]]
    _, s_same, p_same, _, _ = wo.voxelize(same)
    _, s_base, p_base, _, _ = wo.voxelize(base)
    assert np.array_equal(s_same, s_base) and np.array_equal(p_same, p_base)


def test_mirror_z_builds_the_doubled_box_of_the_oracle():
    """mirror_z = 1 makes the handle of the doubled box (method of images) -- voxel set, pads and
    queries equal those of the oracle's own mirror_z_desc, for pads on the mirror planes and for a pad away from them."""
    base = reduced_desc(geometry_desc(1), grid=(16, 16, 12), nt=8)
    off = dict(base, columns=[dict(base["columns"][0], z0=50.0, z1=400.0), base["columns"][1]])
    for d in (base, off):
        g = wt.wt_make_geometry(dict(d, mirror_z=1))
        dm = wo.mirror_z_desc(d)
        col_id, _, pads, vpad, _ = wo.voxelize(dm)
        assert g.shape == (16, 16, 24) and wt.wt_query(g, wt.WT_Q_NZ) == 24 and wt.wt_query(g, wt.WT_Q_N_COLUMNS) == 4
        np.testing.assert_array_equal(wt.wt_get_array(g, wt.WT_A_COLUMN_ID), col_id.astype(np.int8))
        np.testing.assert_array_equal(wt.wt_get_array(g, wt.WT_A_PAD_NODES), pads.astype(np.int32))
        np.testing.assert_array_equal(wt.wt_get_array(g, wt.WT_A_PAD_POTENTIAL), vpad)
        assert wt.wt_query(g, wt.WT_Q_H_BYTES) == 16 * 16 * 24 * 8 * 12
    with pytest.raises(wt.WtideError) as e:
        wt.wt_make_geometry(dict(reduced_desc(geometry_desc(0), grid=(16, 16, 768), nt=8), mirror_z=1))
    assert e.value.code == wt.WT_EINVAL
