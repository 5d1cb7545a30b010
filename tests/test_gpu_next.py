"""GPU parity of the stages around the hot path against the oracle through the C ABI:
static field, carrier transport (step counts and positions bit-exact: fp32 arithmetic in a fixed order, R35),
electronics stage."""
import numpy as np
import pytest
import torch

import paper_2605_13987_b200 as wt
from oracle import wtide_oracle as wo
from wtide_inputs import carriers_on_tracks, geometry_desc, make_tracks, reduced_desc
from wtide_inputs.tracks import bias_voltage

pytestmark = pytest.mark.gpu
DEV = "cuda:0"
MU_E, MU_H, V_SAT = 180.0, 150.0, 150.0


def test_static_field_of_a_solved_table_and_of_a_random_table():
    d = reduced_desc(geometry_desc(0), grid=(16, 16, 8), nt=16)
    g = wt.wt_make_geometry(d)
    (H,) = wt.wt_solve_H([g])
    es = wt.wt_static_field(g, H)
    torch.cuda.synchronize()
    ref = wo.static_field(H.cpu().numpy(), d["dt"])
    assert np.abs(es.cpu().numpy() - ref).max() <= 2e-6 * np.abs(ref).max()
    # ragged nt (not a multiple of 128) and values with cancellation
    d2 = reduced_desc(geometry_desc(0), grid=(12, 8, 6), nt=36)
    g2 = wt.wt_make_geometry(d2)
    H2 = torch.randn((12, 8, 6, 36, 3), device=DEV)
    es2 = wt.wt_static_field(g2, H2)
    torch.cuda.synchronize()
    ref2 = wo.static_field(H2.cpu().numpy(), d2["dt"])
    assert np.abs(es2.cpu().numpy() - ref2).max() <= 1e-5 * np.abs(H2.cpu().numpy()).sum(axis=3).max() * d2["dt"]


@pytest.mark.parametrize("config,grid,n_tracks,n_per", [(1, (32, 32, 64), 6, 40), (2, (32, 32, 16), 4, 30), (4, (24, 24, 48), 4, 30)])
def test_drift_trajectories_are_bit_exact(config, grid, n_tracks, n_per):
    """Carriers of seeded MIP tracks drifted in the static field of the SOLVED table of the config's geometry (reduced grid):
    CSR offsets (step counts), positions and velocities equal the oracle's bit for bit; includes carriers that start inside
    a column (no step), reach a column, leave through a z face, or hit the step cap."""
    nt = 48
    d = reduced_desc(geometry_desc(config), grid=grid, nt=nt)
    g = wt.wt_make_geometry(d)
    (H,) = wt.wt_solve_H([g])
    es = wt.wt_static_field(g, H)
    tracks = make_tracks(config, n_tracks, d, 10.0)
    start, sign, charge, toff = carriers_on_tracks(tracks, n_per, d)
    start = np.concatenate([start, [[d["columns"][0]["cx"], d["columns"][0]["cy"], 0.5 * d["lz"]], [1.0, 1.0, -0.5], [np.nan, 1.0, 1.0]]]).astype(np.float32)
    sign = np.concatenate([sign, [1, -1, 1]]).astype(np.int8)
    vb = bias_voltage(d)
    off, pos, vel = wt.wt_drift_carriers(g, es, torch.as_tensor(start).to(DEV), torch.as_tensor(sign).to(DEV), vb, MU_E, MU_H, V_SAT, max_steps=nt)
    torch.cuda.synchronize()
    o_off, o_pos, o_vel = wo.drift_trajectories(es.cpu().numpy(), d, start, sign, vb, MU_E, MU_H, V_SAT, nt)
    assert np.array_equal(off.cpu().numpy(), o_off)
    assert o_off[-1] > 10 * len(start) // 2 and (np.diff(o_off)[-3:] == 0).all() and np.diff(o_off).max() == nt
    assert np.array_equal(pos.cpu().numpy().view(np.uint32), o_pos.view(np.uint32))
    assert np.array_equal(vel.cpu().numpy().view(np.uint32), o_vel.view(np.uint32))


def test_drift_feeds_eq_1_1_without_leaving_the_device():
    """wt_solve_H -> wt_static_field -> wt_drift_carriers -> wt_convolve_currents chained on device buffers; the currents
    equal the oracle's Eq. 1.1 on the oracle's trajectories (same table)."""
    d = reduced_desc(geometry_desc(1), grid=(32, 32, 64), nt=32)
    g = wt.wt_make_geometry(d)
    (H,) = wt.wt_solve_H([g])
    es = wt.wt_static_field(g, H)
    tracks = make_tracks(1, 3, d, 10.0)
    start, sign, charge, toff = carriers_on_tracks(tracks, 20, d)
    off, pos, vel = wt.wt_drift_carriers(g, es, torch.as_tensor(start).to(DEV), torch.as_tensor(sign).to(DEV), bias_voltage(d))
    cur = wt.wt_convolve_currents(g, H, torch.as_tensor(toff).to(DEV), off, pos, vel, torch.as_tensor(charge).to(DEV), per_track=True)
    torch.cuda.synchronize()
    o_off, o_pos, o_vel = wo.drift_trajectories(es.cpu().numpy(), d, start, sign, bias_voltage(d), MU_E, MU_H, V_SAT, d["nt"])
    ref = wo.convolve_currents(H.cpu().numpy(), (d["nx"], d["ny"], d["nz"]), (d["lx"], d["ly"], d["lz"]), d["nt"], d["dt"], d["v_w"],
                               o_off, o_pos, o_vel, charge, toff)
    l2, mx = wo.current_error(cur.cpu().numpy(), ref)
    assert l2 <= 2e-4 and mx <= 1e-3, (l2, mx)


def test_offsets_scan_on_many_carriers():
    n = 1_000_003
    rng = np.random.default_rng(2)
    counts = rng.integers(0, 600, size=n).astype(np.int64)
    c = torch.as_tensor(counts).to(DEV)
    offs = torch.empty(n + 1, dtype=torch.int64, device=DEV)
    wt._run_on_side_stream(DEV, lambda s: wt._lib.wt_offsets_from_counts(n, c.data_ptr(), offs.data_ptr(), s))
    torch.cuda.synchronize()
    assert np.array_equal(offs.cpu().numpy(), np.concatenate([[0], np.cumsum(counts)]))


def test_electronics_stage_matches_the_oracle():
    rng = np.random.default_rng(4)
    nt = 256
    n = np.arange(nt)
    cur = np.stack([a * np.exp(-0.5 * ((n - c) / w) ** 2) for a, c, w in ((1.0, 60, 9), (-2.5, 100, 20), (0.7, 30, 4), (0.0, 1, 1))]).astype(np.float32)
    cur[:3] += (1e-3 * rng.standard_normal((3, nt))).astype(np.float32)
    h = (np.exp(-np.arange(40) / 6.0) - np.exp(-np.arange(40) / 2.0)).astype(np.float32)
    noise = (0.01 * rng.standard_normal((4, nt))).astype(np.float32)
    for nz_ in (None, noise):
        out, tc = wt.wt_electronics(torch.as_tensor(cur).to(DEV), torch.as_tensor(h).to(DEV), 0.005,
                                    noise=None if nz_ is None else torch.as_tensor(nz_).to(DEV), cfd_fraction=0.3)
        torch.cuda.synchronize()
        ro, rt = wo.electronics(cur, h, 0.005, noise=nz_, cfd_fraction=0.3)
        assert np.abs(out.cpu().numpy() - ro).max() <= 2e-6 * np.abs(ro).max()
        if nz_ is None:
            assert rt[3] == -1.0 and tc[3].item() == -1.0
            assert np.abs(tc.cpu().numpy()[:3] - rt[:3]).max() <= 2e-3, (tc, rt)     # crossing times agree to a fraction of a sample
