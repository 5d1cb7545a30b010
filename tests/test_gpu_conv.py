"""GPU parity of wt_convolve_currents / wt_trajectory_nodes (steps a9-a12) against the oracle,
element by element on the same seeded inputs, through the C ABI.

Tolerance (north_star / R27): currents within 2e-4 of the oracle, normalised to the row's peak;
indices bit-exact."""
import numpy as np
import pytest
import torch

import paper_2605_13987_b200 as wt
from oracle import wtide_oracle as wo
from wtide_inputs import (carriers_on_tracks, geometry_desc, make_tracks, reduced_desc,
                          straight_drift_cfg0)

pytestmark = pytest.mark.gpu
TOL = 2e-4
DEV = "cuda:0"


def _to_dev(csr):
    return {k: torch.as_tensor(np.asarray(v)).to(DEV) for k, v in csr.items()}


def _run(g, H, csr, per_track):
    c = _to_dev(csr)
    out = wt.wt_convolve_currents(g, H, c["track_carrier_offsets"], c["carrier_step_offsets"], c["pos"], c["vel"],
                                  c["charge"], per_track=per_track)
    torch.cuda.synchronize()
    return out.cpu().numpy()


def _oracle(d, Hnp, csr, per_track):
    return wo.convolve_currents(Hnp, (d["nx"], d["ny"], d["nz"]), (d["lx"], d["ly"], d["lz"]), d["nt"], d["dt"], d["v_w"],
                                csr["carrier_step_offsets"], csr["pos"], csr["vel"], csr["charge"],
                                csr["track_carrier_offsets"] if per_track else None)


def test_trajectory_nodes_bit_exact():
    d = geometry_desc(1)
    g = wt.wt_make_geometry(reduced_desc(d, grid=(64, 64, 256), nt=8, substeps=100))
    rng = np.random.default_rng(0)
    pos = rng.uniform(-200.0, 700.0, size=(200_000, 3)).astype(np.float32)
    pos[:1000] = rng.uniform(0, 55.0, size=(1000, 3)).astype(np.float32)
    pos[5] = [np.nan, 1, 1]
    pos[6] = [1, np.inf, 1]
    # exact node positions and cell boundaries
    pos[1000:1064, 0] = (np.arange(64) * 55.0 / 64).astype(np.float32)
    n0, n1, fr = wt.wt_trajectory_nodes(g, torch.as_tensor(pos).to(DEV))
    torch.cuda.synchronize()
    i0, i1, f, fin = wo.trajectory_nodes((64, 64, 256), (55.0, 55.0, 500.0), pos)
    n0, n1, fr = n0.cpu().numpy(), n1.cpu().numpy(), fr.cpu().numpy()
    assert np.array_equal(n0[fin], i0[fin].astype(np.int32))
    assert np.array_equal(n1[fin], i1[fin].astype(np.int32))
    assert np.array_equal(fr[fin].view(np.uint32), f[fin].view(np.uint32))       # bit-exact fractions
    assert (n0[~fin] == -1).all() and (n1[~fin] == -1).all()


def test_cfg0_currents_match_the_oracle():
    """Config 0 workload (256 carriers on one perpendicular track, straight drift, R28) on a random
    fp32 table (conv parity is decoupled from solver parity): per-carrier and per-track outputs."""
    d = geometry_desc(0)
    g = wt.wt_make_geometry(d)
    rng = np.random.default_rng(1)
    Hnp = rng.standard_normal((d["nx"], d["ny"], d["nz"], d["nt"], 3)).astype(np.float32)
    H = torch.as_tensor(Hnp).to(DEV)
    tracks = make_tracks(0, 1, d, 0.0)
    start, sign, charge, toff = carriers_on_tracks(tracks, 256, d, unit_charge=True)
    csr = straight_drift_cfg0(d, start, sign, charge, toff)
    assert csr["carrier_step_offsets"][-1] > 1000
    for per_track in (False, True):
        got = _run(g, H, csr, per_track)
        ref = _oracle(d, Hnp, csr, per_track)
        l2, mx = wo.current_error(got, ref)
        assert l2 <= TOL and mx <= 5 * TOL, (per_track, l2, mx)


def test_ragged_and_degenerate_inputs():
    """Empty carriers, a carrier longer than nt (R26), steps outside the box, non-finite steps,
    a track without carriers, nt = 1024 (eight warps per carrier), nt = 1028 (beyond the systolic kernel's range:
    the one-CTA-per-carrier kernel), nt = 4 and nt = 36 (partly filled last warp)."""
    for nt in (1024, 1028, 4, 36):
        d = reduced_desc(geometry_desc(0), grid=(12, 8, 6), nt=nt)
        g = wt.wt_make_geometry(d)
        rng = np.random.default_rng(nt)
        Hnp = rng.standard_normal((12, 8, 6, nt, 3)).astype(np.float32)
        H = torch.as_tensor(Hnp).to(DEV)
        lens = [0, 3, nt + 7, 1, 0, 40, 5, 0]
        off = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
        S = int(off[-1])
        pos = rng.uniform(-100, 150, size=(S, 3)).astype(np.float32)
        vel = rng.standard_normal((S, 3)).astype(np.float32)
        pos[off[2] + 1, 1] = np.nan
        vel[off[5] + 2, 0] = np.inf
        csr = dict(track_carrier_offsets=np.array([0, 1, 1, 4, 8], np.int64), carrier_step_offsets=off, pos=pos, vel=vel,
                   charge=rng.standard_normal(len(lens)).astype(np.float32))
        for per_track in (False, True):
            got = _run(g, H, csr, per_track)
            ref = _oracle(d, Hnp, csr, per_track)
            assert np.isfinite(got).all()
            scale = np.abs(ref).max()
            assert np.abs(got - ref).max() <= TOL * scale, (nt, per_track)
            if per_track:
                assert (got[1] == 0).all()
    # zero carriers / zero tracks: a valid call that writes nothing
    out = wt.wt_convolve_currents(g, H, torch.zeros(1, dtype=torch.int64, device=DEV), torch.zeros(1, dtype=torch.int64, device=DEV),
                                  torch.zeros((0, 3), device=DEV), torch.zeros((0, 3), device=DEV), torch.zeros(0, device=DEV))
    assert out.shape == (0, nt)


def test_run_to_run_determinism():
    d = reduced_desc(geometry_desc(0), grid=(16, 16, 8), nt=64)
    g = wt.wt_make_geometry(d)
    H = torch.randn((16, 16, 8, 64, 3), device=DEV)
    tracks = make_tracks(0, 4, d, 5.0)
    start, sign, charge, toff = carriers_on_tracks(tracks, 64, d)
    csr = straight_drift_cfg0(d, start, sign, charge, toff, max_steps=64)
    a = _run(g, H, csr, True)
    b = _run(g, H, csr, True)
    assert np.array_equal(a.view(np.uint32), b.view(np.uint32))


def test_full_size_table_sampled_tracks():
    """BASELINE.json configs[1] sizes (64x64x256 grid, nt = 512, 6.4 GB table) in the launch
    configuration bench.py times; the oracle computes a sample of tracks from rows fetched on demand."""
    d = geometry_desc(1)
    g = wt.wt_make_geometry(reduced_desc(d, substeps=100))
    gen = torch.Generator(device=DEV).manual_seed(3)
    H = torch.randn((64, 64, 256, 512, 3), device=DEV, generator=gen)
    tracks = make_tracks(1, 3, d, 10.0)
    start, sign, charge, toff = carriers_on_tracks(tracks, 40, d)
    # curved synthetic paths of ragged length (the solver-driven drift is exercised in test_gpu_solve)
    rng = np.random.default_rng(5)
    lens = rng.integers(0, 90, size=len(start))
    off = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
    pos = np.concatenate([start[c] + np.cumsum(rng.normal(0.3, 0.3, size=(lens[c], 3)), axis=0) for c in range(len(start))]).astype(np.float32)
    vel = rng.standard_normal((int(off[-1]), 3)).astype(np.float32) * 100
    csr = dict(track_carrier_offsets=toff, carrier_step_offsets=off, pos=pos, vel=vel, charge=charge)
    got = _run(g, H, csr, True)
    cache = {}

    def rows(ix, iy, iz):
        key = (ix, iy, iz)
        if key not in cache:
            cache[key] = H[ix, iy, iz].cpu().numpy()
        return cache[key]
    ref = _oracle(d, rows, csr, True)
    l2, mx = wo.current_error(got, ref)
    assert l2 <= TOL and mx <= 5 * TOL, (l2, mx)


def test_many_carriers_ragged_tracks_grouped_path():
    """Enough carriers for the grouped launch (8 carriers per CTA, interleaved over 32 CTAs, partial rows
    per track segment): ragged tracks incl. empty ones, carriers before the first and after the last
    track, empty carriers; per-track and per-carrier outputs against the oracle."""
    nt = 20
    d = reduced_desc(geometry_desc(0), grid=(8, 8, 6), nt=nt)
    g = wt.wt_make_geometry(d)
    rng = np.random.default_rng(7)
    Hnp = rng.standard_normal((8, 8, 6, nt, 3)).astype(np.float32)
    H = torch.as_tensor(Hnp).to(DEV)
    n_car = 12_000
    lens = rng.integers(0, 5, size=n_car)
    lens[100] = nt + 3
    off = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
    S = int(off[-1])
    pos = rng.uniform(-20, 70, size=(S, 3)).astype(np.float32)
    vel = rng.standard_normal((S, 3)).astype(np.float32)
    # tracks: a few carriers before the first track and after the last belong to no track
    cuts = np.sort(rng.choice(np.arange(5, n_car - 5), size=60, replace=False))
    toff = np.concatenate([[3], cuts, cuts[10:13], [n_car - 4]]).astype(np.int64)   # repeated cuts = empty tracks
    toff.sort()
    csr = dict(track_carrier_offsets=toff, carrier_step_offsets=off, pos=pos, vel=vel,
               charge=rng.standard_normal(n_car).astype(np.float32))
    ref_c = _oracle(d, Hnp, csr, False)
    got_c = _run(g, H, csr, False)
    scale = np.abs(ref_c).max()
    assert np.abs(got_c - ref_c).max() <= TOL * scale
    got_t = _run(g, H, csr, True)
    ref_t = np.stack([ref_c[toff[i]:toff[i + 1]].sum(axis=0) for i in range(len(toff) - 1)])
    assert got_t.shape == ref_t.shape
    assert np.abs(got_t - ref_t).max() <= TOL * np.abs(ref_t).max()
    empty = np.nonzero(np.diff(toff) == 0)[0]
    assert len(empty) >= 3 and (got_t[empty] == 0).all()


@pytest.mark.parametrize("config", [2, 4])
def test_tables_beyond_2_31_floats_sampled_tracks(config):
    """BASELINE.json configs[2] (128x128x256, nt = 1024: 51.5 GB, 1.29e10 floats) and configs[4] (96x96x384, nt = 1024:
    43.5 GB) table sizes in the launch configuration bench.py times (eight warps per carrier): row offsets beyond 2^31
    floats / 2^32 bytes.  Tracks are placed so that the highest node indices of the table are read; the oracle computes
    them from rows fetched on demand from the same fp32 table."""
    d = geometry_desc(config)
    nx, ny, nz, nt = d["nx"], d["ny"], d["nz"], d["nt"]
    g2 = wt.wt_make_geometry(d)
    H = torch.empty((nx, ny, nz, nt, 3), dtype=torch.float32, device=DEV)
    flat = H.view(-1)
    gen = torch.Generator(device=DEV).manual_seed(11 + config)
    step = 1 << 28
    for a in range(0, flat.numel(), step):
        flat[a:a + step].normal_(generator=gen)
    assert flat.numel() > 2 ** 31
    rng = np.random.default_rng(13 + config)
    n_car = 24
    lens = rng.integers(1, 120, size=n_car)
    lens[3] = nt + 5                                  # longer than the table's time axis (R26)
    off = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
    # starts spread over the box, half of them in the last x-planes (node index close to nx*ny*nz)
    start = np.stack([rng.uniform(0, d["lx"], n_car), rng.uniform(0, d["ly"], n_car), rng.uniform(0, d["lz"], n_car)], axis=1)
    start[::2, 0] = d["lx"] * (1.0 - rng.uniform(0, 2.5 / nx, size=len(start[::2])))
    start[::4, 1] = d["ly"] * (1.0 - rng.uniform(0, 2.5 / ny, size=len(start[::4])))
    start[::4, 2] = d["lz"] * (1.0 - rng.uniform(0, 2.5 / nz, size=len(start[::4])))
    pos = np.concatenate([start[c] + np.cumsum(rng.normal(0.0, 0.4, size=(lens[c], 3)), axis=0) for c in range(n_car)]).astype(np.float32)
    vel = (rng.standard_normal((int(off[-1]), 3)) * 100).astype(np.float32)
    csr = dict(track_carrier_offsets=np.array([0, 5, 5, 17, n_car], np.int64), carrier_step_offsets=off, pos=pos, vel=vel,
               charge=rng.standard_normal(n_car).astype(np.float32))
    i0, i1, _, _ = wo.trajectory_nodes((nx, ny, nz), (d["lx"], d["ly"], d["lz"]), pos)
    top = ((i1[:, 0] * ny + i1[:, 1]) * nz + i1[:, 2]).max()
    assert top * nt * 3 > 2 ** 31 and top >= nx * ny * nz - 3 * ny * nz
    cache = {}

    def rows(ix, iy, iz):
        key = (ix, iy, iz)
        if key not in cache:
            cache[key] = H[ix, iy, iz].cpu().numpy()
        return cache[key]
    for per_track in (True, False):
        got = _run(g2, H, csr, per_track)
        ref = _oracle(d, rows, csr, per_track)
        l2, mx = wo.current_error(got, ref)
        assert np.isfinite(got).all()
        assert l2 <= TOL and mx <= 5 * TOL, (config, per_track, l2, mx)
    del H
    torch.cuda.empty_cache()


@pytest.mark.parametrize("cache", ["0", "1"])
def test_row_cache_kernel_and_plain_kernel_agree_with_the_oracle(cache, monkeypatch):
    """k_conv_systolic<CACHE> keeps the rows of the current cell in registers while a carrier stays in it; both kernels
    (WTIDE_CONV_CACHE=0/1) on slow carriers that spend several steps per cell, stationary carriers, a skipped (non-finite)
    step followed by steps in the cell at node (0, 0, 0), and cell changes across the periodic wrap and the z clamp."""
    monkeypatch.setenv("WTIDE_CONV_CACHE", cache)
    for nt in (128, 1024, 36):
        d = reduced_desc(geometry_desc(0), grid=(12, 8, 6), nt=nt)
        g = wt.wt_make_geometry(d)
        rng = np.random.default_rng(100 + nt)
        Hnp = rng.standard_normal((12, 8, 6, nt, 3)).astype(np.float32)
        H = torch.as_tensor(Hnp).to(DEV)
        cell = np.array([d["lx"] / 12, d["ly"] / 8, d["lz"] / 6])
        lens = [60, 90, 33, 50, 1, 70]
        off = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
        pos = []
        for c, n in enumerate(lens):
            x0 = rng.uniform(0, 1, 3) * np.array([d["lx"], d["ly"], d["lz"]])
            step = rng.normal(0, 0.15, size=(n, 3)) * cell           # several steps per cell
            if c == 1:
                step[:] = 0.0                                        # stationary carrier
            if c == 2:
                x0 = np.array([d["lx"] - 0.2 * cell[0], 0.1 * cell[1], d["lz"] - 0.3 * cell[2]])   # wraps in x, y; clamps in z
                step = np.abs(step) * np.array([1, -1, 1])
            pos.append(x0 + np.cumsum(step, axis=0))
        pos = np.concatenate(pos).astype(np.float32)
        # carrier 3: a non-finite step, then steps inside the cell whose corner 0 is node (0, 0, 0)
        a = off[3]
        pos[a] = [np.nan, 1.0, 1.0]
        pos[a + 1:a + 6] = (rng.uniform(0.1, 0.9, size=(5, 3)) * cell).astype(np.float32)
        vel = rng.standard_normal((int(off[-1]), 3)).astype(np.float32)
        csr = dict(track_carrier_offsets=np.array([0, 2, 6], np.int64), carrier_step_offsets=off, pos=pos, vel=vel,
                   charge=rng.standard_normal(len(lens)).astype(np.float32))
        for per_track in (False, True):
            got = _run(g, H, csr, per_track)
            ref = _oracle(d, Hnp, csr, per_track)
            assert np.isfinite(got).all()
            assert np.abs(got - ref).max() <= TOL * np.abs(ref).max(), (nt, per_track)


@pytest.mark.parametrize("nt", [1024, 896, 1000, 260])
def test_long_carriers_share_the_causal_triangle(nt, monkeypatch):
    """Cached kernel: the (lag block, step) pairs of every 128-step table are dealt out evenly to the warps (more warps than
    blocks), pieces start with empty sums.  Carriers of 127 ... nt + 300 steps (tables at which 0 ... all but one block have
    run past nt, a ragged last table), nt a multiple of 128 or not, against the oracle; twice for the same bits (R25)."""
    monkeypatch.setenv("WTIDE_CONV_CACHE", "1")
    d = reduced_desc(geometry_desc(0), grid=(12, 8, 6), nt=nt)
    g = wt.wt_make_geometry(d)
    rng = np.random.default_rng(200 + nt)
    Hnp = rng.standard_normal((12, 8, 6, nt, 3)).astype(np.float32)
    H = torch.as_tensor(Hnp).to(DEV)
    cell = np.array([d["lx"] / 12, d["ly"] / 8, d["lz"] / 6])
    lens = [127, 128, 129, 300, min(640, nt - 1), nt, nt + 300, 2, 385]
    off = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
    pos = np.concatenate([rng.uniform(0, 1, 3) * np.array([d["lx"], d["ly"], d["lz"]]) + np.cumsum(rng.normal(0, 0.2, size=(n, 3)) * cell, axis=0)
                          for n in lens]).astype(np.float32)
    vel = rng.standard_normal((int(off[-1]), 3)).astype(np.float32)
    csr = dict(track_carrier_offsets=np.array([0, 4, 7, 9], np.int64), carrier_step_offsets=off, pos=pos, vel=vel,
               charge=rng.standard_normal(len(lens)).astype(np.float32))
    for per_track in (False, True):
        got = _run(g, H, csr, per_track)
        ref = _oracle(d, Hnp, csr, per_track)
        assert np.isfinite(got).all()
        assert np.abs(got - ref).max() <= TOL * np.abs(ref).max(), (nt, per_track)
        again = _run(g, H, csr, per_track)
        assert np.array_equal(got.view(np.uint32), again.view(np.uint32))
