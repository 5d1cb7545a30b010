"""wt_convolve_tracks_noalloc (include/wtide.h): Eq. 1.1 summed per track with the library's built-in scratch instead of a
caller workspace, for callers that cannot allocate device memory.  Checked against the existing path
(wt_convolve_currents, per_track = 1, itself held to the oracle in test_gpu_conv.py) on two calls in a row that share the
scratch, within the tolerance of the Eq. 1.1 tests (2e-4 of the peak; the kernels and the order of summation are the same,
so the results are in fact bit-identical).  This file is collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest
import torch

import paper_2605_13987_b200 as wt
from wtide_inputs import carriers_on_tracks, geometry_desc, make_tracks, reduced_desc, straight_drift_cfg0

pytestmark = pytest.mark.gpu
TOL = 2e-4
DEV = "cuda:0"


def _dev(csr):
    return {k: torch.as_tensor(np.asarray(v)).to(DEV) for k, v in csr.items()}


def _both(g, H, csr):
    c = _dev(csr)
    n_trk = c["track_carrier_offsets"].numel() - 1
    ref = wt.wt_convolve_currents(g, H, c["track_carrier_offsets"], c["carrier_step_offsets"], c["pos"], c["vel"], c["charge"],
                                  per_track=True)
    out = torch.full((n_trk, g.nt), float("nan"), dtype=torch.float32, device=DEV)
    torch.cuda.synchronize()
    free0, alloc0 = torch.cuda.mem_get_info(DEV)[0], torch.cuda.memory_allocated(DEV)
    wt.wt_convolve_tracks_noalloc(g, H, c["track_carrier_offsets"], c["carrier_step_offsets"], c["pos"], c["vel"], c["charge"], out)
    torch.cuda.synchronize()
    free1, alloc1 = torch.cuda.mem_get_info(DEV)[0], torch.cuda.memory_allocated(DEV)
    return ref, out, (free0 - free1, alloc1 - alloc0)


def _check(ref, out):
    assert torch.isfinite(out).all()
    peak = float(ref.abs().max())
    assert peak > 0
    assert float((out - ref).abs().max()) <= TOL * peak
    assert torch.equal(out, ref)          # same kernels, same order of summation (R25)


def _straight(d, n_tracks, per_track, seed):
    tracks = make_tracks(0, n_tracks, d, 5.0, seed=seed)
    start, sign, charge, toff = carriers_on_tracks(tracks, per_track, d)
    return straight_drift_cfg0(d, start, sign, charge, toff, max_steps=d["nt"])


def _ragged(rng, n_car, nt, box):
    lens = rng.integers(0, 5, size=n_car)
    lens[7] = nt + 3
    off = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
    steps = int(off[-1])
    cuts = np.sort(rng.choice(np.arange(5, n_car - 5), size=40, replace=False))
    toff = np.sort(np.concatenate([[3], cuts, cuts[5:8], [n_car - 4]])).astype(np.int64)     # repeated cuts: empty tracks
    return dict(track_carrier_offsets=toff, carrier_step_offsets=off, pos=rng.uniform(-0.3 * box, 1.3 * box, size=(steps, 3)).astype(np.float32),
                vel=rng.standard_normal((steps, 3)).astype(np.float32), charge=rng.standard_normal(n_car).astype(np.float32))


def test_two_calls_in_a_row_match_the_workspace_path():
    """One row per carrier (nt = 64): a call that fills most of the scratch, then a smaller one with other carriers that
    finds the first call's rows in it."""
    d = reduced_desc(geometry_desc(0), grid=(16, 16, 8), nt=64)
    g = wt.wt_make_geometry(d)
    H = torch.randn((16, 16, 8, 64, 3), device=DEV, generator=torch.Generator(device=DEV).manual_seed(21))
    first = _straight(d, 8, 2000, seed=0)                 # 16 000 carriers x 64 = 1 024 000 floats of the 1 048 576
    assert 0.9 * wt.WT_NOALLOC_MAX_FLOATS < (len(first["charge"]) * 64) <= wt.WT_NOALLOC_MAX_FLOATS
    ref, out, _ = _both(g, H, first)
    _check(ref, out)
    second = _straight(d, 3, 50, seed=1)
    ref2, out2, grew = _both(g, H, second)
    _check(ref2, out2)
    assert grew == (0, 0), grew                           # the second call took no device memory (driver's and torch's count)
    assert not torch.equal(out2[:3], out[:3])
    # and the first again: the same bits as before
    ref3, out3, grew = _both(g, H, first)
    assert torch.equal(out3, out) and grew == (0, 0)


def test_grouped_launch_and_ragged_tracks_twice():
    """Enough carriers for the grouped launch (8 carriers per CTA, one partial row per track segment), ragged tracks with
    empty ones and carriers outside every track; twice with different carriers."""
    nt = 20
    d = reduced_desc(geometry_desc(0), grid=(8, 8, 6), nt=nt)
    g = wt.wt_make_geometry(d)
    H = torch.randn((8, 8, 6, nt, 3), device=DEV, generator=torch.Generator(device=DEV).manual_seed(22))
    rng = np.random.default_rng(23)
    for n_car in (12_000, 10_500):
        csr = _ragged(rng, n_car, nt, d["lx"])
        ref, out, _ = _both(g, H, csr)
        _check(ref, out)
        empty = np.nonzero(np.diff(csr["track_carrier_offsets"]) == 0)[0]
        assert len(empty) >= 3 and (out[empty] == 0).all()


def test_sizes_beyond_the_scratch_are_refused_and_the_limit_itself_is_served():
    d = reduced_desc(geometry_desc(0), grid=(8, 8, 6), nt=1024)
    g = wt.wt_make_geometry(d)
    H = torch.randn((8, 8, 6, 1024, 3), device=DEV, generator=torch.Generator(device=DEV).manual_seed(24))
    rng = np.random.default_rng(25)

    def call(n_car):
        off = torch.arange(n_car + 1, dtype=torch.int64, device=DEV)            # one step per carrier
        toff = torch.tensor([0, n_car], dtype=torch.int64, device=DEV)
        pos = torch.as_tensor(rng.uniform(0, d["lx"], size=(n_car, 3)).astype(np.float32)).to(DEV)
        vel = torch.ones((n_car, 3), device=DEV)
        out = torch.full((1, 1024), -7.0, device=DEV)
        wt.wt_convolve_tracks_noalloc(g, H, toff, off, pos, vel, torch.ones(n_car, device=DEV), out)
        torch.cuda.synchronize()
        return out, (toff, off, pos, vel)

    limit = wt.WT_NOALLOC_MAX_FLOATS // 1024
    with pytest.raises(wt.WtideError) as ei:
        call(limit + 1)
    assert ei.value.code == wt.WT_ENOMEM and "WT_NOALLOC_MAX_FLOATS" in str(ei.value) and str(wt.WT_NOALLOC_MAX_FLOATS) in str(ei.value)
    out, (toff, off, pos, vel) = call(limit)              # exactly the limit is served (nt = 1024: eight warps per carrier)
    ref = wt.wt_convolve_currents(g, H, toff, off, pos, vel, torch.ones(limit, device=DEV), per_track=True)
    _check(ref, out)
    # no carriers: a valid call, the track's row is zero
    z = torch.zeros(1, dtype=torch.int64, device=DEV)
    out0 = torch.full((1, 1024), -7.0, device=DEV)
    wt.wt_convolve_tracks_noalloc(g, H, torch.zeros(2, dtype=torch.int64, device=DEV), z, torch.zeros((0, 3), device=DEV),
                                  torch.zeros((0, 3), device=DEV), torch.zeros(0, device=DEV), out0)
    torch.cuda.synchronize()
    assert (out0 == 0).all()
