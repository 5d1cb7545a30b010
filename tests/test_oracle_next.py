"""Pins of the oracle functions for SURVEY 8(f) rows 2 and 3 (carrier transport, electronics stage): closed forms,
hand-computed cases and library routines the functions must reduce to.  CPU only."""
import math

import numpy as np

from oracle import wtide_oracle as wo
from wtide_inputs.configs import square_cell

MU_E, MU_H, V_SAT = 180.0, 150.0, 150.0      # um^2/(V ns), um/ns (BASELINE.json configs[1]: 1800, 1500 cm^2/Vs, 1.5e7 cm/s)


def _desc():
    return square_cell(40.0, 30.0, (16, 16, 12), 64, 0.005, 4.0, 0.5, 4.0, 0.5)


def test_static_field_is_the_telescoped_sum():
    """sum_n H[n] dt: for H[n] = a_n * F(x) the result is (sum a_n) dt F(x); and for the solver's table it equals
    -grad_s W[nt-1] (the pin 'telescoping' of test_oracle_solve) -- here the plain-sum form."""
    rng = np.random.default_rng(0)
    F = rng.standard_normal((4, 3, 2, 3))
    a = rng.standard_normal(5)
    H = F[:, :, :, None, :] * a[None, None, None, :, None]
    assert np.allclose(wo.static_field(H, 0.25), a.sum() * 0.25 * F, rtol=1e-13, atol=1e-13)


def test_uniform_field_gives_uniform_saturated_drift():
    """Uniform E along z: v = mu E / (1 + mu E / v_sat) (BASELINE.json configs[1] formula), holes along +E, electrons along -E,
    positions on a straight line, step count = number of dt steps needed to leave through the z face."""
    d = _desc()
    es = np.zeros((16, 16, 12, 3), np.float32)
    es[..., 2] = 0.02                                    # 1/um per volt
    vb = 100.0                                           # E = 2 V/um
    start = np.array([[10.0, 30.0, 15.0], [10.0, 30.0, 15.0]], np.float32)
    sign = np.array([1, -1], np.int8)
    off, pos, vel = wo.drift_trajectories(es, d, start, sign, vb, MU_E, MU_H, V_SAT, 1000)
    for c, (mu, sg) in enumerate(((MU_H, 1.0), (MU_E, -1.0))):
        v = sg * mu * 2.0 / (1.0 + mu * 2.0 / V_SAT)
        p, w = pos[off[c]:off[c + 1]], vel[off[c]:off[c + 1]]
        assert np.allclose(w[:, 2], v, rtol=2e-5) and np.abs(w[:, :2]).max() == 0
        assert np.allclose(p[:, 2], 15.0 + v * d["dt"] * np.arange(len(p)), rtol=0, atol=2e-3)
        n_expected = math.ceil(((30.0 - 15.0) if sg > 0 else 15.0) / (abs(v) * d["dt"]))
        assert abs(len(p) - n_expected) <= 1 and len(p) < 1000
        assert abs(v) < V_SAT


def test_low_and_high_field_limits_and_the_step_cap():
    d = _desc()
    start = np.array([[10.0, 30.0, 15.0]], np.float32)
    for e_field, expect in ((1e-4, MU_H * 1e-4), (1e4, V_SAT)):      # v -> mu E and v -> v_sat
        es = np.zeros((16, 16, 12, 3), np.float32)
        es[..., 0] = e_field
        off, pos, vel = wo.drift_trajectories(es, d, start, np.array([1], np.int8), 1.0, MU_E, MU_H, V_SAT, 3)
        assert off[-1] == 3 or expect == V_SAT                      # (at v_sat the carrier may reach a column within 3 steps)
        assert np.allclose(vel[0, 0], expect, rtol=2e-2)


def test_a_linear_field_is_interpolated_exactly_and_columns_stop_the_carrier():
    """Trilinear interpolation reproduces a field that is linear in the node coordinates (away from the periodic seam);
    a carrier that starts inside a column records nothing; one that walks into a column stops at the first position inside."""
    d = _desc()
    x = np.arange(16) * 40.0 / 16
    z = np.arange(12) * 30.0 / 12
    es = np.zeros((16, 16, 12, 3), np.float32)
    es[..., 0] = (0.01 + 0.002 * x[:, None, None] + 0.001 * x[None, :, None] - 0.003 * z[None, None, :]).astype(np.float32)
    p0 = np.array([[13.3, 7.7, 11.1]], np.float32)
    off, pos, vel = wo.drift_trajectories(es, d, p0, np.array([1], np.int8), 1.0, MU_E, MU_H, V_SAT, 1)
    e0 = 0.01 + 0.002 * 13.3 + 0.001 * 7.7 - 0.003 * 11.1
    assert np.allclose(vel[0, 0], MU_H * e0 / (1 + MU_H * abs(e0) / V_SAT), rtol=1e-4)
    inside = np.array([[20.5, 20.5, 10.0], [0.5, 39.8, 20.0]], np.float32)          # readout column at the centre, bias at the corner
    off, pos, vel = wo.drift_trajectories(es, d, inside, np.array([1, -1], np.int8), 1.0, MU_E, MU_H, V_SAT, 10)
    assert off[-1] == 0
    es2 = np.zeros((16, 16, 12, 3), np.float32)
    es2[..., 0] = 1.0                                                               # holes drift along +x at ~v_sat towards the centre column
    off, pos, vel = wo.drift_trajectories(es2, d, np.array([[10.0, 20.0, 10.0]], np.float32), np.array([1], np.int8), 100.0, MU_E, MU_H, V_SAT, 500)
    assert 0 < off[-1] < 500
    assert pos[-1, 0] < 16.0 and pos[-1, 0] + vel[-1, 0] * d["dt"] >= 16.0 - 1e-3    # the next position is inside r = 4 around x = 20


def test_electronics_is_a_causal_fir_plus_noise_with_a_cfd_time():
    rng = np.random.default_rng(3)
    cur = rng.standard_normal((3, 40))
    h = np.exp(-np.arange(12) / 3.0)
    out, tc = wo.electronics(cur, h, 0.5)
    for t in range(3):
        assert np.allclose(out[t], np.convolve(cur[t], h)[:40] * 0.5, rtol=1e-12, atol=1e-12)
    noise = rng.standard_normal((3, 40))
    out2, _ = wo.electronics(cur, h, 0.5, noise=noise)
    assert np.allclose(out2, out + noise)
    # constant-fraction time of a ramp 0, 1, 2, ... with fraction 0.25 of its peak 8: crossing at n = 2
    ramp = np.zeros((1, 16))
    ramp[0, :9] = np.arange(9)
    o3, t3 = wo.electronics(ramp, np.array([1.0]), 1.0, cfd_fraction=0.25)
    assert np.allclose(o3, ramp) and abs(t3[0] - 2.0) < 1e-12
    o4, t4 = wo.electronics(-ramp, np.array([1.0]), 1.0, cfd_fraction=0.3)          # negative pulses: same time
    assert abs(t4[0] - 2.4) < 1e-12
    assert wo.electronics(np.zeros((1, 8)), h, 1.0)[1][0] == -1.0
