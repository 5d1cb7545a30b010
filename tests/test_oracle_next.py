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


# ---- the electrostatic (Laplace) field ---------------------------------------------------------------
def _cell(grid=(16, 16, 8)):
    return square_cell(40.0, 30.0, grid, 8, 0.01, 4.0, 0.5, 4.0, 0.5)


def test_static_potential_reproduces_the_electrode_values_and_is_neutral():
    d = _cell()
    col_id, _, _, _, _ = wo.voxelize(d)
    v, e, q = wo.static_potential(d, [1.0, -2.0])
    assert np.abs(v[col_id == 0] - 1.0).max() <= 1e-10 and np.abs(v[col_id == 1] + 2.0).max() <= 1e-10
    assert abs(q.sum()) <= 1e-9 * np.abs(q).sum() and (q[col_id < 0] == 0).all()
    # between the electrodes the potential stays between their values (up to the ringing of the spectral operator)
    assert v.min() >= -2.0 - 0.3 and v.max() <= 1.0 + 0.3


def test_static_potential_is_linear_and_constant_when_all_electrodes_agree():
    d = _cell()
    v1, e1, _ = wo.static_potential(d, [1.0, 0.0])
    v2, e2, _ = wo.static_potential(d, [0.0, 1.0])
    v3, e3, _ = wo.static_potential(d, [3.0, -0.5])
    assert np.abs(3.0 * v1 - 0.5 * v2 - v3).max() <= 1e-9
    assert np.abs(3.0 * e1 - 0.5 * e2 - e3).max() <= 1e-9
    vc, ec, qc = wo.static_potential(d, [0.7, 0.7])
    assert np.abs(vc - 0.7).max() <= 1e-9 and np.abs(ec).max() <= 1e-9
    assert np.abs((v1 + v2) - 1.0).max() <= 1e-9          # north_star check 2 in its static form


def test_static_potential_has_the_logarithmic_profile_of_a_line_charge_near_a_thin_column():
    """A thin full-depth column in a z-invariant cell: between a few grid spacings and a fraction of the pitch the potential
    falls like -(lambda / 2 pi eps) ln r (coaxial textbook profile), lambda = charge per unit length of the column."""
    d = dict(lx=64.0, ly=64.0, lz=8.0, nx=64, ny=64, nz=4, nt=4, dt=0.01, eps_r=5.7, v_w=1.0, substeps=0, columns=[
        dict(cx=32.0, cy=32.0, radius=0.4, resistivity=0.5, z0=0.0, z1=8.0, role=wo.WT_READOUT, pad_at_z1=0),
        dict(cx=0.0, cy=0.0, radius=0.4, resistivity=0.5, z0=0.0, z1=8.0, role=wo.WT_BIAS, pad_at_z1=0)])
    v, e, q = wo.static_potential(d, [1.0, 0.0])
    assert np.abs(v - v[:, :, :1]).max() <= 1e-9                                   # z-invariant
    lam = q[32, 32, :].sum() / d["lz"]                                             # e per um
    eps = d["eps_r"] * wo.EPS0
    r1, r2 = 4, 10
    slope = (v[32 + r2, 32, 0] - v[32 + r1, 32, 0]) / math.log(r2 / r1)
    assert abs(slope / (-lam / (2 * math.pi * eps)) - 1.0) <= 0.05
    # and the radial field there is lambda / (2 pi eps r).  The spectral gradient of the potential of a one-node-wide charge
    # carries a two-node saw-tooth (the Nyquist plane is removed, R11/R14: part of the defined result), so the field is
    # compared after the (1/4, 1/2, 1/4) average over neighbouring nodes that removes that component
    ex = e[:, 32, 0, 0]
    smooth = 0.25 * ex[32 + 5] + 0.5 * ex[32 + 6] + 0.25 * ex[32 + 7]
    assert abs(smooth / (lam / (2 * math.pi * eps * 6.0)) - 1.0) <= 0.05
    assert abs(-(v[32 + 7, 32, 0] - v[32 + 5, 32, 0]) / 2.0 / (lam / (2 * math.pi * eps * 6.0)) - 1.0) <= 0.03    # central difference of V


def test_static_potential_equals_the_stationary_state_on_the_columns():
    """The quasi-static solver's stationary state (tests/test_oracle_solve.py) and the Laplace solution hold the same
    Dirichlet data: both put every column node at its electrode's potential."""
    d = _cell((12, 12, 6))
    col_id, _, _, _, _ = wo.voxelize(d)
    v, _, _ = wo.static_potential(d, [d["v_w"], 0.0])
    assert np.abs(v[col_id == 0] - d["v_w"]).max() <= 1e-10 and np.abs(v[col_id == 1]).max() <= 1e-10


# ---- mirror (Neumann) surfaces by the method of images ---------------------------------------------------
def _mirror_cell(grid=(8, 8, 6), nt=3):
    return square_cell(40.0, 30.0, grid, nt, 0.01, 6.0, 0.5, 6.0, 0.5)


def test_even_extension_is_the_neumann_problem_cosine_transform_route():
    """Independent route: with mirror planes at z = 0 and z = lz the potential of a charge is a cosine series in z.  DCT-I over
    the layers 0 .. nz (scipy) with the same 1/(eps |kappa|^2), kappa_z = pi m / lz, and the highest cosine mode removed (it
    is the Nyquist mode of the doubled box, R11) must equal the oracle's periodic potential of the evenly extended charge."""
    import scipy.fft
    d = wo.mirror_z_desc(_mirror_cell())
    prob = wo.problem_from_desc(d)
    nx, ny, nz2 = prob.shape
    nz = nz2 // 2
    rng = np.random.default_rng(5)
    q_half = rng.standard_normal((nx, ny, nz + 1))
    q = np.zeros(prob.shape)
    q[:, :, :nz + 1] = q_half
    q[:, :, nz + 1:] = q_half[:, :, nz - 1:0:-1]                      # node 2 nz - k mirrors node k
    v = prob.potential_of_charge(q)
    kx, rx = wo.wavenumbers(nx, d["lx"])
    ky, ry = wo.wavenumbers(ny, d["ly"])
    m = np.arange(nz + 1)
    kz = np.pi * m / (d["lz"] / 2)
    ret = rx[:, None, None] & ry[None, :, None] & (m < nz)[None, None, :]
    k2 = kx[:, None, None] ** 2 + ky[None, :, None] ** 2 + kz[None, None, :] ** 2
    g = np.zeros(k2.shape)
    ok = ret & (k2 > 0)
    g[ok] = 1.0 / (prob.eps * k2[ok])
    qh = scipy.fft.dct(np.fft.fftn(q_half, axes=(0, 1)), type=1, axis=2)
    v_cos = np.real(np.fft.ifftn(scipy.fft.idct(g * qh, type=1, axis=2), axes=(0, 1))) / prob.vol
    assert np.abs(v[:, :, :nz + 1] - v_cos).max() <= 1e-11 * np.abs(v).max()
    ez = -prob.grad_s(v)[2]
    assert np.abs(ez[:, :, [0, nz]]).max() <= 1e-10 * np.abs(ez).max()     # no normal field on the mirror planes


def test_mirrored_geometry_and_its_table_are_even_about_both_planes():
    base = _mirror_cell()
    d = wo.mirror_z_desc(base)
    nz = base["nz"]
    col_id, _, pad_nodes, pad_pot, pad_col = wo.voxelize(d)
    occ = col_id >= 0
    assert (occ[:, :, 1:] == occ[:, :, :0:-1]).all()                      # node 2 nz - k mirrors node k
    # pads of the BASELINE-type columns (readout from z = 0, bias up to z = lz) sit on the mirror planes: their images carry none
    assert set(pad_nodes[:, 2]) == {0, nz} and set(pad_col) == {0, 1}
    assert [c["role"] for c in d["columns"]] == [wo.WT_READOUT, wo.WT_BIAS, wo.WT_SEGMENT, wo.WT_SEGMENT]
    H = wo.solve_H_from_desc(d)
    scale = np.abs(H).max()
    assert np.abs(H[:, :, 1:, :, :2] - H[:, :, :0:-1, :, :2]).max() <= 1e-9 * scale      # H_x, H_y even
    assert np.abs(H[:, :, 1:, :, 2] + H[:, :, :0:-1, :, 2]).max() <= 1e-9 * scale        # H_z odd
    assert np.abs(H[:, :, [0, nz], :, 2]).max() <= 1e-9 * scale                          # and zero on the planes (Neumann)
    # it is a different problem from the periodic one: the table of the plain cell differs by far more than any tolerance
    Hp = wo.solve_H_from_desc(base)
    assert wo.h_rel_l2(H[:, :, :nz], Hp) > 1e-2
    # a pad away from the planes is imaged as a pad
    off = dict(base, columns=[dict(base["columns"][0], z0=6.0, z1=20.0), base["columns"][1]])
    dm = wo.mirror_z_desc(off)
    assert dm["columns"][2]["role"] == wo.WT_READOUT and dm["columns"][2]["pad_at_z1"] == 1
    _, _, pn, _, pc = wo.voxelize(dm)
    k0, k2 = set(pn[pc == 0][:, 2]), set(pn[pc == 2][:, 2])
    assert len(k0) == 1 and len(k2) == 1 and list(k0)[0] + list(k2)[0] == 2 * nz
