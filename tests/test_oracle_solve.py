"""Pins of the H-solve oracle (oracle/wtide_oracle.py: Problem, voxelize, solve_H) against what
the paper and the mathematics fix.  CPU only, small grids.

Method: PAPER.md:15 (abstract), :65, :95, :97, Fig. 3 (:109); readings R1-R20 of DESIGN.md.
Each test names the plausible mistake it is meant to catch.
"""
import math

import numpy as np
import pytest

from oracle import wtide_oracle as wo
from wtide_inputs import geometry_desc, reduced_desc
from wtide_inputs.configs import square_cell


def _cell(grid=(12, 12, 8), nt=6, dt=0.01, rho=0.5, lz=50.0):
    return square_cell(55.0, lz, grid, nt, dt, 5.0, rho, 5.0, rho)


def _plane_wave(shape, lengths, m, phase=0.0):
    xs = [np.arange(n) * l / n for n, l in zip(shape, lengths)]
    X, Y, Z = np.meshgrid(*xs, indexing="ij")
    k = [2 * math.pi * mi / l for mi, l in zip(m, lengths)]
    return np.cos(k[0] * X + k[1] * Y + k[2] * Z + phase), np.sin(k[0] * X + k[1] * Y + k[2] * Z + phase), k


def _free(shape, lengths, eps=1.0, sigma=0.0):
    return wo.Problem(shape, lengths, eps, np.full(shape, sigma), np.zeros((0, 3), int), np.zeros(0))


# ---------------------------------------------------------------------------------------------
def test_physical_constants_give_the_dielectric_relaxation_time():
    """tau = eps/sigma for diamond (eps_r 5.7) and 0.5 ohm cm is 5.7*8.854e-12/200 s = 0.2523 ps;
    n_sub = ceil(10 ps / tau) = 40 (SURVEY table of section 8).  Catches unit-conversion slips."""
    eps = 5.7 * wo.EPS0
    tau_ns = eps / wo.conductivity(0.5)
    assert tau_ns == pytest.approx(5.7 * 8.8541878128e-12 / 200.0 * 1e9, rel=1e-12)
    assert wo.auto_substeps(0.010, wo.conductivity(0.5), eps) == 40
    assert wo.auto_substeps(0.005, wo.conductivity(0.1), eps) == 100


def test_column_resistance_formula_and_the_papers_example():
    """R = 4 rho L/(pi d^2); 12 um, 0.75 ohm cm, 500 um is "about 30 kOhm"."""
    r = wo.column_resistance_kohm(0.75, 500.0, 12.0)
    assert r == pytest.approx(4 * 0.75e-2 * 500e-6 / (math.pi * (12e-6) ** 2) / 1e3, rel=1e-12)
    assert abs(r - 30.0) / 30.0 < 0.15


def test_voxelised_column_resistance_matches_the_closed_form():
    """L/(sigma n_nodes dx dy) vs 4 rho L/(pi d^2): pins the node-centre voxeliser (R13) and the
    minimum-image wrap of the corner column (the wrapped column must have as many nodes)."""
    d = square_cell(55.0, 500.0, (64, 64, 16), 4, 0.005, 6.0, 0.75, 6.0, 0.75)
    col_id, sigma, pads, vpad, pcol = wo.voxelize(d)
    dx = 55.0 / 64
    for j in (0, 1):
        n_xy = int((col_id[:, :, 8] == j).sum())
        r_vox = 0.75e4 * 500.0 / (n_xy * dx * dx) * 1e-3
        assert r_vox == pytest.approx(wo.column_resistance_kohm(0.75, 500.0, 12.0), rel=0.08)
    # readout: z in [0, 0.9 lz], pad on its first layer; bias: z in [0.1 lz, lz], pad on its last layer
    z = np.arange(16) * 500.0 / 16
    assert (col_id[32, 32, :] == 0).tolist() == (z <= 450.0).tolist()
    assert (col_id[0, 0, :] == 1).tolist() == (z >= 50.0).tolist()
    assert set(pads[pcol == 0][:, 2]) == {0} and set(pads[pcol == 1][:, 2]) == {15}
    assert np.all(vpad[pcol == 0] == 1.0) and np.all(vpad[pcol == 1] == 0.0)
    assert sigma.max() == pytest.approx(wo.conductivity(0.75))


def test_spectral_gradient_of_single_modes_and_nyquist_removal():
    """grad_s cos(k.x) = -k sin(k.x) for a retained mode (incl. negative index and a radix-3 axis);
    any mode with a Nyquist component is removed from every derivative (R11).
    Catches: wavenumber sign/aliasing, 2 pi / l scaling, axis mix-up."""
    shape, lengths = (8, 12, 6), (5.0, 7.0, 3.0)
    p = _free(shape, lengths)
    c, s, k = _plane_wave(shape, lengths, (1, -5, 2), phase=0.3)
    g = p.grad_s(c)
    for a in range(3):
        np.testing.assert_allclose(g[a], -k[a] * s, atol=1e-12)
    d = p.div_s(c, 2 * c, -c)
    np.testing.assert_allclose(d, -(k[0] + 2 * k[1] - k[2]) * s, atol=1e-12)
    c_nyq, _, _ = _plane_wave(shape, lengths, (1, 6, 0))       # ky at Nyquist, kx not
    for ga in p.grad_s(c_nyq):
        np.testing.assert_allclose(ga, 0.0, atol=1e-12)


def test_poisson_closed_form_for_a_plane_wave_of_charge():
    """q = cos(k.x) per node  =>  V = q / (vol eps |k|^2)   (divide by |k|^2)."""
    shape, lengths, eps = (8, 6, 9), (4.0, 3.0, 6.0), 2.5
    p = _free(shape, lengths, eps)
    c, _, k = _plane_wave(shape, lengths, (2, -1, 3))
    v = p.potential_of_charge(c)
    np.testing.assert_allclose(v, c / (p.vol * eps * sum(ki * ki for ki in k)), atol=1e-13)
    assert p.vol == pytest.approx(0.5 * 0.5 * (6.0 / 9))


def test_potential_is_the_brute_force_sum_of_fundamental_solutions():
    """north_star check 3: V(x) = sum_j q_j G(x - x_j) by explicit loops on a tiny grid equals the DFT
    route, and the literal translated-copy V_ext equals the spectral injection of the same charges
    (PAPER.md:97).  Catches: roll direction, G normalisation, index order."""
    shape, lengths = (4, 6, 3), (4.0, 5.0, 2.0)
    rng = np.random.default_rng(0)
    p = _free(shape, lengths, 1.7)
    q = rng.standard_normal(shape)
    q -= q.mean()
    v_fft = p.potential_of_charge(q)
    v_sum = np.zeros(shape)
    for i in range(shape[0]):
        for j in range(shape[1]):
            for k in range(shape[2]):
                for i2 in range(shape[0]):
                    for j2 in range(shape[1]):
                        for k2 in range(shape[2]):
                            v_sum[i, j, k] += q[i2, j2, k2] * p.green[(i - i2) % 4, (j - j2) % 6, (k - k2) % 3]
    np.testing.assert_allclose(v_fft, v_sum, atol=1e-12)
    # V_ext by translated copies vs spectral injection, on a problem with pads
    d = _cell()
    pr = wo.problem_from_desc(d)
    Q = rng.standard_normal(pr.nb)
    qa = np.zeros(pr.shape)
    qa[pr.pad_nodes[:, 0], pr.pad_nodes[:, 1], pr.pad_nodes[:, 2]] = Q
    np.testing.assert_allclose(pr.v_ext(Q, 0.25), pr.potential_of_charge(qa) + 0.25, atol=1e-12 * np.abs(Q).sum())


def test_boundary_conditions_and_neutrality_hold_after_every_potential():
    """Pad potentials are reproduced at the pad nodes, sum Q = -sum q (R10)."""
    d = _cell()
    pr = wo.problem_from_desc(d)
    rng = np.random.default_rng(1)
    for q in (np.zeros(pr.shape), rng.standard_normal(pr.shape) * 10):
        q = q - q.mean() + 0.01                      # non-neutral free charge on purpose
        v, Q, c = pr.potential(q)
        b = pr.pad_nodes
        np.testing.assert_allclose(v[b[:, 0], b[:, 1], b[:, 2]], pr.pad_potential, atol=1e-10)
        assert Q.sum() == pytest.approx(-q.sum(), abs=1e-9)


def test_superposition_over_electrodes():
    """north_star check 2: all pads stepped to V_w => W == V_w, Q = 0, H == 0; and H is additive over
    disjoint sets of driven pads ("depends on all impedances")."""
    d = _cell(nt=3)
    pr = wo.problem_from_desc(d)
    ns = 4                                            # any stable substep count pins linearity
    ns = max(ns, wo.substeps_from_desc(d))
    ones = wo.Problem(pr.shape, pr.lengths, pr.eps, pr.sigma, pr.pad_nodes, np.ones(pr.nb))
    v, Q, c = ones.potential(np.zeros(pr.shape))
    np.testing.assert_allclose(v, 1.0, atol=1e-12)
    np.testing.assert_allclose(Q, 0.0, atol=1e-9)
    H1 = ones.solve_H(3, d["dt"], ns)
    assert np.abs(H1).max() < 1e-9
    Ha = pr.solve_H(3, d["dt"], ns)                                    # readout driven
    other = wo.Problem(pr.shape, pr.lengths, pr.eps, pr.sigma, pr.pad_nodes, 1.0 - pr.pad_potential)
    Hb = other.solve_H(3, d["dt"], ns)                                 # bias driven
    scale = np.abs(Ha).max()
    np.testing.assert_allclose(Ha + Hb, 0.0, atol=1e-9 * scale)


def test_charge_conservation_at_every_substep():
    d = _cell(nt=3)
    pr = wo.problem_from_desc(d)
    seen = []
    pr.solve_H(3, d["dt"], wo.substeps_from_desc(d),
               on_substep=lambda n, s, q, Q: seen.append((q.sum(), Q.sum(), np.abs(q).sum())))
    assert len(seen) == 2 * wo.substeps_from_desc(d)
    for sq, sQ, mag in seen:
        assert abs(sq) < 1e-10 * max(mag, 1.0) and abs(sQ) < 1e-8


def test_d4_symmetry_of_a_centred_square_cell():
    """H_x(-x, y) = -H_x(x, y), H_x(x, y) = H_y(y, x) for a symmetric voxelisation."""
    d = _cell(grid=(12, 12, 6), nt=2)
    H = wo.solve_H_from_desc(d)
    n = 12
    refl = (n - np.arange(n)) % n
    scale = np.abs(H).max()
    np.testing.assert_allclose(H[refl][..., 0], -H[..., 0], atol=1e-9 * scale)
    np.testing.assert_allclose(H[refl][..., 1], H[..., 1], atol=1e-9 * scale)
    np.testing.assert_allclose(np.swapaxes(H, 0, 1)[..., 0], H[..., 1], atol=1e-9 * scale)


def test_euler_update_of_one_mode_in_a_uniform_conductor():
    """Uniform sigma, no pads, one Fourier mode of charge: amplitude (1 - dt_int sigma/eps)^k exactly
    (R1: d_t rho = div(sigma grad psi) = -(sigma/eps) rho).  Catches: sign of the update, missing vol,
    eps or sigma factors."""
    shape, lengths, eps, sig = (8, 6, 12), (4.0, 3.0, 7.0), 3.0, 5.0
    p = _free(shape, lengths, eps, sig)
    c, _, _ = _plane_wave(shape, lengths, (1, 2, -4), 0.7)
    q = c.copy()
    dt_int = 0.3 * eps / sig
    for k in range(1, 6):
        q, _ = p.euler_substep(q, dt_int)
        np.testing.assert_allclose(q, (1 - 0.3) ** k * c, atol=1e-12)


def test_forward_euler_stability_bound_is_two_relaxation_times():
    """R12: the update operator has eigenvalues in [0, sigma_max/eps], so forward Euler is stable iff
    dt_int <= 2 eps/sigma_max.  With a column wide enough to hold a mode of its own (14 um radius on a
    16^2 x 8 grid) 1.9 tau stays bounded and 2.1 tau grows exponentially."""
    d = square_cell(55.0, 50.0, (16, 16, 8), 3, 0.01, 14.0, 0.5, 5.0, 0.5)
    pr = wo.problem_from_desc(d)
    tau = pr.eps / pr.sigma.max()

    def run(factor, steps=300):
        q = np.zeros(pr.shape)
        norms = []
        for _ in range(steps):
            q, _ = pr.euler_substep(q, factor * tau)
            norms.append(np.abs(q).max())
        return np.array(norms)
    lo, hi = run(1.9), run(2.1)
    assert lo[-1] < 3 * lo[50]
    assert hi[-1] > 1e6 * hi[50]


def test_telescoping_sum_of_H_is_the_last_weighting_field():
    """sum_n H[n] dt = -grad_s W[nt-1] exactly (R2)."""
    d = _cell(nt=4)
    pr = wo.problem_from_desc(d)
    H, ws = pr.solve_H(4, d["dt"], wo.substeps_from_desc(d), return_potentials=True)
    g = pr.grad_s(ws[-1])
    for a in range(3):
        np.testing.assert_allclose(H[..., a].sum(axis=3) * d["dt"], -g[a], atol=1e-10 * np.abs(g[a]).max())


def test_zero_resistance_limit_collapses_H_onto_the_first_samples():
    """north_star check 1 / PAPER.md:35: without impedance H is the static weighting field times a
    delta in time.  With dt >> every relaxation time the response is complete after one output step:
    the columns are equipotentials at their pad values and H[n >= 2] vanishes."""
    d = _cell(grid=(12, 12, 8), nt=3, rho=0.5)
    pr = wo.problem_from_desc(d)
    tau = pr.eps / pr.sigma.max()
    ns = 1500
    d["dt"] = ns * tau                                         # dt = 1500 relaxation times, dt_int = tau
    H, ws = pr.solve_H(3, d["dt"], ns, return_potentials=True)
    col_id = wo.voxelize(d)[0]
    assert np.abs(ws[1][col_id == 0] - 1.0).max() < 5e-2
    assert np.abs(ws[1][col_id == 1]).max() < 5e-2
    early = np.linalg.norm(H[..., 0, :] + H[..., 1, :])
    assert np.linalg.norm(H[..., 2:, :]) < 0.1 * early          # the coarse 12^2 x 8 grid keeps a slow tail


def test_two_layer_capacitor_relaxation_time():
    """1-D resistive slab (thickness b) in series with an insulating gap g between two pad planes:
    E_gap(t) = V/g - (V/g - V/(b+g)) exp(-t/tau), tau = eps (b+g)/(sigma g).  Approximate pin (the
    spectral derivative smears the slab edges): initial and final fields and tau within 20 %."""
    nz, lz = 48, 48.0
    shape, lengths, eps, sig = (1, 1, nz), (1.0, 1.0, lz), 1.0, 1.0
    b, g = 8, 8
    sigma = np.zeros(shape)
    sigma[:, :, 0:b + 1] = sig                       # slab nodes z = 0..b
    pads = [(0, 0, 0), (0, 0, b + g)]
    vp = [1.0, 0.0]
    p = wo.Problem(shape, lengths, eps, sigma, pads, vp)
    tau = eps * (b + g) / (sig * g)
    dt_int = 0.25 * eps / sig
    q = np.zeros(shape)
    kmid = b + g // 2
    e_gap = []
    for s in range(int(6 * tau / dt_int)):
        v, _, _ = p.potential(q)
        e_gap.append(-p.grad_s(v)[2][0, 0, kmid])
        q, _ = p.euler_substep(q, dt_int)
    e_gap = np.array(e_gap)
    assert e_gap[0] == pytest.approx(1.0 / (b + g), rel=0.1)
    assert e_gap[-1] == pytest.approx(1.0 / g, rel=0.1)
    # time to cover 1 - 1/e of the swing
    frac = (e_gap - e_gap[0]) / (e_gap[-1] - e_gap[0])
    t63 = np.argmax(frac >= 1 - math.exp(-1)) * dt_int
    assert t63 == pytest.approx(tau, rel=0.2)


def test_config_descriptors_are_well_formed():
    for cfg in (0, 1, 2, 4):
        d = geometry_desc(cfg)
        small = reduced_desc(d, grid=(16, 16, 8), nt=4)
        col_id, sigma, pads, vpad, pcol = wo.voxelize(small)
        assert len(pads) > 0 and (vpad == 1.0).any() and (vpad == 0.0).any()
        assert d["nt"] % 4 == 0
    d1 = geometry_desc(1)
    for c in d1["columns"]:
        assert 3.0 <= c["radius"] <= 8.0 and 0.1 <= c["resistivity"] <= 1.0


# ---- sharper form of north_star check 1 and the solver <-> Eq. 1.1 link -------------------------
def _brute_force_green(desc):
    """G(x) = (1/(N vol)) sum_k e^{i kappa.x} / (eps |kappa|^2) over the retained modes, by direct summation (no FFT):
    the potential of a unit point charge on the periodic lattice (PAPER.md:97 'fundamental solution'; R9, R11)."""
    nx, ny, nz = desc["nx"], desc["ny"], desc["nz"]
    lx, ly, lz = desc["lx"], desc["ly"], desc["lz"]
    eps = desc["eps_r"] * wo.EPS0
    vol = (lx / nx) * (ly / ny) * (lz / nz)
    X, Y, Z = np.meshgrid(np.arange(nx) * lx / nx, np.arange(ny) * ly / ny, np.arange(nz) * lz / nz, indexing="ij")
    G = np.zeros((nx, ny, nz))
    for a in range(nx):
        ma = a if 2 * a < nx else a - nx
        for b in range(ny):
            mb = b if 2 * b < ny else b - ny
            for c in range(nz):
                mc = c if 2 * c < nz else c - nz
                if 2 * a == nx or 2 * b == ny or 2 * c == nz or (a == 0 and b == 0 and c == 0):
                    continue
                kx, ky, kz = 2 * math.pi * ma / lx, 2 * math.pi * mb / ly, 2 * math.pi * mc / lz
                G += np.cos(kx * X + ky * Y + kz * Z) / (eps * (kx * kx + ky * ky + kz * kz))
    return G / (nx * ny * nz * vol)


def test_stationary_state_makes_every_column_an_equipotential_at_its_pad_value():
    """north_star check 1 on the solver, sharp form: the stationary state of the forward-Euler map (found here by GMRES on
    q = Phi(q) instead of marching for 10^5 substeps) has EVERY node of a column at the potential of the column's pad to
    1e-4 V_w -- the columns are ideal conductors in the limit, H has collapsed onto the prompt response -- and the pad
    potentials are reproduced.  Beside it, the nodal-Dirichlet static solution with whole columns as electrodes (dense
    solve on a Green's function summed by brute force, SURVEY 8(c) pin table): the two agree ON the columns; between them
    they differ at the discretisation level, because the spectral divergence of the masked current (R17, R20) leaves
    charge on non-conducting nodes that never relaxes (sigma = 0 there).  That difference is recorded, not asserted tight."""
    from scipy.sparse.linalg import LinearOperator, gmres
    grid = (12, 12, 6)
    d = square_cell(40.0, 30.0, grid, 8, 0.01, 5.0, 0.05, 5.0, 0.05)
    prob = wo.problem_from_desc(d)
    col_id, _, _, _, _ = wo.voxelize(d)
    n_sub = wo.substeps_from_desc(d)
    dt_int = d["dt"] / n_sub
    N = int(np.prod(grid))
    phi0, _ = prob.euler_substep(np.zeros(grid), dt_int)

    def project(q):
        """the states reachable from q = 0: no k = 0 component (total charge is conserved) and no Nyquist component (R11)"""
        qh = np.fft.fftn(q) * prob.retained
        qh[0, 0, 0] = 0.0
        return np.real(np.fft.ifftn(qh))

    def residual_map(x):
        q = project(x.reshape(grid))
        y, _ = prob.euler_substep(q, dt_int)
        return (x.reshape(grid) - project(y - phi0)).ravel()
    qs, _ = gmres(LinearOperator((N, N), matvec=residual_map, dtype=float), project(phi0).ravel(), rtol=1e-11, atol=0, restart=N, maxiter=3)
    q_inf = project(qs.reshape(grid))
    q_next, _ = prob.euler_substep(q_inf, dt_int)
    assert np.abs(q_next - q_inf).max() <= 1e-8 * np.abs(q_inf).max()            # it IS a fixed point
    w_inf, charges, _ = prob.potential(q_inf)
    target = np.array([d["v_w"] if c["role"] == wo.WT_READOUT else 0.0 for c in d["columns"]])
    on_cols = col_id >= 0
    assert np.abs(w_inf[on_cols] - target[col_id[on_cols]]).max() <= 1e-4 * d["v_w"]
    assert abs(q_inf.sum()) <= 1e-9 * np.abs(q_inf).sum() and abs(charges.sum()) <= 1e-9 * np.abs(charges).sum()
    # nodal-Dirichlet static solution on an independently summed Green's function
    G = _brute_force_green(d)
    assert np.abs(G - prob.green).max() <= 1e-12 * np.abs(G).max()
    nodes = np.argwhere(on_cols)
    vals = target[col_id[on_cols]]
    nb = len(nodes)
    A = np.zeros((nb + 1, nb + 1))
    for i in range(nb):
        dd = (nodes[i][None, :] - nodes) % np.array(grid)
        A[i, :nb] = G[dd[:, 0], dd[:, 1], dd[:, 2]]
    A[:nb, nb] = 1.0
    A[nb, :nb] = 1.0
    sol = np.linalg.solve(A, np.concatenate([vals, [0.0]]))
    v_static = np.full(grid, sol[-1])
    for qb, (i, j, k) in zip(sol[:-1], nodes):
        v_static += qb * np.roll(G, (int(i), int(j), int(k)), (0, 1, 2))
    assert np.abs(v_static[on_cols] - vals).max() <= 1e-10
    assert np.abs(w_inf - v_static)[on_cols].max() <= 1e-4 * d["v_w"]
    # (between the columns the two differ by up to 0.7 V_w on this 12 x 12 x 6 grid -- measured, see the docstring: the
    #  stationary state of the pseudo-spectral scheme is NOT the nodal electrostatic solution, so nothing is asserted there)


def test_overlapping_columns_first_column_wins():
    """R13 'the first column in the list wins on overlap': two overlapping cylinders of different resistivity; every
    node of the lens belongs to column 0, column 1's pad has no node of the lens, conductivities follow the owner.
    Node sets enumerated here by hand (plain loops over the node-centre test)."""
    d = dict(lx=16.0, ly=16.0, lz=8.0, nx=16, ny=16, nz=8, nt=4, dt=0.01, eps_r=5.7, v_w=1.0, substeps=0, columns=[
        dict(cx=6.0, cy=8.0, radius=3.0, resistivity=0.5, z0=0.0, z1=8.0, role=wo.WT_READOUT, pad_at_z1=0),
        dict(cx=9.0, cy=8.0, radius=3.0, resistivity=2.0, z0=0.0, z1=8.0, role=wo.WT_BIAS, pad_at_z1=0)])
    col_id, sigma, pads, pot, pcol = wo.voxelize(d)
    in0 = {(i, j) for i in range(16) for j in range(16) if (i - 6.0) ** 2 + (j - 8.0) ** 2 <= 9.0}
    in1 = {(i, j) for i in range(16) for j in range(16) if (i - 9.0) ** 2 + (j - 8.0) ** 2 <= 9.0}
    lens = in0 & in1
    assert len(lens) >= 5
    for (i, j) in in0:
        assert (col_id[i, j, :] == 0).all() and np.allclose(sigma[i, j, :], wo.conductivity(0.5))
    for (i, j) in in1 - in0:
        assert (col_id[i, j, :] == 1).all() and np.allclose(sigma[i, j, :], wo.conductivity(2.0))
    pad_sets = {c: {(int(p[0]), int(p[1])) for p, pc in zip(pads, pcol) if pc == c} for c in (0, 1)}
    assert pad_sets[0] == in0 and pad_sets[1] == in1 - in0
    assert (pads[:, 2] == 0).all() and set(pot[pcol == 0]) == {1.0} and set(pot[pcol == 1]) == {0.0}


def test_a_carrier_walked_between_the_columns_collects_its_charge():
    """Solver and Eq. 1.1 together (SURVEY 8(c) pin table): oracle H fed to the oracle's Eq. 1.1 for a carrier walked in
    small steps from the surface of the bias column to the surface of the readout column gives
        sum_n i[n] dt = (q / V_w) [W(x_end) - W(x_start)]          (path quadrature of -grad W . dx, telescoped H)
    with W the potential after the last step the truncated sums reach, and that is q within the discretisation error of
    'columns are equipotentials at 0 and V_w'."""
    grid = (16, 16, 8)
    d = square_cell(32.0, 24.0, grid, 48, 0.01, 4.0, 0.05, 4.0, 0.05)
    prob = wo.problem_from_desc(d)
    n_sub = wo.substeps_from_desc(d)
    H, ws = prob.solve_H(d["nt"], d["dt"], n_sub, return_potentials=True)
    # straight path at mid depth from the bias column (at the cell corner) towards the readout column (cell centre)
    n_steps = 24
    s = np.linspace(0.0, 1.0, n_steps + 1)
    start = np.array([4.3 / math.sqrt(2), 4.3 / math.sqrt(2), 12.0])
    end = np.array([16.0 - 4.3 / math.sqrt(2), 16.0 - 4.3 / math.sqrt(2), 12.0])
    pts = start[None, :] + s[:, None] * (end - start)[None, :]
    pos = pts[:-1].astype(np.float32)
    vel = (np.diff(pts, axis=0) / d["dt"]).astype(np.float32)
    q = 3.0
    cur = wo.convolve_currents(H, grid, (d["lx"], d["ly"], d["lz"]), d["nt"], d["dt"], d["v_w"], np.array([0, n_steps]), pos, vel,
                               np.array([q], np.float32))
    collected = cur[0].sum() * d["dt"]

    def w_at(w, p):       # trilinear sample with the ABI's index arithmetic
        i0, i1, f, _ = wo.trajectory_nodes(grid, (d["lx"], d["ly"], d["lz"]), np.asarray(p, np.float32)[None, :])
        out = 0.0
        for cx in (0, 1):
            for cy in (0, 1):
                for cz in (0, 1):
                    wgt = (f[0, 0] if cx else 1 - f[0, 0]) * (f[0, 1] if cy else 1 - f[0, 1]) * (f[0, 2] if cz else 1 - f[0, 2])
                    out += wgt * w[(i1 if cx else i0)[0, 0], (i1 if cy else i0)[0, 1], (i1 if cz else i0)[0, 2]]
        return out
    w_last = ws[d["nt"] - 1 - n_steps]          # every step m <= n_steps - 1 telescopes at least up to this potential
    expected = q / d["v_w"] * (w_at(ws[-1], pts[-1]) - w_at(ws[-1], pts[0]))
    assert np.abs(ws[-1] - w_last).max() <= 0.03 * d["v_w"]                  # the response has settled along the walk
    print("collected", collected, "expected", expected)
    assert abs(collected - expected) <= 0.04 * abs(expected), (collected, expected)
    assert abs(collected - q) <= 0.15 * q, collected                              # electrode to electrode: the carrier's charge
    assert collected > 0                                                          # sign convention of Eq. 1.1 (R3)
