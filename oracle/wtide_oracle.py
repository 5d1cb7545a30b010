"""Plain, slow, double-precision CPU oracle for libwtide.  TEST INFRASTRUCTURE ONLY.

This file restates, step by step and in the paper's order, what the hot path of
arxiv/paper_2605_13987 computes.  It shares no code with the CUDA path
(paper_2605_13987_b200/): neither imports the other.  Only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import it.  numpy.fft and scipy LU are used as library primitives for single
steps (a DFT, a dense solve); there is no blocking, fusion or reordering beyond
what the algorithm states.

What it follows (citations are PAPER.md line + section; "Rn" = reading n listed in
DESIGN.md, taken from SURVEY.md section 8(c) because the paper defers the PDE to its
Ref. [10], which is not available):

* Eq. 1.1, PAPER.md:35-39 (section 1):  i(t) = -(q/V_w) int_0^t H(x(t'),t-t').v(t') dt'
* H solve, PAPER.md:15 (abstract), :65 (section 2), :95, :97 (section 3), Fig. 3 (:109):
  "fundamental solutions to impose boundary conditions and spectral methods to extend
  the solution to the bulk", "iterative forward-Euler procedure", V <-> rho through the
  3-D DFT and |k|^2, V_ext = "rescaled and translated chunks of the fundamental solution".

Pins (tests/test_oracle_*.py, all `-m "not gpu"`): see DESIGN.md section "Oracle pins".
PARITY UNPINNED: the absolute values of H for the paper's sensor (the paper prints none).

Units (R15): length um, time ns, potential V, charge in elementary charges e.
H is in V/(um*ns), velocities in um/ns, currents in e/ns.
"""
from __future__ import annotations

import math

import numpy as np
import scipy.linalg

# eps0 = 8.8541878128e-12 F/m  ->  e / (V um)
EPS0 = 8.8541878128e-12 * 1e-6 / 1.602176634e-19
WT_BIAS = 0
WT_READOUT = 1
WT_SEGMENT = 2       # conductive cylinder without a contact pad (stacked segments: depth-dependent conductivity)


def conductivity(resistivity_ohm_cm: float) -> float:
    """sigma = 1/resistivity in e/(V um ns).  (1/(ohm cm) = 100 S/m = 1e-4 S/um.)"""
    return (1.0 / (resistivity_ohm_cm * 1e-2)) * 1e-6 * 1e-9 / 1.602176634e-19


def column_resistance_kohm(resistivity_ohm_cm: float, length_um: float, diameter_um: float) -> float:
    """R = 4 rho L / (pi d^2), PAPER.md:137 (section 5).  Returned in kOhm."""
    rho_ohm_um = resistivity_ohm_cm * 1e4
    return 4.0 * rho_ohm_um * length_um / (math.pi * diameter_um ** 2) * 1e-3


# ----------------------------------------------------------------------------------------
# grid, wavenumbers (oracle step 1)
# ----------------------------------------------------------------------------------------
def wavenumbers(n: int, length: float):
    """kappa(k) = 2 pi m / l with m = k for k < n/2, k - n for k > n/2.
    Returns (kappa[n], retained[n]); the Nyquist index k = n/2 (even n) is not retained (R11)."""
    k = np.arange(n)
    m = np.where(2 * k < n, k, k - n).astype(np.float64)
    retained = np.ones(n, dtype=bool)
    if n % 2 == 0:
        retained[n // 2] = False
        m[n // 2] = 0.0
    return 2.0 * math.pi * m / length, retained


def node_coordinates(n: int, length: float) -> np.ndarray:
    """x_i = (i * l) / n  (multiply first, then divide: the library uses the same order)."""
    return (np.arange(n, dtype=np.float64) * length) / n


# ----------------------------------------------------------------------------------------
# voxeliser (oracle step 2; "the STL geometry is voxelized"; R13)
# ----------------------------------------------------------------------------------------
def voxelize(desc: dict):
    """Node-centre test for cylinders parallel to z.

    Returns (col_id[nx,ny,nz] int, sigma[nx,ny,nz], pad_nodes[B,3] int, pad_potential[B], pad_col[B]).
    A node belongs to column j iff its minimum-image lateral distance^2 to the axis is <= r^2
    and z0 <= z <= z1; the first column in the list wins on overlap.  Pad nodes of a column =
    its nodes in its first (pad_at_z1 = 0) or last (pad_at_z1 = 1) z-layer; V_pad = v_w for
    readout columns, 0 for bias columns (R4, R8); WT_SEGMENT columns conduct but carry no pad.  Pad order: column
    order, then (ix, iy) row-major.
    """
    nx, ny, nz = desc["nx"], desc["ny"], desc["nz"]
    lx, ly, lz = desc["lx"], desc["ly"], desc["lz"]
    x = node_coordinates(nx, lx)
    y = node_coordinates(ny, ly)
    z = node_coordinates(nz, lz)
    col_id = np.full((nx, ny, nz), -1, dtype=np.int64)
    sigma = np.zeros((nx, ny, nz), dtype=np.float64)
    pad_nodes, pad_pot, pad_col = [], [], []
    for j, col in enumerate(desc["columns"]):
        dxm = np.fmod(np.abs(x - col["cx"]), lx)
        dxm = np.minimum(dxm, lx - dxm)
        dym = np.fmod(np.abs(y - col["cy"]), ly)
        dym = np.minimum(dym, ly - dym)
        inxy = (dxm[:, None] * dxm[:, None] + dym[None, :] * dym[None, :]) <= col["radius"] * col["radius"]
        inz = (col["z0"] <= z) & (z <= col["z1"])
        if not inz.any() or not inxy.any():
            raise ValueError(f"column {j} contains no grid node")
        member = inxy[:, :, None] & inz[None, None, :] & (col_id < 0)
        col_id[member] = j
        sigma[member] = conductivity(col["resistivity"])
        if col["role"] == WT_SEGMENT:
            continue
        layers = np.nonzero(inz)[0]
        kpad = int(layers[-1] if col["pad_at_z1"] else layers[0])
        ij = np.argwhere(member[:, :, kpad])
        if len(ij) == 0:
            raise ValueError(f"column {j} has no pad node")
        for (i, jj) in ij:
            pad_nodes.append((int(i), int(jj), kpad))
            pad_pot.append(desc["v_w"] if col["role"] == WT_READOUT else 0.0)
            pad_col.append(j)
    return (col_id, sigma, np.array(pad_nodes, dtype=np.int64).reshape(-1, 3),
            np.array(pad_pot, dtype=np.float64), np.array(pad_col, dtype=np.int64))


def auto_substeps(dt: float, sigma_max: float, eps: float) -> int:
    """n_sub = ceil(dt * sigma_max / eps)  (R12: dt_int * sigma_max / eps <= 1 < 2 = stability bound)."""
    return max(1, int(math.ceil(dt * (sigma_max / eps))))


# ----------------------------------------------------------------------------------------
# the quasi-static problem (oracle steps 3-7)
# ----------------------------------------------------------------------------------------
class Problem:
    """div[ eps grad d_t psi + sigma grad psi ] = 0 on a periodic box (R1, R5-R7), pads held
    at given potentials by point charges on the pad nodes (R8-R10).

    State q[nx,ny,nz] = free charge per node in e (charge density = q / voxel volume).
    """

    def __init__(self, shape, lengths, eps, sigma, pad_nodes, pad_potential):
        self.shape = tuple(int(s) for s in shape)
        self.lengths = tuple(float(l) for l in lengths)
        self.eps = float(eps)
        self.sigma = np.asarray(sigma, dtype=np.float64).reshape(self.shape)
        self.pad_nodes = np.asarray(pad_nodes, dtype=np.int64).reshape(-1, 3)
        self.pad_potential = np.asarray(pad_potential, dtype=np.float64).reshape(-1)
        nx, ny, nz = self.shape
        lx, ly, lz = self.lengths
        self.vol = (lx / nx) * (ly / ny) * (lz / nz)
        kx, rx = wavenumbers(nx, lx)
        ky, ry = wavenumbers(ny, ly)
        kz, rz = wavenumbers(nz, lz)
        # step 1: a mode with ANY component at the Nyquist index is removed from every field (R11)
        self.retained = rx[:, None, None] & ry[None, :, None] & rz[None, None, :]
        self.kappa = (kx[:, None, None] * self.retained, ky[None, :, None] * self.retained,
                      kz[None, None, :] * self.retained)
        k2 = kx[:, None, None] ** 2 + ky[None, :, None] ** 2 + kz[None, None, :] ** 2
        # step 3: G^(k) = 1/(eps |kappa|^2) on retained non-zero modes, 0 elsewhere
        self.green_hat = np.zeros(self.shape, dtype=np.float64)
        ok = self.retained & (k2 > 0)
        self.green_hat[ok] = 1.0 / (self.eps * k2[ok])
        # the tabulated fundamental solution (R9): potential of a unit point
        # charge at node 0 of the periodic lattice, G = IDFT(G^) / voxel volume
        self.green = np.real(np.fft.ifftn(self.green_hat)) / self.vol
        # step 4: bordered collocation system  [[G(x_b - x_b'), 1], [1^T, 0]]  (R10)
        nb = len(self.pad_nodes)
        self.nb = nb
        a = np.zeros((nb + 1, nb + 1), dtype=np.float64)
        for i in range(nb):
            d = (self.pad_nodes[i][None, :] - self.pad_nodes) % np.array(self.shape)
            a[i, :nb] = self.green[d[:, 0], d[:, 1], d[:, 2]]
        a[:nb, nb] = 1.0
        a[nb, :nb] = 1.0
        self.bordered = a
        self._lu = scipy.linalg.lu_factor(a) if nb > 0 else None

    # -- spectral operators (R14, R20) ---------------------------------------------------
    def grad_s(self, f):
        """Spectral gradient at the nodes: IDFT(i kappa_a DFT(f)), a = x, y, z."""
        fh = np.fft.fftn(f)
        return [np.real(np.fft.ifftn(1j * k * fh)) for k in self.kappa]

    def div_s(self, jx, jy, jz):
        """Spectral divergence: IDFT(sum_a i kappa_a DFT(J_a))."""
        acc = np.zeros(self.shape, dtype=np.complex128)
        for k, j in zip(self.kappa, (jx, jy, jz)):
            acc += 1j * k * np.fft.fftn(j)
        return np.real(np.fft.ifftn(acc))

    # -- step 5 ---------------------------------------------------------------------------
    def potential_of_charge(self, q):
        """V_rho = IDFT(G^ DFT(q)) / vol: "dividing the spectral representation by |k|^2"."""
        return np.real(np.fft.ifftn(self.green_hat * np.fft.fftn(q))) / self.vol

    def boundary_charges(self, v_rho, q_total, pad_potential):
        """Solve A [Q; c] = [V_pad - V_rho|_B ; -sum q]: the point charges "adjusted, in
        magnitude, to enforce the boundary conditions" (R10)."""
        if self.nb == 0:
            return np.zeros(0), 0.0
        b = self.pad_nodes
        rhs = np.concatenate([pad_potential - v_rho[b[:, 0], b[:, 1], b[:, 2]], [-q_total]])
        sol = scipy.linalg.lu_solve(self._lu, rhs)
        return sol[:-1], float(sol[-1])

    def v_ext(self, charges, c):
        """V_ext(x) = c + sum_b Q_b G(x - x_b): literal "rescaled and translated chunks of the
        fundamental solution"."""
        v = np.full(self.shape, c, dtype=np.float64)
        for qb, (i, j, k) in zip(charges, self.pad_nodes):
            v += qb * np.roll(self.green, shift=(int(i), int(j), int(k)), axis=(0, 1, 2))
        return v

    def potential(self, q, pad_potential=None):
        """Returns (V, Q, c) with V = V_rho + V_ext."""
        pp = self.pad_potential if pad_potential is None else np.asarray(pad_potential, dtype=np.float64)
        v_rho = self.potential_of_charge(q)
        charges, c = self.boundary_charges(v_rho, float(np.sum(q)), pp)
        return v_rho + self.v_ext(charges, c), charges, c

    # -- step 7, one forward-Euler substep -------------------------------------------------
    def euler_substep(self, q, dt_int, pad_potential=None):
        """V = potential(q); E = -grad_s V; J = sigma E (nodewise, R17); q <- q - dt_int vol div_s J."""
        v, charges, c = self.potential(q, pad_potential)
        gx, gy, gz = self.grad_s(v)
        jx, jy, jz = self.sigma * (-gx), self.sigma * (-gy), self.sigma * (-gz)
        return q - dt_int * self.vol * self.div_s(jx, jy, jz), charges

    # -- steps 6-8 -------------------------------------------------------------------------
    def solve_H(self, nt, dt, n_sub, on_substep=None, return_potentials=False, dtype=np.float64):
        """H[n] = -grad_s(W[n] - W[n-1]) / dt, W[-1] = 0 (R2), W = step response to V_pad Theta(t).

        Returns H[nx,ny,nz,nt,3] (the ABI layout of include/wtide.h) and optionally the list of W[n].
        """
        nx, ny, nz = self.shape
        H = np.zeros((nx, ny, nz, nt, 3), dtype=dtype)
        q = np.zeros(self.shape, dtype=np.float64)
        dt_int = dt / n_sub
        w_prev = np.zeros(self.shape, dtype=np.float64)
        ws = []
        for n in range(nt):
            if n > 0:
                for s in range(n_sub):
                    q, charges = self.euler_substep(q, dt_int)
                    if on_substep is not None:
                        on_substep(n, s, q, charges)
            w, _, _ = self.potential(q)
            g = self.grad_s(w - w_prev)
            for a in range(3):
                H[:, :, :, n, a] = -g[a] / dt
            w_prev = w
            if return_potentials:
                ws.append(w)
        return (H, ws) if return_potentials else H


def problem_from_desc(desc: dict) -> Problem:
    _, sigma, pad_nodes, pad_pot, _ = voxelize(desc)
    eps = desc["eps_r"] * EPS0
    return Problem((desc["nx"], desc["ny"], desc["nz"]), (desc["lx"], desc["ly"], desc["lz"]),
                   eps, sigma, pad_nodes, pad_pot)


def substeps_from_desc(desc: dict) -> int:
    if desc.get("substeps", 0) > 0:
        return int(desc["substeps"])
    _, sigma, _, _, _ = voxelize(desc)
    return auto_substeps(desc["dt"], float(sigma.max()), desc["eps_r"] * EPS0)


def solve_H_from_desc(desc: dict, nt=None, dtype=np.float64) -> np.ndarray:
    prob = problem_from_desc(desc)
    return prob.solve_H(desc["nt"] if nt is None else nt, desc["dt"], substeps_from_desc(desc), dtype=dtype)


# ----------------------------------------------------------------------------------------
# Eq. 1.1
# ----------------------------------------------------------------------------------------
def trajectory_nodes(shape, lengths, pos):
    """R24 -- the index arithmetic the ABI prescribes, in float32:
    inv = (float)((double)n / l); u = x * inv (one fp32 multiply); i0 = floor(u); f = u - i0.
    x, y wrap periodically; z clamps u to [0, nz-1] and i1 = min(i0 + 1, nz - 1).
    Returns (i0[S,3], i1[S,3], f[S,3] float32, finite[S]).
    """
    pos = np.asarray(pos, dtype=np.float32).reshape(-1, 3)
    i0 = np.zeros(pos.shape, dtype=np.int64)
    i1 = np.zeros(pos.shape, dtype=np.int64)
    f = np.zeros(pos.shape, dtype=np.float32)
    finite = np.isfinite(pos).all(axis=1)
    safe = np.where(finite[:, None], pos, np.float32(0.0)).astype(np.float32)
    for a in range(3):
        n = int(shape[a])
        inv = np.float32(np.float64(n) / np.float64(lengths[a]))
        u = (safe[:, a] * inv).astype(np.float32)
        if a == 2:
            u = np.minimum(np.maximum(u, np.float32(0.0)), np.float32(n - 1))
        fl = np.floor(u)
        f[:, a] = (u - fl).astype(np.float32)
        ifl = fl.astype(np.int64)
        if a < 2:
            i0[:, a] = np.mod(ifl, n)
            i1[:, a] = np.mod(ifl + 1, n)
        else:
            i0[:, a] = ifl
            i1[:, a] = np.minimum(ifl + 1, n - 1)
    return i0, i1, f, finite


def convolve_currents(H, shape, lengths, nt, dt, v_w, carrier_step_offsets, pos, vel, charge,
                      track_carrier_offsets=None):
    """Discrete Eq. 1.1 (R21-R23, R26):
        i_c[n] = -(q_c / V_w) sum_{m <= n, m < M_c} sum_a H~_a(x_c[m], n - m) v_{c,a}[m] dt
    H~ = trilinear blend of the 8 surrounding node rows ("linear interpolation along
    the carrier's trajectory"), indices/fractions by trajectory_nodes (fp32), everything else double.
    A step whose position or velocity is not finite contributes nothing; steps m >= nt are ignored.
    Returns i[n_carriers, nt], or i_track[n_tracks, nt] = sum of its carriers in carrier order.
    H is the table [nx,ny,nz,nt,3] or a callable H(ix, iy, iz) -> row [nt,3] (for tables that do not
    fit in host memory; only data access, no arithmetic).
    """
    nx, ny, nz = (int(s) for s in shape)
    if callable(H):
        rows_of = H
    else:
        Hv = np.asarray(H).reshape(nx, ny, nz, nt, 3)

        def rows_of(ix, iy, iz):
            return Hv[ix, iy, iz]
    off = np.asarray(carrier_step_offsets, dtype=np.int64)
    pos = np.asarray(pos, dtype=np.float32).reshape(-1, 3)
    vel = np.asarray(vel, dtype=np.float32).reshape(-1, 3)
    charge = np.asarray(charge, dtype=np.float32)
    n_car = len(off) - 1
    i0, i1, f, finite = trajectory_nodes(shape, lengths, pos)
    finite = finite & np.isfinite(vel).all(axis=1)
    fd = f.astype(np.float64)
    out = np.zeros((n_car, nt), dtype=np.float64)
    for c in range(n_car):
        qc = float(charge[c])
        for m, s in enumerate(range(off[c], off[c + 1])):
            if m >= nt:
                break
            if not finite[s]:
                continue
            row = np.zeros((nt - m, 3), dtype=np.float64)
            for cx in (0, 1):
                for cy in (0, 1):
                    for cz in (0, 1):
                        w = ((fd[s, 0] if cx else 1.0 - fd[s, 0]) * (fd[s, 1] if cy else 1.0 - fd[s, 1])
                             * (fd[s, 2] if cz else 1.0 - fd[s, 2]))
                        ix = i1[s, 0] if cx else i0[s, 0]
                        iy = i1[s, 1] if cy else i0[s, 1]
                        iz = i1[s, 2] if cz else i0[s, 2]
                        row += w * np.asarray(rows_of(int(ix), int(iy), int(iz)))[: nt - m, :].astype(np.float64)
            v = vel[s].astype(np.float64)
            out[c, m:] += -(qc / v_w) * (row @ v) * dt
    if track_carrier_offsets is None:
        return out
    toff = np.asarray(track_carrier_offsets, dtype=np.int64)
    tr = np.zeros((len(toff) - 1, nt), dtype=np.float64)
    for t in range(len(toff) - 1):
        for c in range(toff[t], toff[t + 1]):
            tr[t] += out[c]
    return tr


# ----------------------------------------------------------------------------------------
# electrostatic field ("An iterative pseudo-spectral method ... is used to solve the Laplace
# equation in the diamond sensor", :95 V <-> rho through the 3-D FFT and |k|^2, Fig. 2 :107)
# ----------------------------------------------------------------------------------------
def static_potential(desc, column_potentials):
    """The Laplace problem the iteration of Fig. 2 converges to, written out as its plain definition (R37 of DESIGN.md):
    every node of column j is held at column_potentials[j] (whole columns are ideal conductors), there is no charge
    anywhere else, the box is periodic and neutral:
        V(x) = c + sum_{s in S} q_s G(x - x_s),   V(x_s) = v_s for s in S,   sum_s q_s = 0,
    S = all column nodes (voxelize), G = the tabulated fundamental solution of the same spectral Laplacian (R9).
    Solved here by one dense least-squares solve; the library iterates (conjugate gradients on the same system).
    Returns (V[nx,ny,nz], E[nx,ny,nz,3] = -grad_s V, q[nx,ny,nz] in e)."""
    col_id, _, _, _, _ = voxelize(desc)
    prob = problem_from_desc(desc)
    shape = prob.shape
    nodes = np.argwhere(col_id >= 0)
    vals = np.asarray(column_potentials, dtype=np.float64)[col_id[col_id >= 0]]
    nb = len(nodes)
    a = np.zeros((nb + 1, nb + 1))
    for i in range(nb):
        dd = (nodes[i][None, :] - nodes) % np.array(shape)
        a[i, :nb] = prob.green[dd[:, 0], dd[:, 1], dd[:, 2]]
    scale = float(prob.green[0, 0, 0])          # border in the units of G (keeps the matrix well scaled); c = scale * last unknown
    a[:nb, nb] = scale
    a[nb, :nb] = scale
    # (charge patterns that lie in the removed Nyquist planes, or deep inside a conductor, barely change V: the system is
    #  consistent but can be singular -- a column that spans every z layer, say -- so the minimum-norm solution is taken;
    #  V and E are unique, q is not)
    sol = scipy.linalg.lstsq(a, np.concatenate([vals, [0.0]]), cond=1e-13)[0]
    q = np.zeros(shape)
    q[nodes[:, 0], nodes[:, 1], nodes[:, 2]] = sol[:-1]
    v = prob.potential_of_charge(q) + scale * sol[-1]
    g = prob.grad_s(v)
    e = np.stack([-g[0], -g[1], -g[2]], axis=-1)
    return v, e, q


# ----------------------------------------------------------------------------------------
# mirror (Neumann) surfaces at z = 0 and z = lz by the method of images
# ----------------------------------------------------------------------------------------
def mirror_z_desc(desc):
    """A field with dV/dz = 0 on the planes z = 0 and z = lz is the restriction to 0 <= z <= lz of a field that is even about
    both planes, hence periodic with period 2 lz: the mirror-surface problem IS the periodic problem (R7) on the doubled box
    lz' = 2 lz, nz' = 2 nz (same node spacing; nodes 0 and nz on the planes) holding every column and its image at
    z in [2 lz - z1, 2 lz - z0].  Columns j < n stay as given, images are columns n + j.  The image of a contact pad is a
    contact pad on the mirrored layer; a pad layer on a mirror plane (layer 0 or nz) is its own image, and the image column
    then carries none (WT_SEGMENT).  Returns the descriptor of the doubled box (mirror_z cleared)."""
    n = len(desc["columns"])
    lz2, nz2 = 2.0 * desc["lz"], 2 * desc["nz"]
    z = node_coordinates(nz2, lz2)
    cols = [dict(c) for c in desc["columns"]]
    for c in desc["columns"]:
        inside = np.nonzero((c["z0"] <= z) & (z <= c["z1"]))[0]
        kpad = int(inside[-1] if c["pad_at_z1"] else inside[0])
        im = dict(c, z0=lz2 - c["z1"], z1=lz2 - c["z0"], pad_at_z1=0 if c["pad_at_z1"] else 1)
        if c["role"] != WT_SEGMENT and kpad in (0, desc["nz"]):
            im["role"] = WT_SEGMENT
        cols.append(im)
    assert len(cols) == 2 * n
    d = dict(desc, lz=lz2, nz=nz2, columns=cols)
    d["mirror_z"] = 0
    return d


# ----------------------------------------------------------------------------------------
# carrier transport in the solved field ("computing the paths of the carriers",
# :101 "dominates the time-to-insight"; BASELINE.json configs[1]: saturated-drift model
# v = mu E / (1 + mu E / v_sat), mu_e = 1800, mu_h = 1500 cm^2/Vs, v_sat = 1.5e7 cm/s, up to nt steps)
# ----------------------------------------------------------------------------------------
def static_field(H, dt):
    """Es[node] = sum_n H[node][n] dt = -grad_s W[nt-1] (R2 telescoped): the static weighting field of the table,
    per volt of V_w.  H: [nx,ny,nz,nt,3]; returns float64 [nx,ny,nz,3] (the library sums in fp32 pairs: compared
    within fp32 rounding)."""
    return np.asarray(H, dtype=np.float64).sum(axis=3) * float(dt)


def drift_trajectories(es, desc, start, sign, v_bias, mu_e, mu_h, v_sat, max_steps):
    """Explicit Euler transport on H's time grid, ALL arithmetic in float32 in the order written here (the library does
    the same operations without FMA contraction, so that step counts -- decided by float comparisons -- and positions are
    bit-exact; R35 of DESIGN.md):
        E   = v_bias * trilinear(Es, x)            indices / fractions by trajectory_nodes (R24); weights w = (wx*wy)*wz;
                                                   sum over the corners k = 4 cx + 2 cy + cz in that order, e += w * Es
        |E| = sqrt((Ex*Ex + Ey*Ey) + Ez*Ez)
        v   = ((sign * mu) * E) / (1 + (mu * |E|) / v_sat)          mu = mu_e for sign < 0 (electron), mu_h for sign > 0
        x'  = x + v * dt ;   recorded pos[m] = x, vel[m] = (x' - x) / dt    (R22: velocity as inferred by the trajectory)
    A carrier is alive at x iff 0 <= z <= lz and, for every column, the minimum-image lateral distance^2 to the axis
    (fmod(|x - cx|, lx), min(d, lx - d), dx*dx + dy*dy) is > r*r; it records a step only while alive, at most max_steps.
    es: [nx,ny,nz,3] (cast to float32); start [C,3]; sign [C] (-1 / +1).
    Returns (carrier_step_offsets int64 [C+1], pos float32 [S,3], vel float32 [S,3])."""
    f32 = np.float32
    nx, ny, nz = desc["nx"], desc["ny"], desc["nz"]
    shape, lengths = (nx, ny, nz), (desc["lx"], desc["ly"], desc["lz"])
    E = np.asarray(es, dtype=f32).reshape(nx, ny, nz, 3)
    lx, ly, lz, dt = f32(desc["lx"]), f32(desc["ly"]), f32(desc["lz"]), f32(desc["dt"])
    cols = [(f32(c["cx"]), f32(c["cy"]), f32(f32(c["radius"]) * f32(c["radius"]))) for c in desc["columns"]]
    vb, vs = f32(v_bias), f32(v_sat)
    start = np.asarray(start, dtype=f32).reshape(-1, 3)
    offs, pos, vel = [0], [], []

    def alive(x):
        if not (x[2] >= f32(0.0) and x[2] <= lz):
            return False
        for (cx, cy, r2) in cols:
            dx = np.fmod(np.abs(f32(x[0] - cx)), lx)
            dx = min(dx, f32(lx - dx))
            dy = np.fmod(np.abs(f32(x[1] - cy)), ly)
            dy = min(dy, f32(ly - dy))
            if not (f32(f32(dx * dx) + f32(dy * dy)) > r2):
                return False
        return True

    for c in range(len(start)):
        x = start[c].copy()
        mu = f32(mu_e) if sign[c] < 0 else f32(mu_h)
        smu = f32(f32(sign[c]) * mu)
        m = 0
        while m < max_steps and np.isfinite(x).all() and alive(x):
            i0, i1, f, _ = trajectory_nodes(shape, lengths, x[None, :])
            e = np.zeros(3, dtype=f32)
            for cx_ in (0, 1):
                wx = f[0, 0] if cx_ else f32(f32(1.0) - f[0, 0])
                for cy_ in (0, 1):
                    wy = f[0, 1] if cy_ else f32(f32(1.0) - f[0, 1])
                    for cz_ in (0, 1):
                        wz = f[0, 2] if cz_ else f32(f32(1.0) - f[0, 2])
                        w = f32(f32(wx * wy) * wz)
                        node = E[(i1 if cx_ else i0)[0, 0], (i1 if cy_ else i0)[0, 1], (i1 if cz_ else i0)[0, 2]]
                        e = (e + (w * node).astype(f32)).astype(f32)
            e = (vb * e).astype(f32)
            en = np.sqrt(f32(f32(f32(e[0] * e[0]) + f32(e[1] * e[1])) + f32(e[2] * e[2])))
            den = f32(f32(1.0) + f32(f32(mu * en) / vs))
            v = ((smu * e).astype(f32) / den).astype(f32)
            xn = (x + (v * dt).astype(f32)).astype(f32)
            pos.append(x.copy())
            vel.append(((xn - x).astype(f32) / dt).astype(f32))
            x = xn
            m += 1
        offs.append(offs[-1] + m)
    return (np.asarray(offs, dtype=np.int64), np.asarray(pos, dtype=f32).reshape(-1, 3), np.asarray(vel, dtype=f32).reshape(-1, 3))


# ----------------------------------------------------------------------------------------
# electronics stage ("the induced signal is convolved with the transfer function of the
# front-end electronics, and noise is added"): causal FIR on H's time grid + additive noise + constant-fraction time
# ----------------------------------------------------------------------------------------
def electronics(currents, transfer, dt, noise=None, cfd_fraction=0.3):
    """out[t][n] = dt * sum_{j <= n, j < len(transfer)} transfer[j] * currents[t][n - j]  (+ noise[t][n]);
    t_cfd[t] = time of the first crossing of cfd_fraction * (extremum of out[t], by absolute value) on the way to that
    extremum, linearly interpolated between samples (n - 1, n), in units of dt; -1 if the row is identically zero.
    Returns (out float64 [T,nt], t_cfd float64 [T])."""
    cur = np.asarray(currents, dtype=np.float64)
    h = np.asarray(transfer, dtype=np.float64)
    T, nt = cur.shape
    out = np.zeros((T, nt))
    for t in range(T):
        for n in range(nt):
            acc = 0.0
            for j in range(min(len(h), n + 1)):
                acc += h[j] * cur[t, n - j]
            out[t, n] = acc * float(dt)
    if noise is not None:
        out = out + np.asarray(noise, dtype=np.float64)
    t_cfd = np.full(T, -1.0)
    for t in range(T):
        k = int(np.argmax(np.abs(out[t])))
        peak = out[t, k]
        if peak == 0.0:
            continue
        thr = cfd_fraction * peak
        s = 1.0 if peak > 0 else -1.0
        for n in range(k + 1):
            if s * out[t, n] >= s * thr:
                if n == 0:
                    t_cfd[t] = 0.0
                else:
                    a, b = s * out[t, n - 1], s * out[t, n]
                    t_cfd[t] = (n - 1) + (s * thr - a) / (b - a)
                break
    return out, t_cfd


# error metrics (R27) ---------------------------------------------------------------------
def h_rel_l2(h_test, h_ref) -> float:
    a = np.asarray(h_test, dtype=np.float64).ravel()
    b = np.asarray(h_ref, dtype=np.float64).ravel()
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def current_error(i_test, i_ref):
    """Per output row: ||di||_2 / (sqrt(nt) max_n |i_ref[n]|); returns (worst row value, max|di|/peak)."""
    a = np.asarray(i_test, dtype=np.float64)
    b = np.asarray(i_ref, dtype=np.float64)
    peak = np.max(np.abs(b), axis=1)
    peak = np.where(peak > 0, peak, 1.0)
    l2 = np.linalg.norm(a - b, axis=1) / (math.sqrt(b.shape[1]) * peak)
    mx = np.max(np.abs(a - b), axis=1) / peak
    return float(l2.max()), float(mx.max())
