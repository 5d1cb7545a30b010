"""Geometry descriptors of the five BASELINE.json configs (synthetic stand-ins).

A descriptor is a plain dict mirroring `wt_geometry_desc` of include/wtide.h:
  lx, ly, lz [um], nx, ny, nz, nt, dt [ns], eps_r, v_w [V], substeps (0 = auto),
  columns = [dict(cx, cy, radius, resistivity [ohm cm], z0, z1, role, pad_at_z1)].

Readings used: R7 column depths (readout z in [0, 0.9 lz], pad at its first
layer; bias z in [0.1 lz, lz], pad at its last layer), R18 hexagonal stand-in, R19 one
(radius, resistivity) draw per column role, R29 swept radius = bias column's, R30.
"""
import math

from .rng import uniform

CONFIG_NAMES = ("cfg0_tiny", "cfg1_pixel", "cfg2_hex", "cfg3_sweep", "cfg4_highstat")
WT_BIAS, WT_READOUT = 0, 1
EPS_R_DIAMOND = 5.7


def _readout(cx, cy, radius, resistivity, lz):
    return dict(cx=cx, cy=cy, radius=radius, resistivity=resistivity, z0=0.0, z1=0.9 * lz,
                role=WT_READOUT, pad_at_z1=0)


def _bias(cx, cy, radius, resistivity, lz):
    return dict(cx=cx, cy=cy, radius=radius, resistivity=resistivity, z0=0.1 * lz, z1=lz,
                role=WT_BIAS, pad_at_z1=1)


def square_cell(pitch, lz, grid, nt, dt, r_read, rho_read, r_bias, rho_bias):
    """One square 3D pixel: central readout column + the 4 corner bias columns, which on the
    periodic lattice are one column at (0, 0) wrapped four ways (R13)."""
    nx, ny, nz = grid
    return dict(lx=pitch, ly=pitch, lz=lz, nx=nx, ny=ny, nz=nz, nt=nt, dt=dt,
                eps_r=EPS_R_DIAMOND, v_w=1.0, substeps=0,
                columns=[_readout(pitch / 2, pitch / 2, r_read, rho_read, lz),
                         _bias(0.0, 0.0, r_bias, rho_bias, lz)])


def hex_cell(grid, nt, dt):
    """R18: centre readout + 6 bias columns at 50 um, 60 deg apart, in a 128 um periodic box."""
    nx, ny, nz = grid
    lz, box = 500.0, 128.0
    cols = [_readout(box / 2, box / 2, 5.0, 0.5, lz)]
    for k in range(6):
        a = math.radians(60.0 * k)
        cols.append(_bias(box / 2 + 50.0 * math.cos(a), box / 2 + 50.0 * math.sin(a), 5.0, 0.5, lz))
    return dict(lx=box, ly=box, lz=lz, nx=nx, ny=ny, nz=nz, nt=nt, dt=dt,
                eps_r=EPS_R_DIAMOND, v_w=1.0, substeps=0, columns=cols)


def _cfg1_draws(seed):
    """R19: radius U[3,8] um and resistivity U[0.1,1] ohm cm, one pair per column role."""
    u = [float(uniform(seed, 1, 0, 0, d)) for d in range(4)]
    return (3.0 + 5.0 * u[0], 0.1 + 0.9 * u[1], 3.0 + 5.0 * u[2], 0.1 + 0.9 * u[3])


def sweep_descs(grid=(64, 64, 256), nt=512, dt=0.005):
    """cfg 3: 32 square cells, pitch {25,55,80,100} x bias radius {2,5,8,10} x resistivity {0.1,1}."""
    out = []
    for pitch in (25.0, 55.0, 80.0, 100.0):
        for r_bias in (2.0, 5.0, 8.0, 10.0):
            for rho in (0.1, 1.0):
                out.append(square_cell(pitch, 500.0, grid, nt, dt, 5.0, rho, r_bias, rho))
    return out


def geometry_desc(config: int, seed: int = 0):
    """Descriptor of config 0, 1, 2, 4 (config 3 is a list: use sweep_descs())."""
    if config == 0:
        return square_cell(55.0, 50.0, (32, 32, 32), 128, 0.010, 5.0, 0.5, 5.0, 0.5)
    if config == 1:
        rr, rhor, rb, rhob = _cfg1_draws(seed)
        return square_cell(55.0, 500.0, (64, 64, 256), 512, 0.005, rr, rhor, rb, rhob)
    if config == 2:
        return hex_cell((128, 128, 256), 1024, 0.0025)
    if config == 4:
        rr, rhor, rb, rhob = _cfg1_draws(seed)
        return square_cell(55.0, 500.0, (96, 96, 384), 1024, 0.0025, rr, rhor, rb, rhob)
    raise ValueError("config must be 0, 1, 2 or 4 (3 is sweep_descs())")


def reduced_desc(desc, grid=None, nt=None, substeps=None):
    """Same geometry on a coarser grid / shorter time axis (parity-test sizes)."""
    d = dict(desc)
    d["columns"] = [dict(c) for c in desc["columns"]]
    if grid is not None:
        d["nx"], d["ny"], d["nz"] = grid
    if nt is not None:
        d["nt"] = nt
    if substeps is not None:
        d["substeps"] = substeps
    return d
