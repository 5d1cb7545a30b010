"""Seeded MIP tracks, macro-carriers and drift trajectories (input recipe of DESIGN.md).

They stand in for the paper's workload (1000 pions of 180 GeV/c along z, HEED deposits,
Garfield++ drift lines -- PAPER.md:59, :73), none of which is available.  Nothing here is part
of the method: the trajectories are INPUTS of Eq. 1.1 and the same arrays are handed to the
oracle and to the library.

Trajectory container ("CSR"): dict with
  track_carrier_offsets int64 [T+1], carrier_step_offsets int64 [C+1],
  pos float32 [S,3] um, vel float32 [S,3] um/ns, charge float32 [C] e.
"""
import math

import numpy as np

from .rng import uniform

MU_E = 180.0     # 1800 cm^2/Vs in um^2/(V ns)
MU_H = 150.0     # 1500 cm^2/Vs
V_SAT = 150.0    # 1.5e7 cm/s in um/ns
PAIRS_PER_UM = 36.0


def _lateral_dist2(x, y, col, lx, ly):
    dx = np.fmod(np.abs(x - col["cx"]), lx)
    dx = np.minimum(dx, lx - dx)
    dy = np.fmod(np.abs(y - col["cy"]), ly)
    dy = np.minimum(dy, ly - dy)
    return dx * dx + dy * dy


def make_tracks(config, n_tracks, desc, theta_max_deg, seed=0):
    """Entry point uniform in the cell on the z = 0 face (redrawn while inside a column),
    polar angle U[0, theta_max], azimuth U[0, 2 pi).  Returns float64 [T,4] = (x0, y0, theta, phi)."""
    t = np.arange(n_tracks)
    out = np.zeros((n_tracks, 4))
    x0 = np.zeros(n_tracks)
    y0 = np.zeros(n_tracks)
    todo = np.ones(n_tracks, dtype=bool)
    attempt = 0
    while todo.any():
        xs = uniform(seed, config, t, attempt, 0) * desc["lx"]
        ys = uniform(seed, config, t, attempt, 1) * desc["ly"]
        x0 = np.where(todo, xs, x0)
        y0 = np.where(todo, ys, y0)
        inside = np.zeros(n_tracks, dtype=bool)
        for col in desc["columns"]:
            inside |= _lateral_dist2(x0, y0, col, desc["lx"], desc["ly"]) <= col["radius"] ** 2
        todo = inside
        attempt += 1
    out[:, 0], out[:, 1] = x0, y0
    out[:, 2] = uniform(seed, config, t, 0, 2) * math.radians(theta_max_deg)
    out[:, 3] = uniform(seed, config, t, 0, 3) * 2.0 * math.pi
    return out


def carriers_on_tracks(tracks, n_per_track, desc, unit_charge=False):
    """n/2 electrons then n/2 holes per track at z = (j + 1/2) lz / (n/2) along the track
    (uniform deposit), charge -/+ 36 pairs/um * lz / (n/2) e (or -/+ 1 with unit_charge).
    Returns start float32 [C,3], sign int8 [C] (-1 electron, +1 hole), charge float32 [C],
    track_carrier_offsets int64 [T+1]."""
    T = len(tracks)
    h = n_per_track // 2
    z = (np.arange(h) + 0.5) * desc["lz"] / h
    tan = np.tan(tracks[:, 2])[:, None]
    x = tracks[:, 0][:, None] + z[None, :] * tan * np.cos(tracks[:, 3])[:, None]
    y = tracks[:, 1][:, None] + z[None, :] * tan * np.sin(tracks[:, 3])[:, None]
    one = np.stack([x, y, np.broadcast_to(z, x.shape)], axis=-1)          # [T,h,3]
    start = np.concatenate([one, one], axis=1).reshape(T * 2 * h, 3).astype(np.float32)
    sign = np.tile(np.concatenate([-np.ones(h, np.int8), np.ones(h, np.int8)]), T)
    w = 1.0 if unit_charge else PAIRS_PER_UM * desc["lz"] / h
    charge = (sign.astype(np.float32) * np.float32(w)).astype(np.float32)
    offsets = (np.arange(T + 1, dtype=np.int64) * (2 * h))
    return start, sign, charge, offsets


def straight_drift_cfg0(desc, start, sign, charge, track_carrier_offsets, max_steps=128, speed=100.0):
    """R28: holes go to the nearest readout column, electrons to the nearest bias column, on a
    straight line in the xy-plane at 100 um/ns (1 um per 10 ps step), stopping at the column
    surface; at most max_steps steps."""
    lx, ly, dt = desc["lx"], desc["ly"], desc["dt"]
    offs = [0]
    pos, vel = [], []
    for c in range(len(start)):
        want = 1 if sign[c] > 0 else 0
        best = None
        for col in desc["columns"]:
            if col["role"] != want:
                continue
            # nearest periodic image of the axis
            ddx = (col["cx"] - float(start[c, 0]) + lx / 2) % lx - lx / 2
            ddy = (col["cy"] - float(start[c, 1]) + ly / 2) % ly - ly / 2
            d = math.hypot(ddx, ddy)
            if best is None or d < best[0]:
                best = (d, ddx, ddy, col["radius"])
        d, ddx, ddy, rad = best
        ux, uy = (ddx / d, ddy / d) if d > 0 else (1.0, 0.0)
        step = speed * dt
        m = 0
        while m < max_steps and d - m * step > rad:
            pos.append((start[c, 0] + m * step * ux, start[c, 1] + m * step * uy, start[c, 2]))
            vel.append((speed * ux, speed * uy, 0.0))
            m += 1
        offs.append(offs[-1] + m)
    return dict(track_carrier_offsets=np.asarray(track_carrier_offsets, dtype=np.int64),
                carrier_step_offsets=np.asarray(offs, dtype=np.int64),
                pos=np.asarray(pos, dtype=np.float32).reshape(-1, 3),
                vel=np.asarray(vel, dtype=np.float32).reshape(-1, 3),
                charge=np.asarray(charge, dtype=np.float32))


def bias_voltage(desc):
    """R30: V_bias = 2 V/um x (smallest readout-to-bias axis distance, minimum image)."""
    best = None
    for a in desc["columns"]:
        if a["role"] != 1:
            continue
        for b in desc["columns"]:
            if b["role"] != 0:
                continue
            d = math.sqrt(float(_lateral_dist2(np.float64(a["cx"]), np.float64(a["cy"]), b, desc["lx"], desc["ly"])))
            best = d if best is None else min(best, d)
    return 2.0 * best


def field_drift(e_static, desc, start, sign, charge, track_carrier_offsets, v_bias=None, nt=None,
                batch_carriers=200_000):
    """Saturated-drift model v = +/- mu E / (1 + mu |E| / v_sat) (BASELINE.json config 1),
    E = V_bias x trilinear sample of the static weighting field `e_static`
    (torch tensor [nx,ny,nz,3], 1/um per volt of V_w; the harness passes sum_n H[n] dt of the
    table under test).  Explicit Euler with the H time step; a carrier stops inside any column
    radius, outside the z faces, or after nt steps.  Recorded: pos[m], vel[m] = (x[m+1]-x[m])/dt (R22).
    Runs on e_static's device; returns the CSR dict with torch tensors on that device."""
    import torch

    dev = e_static.device
    nx, ny, nz = desc["nx"], desc["ny"], desc["nz"]
    lx, ly, lz = desc["lx"], desc["ly"], desc["lz"]
    nt = desc["nt"] if nt is None else nt
    dt = float(desc["dt"])
    vb = bias_voltage(desc) if v_bias is None else v_bias
    E = e_static.to(torch.float32).reshape(nx * ny * nz, 3)
    cols = [(c["cx"], c["cy"], c["radius"]) for c in desc["columns"]]
    start_t = torch.as_tensor(np.asarray(start), dtype=torch.float32, device=dev)
    sign_t = torch.as_tensor(np.asarray(sign), dtype=torch.float32, device=dev)
    counts_all, pos_all, vel_all = [], [], []

    def sample(p):
        u = torch.stack([p[:, 0] * (nx / lx), p[:, 1] * (ny / ly),
                         torch.clamp(p[:, 2] * (nz / lz), 0.0, nz - 1.0)], dim=1)
        fl = torch.floor(u)
        f = u - fl
        i = fl.to(torch.int64)
        out = torch.zeros((p.shape[0], 3), dtype=torch.float32, device=dev)
        for cx in (0, 1):
            ix = torch.remainder(i[:, 0] + cx, nx)
            wx = f[:, 0] if cx else 1.0 - f[:, 0]
            for cy in (0, 1):
                iy = torch.remainder(i[:, 1] + cy, ny)
                wy = f[:, 1] if cy else 1.0 - f[:, 1]
                for cz in (0, 1):
                    iz = torch.clamp(i[:, 2] + cz, max=nz - 1)
                    wz = f[:, 2] if cz else 1.0 - f[:, 2]
                    out += (wx * wy * wz)[:, None] * E[(ix * ny + iy) * nz + iz]
        return out

    def alive(p):
        ok = (p[:, 2] >= 0.0) & (p[:, 2] <= lz)
        for (cx, cy, r) in cols:
            dx = torch.remainder(torch.abs(p[:, 0] - cx), lx)
            dx = torch.minimum(dx, lx - dx)
            dy = torch.remainder(torch.abs(p[:, 1] - cy), ly)
            dy = torch.minimum(dy, ly - dy)
            ok &= (dx * dx + dy * dy) > r * r
        return ok

    for b0 in range(0, len(start_t), batch_carriers):
        p = start_t[b0:b0 + batch_carriers].clone()
        sg = sign_t[b0:b0 + batch_carriers]
        mu = torch.where(sg > 0, torch.tensor(MU_H, device=dev), torch.tensor(MU_E, device=dev))
        act = alive(p)
        count = torch.zeros(p.shape[0], dtype=torch.int64, device=dev)
        rec_pos, rec_vel, rec_idx = [], [], []
        idx = torch.arange(p.shape[0], device=dev)
        for m in range(nt):
            if not bool(act.any()):
                break
            ia = idx[act]
            pa = p[ia]
            e = sample(pa) * vb
            en = torch.linalg.norm(e, dim=1, keepdim=True)
            v = sg[ia][:, None] * mu[ia][:, None] * e / (1.0 + mu[ia][:, None] * en / V_SAT)
            pn = pa + v * dt
            rec_pos.append(pa)
            rec_vel.append((pn - pa) / dt)
            rec_idx.append(ia)
            count[ia] += 1
            p[ia] = pn
            act = torch.zeros_like(act)
            act[ia] = alive(pn)
        if rec_idx:
            cid = torch.cat(rec_idx)
            order = torch.argsort(cid, stable=True)      # carrier-major, step order kept
            pos_all.append(torch.cat(rec_pos)[order])
            vel_all.append(torch.cat(rec_vel)[order])
        counts_all.append(count)
    counts = torch.cat(counts_all) if counts_all else torch.zeros(0, dtype=torch.int64, device=dev)
    offs = torch.zeros(len(counts) + 1, dtype=torch.int64, device=dev)
    offs[1:] = torch.cumsum(counts, 0)
    z3 = torch.zeros((0, 3), dtype=torch.float32, device=dev)
    return dict(track_carrier_offsets=torch.as_tensor(np.asarray(track_carrier_offsets), dtype=torch.int64, device=dev),
                carrier_step_offsets=offs,
                pos=torch.cat(pos_all) if pos_all else z3,
                vel=torch.cat(vel_all) if vel_all else z3,
                charge=torch.as_tensor(np.asarray(charge), dtype=torch.float32, device=dev))


def concat_csr(parts):
    """Concatenate CSR dicts (numpy) of consecutive track batches."""
    toff, coff = [0], [0]
    for p in parts:
        base_c = len(coff) - 1
        toff.extend((np.asarray(p["track_carrier_offsets"])[1:] + base_c).tolist())
        coff.extend((np.asarray(p["carrier_step_offsets"])[1:] + coff[-1]).tolist())
    return dict(track_carrier_offsets=np.asarray(toff, dtype=np.int64),
                carrier_step_offsets=np.asarray(coff, dtype=np.int64),
                pos=np.concatenate([np.asarray(p["pos"]) for p in parts]),
                vel=np.concatenate([np.asarray(p["vel"]) for p in parts]),
                charge=np.concatenate([np.asarray(p["charge"]) for p in parts]))
