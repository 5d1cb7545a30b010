#!/usr/bin/env python
"""bench.py -- throughput of libwtide's hot path on BASELINE.json configs[1].

    python bench.py --gpus 1 --steps 3 --warmup 3          # our arm
    python bench.py --impl reference --steps 1 --warmup 0   # the oracle on the host cores

    python bench.py --config 3 --steps 1 --warmup 1         # the 32-geometry what-if sweep (extra row of BASELINE.md)
    python bench.py --impl cufft                            # cuFFT-composed Euler substep (cross-check baseline only)

A "step" is one pass of the whole hot path over one batch of synthetic input: wt_make_geometry (a0, host) and
wt_solve_H (a1-a8) for the config-1 geometry followed by wt_convolve_currents over all tracks (a9-a12).
  metric / value : carrier-steps x output-samples per second of the Eq. 1.1 stage (inputs resident in HBM)
  setup_s_per_geometry, h_solve_s_per_geometry, h_total_s_per_geometry, stages : the H-solve part of the metric string
                   (host setup a0 timed inside the timed region, once per step; total = setup + solve)
  e2e            : the same Eq. 1.1 throughput with HOST (pinned) trajectory buffers and a host result, and the wall
                   clock of descriptor -> wt_make_geometry -> wt_solve_H -> synchronised table (h_solve_e2e_s)
  roofline       : dominant stage of the step against the measured HBM peak
  cpu_baseline   : the oracle, as it stands, on a bounded sample of the same workload (one core, and all cores for Eq. 1.1)
Prints ONE JSON line (rank 0).
"""
import hashlib
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "carrier_steps_x_output_samples_per_s"
UNIT = "terms/s"


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        j = json.load(open(p))
        return float(j["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def kernel_source_hash():
    """sha256 over the CUDA sources: profiles/r2_traffic.json holds ncu DRAM traffic for exactly one such hash"""
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2605_13987_b200", "csrc")
    for f in sorted(os.listdir(d)):
        if f.endswith((".cu", ".cuh", ".cpp", ".h")):
            h.update(open(os.path.join(d, f), "rb").read())
    return h.hexdigest()[:16]


def measured_traffic():
    """DRAM bytes from the committed ncu --set full captures (profiles/r2_traffic.json: written by hand from the ncu
    raw page of the command named there).  Values are only valid for the kernel sources they were captured with."""
    p = os.path.join(ROOT, "profiles", "r2_traffic.json")
    if not os.path.exists(p):
        return {}
    j = json.load(open(p))
    return j if j.get("kernel_source_hash") == kernel_source_hash() else {"stale": True, "source": j.get("source")}


def workload(args):
    from wtide_inputs import geometry_desc, reduced_desc
    d = geometry_desc(args.config, seed=0)
    if args.grid:
        nx, ny, nz = (int(v) for v in args.grid.split("x"))
        d = reduced_desc(d, grid=(nx, ny, nz))
    if args.nt:
        d = reduced_desc(d, nt=args.nt)
    return d


class ClockSampler:
    """nvidia-smi clocks and throttle reasons during the timed region (B200_PROFILING.md)."""

    def __init__(self, index):
        self.index = index
        self.samples = []
        self.reasons = set()
        self.max_mhz = None
        self._stop = threading.Event()
        self._th = threading.Thread(target=self._run, daemon=True)

    def _run(self):
        q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        while not self._stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--id={self.index}", f"--query-gpu={q}", "--format=csv,noheader,nounits"],
                                     capture_output=True, text=True, timeout=5).stdout.strip().split(",")
                self.samples.append(float(out[0]))
                self.max_mhz = float(out[1])
                for n, v in zip(names, out[2:]):
                    if v.strip().lower().startswith("active"):
                        self.reasons.add(n)
            except Exception:  # noqa: BLE001
                pass
            self._stop.wait(0.2)

    def __enter__(self):
        self._th.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        self._th.join(timeout=5)

    def summary(self):
        return {"sm_mhz": float(np.median(self.samples)) if self.samples else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


def count_terms(offsets, nt):
    """terms = sum_c sum_{m < min(M_c, nt)} (nt - m)"""
    m = np.minimum(np.diff(np.asarray(offsets, dtype=np.int64)), nt)
    return int(np.sum(m * nt - m * (m - 1) // 2))


# --------------------------------------------------------------------------------------------------
# oracle legs (CPU): the only places bench.py executes oracle/
# --------------------------------------------------------------------------------------------------
def oracle_conv_sample(d, rows_of, csr, budget_s):
    """Times oracle.convolve_currents carrier chunk by carrier chunk until budget_s is used."""
    from oracle import wtide_oracle as wo
    off = np.asarray(csr["carrier_step_offsets"])
    n_car = len(off) - 1
    done, terms, t_used, chunk = 0, 0, 0.0, 8
    while done < n_car and t_used < budget_s:
        c1 = min(n_car, done + chunk)
        sub = off[done:c1 + 1] - off[done]
        sl = slice(off[done], off[c1])
        t0 = time.perf_counter()
        wo.convolve_currents(rows_of, (d["nx"], d["ny"], d["nz"]), (d["lx"], d["ly"], d["lz"]), d["nt"], d["dt"], d["v_w"],
                             sub, csr["pos"][sl], csr["vel"][sl], csr["charge"][done:c1])
        t_used += time.perf_counter() - t0
        terms += count_terms(sub, d["nt"])
        done = c1
    return terms, t_used, done


_POOL_TABLE = {}


def _conv_pool_init(table):
    from oracle import wtide_oracle as wo  # noqa: F401  (imported once per worker, outside the timed region)
    _POOL_TABLE["t"] = table


def _conv_chunk(job):
    """(worker process) the oracle's Eq. 1.1 on one chunk of carriers; the table rows were handed over at pool start"""
    from oracle import wtide_oracle as wo
    d, sub, pos, vel, charge = job
    table = _POOL_TABLE["t"]
    t0 = time.perf_counter()
    wo.convolve_currents(lambda ix, iy, iz: table[(ix, iy, iz)], (d["nx"], d["ny"], d["nz"]), (d["lx"], d["ly"], d["lz"]), d["nt"], d["dt"],
                         d["v_w"], sub, pos, vel, charge)
    return time.perf_counter() - t0


def oracle_conv_all_cores(d, table, csr, n_car):
    """The same oracle function over a process pool, carriers split into one chunk per core (tracks and carriers are
    independent units).  Returns (terms, wall seconds, processes)."""
    import concurrent.futures as cf
    import multiprocessing as mp
    cores = os.cpu_count() or 1
    off = np.asarray(csr["carrier_step_offsets"])
    cuts = [n_car * k // cores for k in range(cores + 1)]
    jobs = []
    for k in range(cores):
        c0, c1 = cuts[k], cuts[k + 1]
        if c1 == c0:
            continue
        sl = slice(off[c0], off[c1])
        jobs.append((d, off[c0:c1 + 1] - off[c0], csr["pos"][sl], csr["vel"][sl], csr["charge"][c0:c1]))
    with cf.ProcessPoolExecutor(max_workers=cores, mp_context=mp.get_context("spawn"), initializer=_conv_pool_init, initargs=(table,)) as ex:
        list(ex.map(_conv_chunk, [(d, np.zeros(2, np.int64), np.zeros((0, 3), np.float32), np.zeros((0, 3), np.float32), np.zeros(1, np.float32))] * (2 * cores)))   # workers up
        t0 = time.perf_counter()
        list(ex.map(_conv_chunk, jobs))
        wall = time.perf_counter() - t0
    return count_terms(off[:n_car + 1], d["nt"]), wall, len(jobs)


def oracle_solve_sample(d, budget_s):
    """Times forward-Euler substeps of the oracle on the workload's grid; returns s per substep."""
    from oracle import wtide_oracle as wo
    t0 = time.perf_counter()
    prob = wo.problem_from_desc(d)
    n_sub = wo.substeps_from_desc(d)
    setup = time.perf_counter() - t0
    q = np.zeros(prob.shape)
    n, t_used = 0, 0.0
    while t_used < budget_s or n < 2:
        t0 = time.perf_counter()
        q, _ = prob.euler_substep(q, d["dt"] / n_sub)
        t_used += time.perf_counter() - t0
        n += 1
    return t_used / n, n, n_sub, setup


def synthetic_host_tracks(d, n_tracks, carriers_per_track, track0=0):
    """Trajectories for the reference arm without a GPU table: straight saturated drift towards the
    collecting column (same length statistics as the field drift)."""
    from wtide_inputs import carriers_on_tracks, make_tracks, straight_drift_cfg0
    tracks = make_tracks(1, n_tracks + track0, d, 10.0)[track0:]
    start, sign, charge, toff = carriers_on_tracks(tracks, carriers_per_track, d)
    return straight_drift_cfg0(d, start, sign, charge, toff, max_steps=d["nt"], speed=100.0)


def run_reference(args):
    """--impl reference: the oracle as it stands on the host cores, bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    d = workload(args)
    csr = synthetic_host_tracks(d, 1, 64)
    rng = np.random.default_rng(0)
    cache = {}

    def rows_of(ix, iy, iz):      # a synthetic table row (the oracle's arithmetic does not depend on values)
        key = (ix, iy, iz)
        if key not in cache:
            cache[key] = rng.standard_normal((d["nt"], 3)).astype(np.float32)
        return cache[key]
    budget = args.ref_budget
    for _ in range(args.warmup):
        oracle_conv_sample(d, rows_of, csr, min(1.0, budget))
    terms = t = 0.0
    ts = 0.0
    per_sub = n_sub = None
    for _ in range(max(1, args.steps)):
        a, b, ncar = oracle_conv_sample(d, rows_of, csr, budget)
        terms += a
        t += b
        per_sub, nsubs_timed, n_sub, _ = oracle_solve_sample(d, budget)
        ts += per_sub * nsubs_timed
    steps = max(1, args.steps)
    value = terms / t
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * (t + ts) / steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "configs[1] single pixel cell 64x64x256 nt=512 (bounded sample)", "grid": [d["nx"], d["ny"], d["nz"]],
                       "nt": d["nt"]},
            "h_solve_s_per_geometry": per_sub * n_sub * (d["nt"] - 1), "h_solve_extrapolated": True,
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle",
                             "sample": f"{ncar} carriers of one track per step (Eq. 1.1) + {budget:.0f} s of Euler substeps"},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# --------------------------------------------------------------------------------------------------
# multi-GPU: replicas only.  Tracks are the independent units: rank r
# takes tracks [r * n, (r + 1) * n) of the seeded track list; the only collectives are the timing ones.
# --------------------------------------------------------------------------------------------------
def shard_tracks(tracks_per_rank, world, rank):
    assert 0 <= rank < world
    return slice(rank * tracks_per_rank, (rank + 1) * tracks_per_rank)


def reduce_over_ranks(times_ms, work, world, device):
    """MAX of the per-rank times, SUM of the per-rank work (terms); identity for world == 1."""
    import torch
    vals = torch.tensor(list(times_ms), dtype=torch.float64, device=device)
    tot = torch.tensor([float(work)], dtype=torch.float64, device=device)
    if world > 1:
        import torch.distributed as dist
        dist.all_reduce(vals, op=dist.ReduceOp.MAX)
        dist.all_reduce(tot, op=dist.ReduceOp.SUM)
    return [float(v) for v in vals.cpu()], float(tot.cpu()[0])


# --------------------------------------------------------------------------------------------------
# our arm
# --------------------------------------------------------------------------------------------------
def unique_row_bytes(wt, g, csr_dev, nt, n_nodes, chunk_carriers=50_000):
    """SURVEY 8(d) algorithmic bytes of Eq. 1.1: every distinct (node, lag) element a carrier needs,
    once: sum over carriers c and visited nodes v of 12 (nt - m_first(c, v)), + 24 M_c + 4 in."""
    import torch
    off = csr_dev["carrier_step_offsets"]
    n_car = off.numel() - 1
    total = 0
    for c0 in range(0, n_car, chunk_carriers):
        c1 = min(n_car, c0 + chunk_carriers)
        s0, s1 = int(off[c0]), int(off[c1])
        if s1 == s0:
            continue
        pos = csr_dev["pos"][s0:s1]
        n0, n1, _ = wt.wt_trajectory_nodes(g, pos)
        lens = (off[c0 + 1:c1 + 1] - off[c0:c1])
        car = torch.repeat_interleave(torch.arange(c1 - c0, device=pos.device), lens)
        m = torch.arange(s1 - s0, device=pos.device) - (off[c0:c1] - s0)[car]
        keep = (m < nt) & (n0[:, 0] >= 0)
        keys, ms = [], []
        ny, nz = g.desc["ny"], g.desc["nz"]
        for cx in (0, 1):
            for cy in (0, 1):
                for cz in (0, 1):
                    ix = (n1 if cx else n0)[:, 0].long()
                    iy = (n1 if cy else n0)[:, 1].long()
                    iz = (n1 if cz else n0)[:, 2].long()
                    keys.append((car * n_nodes + (ix * ny + iy) * nz + iz)[keep])
                    ms.append(m[keep])
        keys = torch.cat(keys)
        ms = torch.cat(ms)
        uk, inv = torch.unique(keys, return_inverse=True)
        first = torch.full((uk.numel(),), nt, dtype=torch.int64, device=pos.device)
        first.scatter_reduce_(0, inv, ms, reduce="amin")
        total += int((12 * (nt - first)).sum()) + 24 * (s1 - s0) + 4 * (c1 - c0)
    return total


def run_ours(args):
    import torch
    import torch.distributed as dist

    import paper_2605_13987_b200 as wt
    from wtide_inputs import carriers_on_tracks, field_drift, make_tracks

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dev = f"cuda:{local}"
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(dev))

    if args.config == 3:
        return run_sweep(args, wt, dev, world, rank)
    d = workload(args)
    nt = d["nt"]
    n_nodes = d["nx"] * d["ny"] * d["nz"]
    g = wt.wt_make_geometry(d)
    plan = wt.wt_describe_plan(g)
    n_sub = wt.wt_query(g, wt.WT_Q_SUBSTEPS)
    n_pads = wt.wt_query(g, wt.WT_Q_N_PADS)
    side = wt._stream(dev)

    # ---- inputs (outside the timed region): the table for the drift field, then the trajectories
    K = max(1, args.batch)       # lock-step copies of the geometry in one wt_solve_H call (1 = the bench line)
    gs = [g] * K
    H = [torch.empty((d["nx"], d["ny"], d["nz"], nt, 3), dtype=torch.float32, device=dev) for _ in range(K)]
    ws_solve = torch.empty(K * wt.wt_query(g, wt.WT_Q_SOLVE_WORKSPACE_BYTES) + 256, dtype=torch.uint8, device=dev)
    wt.wt_solve_H(gs, H=H, workspace=ws_solve, device=dev)
    torch.cuda.synchronize()
    # trajectories: the library's own transport in the static field of the table just solved -- inputs of
    # Eq. 1.1 made on the device, outside the timed region
    from wtide_inputs.tracks import MU_E, MU_H, V_SAT, bias_voltage
    t_gen0 = time.perf_counter()
    e_static = wt.wt_static_field(g, H[0])
    theta_max = 15.0 if args.config == 4 else 10.0
    tracks = make_tracks(args.config, args.tracks * world, d, theta_max)[shard_tracks(args.tracks, world, rank)]
    start, sign, charge, toff = carriers_on_tracks(tracks, args.carriers, d)
    c_off, c_pos, c_vel = wt.wt_drift_carriers(g, e_static, torch.as_tensor(start).to(dev), torch.as_tensor(sign).to(dev), bias_voltage(d),
                                               MU_E, MU_H, V_SAT, max_steps=nt)
    csr = {"track_carrier_offsets": torch.as_tensor(toff, dtype=torch.int64).to(dev), "carrier_step_offsets": c_off, "pos": c_pos, "vel": c_vel,
           "charge": torch.as_tensor(charge).to(dev)}
    del e_static
    torch.cuda.synchronize()
    trajectory_gen_s = time.perf_counter() - t_gen0
    off_host = csr["carrier_step_offsets"].cpu().numpy()
    terms = count_terms(off_host, nt)
    n_steps_total = int(off_host[-1])
    n_car = len(off_host) - 1
    alg_conv_bytes = unique_row_bytes(wt, g, csr, nt, n_nodes) + 4 * nt * args.tracks
    ws_conv = torch.empty(wt.wt_conv_workspace_bytes(g, args.tracks, n_car, True) + 256, dtype=torch.uint8, device=dev)
    out = torch.empty((args.tracks, nt), dtype=torch.float32, device=dev)

    setup_times = []

    def step(ev=None):
        # a0: host setup of the geometry, every step (the handle of the previous step is dropped)
        t0 = time.perf_counter()
        gk = wt.wt_make_geometry(d)
        setup_times.append(time.perf_counter() - t0)
        gsk = [gk] * K
        if ev:
            ev[0].record(side)
        wt.wt_solve_H(gsk, H=H, workspace=ws_solve, device=dev)
        if ev:
            ev[1].record(side)
        wt.wt_convolve_currents(g, H[0], csr["track_carrier_offsets"], csr["carrier_step_offsets"], csr["pos"], csr["vel"],
                                csr["charge"], per_track=True, out=out, workspace=ws_conv)
        if ev:
            ev[2].record(side)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    barrier()
    setup_times.clear()
    launches0 = wt.wt_launch_count()
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(args.steps)]
    with ClockSampler(local) as clk:
        t0 = time.perf_counter()
        for k in range(args.steps):
            step(evs[k])
        barrier()
        wall = time.perf_counter() - t0
    launches = wt.wt_launch_count() - launches0
    solve_ms = float(np.mean([e[0].elapsed_time(e[1]) for e in evs]))
    conv_ms = float(np.mean([e[1].elapsed_time(e[2]) for e in evs]))
    step_ms = float(np.mean([e[0].elapsed_time(e[2]) for e in evs]))
    setup_s = float(np.mean(setup_times))
    # end to end for the solve: descriptor -> handle -> synchronised table, wall clock
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    ge = wt.wt_make_geometry(d)
    wt.wt_solve_H([ge], H=H[:1], workspace=ws_solve, device=dev)
    torch.cuda.synchronize()
    first_row = H[0][0, 0, 0].cpu()                      # (device -> host read of a result row)
    h_solve_e2e_s = time.perf_counter() - t0
    del first_row

    # ---- e2e: Eq. 1.1 through the C ABI with host buffers (pinned), copies inside the timed region.
    # The tracks go in batches (they are independent units): the host->device copy of batch b + 1
    # runs on a copy stream while batch b is in wt_convolve_currents; results come back per batch.
    n_batches = max(1, min(8, args.tracks // 64))
    cuts = [args.tracks * b // n_batches for b in range(n_batches + 1)]
    toff_h = csr["track_carrier_offsets"].cpu()
    coff_h = csr["carrier_step_offsets"].cpu()
    host_batches = []
    for b in range(n_batches):
        c0, c1 = int(toff_h[cuts[b]]), int(toff_h[cuts[b + 1]])
        s0, s1 = int(coff_h[c0]), int(coff_h[c1])
        hb = {"track_carrier_offsets": (toff_h[cuts[b]:cuts[b + 1] + 1] - c0), "carrier_step_offsets": (coff_h[c0:c1 + 1] - s0),
              "pos": csr["pos"][s0:s1].cpu(), "vel": csr["vel"][s0:s1].cpu(), "charge": csr["charge"][c0:c1].cpu()}
        host_batches.append({k: v.contiguous().pin_memory() for k, v in hb.items()})
    out_host = torch.empty((args.tracks, nt), dtype=torch.float32).pin_memory()
    h2d = sum(v.numel() * v.element_size() for hb in host_batches for v in hb.values())
    d2h = out_host.numel() * 4
    copy_stream, comp_stream = torch.cuda.Stream(device=dev), torch.cuda.Stream(device=dev)

    def e2e_step():
        ready = []
        dvs = []
        with torch.cuda.stream(copy_stream):
            for hb in host_batches:
                dvs.append({k: v.to(dev, non_blocking=True) for k, v in hb.items()})
                ev = torch.cuda.Event()
                ev.record(copy_stream)
                ready.append(ev)
        with torch.cuda.stream(comp_stream):
            for b, dv in enumerate(dvs):
                comp_stream.wait_event(ready[b])
                ob = out[cuts[b]:cuts[b + 1]]
                wt.wt_convolve_currents(g, H[0], dv["track_carrier_offsets"], dv["carrier_step_offsets"], dv["pos"], dv["vel"],
                                        dv["charge"], per_track=True, out=ob, workspace=ws_conv)
                out_host[cuts[b]:cuts[b + 1]].copy_(ob, non_blocking=True)
                for v in dv.values():
                    v.record_stream(comp_stream)
        torch.cuda.synchronize()
    one_call = out.clone()
    e2e_step()
    # the batched calls group the carriers differently (other partial rows): equal to fp32 rounding of the sums
    e2e_dev = float((out_host.to(dev) - one_call).abs().max() / one_call.abs().max())
    del one_call
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        e2e_step()
    barrier()
    e2e_s = (time.perf_counter() - t0) / args.steps

    # ---- SURVEY 8(f) row 1 beside the step (not part of it): the electrostatic field of the same geometry, readout column at
    # 1 V and the others at 0 V, preconditioned CG to a residual of 1e-7; one cooperative launch, timed with events
    static_info = None
    if rank == 0 and not args.no_static:
        pots = [1.0 if c["role"] == wt.WT_READOUT else 0.0 for c in d["columns"]]
        best = None
        for _ in range(3):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            e0.record(side)
            _, es_lap, info = wt.wt_solve_static(g, pots, precondition=True, max_iter=4000, tol=1e-7, want_v=False, device=dev)
            e1.record(side)
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1)
            best = ms if best is None else min(best, ms)
        info = info.cpu().numpy()
        static_info = {"ms": best, "iterations": int(info[0]), "relative_residual": float(info[1]),
                       "us_per_iteration": 1e3 * best / max(1, int(info[0])), "what": "wt_solve_static, preconditioned CG, two V <-> rho round trips per iteration"}
        del es_lap

    # ---- reduce over ranks (max time, summed work)
    (solve_ms, conv_ms, step_ms, e2e_ms), total_terms = reduce_over_ranks([solve_ms, conv_ms, step_ms, e2e_s * 1e3], terms, world, dev)

    if rank == 0:
        peak, peak_kind = measured_peaks()
        # roofline of the dominant kernel.  Eq. 1.1: algorithmic bytes = per-carrier distinct (node, lag)
        # elements, duration = CUDA events around wt_convolve_currents on its stream.
        # H solve: 60 N bytes per Euler substep + 40 N per output step, duration = events
        # around wt_solve_H.
        N = n_nodes
        alg_solve_bytes = K * ((60 * N * n_sub + 40 * N) * (nt - 1) + 40 * N)
        conv_gbs = alg_conv_bytes / (conv_ms * 1e-3) / 1e9
        solve_gbs = alg_solve_bytes / (solve_ms * 1e-3) / 1e9
        dominant_is_solve = solve_ms >= conv_ms
        # DRAM bytes from the ncu --set full captures of this workload (profiles/r1_solve.md, profiles/r1_conv.md):
        # solve = 35.9 MB per substep in the cold-cache capture of its three kernels (an upper bound: in the replayed
        # graph the working set is L2-resident); Eq. 1.1 = 154.4 GB per call at 1000 tracks x 1000 carriers.
        default_workload = (args.tracks == 1000 and args.carriers == 1000 and not args.grid and not args.nt and K == 1)
        tr = measured_traffic().get("configs[%d]" % args.config, {}) if default_workload else {}
        traffic_solve = tr["solve_dram_bytes_per_substep"] * n_sub * (nt - 1) if "solve_dram_bytes_per_substep" in tr else None
        traffic_conv = tr.get("conv_dram_bytes")
        fma_peak = wt.wt_measure_fp32_fma(dev)
        roof = {"bound": "hbm", "kernel": ("wt_solve_H, all substeps -- " + plan) if dominant_is_solve
                else "k_conv_systolic", "achieved": solve_gbs if dominant_is_solve else conv_gbs, "peak": peak, "unit": "GB/s",
                "frac": (solve_gbs if dominant_is_solve else conv_gbs) / peak,
                "traffic": traffic_solve if dominant_is_solve else traffic_conv, "peak_source": peak_kind,
                "traffic_source": "profiles/r2_traffic.json (ncu --set full, same kernel sources)" if tr else None,
                "algorithmic_bytes": alg_solve_bytes if dominant_is_solve else alg_conv_bytes,
                "fp32_fma_peak_tflops_measured": fma_peak}
        stages = {"solve_ms": solve_ms, "conv_ms": conv_ms,
                  "solve": {"algorithmic_bytes": alg_solve_bytes, "achieved_gbs": solve_gbs, "frac": solve_gbs / peak,
                            "traffic": traffic_solve,
                            "n_sub": n_sub, "substeps": n_sub * (nt - 1), "us_per_substep": 1e3 * solve_ms / (n_sub * (nt - 1)) / K, "pads": n_pads,
                            "lock_step_geometries": K},
                  "conv": {"algorithmic_bytes": alg_conv_bytes, "no_reuse_gather_bytes": 96 * terms, "achieved_gbs": conv_gbs,
                           "frac": conv_gbs / peak, "traffic": traffic_conv,
                           "dram_frac": (traffic_conv / (conv_ms * 1e-3) / 1e9 / peak) if traffic_conv else None,
                           "fp32_flops": 48 * terms, "fp32_frac_of_measured_fma_peak": 48 * terms / (conv_ms * 1e-3) / 1e12 / fma_peak,
                           "carriers": n_car, "carrier_steps": n_steps_total,
                           "mean_steps": n_steps_total / max(1, n_car)}}
        stages["solve"]["plan"] = plan
        if static_info:
            stages["static_field"] = static_info
        stages["setup_s"] = setup_s
        line = {"metric": METRIC, "value": total_terms / (conv_ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": step_ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f32", "data": "synthetic",
                "config": {"workload": "configs[%d] %s, grid %dx%dx%d, nt=%d, dt=%g ns, %d tracks x %d carriers per GPU"
                           % (args.config, {1: "single pixel cell 55um x 500um", 2: "hexagonal stand-in 128um x 500um, 7 columns",
                                            4: "single pixel cell 55um x 500um, high-statistics table", 0: "tiny cell 55um x 50um"}[args.config],
                              d["nx"], d["ny"], d["nz"], nt, d["dt"], args.tracks, args.carriers),
                           "l2": "inputs larger than L2 (H table %.2f GB, trajectories %.2f GB)" % (n_nodes * nt * 12 / 1e9, n_steps_total * 24 / 1e9),
                           "parallelism": "replicas, tracks sharded" if world > 1 else "single GPU"},
                "setup_s_per_geometry": setup_s, "h_solve_s_per_geometry": solve_ms * 1e-3 / K,
                "h_total_s_per_geometry": setup_s + solve_ms * 1e-3 / K,
                "step_value": total_terms / (step_ms * 1e-3 + setup_s), "stages": stages,
                "roofline": roof,
                "e2e": {"value": total_terms / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                        "what": "Eq. 1.1 stage with pinned host trajectories in, host currents out, %d track batches, copies overlapped with the kernels" % n_batches,
                        "max_dev_from_one_call_result_rel_peak": e2e_dev,
                        "h_solve_e2e_s": h_solve_e2e_s,
                        "h_solve_e2e_what": "descriptor -> wt_make_geometry -> wt_solve_H -> synchronize -> one table row on the host, wall clock"},
                "gpu_launches": int(launches), "clocks": clk.summary(), "wall_s_timed_region": wall,
                "inputs": {"trajectories": "wt_static_field + wt_drift_carriers (saturated drift in the solved field, on the device, outside the timed region)",
                           "trajectory_generation_s": trajectory_gen_s}}
        if not args.no_cpu_baseline and world == 1:
            # the oracle on a bounded sample of the same workload (first carriers of track 0), rows of
            # the same fp32 table fetched once
            ncs = min(n_car, 2048)
            s1 = int(off_host[ncs])
            sample = {"carrier_step_offsets": off_host[:ncs + 1], "pos": csr["pos"][:s1].cpu().numpy(), "vel": csr["vel"][:s1].cpu().numpy(),
                      "charge": csr["charge"][:ncs].cpu().numpy()}
            n0, n1, _ = wt.wt_trajectory_nodes(g, csr["pos"][:s1])
            ids = set()
            a0, a1 = n0.cpu().numpy(), n1.cpu().numpy()
            for cx in (a0, a1):
                for cy in (a0, a1):
                    for cz in (a0, a1):
                        ids.update(zip(cx[:, 0].tolist(), cy[:, 1].tolist(), cz[:, 2].tolist()))
            ids = [t for t in ids if t[0] >= 0]
            idx = torch.tensor(ids, device=dev)
            rows = H[0][idx[:, 0], idx[:, 1], idx[:, 2]].cpu().numpy()
            table = {t: rows[i] for i, t in enumerate(ids)}
            o_terms, o_t, o_car = oracle_conv_sample(d, lambda ix, iy, iz: table[(ix, iy, iz)], sample, args.ref_budget)
            per_sub, nsubs, _, _ = oracle_solve_sample(d, args.ref_budget)
            a_terms, a_wall, a_procs = oracle_conv_all_cores(d, table, sample, o_car)
            line["cpu_baseline"] = {"value": o_terms / o_t, "unit": UNIT, "cores": 1, "kind": "oracle",
                                    "all_cores": {"value": a_terms / a_wall, "unit": UNIT, "cores": a_procs,
                                                  "what": "the same carriers of Eq. 1.1 split over one oracle process per host core"},
                                    "sample": "first %d carriers (%.1f s) for Eq. 1.1; %d Euler substeps on the full grid (%.2f s each) "
                                              "-> H solve extrapolated to %.0f s per geometry" % (o_car, o_t, nsubs, per_sub, per_sub * n_sub * (nt - 1)),
                                    "h_solve_s_per_geometry_extrapolated": per_sub * n_sub * (nt - 1), "host_cores_available": os.cpu_count()}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


# --------------------------------------------------------------------------------------------------
# config 3: the 32-geometry what-if sweep (PAPER.md:15 "what-if studies on sensor geometry", :137-141 the bias
# diameter scan).  Every cell: host setup (a0) -> wt_solve_H -> 200 tracks x 1000 carriers through Eq. 1.1.
# The setup of cell i + 1 runs on a host thread while the GPU works on cell i.  One table (6.44 GB) is reused.
# --------------------------------------------------------------------------------------------------
def run_sweep(args, wt, dev, world, rank):
    import concurrent.futures as cf

    import torch
    import torch.distributed as dist

    from wtide_inputs import carriers_on_tracks, make_tracks, reduced_desc
    from wtide_inputs.configs import sweep_descs
    from wtide_inputs.tracks import MU_E, MU_H, V_SAT, bias_voltage
    descs = sweep_descs()
    if args.nt:
        descs = [reduced_desc(dd, nt=args.nt) for dd in descs]
    cells = [int(c) for c in args.cells.split(",")] if args.cells else list(range(len(descs)))
    cells = cells[rank::world]
    n_tracks = 200 if args.tracks == 1000 else args.tracks
    d0 = descs[0]
    nt, n_nodes = d0["nt"], d0["nx"] * d0["ny"] * d0["nz"]
    side = wt._stream(dev)
    H = torch.empty((d0["nx"], d0["ny"], d0["nz"], nt, 3), dtype=torch.float32, device=dev)
    out = torch.empty((n_tracks, nt), dtype=torch.float32, device=dev)
    pool = cf.ThreadPoolExecutor(max_workers=1)

    def timed_setup(dd):
        t0 = time.perf_counter()
        gg = wt.wt_make_geometry(dd)
        return gg, time.perf_counter() - t0

    def one_pass(record):
        rows = []
        fut = pool.submit(timed_setup, descs[cells[0]])
        ws = None
        for k, ci in enumerate(cells):
            g, t_setup = fut.result()
            if k + 1 < len(cells):
                fut = pool.submit(timed_setup, descs[cells[k + 1]])        # overlaps with this cell's GPU work
            dd = descs[ci]
            need = wt.wt_query(g, wt.WT_Q_SOLVE_WORKSPACE_BYTES) + 256
            if ws is None or ws.numel() < need:
                ws = torch.empty(need, dtype=torch.uint8, device=dev)
            e = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
            e[0].record(side)
            wt.wt_solve_H([g], H=[H], workspace=ws, device=dev)
            e[1].record(side)
            torch.cuda.synchronize()
            # inputs of Eq. 1.1 (outside every timed quantity): drift in the static field of this table
            e_static = wt.wt_static_field(g, H)
            tracks = make_tracks(3, n_tracks, dd, 10.0)
            start, sign, charge, toff = carriers_on_tracks(tracks, args.carriers, dd)
            c_off, c_pos, c_vel = wt.wt_drift_carriers(g, e_static, torch.as_tensor(start).to(dev), torch.as_tensor(sign).to(dev), bias_voltage(dd),
                                                       MU_E, MU_H, V_SAT, max_steps=nt)
            csr = {"track_carrier_offsets": torch.as_tensor(toff, dtype=torch.int64).to(dev), "carrier_step_offsets": c_off, "pos": c_pos,
                   "vel": c_vel, "charge": torch.as_tensor(charge).to(dev)}
            del e_static
            n_car = csr["carrier_step_offsets"].numel() - 1
            wsc = torch.empty(wt.wt_conv_workspace_bytes(g, n_tracks, n_car, True) + 256, dtype=torch.uint8, device=dev)
            torch.cuda.synchronize()
            e[2].record(side)
            wt.wt_convolve_currents(g, H, csr["track_carrier_offsets"], csr["carrier_step_offsets"], csr["pos"], csr["vel"], csr["charge"],
                                    per_track=True, out=out, workspace=wsc)
            e[3].record(side)
            torch.cuda.synchronize()
            if record:
                terms = count_terms(csr["carrier_step_offsets"].cpu().numpy(), nt)
                n_sub = wt.wt_query(g, wt.WT_Q_SUBSTEPS)
                rows.append({"cell": ci, "pitch_um": dd["lx"], "bias_radius_um": dd["columns"][1]["radius"], "resistivity_ohm_cm": dd["columns"][0]["resistivity"],
                             "pads": wt.wt_query(g, wt.WT_Q_N_PADS), "n_sub": n_sub, "plan": wt.wt_describe_plan(g).split(":")[0],
                             "setup_s": t_setup, "solve_s": e[0].elapsed_time(e[1]) * 1e-3, "conv_s": e[2].elapsed_time(e[3]) * 1e-3,
                             "terms": terms, "finite": bool(torch.isfinite(out).all())})
        return rows

    for _ in range(min(args.warmup, 1)):
        one_pass(False)
    launches0 = wt.wt_launch_count()
    with ClockSampler(int(dev.split(":")[1])) as clk:
        t0 = time.perf_counter()
        rows = one_pass(True)
        wall = time.perf_counter() - t0
    launches = wt.wt_launch_count() - launches0
    peak, peak_kind = measured_peaks()
    tot = {k: sum(r[k] for r in rows) for k in ("setup_s", "solve_s", "conv_s", "terms")}
    groups = {}
    for r in rows:
        gk = groups.setdefault(str(r["n_sub"]), {"cells": 0, "solve_s": 0.0, "alg_bytes": 0.0, "setup_s": 0.0})
        gk["cells"] += 1
        gk["solve_s"] += r["solve_s"]
        gk["setup_s"] += r["setup_s"]
        gk["alg_bytes"] += (60 * n_nodes * r["n_sub"] + 40 * n_nodes) * (nt - 1) + 40 * n_nodes
    for gk in groups.values():
        gk["solve_frac_of_hbm_roofline"] = gk["alg_bytes"] / gk["solve_s"] / 1e9 / peak
        gk["solve_s_per_geometry"] = gk["solve_s"] / gk["cells"]
    vals = torch.tensor([tot["setup_s"], tot["solve_s"], tot["conv_s"]], dtype=torch.float64, device=dev)
    work = torch.tensor([float(tot["terms"]), float(len(rows))], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(vals, op=dist.ReduceOp.MAX)
        dist.all_reduce(work, op=dist.ReduceOp.SUM)
    if rank == 0:
        setup_s, solve_s, conv_s = (float(v) for v in vals.cpu())
        terms, n_geo = (float(v) for v in work.cpu())
        per_rank_geo = len(rows)
        alg = sum(gk["alg_bytes"] for gk in groups.values())
        line = {"metric": METRIC, "value": terms / conv_s, "unit": UNIT, "n_gpus": world, "steps": 1, "warmup": min(args.warmup, 1),
                "ms_per_step": 1e3 * (setup_s + solve_s + conv_s), "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f32", "data": "synthetic",
                "config": {"workload": "configs[3] what-if sweep: %d square cells (pitch x bias radius x resistivity), grid %dx%dx%d, nt=%d, %d tracks x %d carriers per geometry"
                           % (int(n_geo), d0["nx"], d0["ny"], d0["nz"], nt, n_tracks, args.carriers),
                           "l2": "inputs larger than L2 (H table %.2f GB per geometry)" % (n_nodes * nt * 12 / 1e9),
                           "parallelism": "replicas, geometries sharded" if world > 1 else "single GPU"},
                "setup_s_per_geometry": setup_s / per_rank_geo, "h_solve_s_per_geometry": solve_s / per_rank_geo,
                "conv_s_per_geometry": conv_s / per_rank_geo, "h_total_s_per_geometry": (setup_s + solve_s) / per_rank_geo,
                "s_per_geometry_all_stages": (setup_s + solve_s + conv_s) / per_rank_geo,
                "wall_s_sweep_incl_input_generation": wall,
                "roofline": {"bound": "hbm", "kernel": "wt_solve_H over the sweep (per-cell plans in `cells`)", "achieved": alg / solve_s / 1e9,
                             "peak": peak, "unit": "GB/s", "frac": alg / solve_s / 1e9 / peak, "traffic": None, "peak_source": peak_kind,
                             "algorithmic_bytes": alg},
                "by_n_sub": groups, "cells": rows, "gpu_launches": int(launches), "clocks": clk.summary(),
                "e2e": {"value": terms / (setup_s + solve_s + conv_s), "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0,
                        "what": "terms per second of the whole sweep incl. host setup and the H solves (trajectories are generated on the device "
                                "from each table: no host buffers in this workload)"}}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


# --------------------------------------------------------------------------------------------------
# --impl cufft: the Euler substep composed from cuFFT 3-D transforms (torch.fft) and elementwise kernels, as the
# paper's own port does ("the 3D FFT implementation shipped with CUDA" + a |k|^2 kernel).  A
# cross-check BASELINE for the fused kernels' head-room (~200 N bytes per substep), not product code:
# no boundary solve, fp32 state.
# --------------------------------------------------------------------------------------------------
def run_cufft(args):
    import torch
    if int(os.environ.get("RANK", "0")) != 0:
        return
    d = workload(args)
    dev = "cuda:0"
    nx, ny, nz = d["nx"], d["ny"], d["nz"]
    N = nx * ny * nz
    kx = (2 * np.pi * np.fft.fftfreq(nx, d["lx"] / nx)).astype(np.float32)
    ky = (2 * np.pi * np.fft.fftfreq(ny, d["ly"] / ny)).astype(np.float32)
    kz = (2 * np.pi * np.fft.rfftfreq(nz, d["lz"] / nz)).astype(np.float32)
    KX = torch.tensor(kx, device=dev)[:, None, None]
    KY = torch.tensor(ky, device=dev)[None, :, None]
    KZ = torch.tensor(kz, device=dev)[None, None, :]
    k2 = KX * KX + KY * KY + KZ * KZ
    ginv = torch.where(k2 > 0, 1.0 / k2, torch.zeros_like(k2))
    sig = (torch.rand((nx, ny, nz), device=dev) < 0.08).float() * 1e-2
    rh = torch.fft.rfftn(torch.randn((nx, ny, nz), device=dev))

    def substep(rh):
        vh = rh * ginv
        acc = torch.zeros_like(rh)
        for K in (KX, KY, KZ):
            e = torch.fft.irfftn(-1j * K * vh, s=(nx, ny, nz))
            acc += 1j * K * torch.fft.rfftn(sig * e)
        return rh - acc
    n_rep = 50
    for _ in range(5):
        rh = substep(rh)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(n_rep):
        rh = substep(rh)
    e1.record()
    torch.cuda.synchronize()
    us = e0.elapsed_time(e1) * 1e3 / n_rep
    peak, peak_kind = measured_peaks()
    print(json.dumps({"impl": "cufft", "what": "Euler substep composed from torch.fft (cuFFT) rfftn/irfftn + elementwise kernels, no boundary solve, fp32",
                      "grid": [nx, ny, nz], "us_per_substep": us, "frac_of_60N_hbm_roofline": 60 * N / (us * 1e-6) / 1e9 / peak,
                      "peak": peak, "peak_source": peak_kind}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference", "cufft"])
    ap.add_argument("--no-static", action="store_true", help="skip the timing of wt_solve_static (reported under stages.static_field)")
    ap.add_argument("--tracks", type=int, default=1000, help="MIP tracks per GPU")
    ap.add_argument("--carriers", type=int, default=1000, help="macro-carriers per track")
    ap.add_argument("--config", type=int, default=1, choices=[0, 1, 2, 3, 4],
                    help="BASELINE.json config whose geometry, grid and nt are used (default 1 = the bench line; 2 and 4 are "
                         "measured as extra rows of BASELINE.md with one batch of tracks, see DESIGN.md)")
    ap.add_argument("--batch", type=int, default=1, help="lock-step copies of the geometry per wt_solve_H call (extra measurement; 1 = bench line)")
    ap.add_argument("--grid", default="", help="override grid, e.g. 32x32x64 (debug only; not a bench line)")
    ap.add_argument("--nt", type=int, default=0, help="override nt (debug only)")
    ap.add_argument("--ref-budget", type=float, default=10.0, help="seconds of oracle work per leg")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cells", default="", help="config 3 only: comma-separated indices of the sweep cells to run (default: all 32)")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # launched without torchrun: start the N ranks ourselves (one process per GPU, replicas: DESIGN.md section 9)
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
               "--master-port", str(29500 + os.getpid() % 2000), os.path.abspath(__file__)] + sys.argv[1:]
        sys.exit(subprocess.call(cmd))
    if args.impl == "reference":
        run_reference(args)
    elif args.impl == "cufft":
        run_cufft(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
