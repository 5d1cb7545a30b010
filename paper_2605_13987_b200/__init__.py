"""Thin Python binding of libwtide (include/wtide.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels of libwtide.so; PyTorch is used for device
memory and streams.  There is NO CPU fallback: if the shared library cannot be loaded (or built
with nvcc) importing this package fails, and the compute calls need a CUDA device.

Functions carry the names of the C entry points: wt_make_geometry, wt_solve_H,
wt_convolve_currents, wt_trajectory_nodes, wt_query, wt_get_array, wt_free.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

WT_OK, WT_EINVAL, WT_EGEOM, WT_EUNSTABLE, WT_ENOMEM, WT_ECUDA = 0, -1, -2, -3, -4, -5
WT_BIAS, WT_READOUT, WT_SEGMENT = 0, 1, 2
WT_Q_H_BYTES, WT_Q_SOLVE_WORKSPACE_BYTES, WT_Q_SUBSTEPS, WT_Q_N_PADS = 1, 2, 3, 4
WT_Q_N_NODES, WT_Q_N_CONDUCTING, WT_Q_N_PAD_LAYERS, WT_Q_NT, WT_Q_N_COLUMNS, WT_Q_NZ = 5, 6, 7, 8, 9, 10
WT_A_COLUMN_ID, WT_A_PAD_NODES, WT_A_PAD_POTENTIAL, WT_A_AINV, WT_A_GT, WT_A_GZT = 1, 2, 3, 4, 5, 6

EXPORTS = ("wt_make_geometry", "wt_solve_H", "wt_convolve_currents", "wt_free", "wt_trajectory_nodes",
           "wt_conv_workspace_bytes", "wt_query", "wt_get_array", "wt_last_error", "wt_launch_count", "wt_describe_plan", "wt_measure_fp32_fma", "wt_static_field",
           "wt_drift_workspace_bytes", "wt_drift_count", "wt_offsets_from_counts", "wt_drift_fill", "wt_electronics", "wt_static_workspace_bytes", "wt_solve_static",
           "wt_convolve_tracks_noalloc")


class wt_column(C.Structure):
    _fields_ = [("cx", C.c_double), ("cy", C.c_double), ("radius", C.c_double), ("resistivity", C.c_double),
                ("z0", C.c_double), ("z1", C.c_double), ("role", C.c_int), ("pad_at_z1", C.c_int)]


class wt_geometry_desc(C.Structure):
    _fields_ = [("lx", C.c_double), ("ly", C.c_double), ("lz", C.c_double),
                ("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int), ("nt", C.c_int),
                ("dt", C.c_double), ("eps_r", C.c_double), ("v_w", C.c_double),
                ("substeps", C.c_int), ("n_columns", C.c_int), ("columns", C.POINTER(wt_column)), ("mirror_z", C.c_int)]


class WtideError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libwtide error {code}: {msg}")
        self.code = code


def _load():
    path = _build.LIB
    if not os.path.exists(path) or _build.needs_build():
        try:
            _build.build()
        except Exception as e:  # noqa: BLE001
            if not os.path.exists(path):
                raise ImportError(f"libwtide.so is missing and could not be built with nvcc: {e}") from e
            import warnings
            warnings.warn(f"libwtide.so is older than its sources and the nvcc rebuild failed ({e}); loading the STALE library")
    lib = C.CDLL(path)
    vp, i64, sz = C.c_void_p, C.c_int64, C.c_size_t
    lib.wt_make_geometry.argtypes = [C.POINTER(wt_geometry_desc), C.POINTER(vp)]
    lib.wt_solve_H.argtypes = [C.POINTER(vp), C.c_int, C.POINTER(vp), sz, vp, sz, vp]
    lib.wt_convolve_currents.argtypes = [vp, vp, i64, vp, i64, vp, vp, vp, vp, C.c_int, vp, vp, sz, vp]
    lib.wt_convolve_tracks_noalloc.argtypes = [vp, vp, i64, vp, i64, vp, vp, vp, vp, vp, vp]
    lib.wt_free.argtypes = [vp]
    lib.wt_free.restype = None
    lib.wt_trajectory_nodes.argtypes = [vp, i64, vp, vp, vp, vp, vp]
    lib.wt_conv_workspace_bytes.argtypes = [vp, i64, i64, C.c_int, C.POINTER(sz)]
    lib.wt_query.argtypes = [vp, C.c_int, C.POINTER(i64)]
    lib.wt_get_array.argtypes = [vp, C.c_int, vp, sz]
    lib.wt_describe_plan.argtypes = [vp, C.c_char_p, sz]
    lib.wt_describe_plan.restype = C.c_int
    lib.wt_measure_fp32_fma.argtypes = [vp, sz, vp, C.POINTER(C.c_double)]
    lib.wt_measure_fp32_fma.restype = C.c_int
    dbl = C.c_double
    lib.wt_static_field.argtypes = [vp, vp, vp, vp]
    lib.wt_drift_workspace_bytes.argtypes = [vp, C.POINTER(sz)]
    lib.wt_drift_count.argtypes = [vp, vp, dbl, dbl, dbl, dbl, i64, vp, vp, C.c_int, vp, vp, sz, vp]
    lib.wt_offsets_from_counts.argtypes = [i64, vp, vp, vp]
    lib.wt_drift_fill.argtypes = [vp, vp, dbl, dbl, dbl, dbl, i64, vp, vp, C.c_int, vp, vp, vp, vp, sz, vp]
    lib.wt_electronics.argtypes = [i64, C.c_int, vp, vp, C.c_int, vp, dbl, dbl, vp, vp, vp]
    lib.wt_static_workspace_bytes.argtypes = [vp, C.POINTER(sz)]
    lib.wt_solve_static.argtypes = [vp, C.POINTER(dbl), C.c_int, C.c_int, C.c_int, dbl, vp, vp, vp, vp, sz, vp]
    lib.wt_static_workspace_bytes.restype = C.c_int
    lib.wt_solve_static.restype = C.c_int
    for n in ("wt_static_field", "wt_drift_workspace_bytes", "wt_drift_count", "wt_offsets_from_counts", "wt_drift_fill", "wt_electronics", "wt_static_workspace_bytes", "wt_solve_static"):
        getattr(lib, n).restype = C.c_int
    lib.wt_last_error.restype = C.c_char_p
    lib.wt_launch_count.restype = C.c_int64
    for n in ("wt_make_geometry", "wt_solve_H", "wt_convolve_currents", "wt_trajectory_nodes",
              "wt_conv_workspace_bytes", "wt_query", "wt_get_array"):
        getattr(lib, n).restype = C.c_int
    return lib


_lib = _load()
LIBRARY_PATH = _build.LIB


def _check(rc):
    if rc != WT_OK:
        raise WtideError(rc, _lib.wt_last_error().decode())


class Geometry:
    """Owns a wt_geometry handle (host object)."""

    def __init__(self, handle, desc):
        self.handle = handle
        self.desc = desc

    def __del__(self):
        h, self.handle = getattr(self, "handle", None), None
        if h and _lib is not None:       # (module globals may already be gone at interpreter shutdown)
            _lib.wt_free(h)

    @property
    def shape(self):
        return (self.desc["nx"], self.desc["ny"], self.desc["nz"])

    @property
    def nt(self):
        return self.desc["nt"]


def wt_make_geometry(desc: dict) -> Geometry:
    cols = (wt_column * len(desc["columns"]))()
    for i, c in enumerate(desc["columns"]):
        cols[i] = wt_column(c["cx"], c["cy"], c["radius"], c["resistivity"], c["z0"], c["z1"], c["role"], c["pad_at_z1"])
    d = wt_geometry_desc(desc["lx"], desc["ly"], desc["lz"], desc["nx"], desc["ny"], desc["nz"], desc["nt"],
                         desc["dt"], desc["eps_r"], desc["v_w"], desc.get("substeps", 0), len(cols), cols, int(desc.get("mirror_z", 0)))
    out = C.c_void_p()
    _check(_lib.wt_make_geometry(C.byref(d), C.byref(out)))
    kept = dict(desc)
    if kept.get("mirror_z", 0):       # the handle describes the doubled box (include/wtide.h): shapes follow it
        kept["nz"], kept["lz"] = 2 * desc["nz"], 2.0 * desc["lz"]
    return Geometry(out.value, kept)


def wt_free(geom: Geometry):
    h, geom.handle = geom.handle, None
    if h:
        _lib.wt_free(h)


def wt_query(geom: Geometry, what: int) -> int:
    v = C.c_int64()
    _check(_lib.wt_query(geom.handle, what, C.byref(v)))
    return v.value


def wt_get_array(geom: Geometry, what: int) -> np.ndarray:
    nx, ny, nz = geom.shape
    nb = wt_query(geom, WT_Q_N_PADS)
    if what == WT_A_COLUMN_ID:
        a = np.empty((nx, ny, nz), np.int8)
    elif what == WT_A_PAD_NODES:
        a = np.empty((nb, 3), np.int32)
    elif what == WT_A_PAD_POTENTIAL:
        a = np.empty(nb, np.float64)
    elif what == WT_A_AINV:
        a = np.empty((nb, nb), np.float64)
    elif what in (WT_A_GT, WT_A_GZT):
        a = np.empty((nx, nz, ny // 2), np.float32)
    else:
        raise ValueError("unknown array")
    _check(_lib.wt_get_array(geom.handle, what, a.ctypes.data, a.nbytes))
    return a


# ---- device calls (torch for memory and streams only) ------------------------------------------
_streams = {}


def _stream(device):
    import torch
    key = torch.device(device).index or 0
    if key not in _streams:
        _streams[key] = torch.cuda.Stream(device=device)
    return _streams[key]


def _run_on_side_stream(device, fn):
    """libwtide never touches the default stream: enqueue on a side stream ordered after the
    caller's current stream, then order the current stream after it."""
    import torch
    side = _stream(device)
    cur = torch.cuda.current_stream(device)
    side.wait_stream(cur)
    with torch.cuda.device(device):
        rc = fn(side.cuda_stream)
    cur.wait_stream(side)
    _check(rc)


def wt_solve_H(geoms, H=None, workspace=None, device="cuda:0"):
    """Solves H for a lock-step batch of geometries.  Returns the list of H tensors
    [nx, ny, nz, nt, 3] float32 on `device` (allocated here unless given)."""
    import torch
    geoms = list(geoms)
    g0 = geoms[0]
    nx, ny, nz = g0.shape
    if H is None:
        H = [torch.empty((nx, ny, nz, g0.nt, 3), dtype=torch.float32, device=device) for _ in geoms]
    need = sum(wt_query(g, WT_Q_SOLVE_WORKSPACE_BYTES) for g in geoms)
    if workspace is None:
        workspace = torch.empty(need + 256, dtype=torch.uint8, device=device)
    wptr = (workspace.data_ptr() + 255) // 256 * 256
    wbytes = workspace.numel() - (wptr - workspace.data_ptr())
    hs = (C.c_void_p * len(geoms))(*[g.handle for g in geoms])
    hp = (C.c_void_p * len(geoms))(*[h.data_ptr() for h in H])
    hbytes = H[0].numel() * 4
    _run_on_side_stream(device, lambda s: _lib.wt_solve_H(hs, len(geoms), hp, hbytes, wptr, wbytes, s))
    workspace.record_stream(_stream(device))
    for h in H:
        h.record_stream(_stream(device))
    return H


def wt_conv_workspace_bytes(geom, n_tracks, n_carriers, per_track=True) -> int:
    b = C.c_size_t()
    _check(_lib.wt_conv_workspace_bytes(geom.handle, n_tracks, n_carriers, int(per_track), C.byref(b)))
    return b.value


def wt_convolve_currents(geom, H, track_carrier_offsets, carrier_step_offsets, pos, vel, charge,
                         per_track=True, out=None, workspace=None):
    """Eq. 1.1 for a batch of carriers.  All arguments are CUDA tensors (int64 offsets, float32
    pos/vel [S,3], charge [C]).  Returns out[n_tracks or n_carriers, nt] float32."""
    import torch
    device = H.device
    n_car = carrier_step_offsets.numel() - 1
    n_trk = track_carrier_offsets.numel() - 1 if track_carrier_offsets is not None else 0
    rows = n_trk if per_track else n_car
    if out is None:
        out = torch.empty((rows, geom.nt), dtype=torch.float32, device=device)
    need = wt_conv_workspace_bytes(geom, n_trk, n_car, per_track)
    if workspace is None and need:
        workspace = torch.empty(need + 256, dtype=torch.uint8, device=device)
    wptr = (workspace.data_ptr() + 255) // 256 * 256 if workspace is not None else 0
    wbytes = workspace.numel() - (wptr - workspace.data_ptr()) if workspace is not None else 0
    for t in (pos, vel, charge):
        assert t.dtype == torch.float32 and t.is_contiguous()
    assert carrier_step_offsets.dtype == torch.int64
    tptr = track_carrier_offsets.data_ptr() if track_carrier_offsets is not None else 0
    _run_on_side_stream(device, lambda s: _lib.wt_convolve_currents(
        geom.handle, H.data_ptr(), n_trk, tptr, n_car, carrier_step_offsets.data_ptr(),
        pos.data_ptr(), vel.data_ptr(), charge.data_ptr(), int(per_track), out.data_ptr(), wptr, wbytes, s))
    for t in (out, workspace):
        if t is not None:
            t.record_stream(_stream(device))
    return out


WT_NOALLOC_MAX_FLOATS = 1 << 20


def wt_convolve_tracks_noalloc(geom, H, track_carrier_offsets, carrier_step_offsets, pos, vel, charge, out):
    """Eq. 1.1 summed per track with the library's built-in scratch (include/wtide.h): the call allocates no device memory,
    so `out` [n_tracks, nt] float32 is the caller's.  n_carriers * nt <= WT_NOALLOC_MAX_FLOATS, else WtideError (WT_ENOMEM).
    Calls that overlap on the GPU race on the shared scratch."""
    import torch
    device = H.device
    n_car = carrier_step_offsets.numel() - 1
    n_trk = track_carrier_offsets.numel() - 1
    for t in (pos, vel, charge):
        assert t.dtype == torch.float32 and t.is_contiguous()
    assert carrier_step_offsets.dtype == torch.int64 and track_carrier_offsets.dtype == torch.int64
    assert out.dtype == torch.float32 and out.is_contiguous() and tuple(out.shape) == (n_trk, geom.nt) and out.device == device
    # (_run_on_side_stream makes `device` current for the call, as the header asks)
    _run_on_side_stream(device, lambda s: _lib.wt_convolve_tracks_noalloc(
        geom.handle, H.data_ptr(), n_trk, track_carrier_offsets.data_ptr(), n_car, carrier_step_offsets.data_ptr(),
        pos.data_ptr(), vel.data_ptr(), charge.data_ptr(), out.data_ptr(), s))
    out.record_stream(_stream(device))
    return out


def wt_describe_plan(geom: Geometry) -> str:
    buf = C.create_string_buffer(512)
    _check(_lib.wt_describe_plan(geom.handle, buf, len(buf)))
    return buf.value.decode()


def wt_static_field(geom, H):
    """Es = dt * sum_n H[..., n, :]: float32 [nx, ny, nz, 3] on H's device."""
    import torch
    nx, ny, nz = geom.shape
    es = torch.empty((nx, ny, nz, 3), dtype=torch.float32, device=H.device)
    _run_on_side_stream(H.device, lambda s: _lib.wt_static_field(geom.handle, H.data_ptr(), es.data_ptr(), s))
    es.record_stream(_stream(H.device))
    return es


def wt_solve_static(geom, column_potentials, precondition=True, max_iter=2000, tol=1e-7, want_v=True, want_e=True, device="cuda:0"):
    """Electrostatic potential and field with whole columns as electrodes.
    Returns (V float32 [nx,ny,nz] or None, E float32 [nx,ny,nz,3] or None, info float64 [4] on the device:
    iterations, relative residual, constant c, sum of the charges)."""
    import torch
    nx, ny, nz = geom.shape
    need = C.c_size_t()
    _check(_lib.wt_static_workspace_bytes(geom.handle, C.byref(need)))
    ws = torch.empty(need.value + 256, dtype=torch.uint8, device=device)
    wptr = (ws.data_ptr() + 255) // 256 * 256
    v = torch.empty((nx, ny, nz), dtype=torch.float32, device=device) if want_v else None
    e = torch.empty((nx, ny, nz, 3), dtype=torch.float32, device=device) if want_e else None
    info = torch.empty(4, dtype=torch.float64, device=device)
    pots = (C.c_double * len(column_potentials))(*[float(x) for x in column_potentials])
    _run_on_side_stream(device, lambda s: _lib.wt_solve_static(
        geom.handle, pots, len(column_potentials), int(bool(precondition)), int(max_iter), float(tol),
        v.data_ptr() if want_v else 0, e.data_ptr() if want_e else 0, info.data_ptr(), wptr, need.value, s))
    for t in (ws, v, e, info):
        if t is not None:
            t.record_stream(_stream(device))
    return v, e, info


def wt_drift_carriers(geom, es, start, sign, v_bias, mu_e=180.0, mu_h=150.0, v_sat=150.0, max_steps=None):
    """Saturated-drift transport of carriers in the static field `es` (wt_static_field).  start float32 [C,3], sign int8 [C]
    on es's device.  Returns (carrier_step_offsets int64 [C+1], pos float32 [S,3], vel float32 [S,3]) on the device."""
    import torch
    dev = es.device
    n = start.shape[0]
    max_steps = geom.nt if max_steps is None else max_steps
    assert start.dtype == torch.float32 and start.is_contiguous() and sign.dtype == torch.int8 and sign.is_contiguous()
    need = C.c_size_t()
    _check(_lib.wt_drift_workspace_bytes(geom.handle, C.byref(need)))
    ws = torch.empty(need.value + 256, dtype=torch.uint8, device=dev)
    wptr = (ws.data_ptr() + 255) // 256 * 256
    counts = torch.empty(max(n, 1), dtype=torch.int64, device=dev)
    offs = torch.empty(n + 1, dtype=torch.int64, device=dev)
    args = (geom.handle, es.data_ptr(), float(v_bias), float(mu_e), float(mu_h), float(v_sat), n, start.data_ptr(), sign.data_ptr(), int(max_steps))
    _run_on_side_stream(dev, lambda s: _lib.wt_drift_count(*args, counts.data_ptr(), wptr, need.value, s))
    _run_on_side_stream(dev, lambda s: _lib.wt_offsets_from_counts(n, counts.data_ptr(), offs.data_ptr(), s))
    total = int(offs[-1])                      # (the one host read: sizes of the outputs)
    pos = torch.empty((total, 3), dtype=torch.float32, device=dev)
    vel = torch.empty((total, 3), dtype=torch.float32, device=dev)
    _run_on_side_stream(dev, lambda s: _lib.wt_drift_fill(*args, offs.data_ptr(), pos.data_ptr(), vel.data_ptr(), wptr, need.value, s))
    for t in (ws, counts, offs, pos, vel):
        t.record_stream(_stream(dev))
    return offs, pos, vel


def wt_electronics(currents, transfer, dt, noise=None, cfd_fraction=0.3):
    """Front-end transfer function (causal FIR), optional additive noise, constant-fraction time per row.
    Returns (out float32 [R, nt], t_cfd float32 [R])."""
    import torch
    dev = currents.device
    rows, nt = currents.shape
    assert currents.dtype == torch.float32 and currents.is_contiguous() and transfer.dtype == torch.float32 and transfer.is_contiguous()
    out = torch.empty((rows, nt), dtype=torch.float32, device=dev)
    tc = torch.empty(rows, dtype=torch.float32, device=dev)
    nptr = noise.data_ptr() if noise is not None else 0
    _run_on_side_stream(dev, lambda s: _lib.wt_electronics(rows, nt, currents.data_ptr(), transfer.data_ptr(), transfer.numel(), nptr, float(dt),
                                                            float(cfd_fraction), out.data_ptr(), tc.data_ptr(), s))
    for t in (out, tc):
        t.record_stream(_stream(dev))
    return out, tc


def wt_measure_fp32_fma(device="cuda:0") -> float:
    """Measured FP32 FMA rate of the device in TFLOP/s."""
    import torch
    scratch = torch.empty(4 << 20, dtype=torch.uint8, device=device)
    out = C.c_double()
    with torch.cuda.device(device):
        _check(_lib.wt_measure_fp32_fma(scratch.data_ptr(), scratch.numel(), _stream(device).cuda_stream, C.byref(out)))
    return out.value


def wt_launch_count() -> int:
    return int(_lib.wt_launch_count())


def wt_trajectory_nodes(geom, pos):
    """R24 index arithmetic on the device: returns (node0 int32 [S,3], node1 int32 [S,3], frac float32 [S,3])."""
    import torch
    s = pos.shape[0]
    n0 = torch.empty((s, 3), dtype=torch.int32, device=pos.device)
    n1 = torch.empty((s, 3), dtype=torch.int32, device=pos.device)
    fr = torch.empty((s, 3), dtype=torch.float32, device=pos.device)
    _run_on_side_stream(pos.device, lambda st: _lib.wt_trajectory_nodes(
        geom.handle, s, pos.data_ptr(), n0.data_ptr(), n1.data_ptr(), fr.data_ptr(), st))
    return n0, n1, fr
