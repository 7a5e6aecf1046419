"""CPU oracle of the CBM-MUCH first-level J/psi selection -- TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg
may import this package.  It is independent of the CUDA path (no shared code, headers,
helpers or tables); the product never routes through it.

    run(...)            -> oracle/cbm_oracle.c   (the definition as nested loops, int64)
    run_slope_sorted()  -> oracle/slope_sorted.c (independent sorted/multiplicity route; a pin)
    brute_force         -> oracle/brute_force.py (no short-circuit, explicit S-tuples; a pin)
    selected, unpack_xy20, gather, filter_layers, build_events -> plain Python loops (the definitions of the list of
                           selected events, the packed wire format, the gather, the input filter, the event building)
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = os.path.join(_HERE, "liboracle.so")
_SRCS = [os.path.join(_HERE, "cbm_oracle.c"), os.path.join(_HERE, "slope_sorted.c"), os.path.join(_HERE, "msd_oracle.c")]
MAX_LAYERS = 24


class Geometry(ctypes.Structure):
    _fields_ = [
        ("n_stations", ctypes.c_uint32),
        ("layer_z", ctypes.c_int32 * MAX_LAYERS),
        ("win_in_num", ctypes.c_uint32), ("win_in_den", ctypes.c_uint32),
        ("win_link_num", ctypes.c_uint32), ("win_link_den", ctypes.c_uint32),
        ("min_candidates", ctypes.c_uint32),
    ]


def geometry(layer_z, win_in=(1, 100), win_link=(2, 100), min_candidates=2) -> Geometry:
    g = Geometry()
    assert len(layer_z) % 3 == 0 and 3 <= len(layer_z) <= MAX_LAYERS
    g.n_stations = len(layer_z) // 3
    for i, z in enumerate(layer_z):
        g.layer_z[i] = int(z)
    g.win_in_num, g.win_in_den = win_in
    g.win_link_num, g.win_link_den = win_link
    g.min_candidates = min_candidates
    return g


class MsdParams(ctypes.Structure):
    """Parameters of the paper-literal selection (oracle/msd_oracle.c)."""
    _fields_ = [
        ("n_stations", ctypes.c_uint32),
        ("layer_z", ctypes.c_int32 * MAX_LAYERS),
        ("station", ctypes.c_uint32),
        ("thr_x_num", ctypes.c_uint32), ("thr_x_den", ctypes.c_uint32),
        ("thr_y_num", ctypes.c_uint32), ("thr_y_den", ctypes.c_uint32),
        ("ndf", ctypes.c_uint32),
        ("min_triplets", ctypes.c_uint32),
    ]


def msd_params(layer_z, station=None, thr_x=(3, 100), thr_y=(25, 1000), ndf=2, min_triplets=2) -> MsdParams:
    """MSD thresholds 0.03 (x-z) and 0.025 (y-z); at least two passing triplets."""
    p = MsdParams()
    assert len(layer_z) % 3 == 0 and 3 <= len(layer_z) <= MAX_LAYERS
    p.n_stations = len(layer_z) // 3
    for i, z in enumerate(layer_z):
        p.layer_z[i] = int(z)
    p.station = p.n_stations - 1 if station is None else station
    p.thr_x_num, p.thr_x_den = thr_x
    p.thr_y_num, p.thr_y_den = thr_y
    p.ndf, p.min_triplets = ndf, min_triplets
    return p


def build(force: bool = False) -> str:
    """gcc -O2 (the paper's CPU flags, minus -march=native so the .so is portable)."""
    newest = max(os.path.getmtime(s) for s in _SRCS)
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < newest:
        subprocess.run(["gcc", "-O2", "-fPIC", "-shared", "-std=c11", "-o", _LIB] + _SRCS, check=True)
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_LIB)
        vp, u64 = ctypes.c_void_p, ctypes.c_uint64
        lib.cbm_oracle_run.restype = ctypes.c_int
        lib.cbm_oracle_run.argtypes = [ctypes.POINTER(Geometry), vp, vp, vp, u64, u64, u64, vp, vp, vp]
        lib.cbm_oracle_run_list.restype = ctypes.c_int
        lib.cbm_oracle_run_list.argtypes = [ctypes.POINTER(Geometry), vp, vp, vp, vp, u64, u64, vp, vp, vp]
        lib.cbm_msd_oracle_run.restype = ctypes.c_int
        lib.cbm_msd_oracle_run.argtypes = [ctypes.POINTER(MsdParams), vp, vp, vp, u64, u64, vp, vp]
        lib.cbm_slope_sorted_run.restype = ctypes.c_int
        lib.cbm_slope_sorted_run.argtypes = [ctypes.POINTER(Geometry), vp, vp, vp, u64, u64, vp, vp, vp, vp]
        _lib = lib
    return _lib


def _check_inputs(x, y, off):
    x = np.ascontiguousarray(x, dtype=np.int32)
    y = np.ascontiguousarray(y, dtype=np.int32)
    off = np.ascontiguousarray(off, dtype=np.uint32)
    return x, y, off


def run(geo: Geometry, x, y, off, e_begin=0, e_end=None, max_list_entries=0):
    """Oracle over events [e_begin, e_end).  Returns (n_triplets[n,S], n_candidates[n], accept[n])."""
    lib = _load()
    x, y, off = _check_inputs(x, y, off)
    S = geo.n_stations
    n_events = (off.size - 1) // (3 * S)
    e_end = n_events if e_end is None else e_end
    n = e_end - e_begin
    nt = np.zeros((max(n, 0), S), dtype=np.uint32)
    nc = np.zeros(max(n, 0), dtype=np.uint32)
    ac = np.zeros(max(n, 0), dtype=np.uint8)
    rc = lib.cbm_oracle_run(ctypes.byref(geo), x.ctypes.data, y.ctypes.data, off.ctypes.data, e_begin, e_end,
                            max_list_entries, nt.ctypes.data, nc.ctypes.data, ac.ctypes.data)
    if rc != 0:
        raise RuntimeError(f"cbm_oracle_run failed: {rc}")
    return nt, nc, ac


def run_list(geo: Geometry, x, y, off, event_ids, max_list_entries=0):
    """Oracle over a list of event ids (sampled parity at full size)."""
    lib = _load()
    x, y, off = _check_inputs(x, y, off)
    ids = np.ascontiguousarray(event_ids, dtype=np.uint64)
    S = geo.n_stations
    nt = np.zeros((ids.size, S), dtype=np.uint32)
    nc = np.zeros(ids.size, dtype=np.uint32)
    ac = np.zeros(ids.size, dtype=np.uint8)
    rc = lib.cbm_oracle_run_list(ctypes.byref(geo), x.ctypes.data, y.ctypes.data, off.ctypes.data,
                                 ids.ctypes.data, ids.size, max_list_entries,
                                 nt.ctypes.data, nc.ctypes.data, ac.ctypes.data)
    if rc != 0:
        raise RuntimeError(f"cbm_oracle_run_list failed: {rc}")
    return nt, nc, ac


def run_slope_sorted(geo: Geometry, x, y, off, e_begin=0, e_end=None):
    """Independent sorted/multiplicity implementation.  Returns (n_triplets, n_candidates, accept, n_eval)."""
    lib = _load()
    x, y, off = _check_inputs(x, y, off)
    S = geo.n_stations
    n_events = (off.size - 1) // (3 * S)
    e_end = n_events if e_end is None else e_end
    n = e_end - e_begin
    nt = np.zeros((max(n, 0), S), dtype=np.uint32)
    nc = np.zeros(max(n, 0), dtype=np.uint32)
    ac = np.zeros(max(n, 0), dtype=np.uint8)
    ne = ctypes.c_uint64(0)
    rc = lib.cbm_slope_sorted_run(ctypes.byref(geo), x.ctypes.data, y.ctypes.data, off.ctypes.data, e_begin, e_end,
                                  nt.ctypes.data, nc.ctypes.data, ac.ctypes.data, ctypes.byref(ne))
    if rc != 0:
        raise RuntimeError(f"cbm_slope_sorted_run failed: {rc}")
    return nt, nc, ac, int(ne.value)


def selected(accept):
    """The list of selected events ("the list of selected events is transferred back"): the ids of
    the events with accept != 0 in ascending order.  Written out as the plain loop it is."""
    ids = []
    for e, a in enumerate(np.asarray(accept).ravel().tolist()):
        if a:
            ids.append(e)
    return np.asarray(ids, dtype=np.uint32)


def unpack_xy20(xy20):
    """The packed wire format XY20 (include/cbm_trigger.h), decoded hit by hit:
    bytes 5i..5i+4 of the stream, little endian, hold x in bits 0..19 and y in bits 20..39, each a 20-bit
    two's complement number.  Returns (x, y) as int32 arrays."""
    b = list(bytes(xy20)) if isinstance(xy20, (bytes, bytearray)) else np.asarray(xy20, dtype=np.uint8).ravel().tolist()
    n = len(b) // 5
    xs, ys = [], []
    for i in range(n):
        v = b[5 * i] | (b[5 * i + 1] << 8) | (b[5 * i + 2] << 16) | (b[5 * i + 3] << 24) | (b[5 * i + 4] << 32)
        xv, yv = v & 0xFFFFF, (v >> 20) & 0xFFFFF
        xs.append(xv - (1 << 20) if xv >= (1 << 19) else xv)
        ys.append(yv - (1 << 20) if yv >= (1 << 19) else yv)
    return np.asarray(xs, dtype=np.int32), np.asarray(ys, dtype=np.int32)


def run_msd(par: MsdParams, x, y, off, e_begin=0, e_end=None):
    """The paper's selection, literally: triplets of the trigger station, least-squares line
    through the vertex, MSD cut, at least two passing triplets.  Returns (n_passing[n], accept[n])."""
    lib = _load()
    x, y, off = _check_inputs(x, y, off)
    n_events = (off.size - 1) // (3 * par.n_stations)
    e_end = n_events if e_end is None else e_end
    n = max(e_end - e_begin, 0)
    npass = np.zeros(n, dtype=np.uint32)
    ac = np.zeros(n, dtype=np.uint8)
    rc = lib.cbm_msd_oracle_run(ctypes.byref(par), x.ctypes.data, y.ctypes.data, off.ctypes.data, e_begin, e_end,
                                npass.ctypes.data, ac.ctypes.data)
    if rc != 0:
        raise RuntimeError(f"cbm_msd_oracle_run failed: {rc}")
    return npass, ac


def gather(x, y, off, n_layers, event_ids):
    """The hits of the listed events as a batch of the same layout, event by
    event and layer by layer.  Returns (x, y, off) with off[0] = 0."""
    xs, ys, o = [], [], [0]
    for e in np.asarray(event_ids).ravel().tolist():
        for l in range(n_layers):
            a, b = int(off[e * n_layers + l]), int(off[e * n_layers + l + 1])
            xs.extend(np.asarray(x[a:b]).tolist())
            ys.extend(np.asarray(y[a:b]).tolist())
            o.append(o[-1] + (b - a))
    return np.asarray(xs, dtype=np.int32), np.asarray(ys, dtype=np.int32), np.asarray(o, dtype=np.uint32)


def filter_layers(xyz, ev_off, layer_z):
    """The paper's input filter (implementation "i3"): out of the full-setup hit data of every event
    (STS and MUCH, about 5000 hits per event, records x, y, z as in PAPER.md:166-170) only the hits of the layers the
    selection works on are kept.  A hit belongs to layer l iff its z equals layer_z[l] (z is a per-layer constant,
    DESIGN.md reading R6); every other hit is dropped.  The kept hits of an event are grouped by layer, in the order
    they have in the stream.  Written out as the plain loops it is.

    xyz: int32 [N][3] records; ev_off: [E + 1] record offsets of the events.  Returns (x, y, off) in the batch layout of
    include/cbm_trigger.h (off has E * L + 1 entries)."""
    xyz = np.asarray(xyz, dtype=np.int32).reshape(-1, 3)
    ev_off = np.asarray(ev_off).ravel().tolist()
    lz = [int(z) for z in layer_z]
    xs, ys, off = [], [], [0]
    rec = xyz.tolist()
    for e in range(len(ev_off) - 1):
        for l in range(len(lz)):
            for i in range(ev_off[e], ev_off[e + 1]):
                if rec[i][2] == lz[l]:
                    xs.append(rec[i][0])
                    ys.append(rec[i][1])
            off.append(len(xs))
    return np.asarray(xs, dtype=np.int32), np.asarray(ys, dtype=np.int32), np.asarray(off, dtype=np.uint32)


def build_events(t, t_gap):
    """Event building from a free-streaming, time-ordered hit stream (section 8: the data acquisition
    "will deliver free-streaming data not associated to single event by a hardware trigger ... the time measurement of
    each hit must be considered"; the paper gives no rule, reading B9 fixes one): the records of a timeslice
    come in stream order with an integer time stamp t[i]; record i opens a new event iff i == 0 or
    t[i] - t[i-1] > t_gap.  An event is a maximal run of records without such a gap.  Written out as the plain loop it is.

    Returns ev_off (uint32 [n_events + 1]): ev_off[k] = first record of event k, ev_off[n_events] = number of records
    ([0] for an empty stream)."""
    ts = [int(v) for v in np.asarray(t).ravel().tolist()]
    gap = int(t_gap)
    starts = []
    for i in range(len(ts)):
        if i == 0 or ts[i] - ts[i - 1] > gap:
            starts.append(i)
    return np.asarray(starts + [len(ts)], dtype=np.uint32)
