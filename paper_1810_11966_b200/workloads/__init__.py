"""Seeded synthetic workloads for the CBM-MUCH first-level J/psi trigger.

Input generators only: this module holds none of the trigger's arithmetic and is the
one module that both the CUDA path (tests, bench) and the CPU oracle's tests consume.
The five configurations are BASELINE.json's ``configs`` with the readings R13-R18 of
SURVEY.md section 8(c); they stand in for the paper's simulated samples D1-D3
(PAPER.md:96-99), which are not available.  The recipe is restated in DESIGN.md.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gen.c")
_LIB = os.path.join(_HERE, "libcbmgen.so")
MAX_LAYERS = 24


class _GenParams(ctypes.Structure):
    _fields_ = [
        ("struct_size", ctypes.c_uint32),
        ("n_stations", ctypes.c_uint32),
        ("layer_z", ctypes.c_int32 * MAX_LAYERS),
        ("occupancy_mode", ctypes.c_uint32),
        ("max_bg_per_layer", ctypes.c_uint32),
        ("mean_a", ctypes.c_double),
        ("mean_b", ctypes.c_double),
        ("frac_b", ctypes.c_double),
        ("mean_clamp", ctypes.c_double),
        ("half_aperture", ctypes.c_double),
        ("signal_fraction", ctypes.c_double),
        ("vertex_sigma_cm", ctypes.c_double),
        ("signal_slope_max", ctypes.c_double),
        ("smear_sigma_cm", ctypes.c_double),
        ("layer_efficiency", ctypes.c_double),
    ]


def station_layers_z(bases_cm):
    """Layer z in 10-um units: station base + {0, 10, 20} cm (BASELINE.json configs[0])."""
    return [int(round((b + d) * 1000)) for b in bases_cm for d in (0, 10, 20)]


GEOMETRY_4 = station_layers_z([60, 100, 150, 210])
GEOMETRY_6 = station_layers_z([60, 100, 150, 210, 280, 360])


@dataclass(frozen=True)
class WorkloadConfig:
    """One of BASELINE.json's configurations (synthetic stand-in for the paper's samples)."""

    name: str
    n_events: int
    seed: int
    layer_z: tuple
    occupancy_mode: int  # 0 fixed, 1 log-normal, 2 mixture
    mean_a: float
    mean_b: float = 0.0
    frac_b: float = 0.0
    signal_fraction: float = 0.0
    mean_clamp: float = 2000.0
    half_aperture: float = 0.35
    vertex_sigma_cm: float = 0.1
    signal_slope_max: float = 0.3
    smear_sigma_cm: float = 0.1
    layer_efficiency: float = 0.95
    max_bg_per_layer: int = 4000
    chunk_events: int = 0  # config 4: streamed in chunks of this many events
    # trigger parameters that go with the workload (BASELINE.json configs[0])
    win_in: tuple = (1, 100)
    win_link: tuple = (2, 100)
    min_candidates: int = 2
    max_hits_per_layer: int = 4096

    @property
    def n_stations(self) -> int:
        return len(self.layer_z) // 3

    @property
    def n_layers(self) -> int:
        return len(self.layer_z)


CONFIGS = {
    0: WorkloadConfig("cfg0_tiny", 1_000, 1, tuple(GEOMETRY_4), 0, 20.0, signal_fraction=0.10),
    1: WorkloadConfig("cfg1_central_like", 100_000, 2, tuple(GEOMETRY_4), 0, 60.0, signal_fraction=0.01),
    2: WorkloadConfig("cfg2_timeslice", 1_000_000, 3, tuple(GEOMETRY_6), 1, 40.0, mean_b=0.8,
                      signal_fraction=0.001),
    3: WorkloadConfig("cfg3_imbalance", 1_000_000, 4, tuple(GEOMETRY_4), 2, 5.0, mean_b=300.0, frac_b=0.05,
                      signal_fraction=0.005),
    4: WorkloadConfig("cfg4_streaming", 10_000_000, 5, tuple(GEOMETRY_6), 1, 40.0, mean_b=0.8,
                      signal_fraction=0.001, chunk_events=1_000_000),
}


# The paper's own measurement workload ("about 15 hits per layer", about 45 per event in the
# trigger station; Table 1: 1 000 .. 80 000 events): one station of three layers, background
# Poisson(15) per layer, a planted pair in 1 % of the events.  Synthetic stand-in for the sample D2; used by the
# paper-literal MSD mode only (bench.py --mode msd, tests/test_msd_mode.py).
PAPER_TABLE1 = WorkloadConfig("paper_table1_trigger_station", 40_000, 11, tuple(station_layers_z([210])), 0, 15.0,
                              signal_fraction=0.01)


def build(force: bool = False) -> str:
    """Compile gen.c into libcbmgen.so (gcc, in-tree)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fPIC", "-shared", "-std=c11", "-o", _LIB, _SRC, "-lm", "-lpthread"]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_LIB)
        lib.cbm_gen_offsets.restype = ctypes.c_uint64
        lib.cbm_gen_offsets.argtypes = [ctypes.POINTER(_GenParams), ctypes.c_uint64, ctypes.c_uint64,
                                        ctypes.c_uint32, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int]
        lib.cbm_gen_hits.restype = ctypes.c_int
        lib.cbm_gen_hits.argtypes = [ctypes.POINTER(_GenParams), ctypes.c_uint64, ctypes.c_uint64,
                                     ctypes.c_uint32, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p,
                                     ctypes.c_int]
        _lib = lib
    return _lib


def _params(cfg: WorkloadConfig) -> _GenParams:
    p = _GenParams()
    p.struct_size = ctypes.sizeof(_GenParams)
    p.n_stations = cfg.n_stations
    for i, z in enumerate(cfg.layer_z):
        p.layer_z[i] = z
    p.occupancy_mode = cfg.occupancy_mode
    p.max_bg_per_layer = cfg.max_bg_per_layer
    p.mean_a, p.mean_b, p.frac_b, p.mean_clamp = cfg.mean_a, cfg.mean_b, cfg.frac_b, cfg.mean_clamp
    p.half_aperture = cfg.half_aperture
    p.signal_fraction = cfg.signal_fraction
    p.vertex_sigma_cm = cfg.vertex_sigma_cm
    p.signal_slope_max = cfg.signal_slope_max
    p.smear_sigma_cm = cfg.smear_sigma_cm
    p.layer_efficiency = cfg.layer_efficiency
    return p


@dataclass
class Batch:
    """One CSR-SoA timeslice batch: x[N], y[N] int32 (10-um units), off[E*L+1] uint32."""

    cfg: WorkloadConfig
    first_event: int
    n_events: int
    x: np.ndarray
    y: np.ndarray
    off: np.ndarray
    truth: np.ndarray = field(default=None)  # bit0 planted, bit1 both tracks complete, bit2 class b

    @property
    def n_hits(self) -> int:
        return int(self.off[-1])


def default_threads() -> int:
    return max(1, min(64, os.cpu_count() or 1))


def generate_offsets(cfg: WorkloadConfig, n_events=None, first_event=0, seed=None, n_threads=None,
                     off_out=None):
    """Pass 1: offsets and truth flags.  Returns (off, truth, n_hits)."""
    lib = _load()
    n_events = cfg.n_events if n_events is None else int(n_events)
    seed = cfg.seed if seed is None else int(seed)
    n_threads = default_threads() if n_threads is None else n_threads
    L = cfg.n_layers
    off = np.empty(n_events * L + 1, dtype=np.uint32) if off_out is None else off_out
    assert off.dtype == np.uint32 and off.size >= n_events * L + 1 and off.flags.c_contiguous
    truth = np.zeros(n_events, dtype=np.uint8)
    p = _params(cfg)
    n_hits = lib.cbm_gen_offsets(ctypes.byref(p), seed, first_event, n_events,
                                 off.ctypes.data, truth.ctypes.data, n_threads)
    if n_hits == 2**64 - 1:
        raise RuntimeError("cbm_gen_offsets failed (bad parameters or more than 2^32-1 hits)")
    return off, truth, int(n_hits)


def generate_hits(cfg: WorkloadConfig, off, x_out, y_out, n_events=None, first_event=0, seed=None,
                  n_threads=None):
    """Pass 2: fill x_out / y_out (any int32 buffers of >= n_hits entries, e.g. pinned memory)."""
    lib = _load()
    n_events = cfg.n_events if n_events is None else int(n_events)
    seed = cfg.seed if seed is None else int(seed)
    n_threads = default_threads() if n_threads is None else n_threads
    p = _params(cfg)
    for a in (x_out, y_out):
        assert a.dtype == np.int32 and a.flags.c_contiguous and a.size >= int(off[n_events * cfg.n_layers])
    rc = lib.cbm_gen_hits(ctypes.byref(p), seed, first_event, n_events, off.ctypes.data,
                          x_out.ctypes.data, y_out.ctypes.data, n_threads)
    if rc != 0:
        raise RuntimeError("cbm_gen_hits failed")


def generate(cfg: WorkloadConfig, n_events=None, first_event=0, seed=None, n_threads=None) -> Batch:
    """Generate one batch of ``cfg`` into fresh numpy arrays."""
    n_events = cfg.n_events if n_events is None else int(n_events)
    off, truth, n_hits = generate_offsets(cfg, n_events, first_event, seed, n_threads)
    x = np.empty(max(n_hits, 1), dtype=np.int32)[:n_hits]
    y = np.empty(max(n_hits, 1), dtype=np.int32)[:n_hits]
    if n_hits:
        generate_hits(cfg, off, x, y, n_events, first_event, seed, n_threads)
    return Batch(cfg, first_event, n_events, x, y, off, truth)


def batch_from_layers(layer_z, events) -> tuple:
    """Hand-built events -> (x, y, off).  ``events`` is a list of events, each a list of L layers,
    each a list of (x, y) integer pairs."""
    L = len(layer_z)
    xs, ys, off = [], [], [0]
    for ev in events:
        assert len(ev) == L
        for layer in ev:
            for (hx, hy) in layer:
                xs.append(int(hx))
                ys.append(int(hy))
            off.append(len(xs))
    return (np.asarray(xs, dtype=np.int32).reshape(-1), np.asarray(ys, dtype=np.int32).reshape(-1),
            np.asarray(off, dtype=np.uint32))


XY20_MIN, XY20_MAX = -(1 << 19), (1 << 19) - 1


def pack_xy20(x, y):
    """The packed wire format XY20 of include/cbm_trigger.h (input formatting only): 5 bytes per hit, little
    endian, bits 0..19 = x, bits 20..39 = y, 20-bit two's complement.  Raises if a coordinate does not fit."""
    x = np.ascontiguousarray(x, dtype=np.int32)
    y = np.ascontiguousarray(y, dtype=np.int32)
    if x.size and (min(x.min(), y.min()) < XY20_MIN or max(x.max(), y.max()) > XY20_MAX):
        raise ValueError("coordinate outside the 20-bit range of the XY20 wire format")
    v = (x.astype(np.int64) & 0xFFFFF).astype(np.uint64) | ((y.astype(np.int64) & 0xFFFFF).astype(np.uint64) << np.uint64(20))
    return np.ascontiguousarray(v.astype("<u8").view(np.uint8).reshape(-1, 8)[:, :5]).reshape(-1)


def full_setup_stream(batch: Batch, other_hits_per_event=400, seed=0, other_z=None):
    """A full-setup hit stream around a generated batch (input formatting only; records x, y, z;
    PAPER.md:188: an event holds the hits of the whole setup, of which the selection uses a small fraction): every
    event's batch hits become records (x, y, z of their layer), mixed in random order -- the relative order of the
    hits of one layer is kept -- with `other_hits_per_event` (Poisson) records of other detector planes (z values
    that are not layer z).  Returns (xyz int32 [N][3], ev_off uint32 [E + 1])."""
    cfg = batch.cfg
    L, E = cfg.n_layers, batch.n_events
    rng = np.random.default_rng(seed)
    lz = np.asarray(cfg.layer_z, dtype=np.int32)
    if other_z is None:  # STS-like planes upstream of the absorbers, and planes between the stations
        other_z = np.asarray([z for z in list(range(30_000, 101_000, 10_000)) + [int(v) + 5_000 for v in lz] if z not in set(lz.tolist())],
                             dtype=np.int32)
    cnt = np.diff(batch.off.astype(np.int64)).reshape(E, L)
    n_much = cnt.sum(axis=1)
    n_other = rng.poisson(other_hits_per_event, size=E).astype(np.int64)
    ev_off = np.zeros(E + 1, dtype=np.int64)
    np.cumsum(n_much + n_other, out=ev_off[1:])
    N = int(ev_off[-1])
    assert N < 2**32
    xyz = np.empty((N, 3), dtype=np.int32)
    layer_of_hit = np.repeat(np.tile(np.arange(L), E), cnt.ravel())
    for e in range(E):
        a, b = int(batch.off[e * L]), int(batch.off[e * L + L])
        m, o = int(n_much[e]), int(n_other[e])
        is_much = np.zeros(m + o, dtype=bool)
        is_much[rng.choice(m + o, size=m, replace=False)] = True
        # batch hits in a random layer interleaving that keeps the order inside every layer
        order = np.argsort(rng.random(m) + 0.0, kind="stable") if m else np.zeros(0, dtype=np.int64)
        lay = layer_of_hit[a:b]
        seq = np.empty(m, dtype=np.int64)
        # positions are dealt to layers at random; within a layer the hits keep their order
        perm_lay = lay[order]
        for l in np.unique(lay):
            seq[np.flatnonzero(perm_lay == l)] = a + np.flatnonzero(lay == l)
        rec = xyz[int(ev_off[e]):int(ev_off[e + 1])]
        rec[is_much, 0], rec[is_much, 1], rec[is_much, 2] = batch.x[seq], batch.y[seq], lz[layer_of_hit[seq]]
        rec[~is_much, 0] = rng.integers(-400_000, 400_001, size=o)
        rec[~is_much, 1] = rng.integers(-400_000, 400_001, size=o)
        rec[~is_much, 2] = other_z[rng.integers(0, other_z.size, size=o)]
    return xyz, ev_off.astype(np.uint32)


def timed_stream(batch: Batch, other_hits_per_event=100, mean_dt=100, spread=8, seed=0):
    """A free-streaming timeslice around a generated batch (input formatting only; free-streaming
    data, every hit with a time measurement): the records of full_setup_stream() in their stream order, plus a time
    stamp per record in ns: interaction e happens at T_e (exponential gaps of mean `mean_dt`: 100 ns = CBM's 10 MHz,
    PAPER.md:23), its records lie at T_e + sorted uniform offsets in [0, spread].  Returns (xyz int32 [N][3],
    t int32 [N] non-decreasing, ev_off uint32 [E + 1] of the interactions)."""
    xyz, ev_off = full_setup_stream(batch, other_hits_per_event=other_hits_per_event, seed=seed)
    rng = np.random.default_rng(seed + 1000)
    E = batch.n_events
    T = np.cumsum(rng.exponential(mean_dt, size=E)).astype(np.int64) + np.arange(E, dtype=np.int64)  # strictly increasing
    t = np.empty(xyz.shape[0], dtype=np.int64)
    for e in range(E):
        a, b = int(ev_off[e]), int(ev_off[e + 1])
        t[a:b] = T[e] + np.sort(rng.integers(0, spread + 1, size=b - a))
    t = np.maximum.accumulate(t)  # interactions closer than `spread` overlap: the stream stays time-ordered
    assert t.size == 0 or t[-1] < 2**31
    return xyz, t.astype(np.int32), ev_off
