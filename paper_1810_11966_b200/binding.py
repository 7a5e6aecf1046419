"""Thin ctypes binding of libcbmtrigger.so (include/cbm_trigger.h): argument marshalling only.

Every step of the selection runs in the CUDA kernels behind the C ABI.  There is no CPU fallback:
if the library has not been built, importing the symbols raises.  The functions carry the names
of the C entry points; ``Trigger`` is a small convenience wrapper around a handle.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libcbmtrigger.so")

MAX_LAYERS = 24
N_KERNELS = 6
KERNEL_NAMES = ("classify_kernel", "tile_kernel", "team_kernel_M", "chain_kernel_H", "team_kernel_G", "team_kernel_X")
CBM_OK, CBM_ERR_INVALID_ARG, CBM_ERR_RANGE, CBM_ERR_CAPACITY, CBM_ERR_STATE, CBM_ERR_CUDA = 0, -1, -2, -3, -4, -5
CBM_FLAG_PROFILE, CBM_FLAG_NO_TINY_PATH, CBM_FLAG_PACKED_INPUT, CBM_FLAG_SERIAL = 1, 2, 4, 8
EXPORTS = (
    "cbm_trigger_create", "cbm_trigger_destroy", "cbm_trigger_host_buffers", "cbm_trigger_upload_events",
    "cbm_trigger_run", "cbm_trigger_fetch_results", "cbm_trigger_run_device", "cbm_trigger_device_status",
    "cbm_trigger_get_stats", "cbm_trigger_last_error", "cbm_trigger_version", "cbm_trigger_device_kernel_times",
    "cbm_trigger_fetch_selected", "cbm_trigger_select_device", "cbm_trigger_select_noalloc",
    "cbm_trigger_host_buffers_packed", "cbm_trigger_upload_events_packed", "cbm_trigger_msd_device", "cbm_trigger_gather_device",
    "cbm_trigger_ubench", "cbm_trigger_filter_device", "cbm_trigger_build_events_device", "cbm_trigger_pack_xy20",
)
PROFILE_RING = 32
# scheduler classes (csrc/cbm_trigger.cu, csrc/params.h), restated for bookkeeping in bench.py only
CLASS_CAPS = (128, 448, 4096)
TINY_MAX_LAYER_DEFAULT, TINY_MAX_TOTAL = 24, 96


class Config(ctypes.Structure):
    _fields_ = [
        ("struct_size", ctypes.c_uint32),
        ("n_stations", ctypes.c_uint32),
        ("layer_z", ctypes.c_int32 * MAX_LAYERS),
        ("win_in_num", ctypes.c_uint32), ("win_in_den", ctypes.c_uint32),
        ("win_link_num", ctypes.c_uint32), ("win_link_den", ctypes.c_uint32),
        ("min_candidates", ctypes.c_uint32),
        ("max_events", ctypes.c_uint32),
        ("max_hits", ctypes.c_uint64),
        ("max_hits_per_layer", ctypes.c_uint32),
        ("n_slots", ctypes.c_uint32),
        ("device", ctypes.c_int32),
        ("tiny_max_layer_hits", ctypes.c_uint32),
        ("flags", ctypes.c_uint32),
    ]


class Stats(ctypes.Structure):
    _fields_ = [
        ("struct_size", ctypes.c_uint32),
        ("n_events", ctypes.c_uint32),
        ("n_hits", ctypes.c_uint64),
        ("n_class", ctypes.c_uint32 * 4),
        ("n_redone", ctypes.c_uint32),
        ("n_invalid", ctypes.c_uint32),
        ("first_invalid", ctypes.c_uint32),
        ("n_launches", ctypes.c_uint32),
        ("kernel_ms", ctypes.c_float * N_KERNELS),
        ("h2d_ms", ctypes.c_float), ("d2h_ms", ctypes.c_float),
    ]

    def as_dict(self):
        return {"n_events": self.n_events, "n_hits": self.n_hits, "n_class": list(self.n_class), "n_redone": self.n_redone,
                "n_invalid": self.n_invalid, "first_invalid": self.first_invalid, "n_launches": self.n_launches,
                "kernel_ms": [float(v) for v in self.kernel_ms], "h2d_ms": float(self.h2d_ms),
                "d2h_ms": float(self.d2h_ms)}


class Ubench(ctypes.Structure):
    _fields_ = [
        ("struct_size", ctypes.c_uint32),
        ("n_sm", ctypes.c_uint32),
        ("alu_lane_ops_per_s", ctypes.c_double),
        ("imad_lane_ops_per_s", ctypes.c_double),
        ("window_evals_per_s", ctypes.c_double),
        ("packed_tests_per_s", ctypes.c_double),
    ]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_ if k != "struct_size"}


class MsdParams(ctypes.Structure):
    _fields_ = [
        ("struct_size", ctypes.c_uint32),
        ("station", ctypes.c_uint32),
        ("thr_x_num", ctypes.c_uint32), ("thr_x_den", ctypes.c_uint32),
        ("thr_y_num", ctypes.c_uint32), ("thr_y_den", ctypes.c_uint32),
        ("ndf", ctypes.c_uint32),
        ("min_triplets", ctypes.c_uint32),
    ]


def make_msd_params(station=None, thr_x=(3, 100), thr_y=(25, 1000), ndf=2, min_triplets=2) -> MsdParams:
    m = MsdParams()
    m.struct_size = ctypes.sizeof(MsdParams)
    m.station = 0xFFFFFFFF if station is None else station
    m.thr_x_num, m.thr_x_den = thr_x
    m.thr_y_num, m.thr_y_den = thr_y
    m.ndf, m.min_triplets = ndf, min_triplets
    return m


class CbmTriggerError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"cbm_trigger error {code}: {msg}")
        self.code = code


_lib = None


def load_library():
    """dlopen libcbmtrigger.so.  Raises if it is missing: the product has no other path."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_1810_11966_b200.build` "
                               "(nvcc, sm_100a); there is no CPU fallback")
        lib = ctypes.CDLL(LIB_PATH)
        vp, u32, u64, i32 = ctypes.c_void_p, ctypes.c_uint32, ctypes.c_uint64, ctypes.c_int
        lib.cbm_trigger_create.restype = i32
        lib.cbm_trigger_create.argtypes = [ctypes.POINTER(Config), ctypes.POINTER(vp)]
        lib.cbm_trigger_destroy.restype = None
        lib.cbm_trigger_destroy.argtypes = [vp]
        lib.cbm_trigger_host_buffers.restype = i32
        lib.cbm_trigger_host_buffers.argtypes = [vp, u32, ctypes.POINTER(vp), ctypes.POINTER(vp), ctypes.POINTER(vp)]
        lib.cbm_trigger_upload_events.restype = i32
        lib.cbm_trigger_upload_events.argtypes = [vp, u32, u32, u64, vp, vp, vp]
        lib.cbm_trigger_host_buffers_packed.restype = i32
        lib.cbm_trigger_host_buffers_packed.argtypes = [vp, u32, ctypes.POINTER(vp), ctypes.POINTER(vp)]
        lib.cbm_trigger_upload_events_packed.restype = i32
        lib.cbm_trigger_upload_events_packed.argtypes = [vp, u32, u32, u64, vp, vp]
        lib.cbm_trigger_run.restype = i32
        lib.cbm_trigger_run.argtypes = [vp, u32]
        lib.cbm_trigger_fetch_results.restype = i32
        lib.cbm_trigger_fetch_results.argtypes = [vp, u32, vp, vp, vp]
        lib.cbm_trigger_run_device.restype = i32
        lib.cbm_trigger_run_device.argtypes = [vp, u32, u64, vp, vp, vp, vp, vp, vp, vp]
        lib.cbm_trigger_device_status.restype = i32
        lib.cbm_trigger_device_status.argtypes = [vp, vp, ctypes.POINTER(Stats)]
        lib.cbm_trigger_device_kernel_times.restype = i32
        lib.cbm_trigger_device_kernel_times.argtypes = [vp, vp, u32, vp]
        lib.cbm_trigger_fetch_selected.restype = i32
        lib.cbm_trigger_fetch_selected.argtypes = [vp, u32, vp, u32, ctypes.POINTER(u32)]
        lib.cbm_trigger_select_device.restype = i32
        lib.cbm_trigger_select_device.argtypes = [vp, u32, vp, vp, vp, vp]
        lib.cbm_trigger_pack_xy20.restype = i32
        lib.cbm_trigger_pack_xy20.argtypes = [vp, vp, u64, vp, ctypes.POINTER(u64)]
        lib.cbm_trigger_select_noalloc.restype = i32
        lib.cbm_trigger_select_noalloc.argtypes = [u32, vp, vp, vp, vp]
        lib.cbm_trigger_gather_device.restype = i32
        lib.cbm_trigger_gather_device.argtypes = [vp, u32, u64, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp]
        lib.cbm_trigger_msd_device.restype = i32
        lib.cbm_trigger_msd_device.argtypes = [vp, ctypes.POINTER(MsdParams), u32, u64, vp, vp, vp, vp, vp, vp]
        lib.cbm_trigger_filter_device.restype = i32
        lib.cbm_trigger_filter_device.argtypes = [vp, u32, u64, vp, vp, vp, vp, vp, vp]
        lib.cbm_trigger_build_events_device.restype = i32
        lib.cbm_trigger_build_events_device.argtypes = [vp, u64, vp, u32, vp, ctypes.POINTER(u32), vp]
        lib.cbm_trigger_ubench.restype = i32
        lib.cbm_trigger_ubench.argtypes = [vp, ctypes.POINTER(Ubench)]
        lib.cbm_trigger_get_stats.restype = i32
        lib.cbm_trigger_get_stats.argtypes = [vp, u32, ctypes.POINTER(Stats)]
        lib.cbm_trigger_last_error.restype = ctypes.c_char_p
        lib.cbm_trigger_last_error.argtypes = [vp]
        lib.cbm_trigger_version.restype = ctypes.c_char_p
        lib.cbm_trigger_version.argtypes = []
        _lib = lib
    return _lib


def make_config(layer_z, max_events, max_hits, win_in=(1, 100), win_link=(2, 100), min_candidates=2,
                max_hits_per_layer=4096, n_slots=2, device=0, tiny_max_layer_hits=0,
                flags=0) -> Config:
    c = Config()
    c.struct_size = ctypes.sizeof(Config)
    c.n_stations = len(layer_z) // 3
    for i, z in enumerate(layer_z[:MAX_LAYERS]):
        c.layer_z[i] = int(z)
    c.win_in_num, c.win_in_den = win_in
    c.win_link_num, c.win_link_den = win_link
    c.min_candidates = min_candidates
    c.max_events, c.max_hits = int(max_events), int(max_hits)
    c.max_hits_per_layer = max_hits_per_layer
    c.n_slots, c.device = n_slots, device
    c.tiny_max_layer_hits, c.flags = tiny_max_layer_hits, flags
    return c


# ------------------------------------------------------------------ the C entry points, same names
def cbm_trigger_version() -> str:
    return load_library().cbm_trigger_version().decode()


def cbm_trigger_last_error(handle) -> str:
    return load_library().cbm_trigger_last_error(handle).decode()


def _check(rc, handle):
    if rc != CBM_OK:
        raise CbmTriggerError(rc, cbm_trigger_last_error(handle))


def cbm_trigger_create(cfg: Config):
    h = ctypes.c_void_p()
    rc = load_library().cbm_trigger_create(ctypes.byref(cfg), ctypes.byref(h))
    _check(rc, None)
    return h


def cbm_trigger_destroy(handle):
    load_library().cbm_trigger_destroy(handle)


def cbm_trigger_host_buffers(handle, slot, max_hits, n_off):
    """numpy views (no copy) of the slot's pinned staging buffers."""
    px, py, po = ctypes.c_void_p(), ctypes.c_void_p(), ctypes.c_void_p()
    _check(load_library().cbm_trigger_host_buffers(handle, slot, ctypes.byref(px), ctypes.byref(py), ctypes.byref(po)),
           handle)
    x = np.ctypeslib.as_array(ctypes.cast(px, ctypes.POINTER(ctypes.c_int32)), shape=(max(int(max_hits), 1),))
    y = np.ctypeslib.as_array(ctypes.cast(py, ctypes.POINTER(ctypes.c_int32)), shape=(max(int(max_hits), 1),))
    off = np.ctypeslib.as_array(ctypes.cast(po, ctypes.POINTER(ctypes.c_uint32)), shape=(int(n_off),))
    return x, y, off


def _host_ptr(a, dtype):
    assert isinstance(a, np.ndarray) and a.dtype == dtype and a.flags.c_contiguous, (type(a), getattr(a, "dtype", None))
    return a.ctypes.data


def cbm_trigger_upload_events(handle, slot, n_events, n_hits, x, y, off):
    _check(load_library().cbm_trigger_upload_events(handle, slot, n_events, n_hits, _host_ptr(x, np.int32),
                                                    _host_ptr(y, np.int32), _host_ptr(off, np.uint32)), handle)


def cbm_trigger_host_buffers_packed(handle, slot, max_hits, n_off):
    """numpy views (no copy) of the slot's pinned staging buffers of the packed wire format XY20."""
    pp, po = ctypes.c_void_p(), ctypes.c_void_p()
    _check(load_library().cbm_trigger_host_buffers_packed(handle, slot, ctypes.byref(pp), ctypes.byref(po)), handle)
    xy = np.ctypeslib.as_array(ctypes.cast(pp, ctypes.POINTER(ctypes.c_uint8)), shape=(max(int(max_hits), 1) * 5,))
    off = np.ctypeslib.as_array(ctypes.cast(po, ctypes.POINTER(ctypes.c_uint32)), shape=(int(n_off),))
    return xy, off


def cbm_trigger_upload_events_packed(handle, slot, n_events, n_hits, xy20, off):
    _check(load_library().cbm_trigger_upload_events_packed(handle, slot, n_events, n_hits, _host_ptr(xy20, np.uint8),
                                                           _host_ptr(off, np.uint32)), handle)


def cbm_trigger_run(handle, slot):
    _check(load_library().cbm_trigger_run(handle, slot), handle)


def cbm_trigger_fetch_results(handle, slot, n_triplets, n_candidates, accept):
    """Fills the caller's numpy arrays.  Returns the C return code (CBM_OK or CBM_ERR_RANGE), raises on others."""
    rc = load_library().cbm_trigger_fetch_results(
        handle, slot, None if n_triplets is None else _host_ptr(n_triplets, np.uint32),
        _host_ptr(n_candidates, np.uint32), None if accept is None else _host_ptr(accept, np.uint8))
    if rc not in (CBM_OK, CBM_ERR_RANGE):
        _check(rc, handle)
    return rc


def cbm_trigger_fetch_selected(handle, slot, event_ids):
    """Fills event_ids (uint32 numpy array = the capacity); returns the number of selected events."""
    n = ctypes.c_uint32(0)
    rc = load_library().cbm_trigger_fetch_selected(handle, slot, _host_ptr(event_ids, np.uint32) if event_ids.size else None,
                                                   event_ids.size, ctypes.byref(n))
    _check(rc, handle)
    return int(n.value)


def cbm_trigger_select_device(handle, n_events, d_accept, d_event_ids, d_n_selected, stream=0):
    """d_* are raw device addresses (ints); stream is a cudaStream_t as int."""
    _check(load_library().cbm_trigger_select_device(handle, n_events, d_accept, d_event_ids, d_n_selected, stream), handle)


def cbm_trigger_pack_xy20(x, y, out=None):
    """The library's host packer of the wire format XY20 (no CUDA): int32 numpy arrays -> 5 bytes per hit.  `out` may be
    a slot's pinned buffer (cbm_trigger_host_buffers_packed).  Raises CbmTriggerError(CBM_ERR_RANGE) for a coordinate
    outside the 20-bit range; the exception carries `first_bad`."""
    n = int(x.size)
    if out is None:
        out = np.empty(5 * n, dtype=np.uint8)
    assert out.dtype == np.uint8 and out.flags.c_contiguous and out.size >= 5 * n
    bad = ctypes.c_uint64(0)
    rc = load_library().cbm_trigger_pack_xy20(_host_ptr(x, np.int32), _host_ptr(y, np.int32), n, out.ctypes.data, ctypes.byref(bad))
    if rc != CBM_OK:
        err = CbmTriggerError(rc, cbm_trigger_last_error(None))
        err.first_bad = int(bad.value)
        raise err
    return out[:5 * n]


NOALLOC_MAX_EVENTS = 1 << 24  # CBM_TRIGGER_NOALLOC_MAX_EVENTS


def cbm_trigger_select_noalloc(n_events, d_accept, d_event_ids, d_n_selected, stream=0):
    """The list of selected events without a handle and without any allocation, for callers that may not allocate
    device memory (a readout loop after start of run, a plug-in that only gets pointers and a stream): same result as
    cbm_trigger_select_device.  d_* are raw device addresses (ints) on the current device; stream is a cudaStream_t
    as int.  At most NOALLOC_MAX_EVENTS events; calls on one device share one fixed scratch array, so they must not
    overlap on the GPU (include/cbm_trigger.h)."""
    _check(load_library().cbm_trigger_select_noalloc(n_events, d_accept, d_event_ids, d_n_selected, stream), None)


def cbm_trigger_gather_device(handle, n_events, n_hits, d_x, d_y, d_off, d_ids, d_n_sel, d_out_x, d_out_y, d_out_off,
                              d_out_n_hits, stream=0):
    """d_* are raw device addresses (ints); stream is a cudaStream_t as int."""
    _check(load_library().cbm_trigger_gather_device(handle, n_events, n_hits, d_x, d_y, d_off, d_ids, d_n_sel, d_out_x, d_out_y,
                                                    d_out_off, d_out_n_hits, stream), handle)


def cbm_trigger_filter_device(handle, n_events, n_records, d_xyz, d_ev_off, d_out_x, d_out_y, d_out_off, stream=0):
    """d_* are raw device addresses (ints); stream is a cudaStream_t as int."""
    _check(load_library().cbm_trigger_filter_device(handle, n_events, n_records, d_xyz, d_ev_off, d_out_x, d_out_y, d_out_off,
                                                    stream), handle)


def cbm_trigger_build_events_device(handle, n_records, d_t, t_gap, d_ev_off, stream=0) -> int:
    """d_* are raw device addresses (ints); blocks; returns the number of events built."""
    n = ctypes.c_uint32(0)
    _check(load_library().cbm_trigger_build_events_device(handle, n_records, d_t, t_gap, d_ev_off, ctypes.byref(n), stream), handle)
    return int(n.value)


def cbm_trigger_ubench(handle) -> dict:
    """The integer-pipe micro-benchmarks (blocking); returns the rates as a dict."""
    u = Ubench()
    u.struct_size = ctypes.sizeof(Ubench)
    _check(load_library().cbm_trigger_ubench(handle, ctypes.byref(u)), handle)
    return u.as_dict()


def cbm_trigger_msd_device(handle, params, n_events, n_hits, d_x, d_y, d_off, d_n_passing, d_accept, stream=0):
    """d_* are raw device addresses (ints); stream is a cudaStream_t as int."""
    _check(load_library().cbm_trigger_msd_device(handle, ctypes.byref(params), n_events, n_hits, d_x, d_y, d_off,
                                                 d_n_passing, d_accept, stream), handle)


def cbm_trigger_get_stats(handle, slot) -> Stats:
    st = Stats()
    _check(load_library().cbm_trigger_get_stats(handle, slot, ctypes.byref(st)), handle)
    return st


def cbm_trigger_run_device(handle, n_events, n_hits, d_x, d_y, d_off, d_n_triplets, d_n_candidates, d_accept,
                           stream=0):
    """d_* are raw device addresses (ints); stream is a cudaStream_t as int."""
    _check(load_library().cbm_trigger_run_device(handle, n_events, n_hits, d_x, d_y, d_off, d_n_triplets,
                                                 d_n_candidates, d_accept, stream), handle)


def cbm_trigger_device_status(handle, stream=0):
    st = Stats()
    rc = load_library().cbm_trigger_device_status(handle, stream, ctypes.byref(st))
    if rc not in (CBM_OK, CBM_ERR_RANGE):
        _check(rc, handle)
    return rc, st


def cbm_trigger_device_kernel_times(handle, stream=0, n_last=PROFILE_RING):
    """(n, N_KERNELS) float32 array: device ms of every kernel of the last n run_device calls, oldest first."""
    buf = np.zeros((PROFILE_RING, N_KERNELS), dtype=np.float32)
    n = load_library().cbm_trigger_device_kernel_times(handle, stream, min(n_last, PROFILE_RING), buf.ctypes.data)
    if n < 0:
        _check(n, handle)
    return buf[:n]


# ------------------------------------------------------------------ convenience wrapper
class Trigger:
    """Owns one handle.  Host-path: upload/run/fetch on slots.  Device path: run_device on torch tensors."""

    def __init__(self, layer_z, max_events, max_hits, **kw):
        self.cfg = make_config(layer_z, max_events, max_hits, **kw)
        self.S = self.cfg.n_stations
        self.L = 3 * self.S
        self.handle = cbm_trigger_create(self.cfg)

    def close(self):
        if self.handle is not None:
            cbm_trigger_destroy(self.handle)
            self.handle = None

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def host_buffers(self, slot):
        return cbm_trigger_host_buffers(self.handle, slot, self.cfg.max_hits, self.cfg.max_events * self.L + 1)

    def upload_events(self, slot, x, y, off, n_events=None, n_hits=None):
        n_events = (off.size - 1) // self.L if n_events is None else n_events
        n_hits = int(off[n_events * self.L]) if n_hits is None else n_hits
        cbm_trigger_upload_events(self.handle, slot, n_events, n_hits, x, y, off)
        return n_events, n_hits

    def host_buffers_packed(self, slot):
        return cbm_trigger_host_buffers_packed(self.handle, slot, self.cfg.max_hits, self.cfg.max_events * self.L + 1)

    def upload_events_packed(self, slot, xy20, off, n_events=None, n_hits=None):
        n_events = (off.size - 1) // self.L if n_events is None else n_events
        n_hits = int(off[n_events * self.L]) if n_hits is None else n_hits
        cbm_trigger_upload_events_packed(self.handle, slot, n_events, n_hits, xy20, off)
        return n_events, n_hits

    def run(self, slot):
        cbm_trigger_run(self.handle, slot)

    def fetch_results(self, slot, n_events, out=None, check=True):
        if out is None:
            out = (np.empty((n_events, self.S), dtype=np.uint32), np.empty(n_events, dtype=np.uint32),
                   np.empty(n_events, dtype=np.uint8))
        rc = cbm_trigger_fetch_results(self.handle, slot, out[0], out[1], out[2])
        if check and rc != CBM_OK:
            raise CbmTriggerError(rc, cbm_trigger_last_error(self.handle))
        return out if check else (out, rc)

    def stats(self, slot) -> Stats:
        return cbm_trigger_get_stats(self.handle, slot)

    def fetch_selected(self, slot, capacity=None):
        """Ascending ids of the accepted events of the slot's last run."""
        ids = np.empty(self.cfg.max_events if capacity is None else capacity, dtype=np.uint32)
        n = cbm_trigger_fetch_selected(self.handle, slot, ids)
        return ids[:n].copy()

    def select_device(self, n_events, d_ac, d_ids, d_n, stream=None):
        import torch
        st = torch.cuda.current_stream().cuda_stream if stream is None else stream
        cbm_trigger_select_device(self.handle, n_events, d_ac.data_ptr(), d_ids.data_ptr(), d_n.data_ptr(), st)

    def select(self, x, y, off, slot=0):
        """upload + run + fetch of one host batch (numpy arrays)."""
        n_events, _ = self.upload_events(slot, x, y, off)
        self.run(slot)
        return self.fetch_results(slot, n_events)

    def run_device(self, n_events, n_hits, d_x, d_y, d_off, d_nt, d_nc, d_ac, stream=None):
        """torch CUDA tensors in, torch CUDA tensors out (PyTorch supplies memory and the stream)."""
        import torch
        st = torch.cuda.current_stream().cuda_stream if stream is None else stream
        cbm_trigger_run_device(self.handle, n_events, n_hits, d_x.data_ptr(), d_y.data_ptr(), d_off.data_ptr(),
                               d_nt.data_ptr(), d_nc.data_ptr(), d_ac.data_ptr(), st)

    def gather_device(self, n_events, n_hits, d_x, d_y, d_off, d_ids, d_n, d_ox, d_oy, d_ooff, d_on, stream=None):
        """The selected events' hits as a compact batch (torch CUDA tensors)."""
        import torch
        st = torch.cuda.current_stream().cuda_stream if stream is None else stream
        cbm_trigger_gather_device(self.handle, n_events, n_hits, d_x.data_ptr(), d_y.data_ptr(), d_off.data_ptr(), d_ids.data_ptr(),
                                  d_n.data_ptr(), d_ox.data_ptr(), d_oy.data_ptr(), d_ooff.data_ptr(), d_on.data_ptr(), st)

    def filter_device(self, n_events, n_records, d_xyz, d_ev_off, d_ox, d_oy, d_ooff, stream=None):
        """The input filter on torch CUDA tensors: full-setup records -> the batch layout."""
        import torch
        st = torch.cuda.current_stream().cuda_stream if stream is None else stream
        cbm_trigger_filter_device(self.handle, n_events, n_records, d_xyz.data_ptr(), d_ev_off.data_ptr(), d_ox.data_ptr(),
                                  d_oy.data_ptr(), d_ooff.data_ptr(), st)

    def build_events_device(self, n_records, d_t, t_gap, d_ev_off, stream=None) -> int:
        """Event building from time stamps on torch CUDA tensors; returns the number of events."""
        import torch
        st = torch.cuda.current_stream().cuda_stream if stream is None else stream
        return cbm_trigger_build_events_device(self.handle, n_records, d_t.data_ptr(), t_gap, d_ev_off.data_ptr(), st)

    def ubench(self) -> dict:
        return cbm_trigger_ubench(self.handle)

    def msd_device(self, params, n_events, n_hits, d_x, d_y, d_off, d_np, d_ac, stream=None):
        """The paper-literal selection on torch CUDA tensors."""
        import torch
        st = torch.cuda.current_stream().cuda_stream if stream is None else stream
        cbm_trigger_msd_device(self.handle, params, n_events, n_hits, d_x.data_ptr(), d_y.data_ptr(), d_off.data_ptr(),
                               d_np.data_ptr(), d_ac.data_ptr(), st)

    def device_kernel_times(self, stream=None, n_last=PROFILE_RING):
        import torch
        st = torch.cuda.current_stream().cuda_stream if stream is None else stream
        return cbm_trigger_device_kernel_times(self.handle, st, n_last)

    def device_status(self, stream=None):
        import torch
        st = torch.cuda.current_stream().cuda_stream if stream is None else stream
        return cbm_trigger_device_status(self.handle, st)
