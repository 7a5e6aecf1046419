"""Shared helpers of the parity tests: a multi-threaded driver of the CPU oracle (events are
independent) and a one-call wrapper of the CUDA path through the C ABI."""
import os
from concurrent.futures import ThreadPoolExecutor

import numpy as np

import oracle
from paper_1810_11966_b200 import binding as K


def oracle_mt(geo, x, y, off, e_begin=0, e_end=None, n_threads=None, chunk=2000):
    """oracle.run over [e_begin, e_end) on all host cores (ctypes releases the GIL)."""
    S = geo.n_stations
    n_events = (off.size - 1) // (3 * S)
    e_end = n_events if e_end is None else e_end
    n = e_end - e_begin
    nt = np.zeros((n, S), dtype=np.uint32)
    nc = np.zeros(n, dtype=np.uint32)
    ac = np.zeros(n, dtype=np.uint8)
    n_threads = n_threads or min(32, os.cpu_count() or 1)
    ranges = [(a, min(a + chunk, e_end)) for a in range(e_begin, e_end, chunk)]

    def work(r):
        a, b = r
        t, c, k = oracle.run(geo, x, y, off, a, b)
        nt[a - e_begin:b - e_begin] = t
        nc[a - e_begin:b - e_begin] = c
        ac[a - e_begin:b - e_begin] = k

    with ThreadPoolExecutor(n_threads) as ex:
        list(ex.map(work, ranges))
    return nt, nc, ac


def gpu_select(layer_z, x, y, off, win_in=(1, 100), win_link=(2, 100), min_candidates=2, max_hits_per_layer=4096,
               flags=0, tiny_max_layer_hits=0, check=True):
    """One batch through cbm_trigger_create / upload_events / run / fetch_results."""
    L = len(layer_z)
    n_events = (off.size - 1) // L
    n_hits = int(off[-1])
    trig = K.Trigger(layer_z, max(n_events, 1), max(n_hits, 1), win_in=win_in, win_link=win_link,
                     min_candidates=min_candidates, max_hits_per_layer=max_hits_per_layer, n_slots=1, flags=flags,
                     tiny_max_layer_hits=tiny_max_layer_hits)
    try:
        x = np.ascontiguousarray(x, dtype=np.int32)
        y = np.ascontiguousarray(y, dtype=np.int32)
        off = np.ascontiguousarray(off, dtype=np.uint32)
        trig.upload_events(0, x, y, off, n_events, n_hits)
        trig.run(0)
        if check:
            out = trig.fetch_results(0, n_events)
            return out + (trig.stats(0).as_dict(),)
        out, rc = trig.fetch_results(0, n_events, check=False)
        return out + (trig.stats(0).as_dict(), rc, K.cbm_trigger_last_error(trig.handle))
    finally:
        trig.close()


def assert_same(got, want, what=""):
    for name, g, w in zip(("n_triplets", "n_candidates", "accept"), got[:3], want[:3]):
        g = np.asarray(g)
        w = np.asarray(w).reshape(g.shape)
        if not np.array_equal(g, w):
            bad = np.argwhere(g != w)
            first = tuple(bad[0])
            raise AssertionError(f"{what}: {name} differs at {len(bad)} places; first {first}: gpu {g[first]} oracle {w[first]}")


def oracle_msd_mt(par, x, y, off, n_threads=None, chunk=20000):
    """oracle.run_msd over all events on all host cores."""
    n_events = (off.size - 1) // (3 * par.n_stations)
    npass = np.zeros(n_events, dtype=np.uint32)
    ac = np.zeros(n_events, dtype=np.uint8)
    n_threads = n_threads or min(32, os.cpu_count() or 1)
    ranges = [(a, min(a + chunk, n_events)) for a in range(0, n_events, chunk)]

    def work(r):
        a, b = r
        npass[a:b], ac[a:b] = oracle.run_msd(par, x, y, off, a, b)

    with ThreadPoolExecutor(n_threads) as ex:
        list(ex.map(work, ranges))
    return npass, ac


def device_run(cfg, b, flags=0):
    """One batch through cbm_trigger_run_device on torch-owned device arrays (bench.py's launch configuration).
    Returns (n_triplets[E][S], n_candidates[E], accept[E], stats dict)."""
    import torch
    E, S = b.n_events, cfg.n_stations
    dev = torch.device("cuda:0")
    pad = (-b.n_hits) % 4 + 4
    dx = torch.zeros(b.n_hits + pad, dtype=torch.int32, device=dev)
    dy = torch.zeros(b.n_hits + pad, dtype=torch.int32, device=dev)
    dx[:b.n_hits] = torch.from_numpy(b.x).to(dev)
    dy[:b.n_hits] = torch.from_numpy(b.y).to(dev)
    doff = torch.from_numpy(b.off.view(np.int32)).to(dev)
    dnt = torch.full((E * S,), -1, dtype=torch.int32, device=dev)
    dnc = torch.full((E,), -1, dtype=torch.int32, device=dev)
    dac = torch.full((E,), 255, dtype=torch.uint8, device=dev)
    with K.Trigger(cfg.layer_z, E, b.n_hits, win_in=cfg.win_in, win_link=cfg.win_link, min_candidates=cfg.min_candidates,
                   max_hits_per_layer=cfg.max_hits_per_layer, n_slots=0, flags=flags) as trig:
        trig.run_device(E, b.n_hits, dx, dy, doff, dnt, dnc, dac)
        rc, st = trig.device_status()
        assert rc == K.CBM_OK
    return (dnt.cpu().numpy().view(np.uint32).reshape(-1, S), dnc.cpu().numpy().view(np.uint32), dac.cpu().numpy(), st.as_dict())
