"""bench.py -- throughput of the CBM-MUCH first-level J/psi selection on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl ours|reference]

A "step" is one pass of the whole hot path (a3..a8: classify, stage, triplet search, compaction, linking,
decision, result write) over one synthetic timeslice batch.  Default workload: BASELINE.json
configs[3] (load-imbalance stress, 1,000,000 events) -- the configuration the north_star's roofline target
is stated on.  `value` is measured with the batch resident in HBM (cbm_trigger_run_device);
`e2e` is measured through cbm_trigger_upload_events / run / fetch_results with pinned HOST buffers, the
H2D and D2H copies inside the timed region, two slots in flight.

Prints ONE JSON line (rank 0).  `--impl reference` times the CPU oracle (oracle/) on the host cores.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "events_per_second"
UNIT = "events/s"
CBM_INTERACTION_RATE_HZ = 1.0e7


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json configs index (0..3; 4 = streaming of config-2 chunks)")
    ap.add_argument("--events", type=int, default=0, help="events per batch (0 = the config's size)")
    ap.add_argument("--e2e-steps", type=int, default=0, help="steps of the end-to-end leg (0 = min(steps, 10))")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--serial", action="store_true", help="CBM_FLAG_SERIAL: the kernels of a step one after the other")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-packed", action="store_true", help="skip the end-to-end leg with the packed wire format XY20")
    return ap.parse_args()


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            with open(path) as f:
                return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""

    QUERY = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")

    def __init__(self, device_index=0):
        self.device_index = device_index
        self.samples = []
        self.proc = None
        self.thread = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.device_index}", f"--query-gpu={self.QUERY}", "--format=csv,noheader,nounits",
                 "-lms", "20"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._read, daemon=True)
        self.thread.start()

    def _read(self):
        for line in self.proc.stdout:
            parts = [p.strip() for p in line.split(",")]
            if len(parts) >= 7:
                self.samples.append((time.perf_counter(), parts))

    def stop(self, t0=None, t1=None):
        """Samples taken inside the timed region [t0, t1] (host clock); if the region was shorter than the
        sampling interval, the samples of the surrounding loaded phase (warm-up included) are used."""
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        inside = [p for (t, p) in self.samples if t0 is not None and t0 <= t <= t1 + 0.03]
        window = "timed region"
        if len(inside) < 2:
            inside, window = [p for (_, p) in self.samples], "warm-up + timed region"
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        self.window = window
        for p in inside:
            try:
                sm.append(float(p[0]))
                mx.append(float(p[1]))
            except ValueError:
                continue
            for name, v in zip(names, p[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm), "window": window}


# ---------------------------------------------------------------------------------------------- accounting
def algorithmic_bytes(n_events, n_hits, S):
    """hits read once (8 B), offsets read once, results written once."""
    L = 3 * S
    return 8 * n_hits + 4 * (n_events * L + 1) + n_events * (4 * S + 5)


def class_accounting(off, S, tiny_max_layer, tiny_max_total, caps):
    """Events, hits and algorithmic bytes per scheduler class (tile, team_M, team_H, team_G), from the offsets.
    Restates the scheduler's rule for the roofline bookkeeping only; the counts are
    checked against the library's own statistics."""
    L = 3 * S
    n_events = (off.size - 1) // L
    cnt = np.diff(off.astype(np.int64)).reshape(n_events, L)
    mx = cnt.max(axis=1) if n_events else np.zeros(0, dtype=np.int64)
    tot = cnt.sum(axis=1)
    cls = np.full(n_events, 3, dtype=np.int64)
    cls[mx <= caps[1]] = 2
    cls[mx <= caps[0]] = 1
    cls[(mx <= tiny_max_layer) & (tot <= tiny_max_total)] = 0
    out = []
    for c in range(4):
        sel = cls == c
        ne, nh = int(sel.sum()), int(tot[sel].sum())
        out.append({"events": ne, "hits": nh, "bytes": 8 * nh + ne * (4 * L + 4 * S + 5)})
    return out


def oracle_events_per_second(cfg, batch, n_sample, n_threads):
    """The CPU oracle, as it stands, on the first n_sample events of the batch over n_threads host threads
    (events are independent: the paper's pthread scheme)."""
    from concurrent.futures import ThreadPoolExecutor
    import oracle
    g = oracle.geometry(cfg.layer_z, cfg.win_in, cfg.win_link, cfg.min_candidates)
    n_sample = min(n_sample, batch.n_events)
    chunk = max(1, min(2000, n_sample // (4 * n_threads) or 1))
    ranges = [(a, min(a + chunk, n_sample)) for a in range(0, n_sample, chunk)]
    oracle.run(g, batch.x, batch.y, batch.off, 0, min(64, n_sample))  # load the library outside the timing
    t0 = time.perf_counter()
    with ThreadPoolExecutor(n_threads) as ex:
        acc = sum(int(r[2].sum()) for r in ex.map(lambda r: oracle.run(g, batch.x, batch.y, batch.off, r[0], r[1]), ranges))
    dt = time.perf_counter() - t0
    return n_sample / dt, dt, acc


def cpu_sample_size(cid):
    # about 10-30 s of CPU work at the oracle's measured single-core rates
    return {0: 1000, 1: 200_000, 2: 100_000, 3: 500_000, 4: 100_000}[cid]


def run_reference(args, cfg, cid):
    """--impl reference: the oracle on the host cores, each step a bounded sample of the same workload."""
    from paper_1810_11966_b200 import workloads as W
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    n_threads = os.cpu_count() or 1
    n_events = args.events or (cfg.chunk_events or cfg.n_events)
    per_step = max(1, min(n_events, cpu_sample_size(cid) // 4))
    batch = W.generate(cfg, n_events=per_step)
    for _ in range(args.warmup):
        oracle_events_per_second(cfg, batch, max(1, per_step // 8), n_threads)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle_events_per_second(cfg, batch, per_step, n_threads)
    dt = time.perf_counter() - t0
    value = per_step * args.steps / dt
    sample = f"first {per_step} events of {cfg.name} per step, oracle/cbm_oracle.c over {n_threads} threads"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "int64", "data": "synthetic",
        "config": {"workload": cfg.name, "events_per_step": per_step, "hits_per_step": batch.n_hits},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": n_threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "hits_per_second": batch.n_hits * args.steps / dt,
    }))


# ---------------------------------------------------------------------------------------------- multi-rank
def rank_event_range(rank, events_per_rank):
    """Events are independent: rank r owns the contiguous range
    [r*E, (r+1)*E) of the synthetic event stream -- weak scaling, no exchange step, no collective
    in the data path (replicas only)."""
    return rank * events_per_rank, (rank + 1) * events_per_rank


def reduce_over_ranks(dist, device, times, counts):
    """Whole-job bookkeeping of one bench run: MAX over ranks of every entry of `times` (device
    time of the slowest rank), SUM over ranks of every entry of `counts` (events, hits).
    `dist` is torch.distributed or None (single process)."""
    import torch
    t = torch.tensor([float(v) for v in times], dtype=torch.float64, device=device)
    c = torch.tensor([float(v) for v in counts], dtype=torch.float64, device=device)
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(c, op=dist.ReduceOp.SUM)
    return [float(v) for v in t], [float(v) for v in c]


def whole_job_rate(total_units, steps, seconds_max):
    """`value` of the JSON line: units all ranks processed / time of the slowest rank."""
    return total_units * steps / seconds_max


# ---------------------------------------------------------------------------------------------- our arm
def to_device_padded(torch, a, dev):
    """int32 device copy with the 16-byte tail padding the staging copies may over-read."""
    n = a.size
    t = torch.zeros(n + ((-n) % 4) + 4, dtype=torch.int32, device=dev)
    t[:n] = torch.from_numpy(a.view(np.int32)).to(dev)
    return t


def run_ours(args, cfg, cid):
    import torch
    from paper_1810_11966_b200 import binding as K
    from paper_1810_11966_b200 import workloads as W

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product has no CPU path (use --impl reference for the oracle)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- workload: each rank owns its own batch (weak scaling; events are independent, no collective)
    E = args.events or (cfg.chunk_events or cfg.n_events)
    S = cfg.n_stations
    t_gen = time.perf_counter()
    batch = W.generate(cfg, n_events=E, first_event=rank_event_range(rank, E)[0])
    t_gen = time.perf_counter() - t_gen
    n_hits = batch.n_hits
    B_alg = algorithmic_bytes(E, n_hits, S)

    dx = to_device_padded(torch, batch.x, dev)
    dy = to_device_padded(torch, batch.y, dev)
    doff = torch.from_numpy(batch.off.view(np.int32)).to(dev)
    dnt = torch.zeros(E * S, dtype=torch.int32, device=dev)
    dnc = torch.zeros(E, dtype=torch.int32, device=dev)
    dac = torch.zeros(E, dtype=torch.uint8, device=dev)

    trig = K.Trigger(cfg.layer_z, E, n_hits, win_in=cfg.win_in, win_link=cfg.win_link,
                     min_candidates=cfg.min_candidates, max_hits_per_layer=cfg.max_hits_per_layer, n_slots=0,
                     device=local_rank, flags=K.CBM_FLAG_PROFILE | (K.CBM_FLAG_SERIAL if args.serial else 0))
    stream = torch.cuda.Stream(device=dev)
    sampler = ClockSampler(local_rank)
    sampler.start()  # nvidia-smi needs ~0.1 s to deliver its first sample: started before the warm-up
    with torch.cuda.stream(stream):
        t_load = time.perf_counter()
        n_warm = 0
        while n_warm < args.warmup or (time.perf_counter() - t_load < 0.25 and n_warm < 1000):
            trig.run_device(E, n_hits, dx, dy, doff, dnt, dnc, dac)  # untimed: W steps, and at least 0.25 s of load
            n_warm += 1
            if n_warm >= args.warmup:
                torch.cuda.synchronize()
        rc, st = trig.device_status()
        if rc != K.CBM_OK:
            raise SystemExit("bench.py: the device rejected events of a generated batch")
        barrier()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t_region0 = time.perf_counter()
        ev0.record(stream)
        for _ in range(args.steps):
            trig.run_device(E, n_hits, dx, dy, doff, dnt, dnc, dac)
        ev1.record(stream)
        barrier()
        clocks = sampler.stop(t_region0, time.perf_counter())
        ms_total = ev0.elapsed_time(ev1)
        ktimes = trig.device_kernel_times(n_last=args.steps)
    n_accept = int(dac.sum().item())
    n_cand_events = int((dnc != 0).sum().item())
    stats = st.as_dict()
    trig.close()

    # ---- end-to-end leg: pinned HOST buffers -> H2D -> kernels -> D2H, two slots in flight
    e2e = e2e_packed = None
    if not args.no_e2e:
        e2e = run_e2e(args, cfg, cid, batch, K, W, local_rank, rank, barrier)
        if not args.no_packed:
            e2e_packed = run_e2e(args, cfg, cid, batch, K, W, local_rank, rank, barrier, packed=True)
    del dx, dy, doff

    # max over ranks (device time), whole-job aggregate
    (ms_total_max, e2e_s_max), (events_all, hits_all) = reduce_over_ranks(
        dist, dev, [ms_total, e2e["seconds"] if e2e else 0.0], [E, n_hits])
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    if rank != 0:
        return

    ms_per_step = ms_total_max / args.steps
    value = whole_job_rate(events_all, args.steps, ms_total_max * 1e-3)
    peak, peak_src = measured_peaks()

    # ---- roofline of the dominant kernel: algorithmic bytes of the events it processes / its mean launch time
    acct = class_accounting(batch.off, S, K.TINY_MAX_LAYER_DEFAULT, K.TINY_MAX_TOTAL, K.CLASS_CAPS)
    kmean = ktimes.mean(axis=0) if len(ktimes) else np.zeros(K.N_KERNELS)
    # kernels: classify (reads every event's offsets), tile, team_M, team_H, team_G, team_X (events handed on)
    zero = {"events": 0, "hits": 0, "bytes": 0}
    acct = [{"events": E, "hits": 0, "bytes": 4 * (E * 3 * S + 1)}] + acct + [zero]
    kbytes = [a["bytes"] for a in acct]
    # dominant kernel = the one that moves the most algorithmic bytes.  (The three class kernels run side by
    # side on their own streams after the tile kernel, so the event-to-event time of a small class also counts
    # its wait for SMs; the times of the tile kernel and of the dominant class kernel are their own.)
    dom = int(np.argmax(kbytes))
    dom_ms = float(kmean[dom])
    achieved = kbytes[dom] / (dom_ms * 1e-3) / 1e9 if dom_ms > 0 else 0.0
    roofline = {"bound": "hbm", "kernel": K.KERNEL_NAMES[dom], "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": NCU_TRAFFIC_BYTES.get((cfg.name, K.KERNEL_NAMES[dom])),
                "peak_source": peak_src, "algorithmic_bytes_per_launch": kbytes[dom], "ms_per_launch": dom_ms,
                "share_of_step": dom_ms / ms_per_step if ms_per_step > 0 else None}
    step_gbs = B_alg / (ms_per_step * 1e-3) / 1e9
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "int64", "data": "synthetic",
        "config": {"workload": cfg.name, "baseline_config_index": cid, "events_per_batch": E, "hits_per_batch": n_hits,
                   "stations": S, "bytes_per_batch": B_alg, "l2": "inputs larger than L2 (no flush needed)"
                   if B_alg > 200e6 else "inputs smaller than L2: L2-resident between steps", "parallelism": f"replicas x{world}"},
        "hits_per_second": hits_all * args.steps / (ms_total_max * 1e-3),
        "vs_10MHz": value / CBM_INTERACTION_RATE_HZ,
        "gpu_launches": K.N_KERNELS * args.steps,
        "kernels": {name: {"ms": float(kmean[i]), "events": acct[i]["events"], "hits": acct[i]["hits"],
                           "algorithmic_bytes": kbytes[i]} for i, name in enumerate(K.KERNEL_NAMES)},
        "classes": stats["n_class"], "accepted_events": n_accept, "events_with_candidates": n_cand_events,
        "roofline": roofline,
        "roofline_step": {"bound": "hbm", "achieved": step_gbs, "peak": peak, "unit": "GB/s", "frac": step_gbs / peak,
                          "frac_of_8TBs_nominal": step_gbs / 8000.0, "algorithmic_bytes_per_step": B_alg},
        "clocks": clocks, "warmup_steps_run": n_warm, "generation_s": t_gen,
    }
    if e2e:
        e2e_value = whole_job_rate(events_all, e2e["steps"], e2e_s_max)
        out["e2e"] = {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": e2e["h2d_bytes"],
                      "d2h_bytes_per_step": e2e["d2h_bytes"], "steps": e2e["steps"], "slots": 2,
                      "ms_per_step": 1e3 * e2e_s_max / e2e["steps"], "h2d_gbs": e2e["h2d_bytes"] * e2e["steps"] / e2e_s_max / 1e9,
                      "vs_10MHz": e2e_value / CBM_INTERACTION_RATE_HZ, "h2d_ms_last": e2e["h2d_ms"], "kernel_ms_last": e2e["kernel_ms"]}
    if e2e_packed and world == 1:  # extra: the same pipeline fed with the 5-byte-per-hit wire format
        v = whole_job_rate(E, e2e_packed["steps"], e2e_packed["seconds"])
        out["e2e_packed_xy20"] = {"value": v, "unit": UNIT, "h2d_bytes_per_step": e2e_packed["h2d_bytes"],
                                  "d2h_bytes_per_step": e2e_packed["d2h_bytes"], "steps": e2e_packed["steps"],
                                  "ms_per_step": 1e3 * e2e_packed["seconds"] / e2e_packed["steps"],
                                  "h2d_gbs": e2e_packed["h2d_bytes"] * e2e_packed["steps"] / e2e_packed["seconds"] / 1e9,
                                  "vs_10MHz": v / CBM_INTERACTION_RATE_HZ, "accepted": e2e_packed["accepted"]}
    if world == 1 and not args.no_cpu_baseline:
        n_threads = os.cpu_count() or 1
        n_sample = min(E, cpu_sample_size(cid))
        v, dt, _ = oracle_events_per_second(cfg, batch, n_sample, n_threads)
        out["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": n_threads, "kind": "oracle", "seconds": dt,
                               "sample": f"first {n_sample} events of the same batch, oracle/cbm_oracle.c over {n_threads} threads"}
    print(json.dumps(out))


# per-launch DRAM traffic (dram__bytes_read.sum + dram__bytes_write.sum) of one `ncu --set full` capture,
# copied by hand from profiles/ (see the .md there); None until a capture exists for that kernel.
NCU_TRAFFIC_BYTES = {
    ("cfg3_imbalance", "team_kernel_H"): 1_754_425_000 + 8_558_848,   # profiles/r1_team_kernel_H.md
    ("cfg3_imbalance", "tile_kernel"): 519_462_144 + 20_825_856,      # profiles/r1_tile_kernel.md
}


def run_e2e(args, cfg, cid, batch, K, W, local_rank, rank, barrier, packed=False):
    """K2 batches through upload_events / run / fetch_results, inputs in the slots' pinned HOST buffers
    (cbm_trigger_host_buffers: the producer writes there), two slots in flight so that the H2D of batch i+1
    overlaps the kernels and the D2H of batch i.  Wall clock between device synchronisations."""
    import torch
    E, S, L = batch.n_events, cfg.n_stations, cfg.n_layers
    steps = args.e2e_steps or min(max(args.steps, 2), 10)
    batches = [batch]
    if cfg.chunk_events:  # config 4: distinct chunks in the two slots
        batches.append(W.generate(cfg, n_events=E, first_event=(rank + 1) * E + 7 * E))
    max_hits = max(b.n_hits for b in batches)
    trig = K.Trigger(cfg.layer_z, E, max_hits, win_in=cfg.win_in, win_link=cfg.win_link,
                     min_candidates=cfg.min_candidates, max_hits_per_layer=cfg.max_hits_per_layer, n_slots=2,
                     device=local_rank, flags=K.CBM_FLAG_PROFILE | (K.CBM_FLAG_PACKED_INPUT if packed else 0))
    bufs, nh = [], []
    for s in (0, 1):  # the producer (DAQ / generator) writes the batch into the slot's pinned staging, untimed
        b = batches[s % len(batches)]
        if packed:
            hp, ho = trig.host_buffers_packed(s)
            hp[:5 * b.n_hits] = W.pack_xy20(b.x, b.y)
            ho[:b.off.size] = b.off
            bufs.append((hp, ho))
        else:
            hx, hy, ho = trig.host_buffers(s)
            hx[:b.n_hits] = b.x
            hy[:b.n_hits] = b.y
            ho[:b.off.size] = b.off
            bufs.append((hx, hy, ho))
        nh.append(b.n_hits)
    out = [(np.empty((E, S), dtype=np.uint32), np.empty(E, dtype=np.uint32), np.empty(E, dtype=np.uint8)) for _ in (0, 1)]

    def pipeline(n):
        for i in range(n):
            s = i & 1
            if i >= 2:
                trig.fetch_results(s, E, out=out[s])
            if packed:
                trig.upload_events_packed(s, bufs[s][0], bufs[s][1], E, nh[s])
            else:
                trig.upload_events(s, bufs[s][0], bufs[s][1], bufs[s][2], E, nh[s])
            trig.run(s)
        for i in range(max(0, n - 2), n):
            trig.fetch_results(i & 1, E, out=out[i & 1])

    pipeline(max(2, min(args.warmup, 3)))
    barrier()
    t0 = time.perf_counter()
    pipeline(steps)
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    st = trig.stats(0)
    hit_bytes = 20 * ((nh[0] + 3) // 4) if packed else 8 * nh[0]
    res = {"seconds": dt, "steps": steps, "h2d_bytes": hit_bytes + 4 * (E * L + 1), "d2h_bytes": E * (4 * S + 5) + 64 + 4,
           "h2d_ms": float(st.h2d_ms), "kernel_ms": [float(v) for v in st.kernel_ms], "accepted": int(out[0][2].sum())}
    trig.close()
    return res


def main():
    args = parse_args()
    from paper_1810_11966_b200 import workloads as W
    cfg = W.CONFIGS[args.config]
    if args.impl == "reference":
        run_reference(args, cfg, args.config)
    else:
        run_ours(args, cfg, args.config)


if __name__ == "__main__":
    main()
