"""bench.py -- throughput of the CBM-MUCH first-level J/psi selection on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--mode selection|msd] [--impl ours|reference]

A "step" is one pass of the whole hot path (a3..a8: classify, stage, triplet search, compaction, linking,
decision, result write) over one synthetic timeslice batch.  Default workload: BASELINE.json
configs[3] (load-imbalance stress, 1,000,000 events) -- the configuration the north_star's roofline target
is stated on.

  value        events/s with the batch resident in HBM (cbm_trigger_run_device), `value_kind` says so
  e2e          events/s through cbm_trigger_upload_events / run / fetch_results from the slots' pinned HOST
               buffers, the H2D and D2H copies inside the timed region; `sustained_value` repeats it
  kernels      per-kernel device times of a CBM_FLAG_SERIAL pass (one kernel after the other: kernel times)
  roofline     dominant kernel against the measured HBM copy bandwidth; roofline_step = the whole step against
               max(t_HBM, t_INT), t_INT from the measured window-evaluation rate (cbm_trigger_ubench) and the
               oracle-side N_eval of a sample
  cpu_baseline the CPU oracle on the host cores (all cores, and one core)
  config4_streaming  (default run only) the key figures of `--config 4`, run in a process of its own: a ring of
               three distinct 10^6-event chunks, ten chunk-iterations, int32 and packed wire format, against 10 MHz

Prints ONE JSON line (rank 0).  `--impl reference` times the CPU oracle (oracle/) on the host cores.
"""
from __future__ import annotations

import argparse
import csv
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
TRAFFIC_CSV = os.path.join("profiles", "r3_traffic.csv")  # ncu --set full captures, per kernel and workload
INST_CSV = os.path.join("profiles", "r3_inst.csv")
# the source files a kernel is compiled from (beside the shared ptx.cuh / params.h / classify.cuh): a committed ncu
# figure is quoted as this run's only while these files are byte-identical to the ones the capture was taken from
KERNEL_SOURCES = {"classify_kernel": ("classify.cuh",), "tile_kernel": ("tile.cuh",), "team_kernel_M": ("team.cuh",),
                  "chain_kernel_H": ("chain.cuh",), "team_kernel_G": ("team.cuh",), "team_kernel_X": ("team.cuh",),
                  "msd_kernel": ("msd.cuh",)}
SHARED_SOURCES = ("ptx.cuh", "params.h", "classify.cuh")


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--mode", default="selection", choices=["selection", "msd"],
                    help="selection: the north_star path; msd: the paper-literal cut on the Table-1-shaped workload")
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json configs index (0..3; 4 = streaming of config-2 chunks)")
    ap.add_argument("--events", type=int, default=0, help="events per batch (0 = the config's size)")
    ap.add_argument("--e2e-steps", type=int, default=0, help="steps of the end-to-end leg (0 = min(steps, 10))")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-packed", action="store_true", help="skip the end-to-end leg with the packed wire format XY20")
    ap.add_argument("--no-ubench", action="store_true", help="skip the integer-pipe micro-benchmarks")
    ap.add_argument("--no-caller-memory", action="store_true", help="skip the end-to-end leg from pageable caller arrays")
    ap.add_argument("--no-streaming-leg", action="store_true",
                    help="default run (config 3, 1 GPU): do not add the streaming configuration (config 4) to the line")
    ap.add_argument("--serial", action="store_true", help="CBM_FLAG_SERIAL also in the timed leg (kernels one after the other)")
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


def kernel_source_sha(kernel):
    """First 16 hex digits of the SHA-256 over the files `kernel` is compiled from (KERNEL_SOURCES + SHARED_SOURCES,
    in that order).  The ncu CSVs under profiles/ store the value of the build they were captured from; .git does not
    travel to the GPU box, so this - not a commit id - is what the bench can check at run time."""
    import hashlib
    h = hashlib.sha256()
    csrc = os.path.join(ROOT, "paper_1810_11966_b200", "csrc")
    for fn in KERNEL_SOURCES.get(kernel, ()) + SHARED_SOURCES:
        with open(os.path.join(csrc, fn), "rb") as f:
            h.update(f.read())
    return h.hexdigest()[:16]


def _capture_row(row, kernel):
    """Provenance of one committed ncu figure; "stale" = the kernel's sources changed since the capture."""
    sha = row.get("source_sha16") or ""
    return {"kind": "committed_capture", "capture": row.get("capture"), "commit": row.get("commit"), "source_sha16": sha,
            "stale": sha != kernel_source_sha(kernel)}


def ncu_traffic(workload, kernel):
    """dram__bytes_read.sum + dram__bytes_write.sum of one committed `ncu --set full` capture of this kernel on
    this workload (profiles/r3_traffic.csv names the capture, its commit and the hash of the kernel's sources), else
    None.  A figure whose kernel sources have changed since is returned with "stale": True and must not be quoted."""
    path = os.path.join(ROOT, TRAFFIC_CSV)
    if not os.path.exists(path):
        return None
    with open(path) as f:
        for row in csv.DictReader(f):
            if row.get("workload") == workload and row.get("kernel") == kernel:
                return dict(_capture_row(row, kernel), bytes=int(row["dram_bytes_read"]) + int(row["dram_bytes_write"]),
                            source=TRAFFIC_CSV)
    return None


def ncu_instructions(workload):
    """smsp__inst_executed.sum of the committed `ncu --set full` captures of this workload's kernels
    (profiles/r3_inst.csv): {kernel: warp-instructions per launch, provenance, "stale"}."""
    path = os.path.join(ROOT, INST_CSV)
    res = {}
    if os.path.exists(path):
        with open(path) as f:
            for row in csv.DictReader(f):
                if row.get("workload") == workload:
                    res[row["kernel"]] = dict(_capture_row(row, row["kernel"]), warp_instructions=int(row["warp_instructions"]))
    return res


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
    Restates the scheduler's rule for the roofline bookkeeping only; the event counts are
    checked against the library's own statistics (the tile's staging capacity moves a few events from tiny to M)."""
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


# ---------------------------------------------------------------------------------------------- CPU oracle legs
def oracle_events_per_second(cfg, batch, n_sample, n_threads, msd_params=None):
    """The CPU oracle, as it stands, on the first n_sample events of the batch over n_threads host threads
    (events are independent: the paper's pthread scheme)."""
    from concurrent.futures import ThreadPoolExecutor
    import oracle
    if msd_params is None:
        g = oracle.geometry(cfg.layer_z, cfg.win_in, cfg.win_link, cfg.min_candidates)
        call = lambda a, b: oracle.run(g, batch.x, batch.y, batch.off, a, b)[2]
    else:
        call = lambda a, b: oracle.run_msd(msd_params, batch.x, batch.y, batch.off, a, b)[1]
    n_sample = min(n_sample, batch.n_events)
    chunk = max(1, min(2000, n_sample // (4 * n_threads) or 1))
    ranges = [(a, min(a + chunk, n_sample)) for a in range(0, n_sample, chunk)]
    call(0, min(64, n_sample))  # load the library outside the timing
    t0 = time.perf_counter()
    if n_threads == 1:
        acc = sum(int(call(a, b).sum()) for (a, b) in ranges)
    else:
        with ThreadPoolExecutor(n_threads) as ex:
            acc = sum(int(r.sum()) for r in ex.map(lambda r: call(r[0], r[1]), ranges))
    dt = time.perf_counter() - t0
    return n_sample / dt, dt, acc


def cpu_sample_size(cid):
    # about 10-30 s of CPU work at the oracle's measured all-core rates
    return {0: 1000, 1: 200_000, 2: 100_000, 3: 500_000, 4: 100_000}[cid]


def cpu_baseline_block(cfg, cid, batch, msd_params=None, what="oracle/cbm_oracle.c"):
    """cpu_baseline of the JSON line: all host cores on a bounded sample, and one core on a smaller one."""
    n_threads = os.cpu_count() or 1
    n_sample = min(batch.n_events, cpu_sample_size(cid) if msd_params is None else 400_000)
    v, dt, _ = oracle_events_per_second(cfg, batch, n_sample, n_threads, msd_params)
    n1 = max(1, min(batch.n_events, n_sample // max(2, n_threads // 2)))
    v1, dt1, _ = oracle_events_per_second(cfg, batch, n1, 1, msd_params)
    return {"value": v, "unit": UNIT, "cores": n_threads, "kind": "oracle", "seconds": dt,
            "sample": f"first {n_sample} events of the same batch, {what} over {n_threads} threads",
            "single_thread": {"value": v1, "unit": UNIT, "cores": 1, "seconds": dt1,
                              "sample": f"first {n1} events of the same batch, {what}, one thread"}}


def n_eval_per_event(cfg, batch, n_sample=4000):
    """Algorithmic window evaluations per event from the independent slope-sorted CPU counter on a
    sample of the batch (part of the CPU-baseline leg: it runs oracle/ code)."""
    import oracle
    n = min(batch.n_events, n_sample)
    g = oracle.geometry(cfg.layer_z, cfg.win_in, cfg.win_link, cfg.min_candidates)
    return float(oracle.run_slope_sorted(g, batch.x, batch.y, batch.off, 0, n)[3]) / max(n, 1), n


def run_reference(args, cfg, cid):
    """--impl reference: the oracle on the host cores, each step a bounded sample of the same workload."""
    from paper_1810_11966_b200 import workloads as W
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    n_threads = os.cpu_count() or 1
    msd = None
    if args.mode == "msd":
        import oracle
        cfg = W.PAPER_TABLE1
        msd = oracle.msd_params(cfg.layer_z)
    n_events = args.events or (cfg.chunk_events or cfg.n_events)
    per_step = max(1, min(n_events, (cpu_sample_size(cid) if msd is None else 400_000) // 4))
    batch = W.generate(cfg, n_events=per_step)
    for _ in range(args.warmup):
        oracle_events_per_second(cfg, batch, max(1, per_step // 8), n_threads, msd)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle_events_per_second(cfg, batch, per_step, n_threads, msd)
    dt = time.perf_counter() - t0
    value = per_step * args.steps / dt
    src = "oracle/msd_oracle.c" if msd is not None else "oracle/cbm_oracle.c"
    sample = f"first {per_step} events of {cfg.name} per step, {src} over {n_threads} threads"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "int64", "data": "synthetic",
        "config": {"workload": cfg.name, "events_per_step": per_step, "hits_per_step": batch.n_hits, "mode": args.mode},
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


def setup_rank():
    import torch
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

    return torch, rank, world, local_rank, dev, dist, barrier


def timed_device_loop(torch, args, sampler, barrier, step):
    """W untimed warm-up steps (and at least 0.25 s of load), then exactly K timed steps between CUDA events on the
    launching stream.  Returns (ms_total, n_warm, clocks)."""
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        t_load = time.perf_counter()
        n_warm = 0
        while n_warm < args.warmup or (time.perf_counter() - t_load < 0.25 and n_warm < 1000):
            step()
            n_warm += 1
            if n_warm >= args.warmup:
                torch.cuda.synchronize()
        barrier()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0 = time.perf_counter()
        ev0.record(stream)
        for _ in range(args.steps):
            step()
        ev1.record(stream)
        barrier()
        clocks = sampler.stop(t0, time.perf_counter())
        return ev0.elapsed_time(ev1), n_warm, clocks


def run_ours(args, cfg, cid):
    from paper_1810_11966_b200 import binding as K
    from paper_1810_11966_b200 import workloads as W
    torch, rank, world, local_rank, dev, dist, barrier = setup_rank()

    # ---- workload: each rank owns its own batch (weak scaling; events are independent, no collective)
    E = args.events or (cfg.chunk_events or cfg.n_events)
    S, L = cfg.n_stations, cfg.n_layers
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
    make = lambda flags: K.Trigger(cfg.layer_z, E, n_hits, win_in=cfg.win_in, win_link=cfg.win_link,
                                   min_candidates=cfg.min_candidates, max_hits_per_layer=cfg.max_hits_per_layer, n_slots=0,
                                   device=local_rank, flags=flags)

    # ---- the timed leg: K steps back to back on device-resident inputs
    trig = make(K.CBM_FLAG_PROFILE | (K.CBM_FLAG_SERIAL if args.serial else 0))
    sampler = ClockSampler(local_rank)
    sampler.start()  # nvidia-smi needs ~0.1 s to deliver its first sample: started before the warm-up
    ms_total, n_warm, clocks = timed_device_loop(
        torch, args, sampler, barrier, lambda: trig.run_device(E, n_hits, dx, dy, doff, dnt, dnc, dac))
    rc, st = trig.device_status()
    if rc != K.CBM_OK:
        raise SystemExit("bench.py: the device rejected events of a generated batch")
    stats = st.as_dict()
    ubench = None
    if rank == 0 and not args.no_ubench:
        ubench = trig.ubench()
    trig.close()
    ref = (dnt.cpu().numpy().view(np.uint32).reshape(E, S).copy(), dnc.cpu().numpy().view(np.uint32).copy(), dac.cpu().numpy().copy())
    n_accept, n_cand_events = int(ref[2].sum()), int((ref[1] != 0).sum())

    # ---- kernel times: the same step with the kernels one after the other (CBM_FLAG_SERIAL), so that every
    # CUDA-event pair brackets its kernel alone
    trig = make(K.CBM_FLAG_PROFILE | K.CBM_FLAG_SERIAL)
    n_ser = max(3, min(args.steps, 10))
    with torch.cuda.stream(torch.cuda.Stream()):
        for _ in range(2 + n_ser):
            trig.run_device(E, n_hits, dx, dy, doff, dnt, dnc, dac)
        ktimes = trig.device_kernel_times(n_last=n_ser)
    trig.close()
    got = (dnt.cpu().numpy().view(np.uint32).reshape(E, S), dnc.cpu().numpy().view(np.uint32), dac.cpu().numpy())
    if not all(np.array_equal(a, b) for a, b in zip(ref, got)):
        raise SystemExit("bench.py: the serial and the side-by-side launch sequences disagree")

    # ---- end-to-end legs: pinned HOST buffers -> H2D -> kernels -> D2H, slots in flight; every fetched batch is
    # compared with the device-resident results (outside the timed region)
    e2e = e2e_packed = e2e_caller = None
    if not args.no_e2e:
        e2e = run_e2e(args, cfg, batch, ref, K, W, local_rank, rank, barrier)
        if not args.no_packed and world == 1:
            e2e_packed = run_e2e(args, cfg, batch, ref, K, W, local_rank, rank, barrier, packed=True)
        if world == 1 and not args.no_caller_memory:
            e2e_caller = run_e2e(args, cfg, batch, ref, K, W, local_rank, rank, barrier, caller_memory=True)
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

    # ---- per-kernel accounting: algorithmic bytes of the events a kernel processes / its mean (serial) time
    acct = class_accounting(batch.off, S, K.TINY_MAX_LAYER_DEFAULT, K.TINY_MAX_TOTAL, K.CLASS_CAPS)
    kmean = ktimes.mean(axis=0) if len(ktimes) else np.zeros(K.N_KERNELS)
    zero = {"events": 0, "hits": 0, "bytes": 0}
    # classify reads every event's offsets; tile, team_M, team_H, team_G their events; team_X the events handed on
    acct = [{"events": E, "hits": 0, "bytes": 4 * (E * L + 1)}] + acct + [dict(zero, events=stats["n_redone"])]
    kbytes = [a["bytes"] for a in acct]
    dom = int(np.argmax(kmean))  # the kernel that takes the most time
    dom_ms = float(kmean[dom])
    achieved = kbytes[dom] / (dom_ms * 1e-3) / 1e9 if dom_ms > 0 else 0.0
    traffic = ncu_traffic(cfg.name, K.KERNEL_NAMES[dom])
    roofline = {"bound": "hbm", "kernel": K.KERNEL_NAMES[dom], "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": traffic["bytes"] if traffic and not traffic["stale"] else None,
                "traffic_source": traffic,  # a committed capture, not a counter of this run; null above when stale
                "peak_source": peak_src, "algorithmic_bytes_per_launch": kbytes[dom], "ms_per_launch": dom_ms,
                "share_of_serial_step": dom_ms / float(kmean.sum()) if kmean.sum() > 0 else None,
                "timing": "CUDA events around the kernel on its stream, kernels launched one after the other (CBM_FLAG_SERIAL)"}
    step_gbs = B_alg / (ms_per_step * 1e-3) / 1e9
    t_hbm_ms = B_alg / (peak * 1e9) * 1e3
    out = {
        "metric": METRIC, "value": value, "value_kind": "hbm_resident", "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "int64", "data": "synthetic",
        "config": {"workload": cfg.name, "baseline_config_index": cid, "events_per_batch": E, "hits_per_batch": n_hits,
                   "stations": S, "bytes_per_batch": B_alg, "l2": "inputs larger than L2 (no flush needed)"
                   if B_alg > 200e6 else "inputs smaller than L2: L2-resident between steps", "parallelism": f"replicas x{world}",
                   "launch": "serial" if args.serial else "side by side"},
        "hits_per_second": hits_all * args.steps / (ms_total_max * 1e-3),
        "vs_10MHz": value / CBM_INTERACTION_RATE_HZ,
        # kernels launched in the timed region: the library's own count of the last run (cbm_trigger_stats_t.n_launches),
        # the same for every step of a fixed batch
        "gpu_launches": int(stats["n_launches"]) * args.steps,
        "kernels": {name: {"ms": float(kmean[i]), "events": acct[i]["events"], "hits": acct[i]["hits"],
                           "algorithmic_bytes": kbytes[i],
                           "frac": kbytes[i] / (float(kmean[i]) * 1e-3) / 1e9 / peak if kmean[i] > 0 else None}
                    for i, name in enumerate(K.KERNEL_NAMES)},
        "serial_step_ms": float(kmean.sum()),
        "classes": stats["n_class"], "events_redone": stats["n_redone"], "accepted_events": n_accept,
        "events_with_candidates": n_cand_events,
        "roofline": roofline,
        "roofline_step": {"bound": "hbm", "achieved": step_gbs, "peak": peak, "unit": "GB/s", "frac": step_gbs / peak,
                          "frac_of_8TBs_nominal": step_gbs / 8000.0, "algorithmic_bytes_per_step": B_alg, "t_hbm_ms": t_hbm_ms},
        "clocks": clocks, "warmup_steps_run": n_warm, "generation_s": t_gen,
    }
    # What the kernels are bound by in fact: instruction issue.  The warp-instructions of the
    # captured kernels of this workload (committed ncu captures) at one instruction per scheduler and cycle.
    inst = {k: v for k, v in ncu_instructions(cfg.name).items() if not v["stale"]}
    if inst and clocks.get("sm_mhz"):
        n_sched = 4 * torch.cuda.get_device_properties(local_rank).multi_processor_count
        wi = sum(v["warp_instructions"] for v in inst.values())
        t_issue_ms = wi / (n_sched * clocks["sm_mhz"] * 1e6) * 1e3
        out["roofline_step"]["issue"] = {
            "warp_instructions_per_step": wi, "kernels": inst, "schedulers": n_sched, "sm_mhz": clocks["sm_mhz"],
            "t_issue_ms": t_issue_ms, "frac": t_issue_ms / ms_per_step,
            "kind": "committed_capture",
            "note": "instruction counts from committed ncu captures whose kernel sources are unchanged (not counters of "
                    "this run); captured kernels only; the step cannot be shorter than t_issue_ms at this instruction count"}
    if ubench:
        out["ubench"] = dict(ubench, note="cbm_trigger_ubench: measured on this GPU in this run, 8 chains per thread")
    if e2e:
        e2e_value = whole_job_rate(events_all, e2e["steps"], e2e_s_max)
        h2d_gbs = e2e["h2d_bytes"] * e2e["steps"] / e2e_s_max / 1e9
        out["e2e"] = {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": e2e["h2d_bytes"],
                      "d2h_bytes_per_step": e2e["d2h_bytes"], "steps": e2e["steps"], "slots": e2e["slots"],
                      "distinct_chunks": e2e["distinct"], "ms_per_step": 1e3 * e2e_s_max / e2e["steps"], "h2d_gbs": h2d_gbs,
                      "h2d_copy_gbs": e2e["h2d_copy_gbs"], "frac_of_h2d_ceiling": h2d_gbs / e2e["h2d_copy_gbs"] if e2e["h2d_copy_gbs"] else None,
                      "vs_10MHz": e2e_value / CBM_INTERACTION_RATE_HZ, "parity": e2e["parity"]}
        out["sustained_value"] = e2e_value
    for key, leg in (("e2e_packed_xy20", e2e_packed), ("e2e_caller_memory", e2e_caller)):
        if leg:  # extras: 5-byte-per-hit wire format; pageable caller arrays memcpy'd into the staging
            v = whole_job_rate(E, leg["steps"], leg["seconds"])
            out[key] = {"value": v, "unit": UNIT, "h2d_bytes_per_step": leg["h2d_bytes"], "d2h_bytes_per_step": leg["d2h_bytes"],
                        "steps": leg["steps"], "ms_per_step": 1e3 * leg["seconds"] / leg["steps"],
                        "h2d_gbs": leg["h2d_bytes"] * leg["steps"] / leg["seconds"] / 1e9,
                        "vs_10MHz": v / CBM_INTERACTION_RATE_HZ, "parity": leg["parity"]}
    if world == 1 and not args.no_cpu_baseline:
        out["cpu_baseline"] = cpu_baseline_block(cfg, cid, batch)
        # the stated roofline (north_star): the slower of hit bytes at HBM peak and window evaluations at the
        # measured integer rate
        nev, n_smp = n_eval_per_event(cfg, batch)
        rs = out["roofline_step"]
        rs["n_eval_per_event"] = nev
        rs["n_eval_sample"] = f"oracle/slope_sorted.c on the first {n_smp} events"
        if ubench:
            # t_INT = N_eval * c_eval / R_int: c_eval = 6 ALU lane-instructions per evaluation (x and y:
            # 4 ISETP + 2 SEL/LOP3 in the SASS of the walks; the two IMAD.WIDE run on the FMA pipe), R_int = the measured
            # integer lane-ops/s.  Beside it the same work at the measured rate of the whole test as compiled.
            c_eval = 6
            t_int_ms = nev * E * c_eval / ubench["alu_lane_ops_per_s"] * 1e3
            rs["c_eval"] = c_eval
            rs["t_int_ms"] = t_int_ms
            rs["t_int_ms_at_measured_window_rate"] = nev * E / ubench["window_evals_per_s"] * 1e3
            rs["bound"] = "hbm" if t_hbm_ms >= t_int_ms else "alu"
            rs["frac_of_stated_roofline"] = max(t_hbm_ms, t_int_ms) / ms_per_step
    return out


def run_e2e(args, cfg, batch, ref, K, W, local_rank, rank, barrier, packed=False, caller_memory=False):
    """Batches through upload_events / run / fetch_results with all slots in flight, so that the H2D of batch i+1
    overlaps the kernels and the D2H of batch i.  Inputs lie in the slots' pinned HOST buffers
    (cbm_trigger_host_buffers: the producer writes there) -- or, with caller_memory, in ordinary numpy arrays that
    upload_events memcpy's into the staging inside the timed region.  Every slot holds a DISTINCT chunk of events
    (two slots; config 4, streaming: a ring of three, ten chunk-iterations).  Wall clock between device synchronisations.
    Every slot's results are compared with device-resident results of the same chunk, outside the timed region."""
    import torch
    E, S, L = batch.n_events, cfg.n_stations, cfg.n_layers
    streaming = bool(cfg.chunk_events)
    n_slots = 3 if streaming else 2
    steps = args.e2e_steps or (10 if streaming else min(max(args.steps, 2), 10))
    if caller_memory:
        steps = min(steps, 3)
    # every slot holds a chunk of its own (distinct events), so that no step re-uploads what the previous one sent
    chunks = [batch] + [other_chunk(W, cfg, E, (rank + 1) * E + (7 + k) * E) for k in range(1, n_slots)]
    max_hits = max(b.n_hits for b in chunks)
    trig = K.Trigger(cfg.layer_z, E, max_hits, win_in=cfg.win_in, win_link=cfg.win_link,
                     min_candidates=cfg.min_candidates, max_hits_per_layer=cfg.max_hits_per_layer, n_slots=n_slots,
                     device=local_rank, flags=K.CBM_FLAG_PROFILE | (K.CBM_FLAG_PACKED_INPUT if packed else 0))
    bufs, nh = [], []
    for s in range(n_slots):  # the producer (DAQ / generator) writes the batch into the slot's pinned staging, untimed
        b = chunks[s % len(chunks)]
        if caller_memory:
            bufs.append((b.x, b.y, b.off))
        elif packed:
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
    out = [(np.empty((E, S), dtype=np.uint32), np.empty(E, dtype=np.uint32), np.empty(E, dtype=np.uint8)) for _ in range(n_slots)]

    def pipeline(n):
        for i in range(n):
            s = i % n_slots
            if i >= n_slots:
                trig.fetch_results(s, E, out=out[s])
            if packed:
                trig.upload_events_packed(s, bufs[s][0], bufs[s][1], E, nh[s])
            else:
                trig.upload_events(s, bufs[s][0], bufs[s][1], bufs[s][2], E, nh[s])
            trig.run(s)
        for i in range(max(0, n - n_slots), n):
            trig.fetch_results(i % n_slots, E, out=out[i % n_slots])

    pipeline(max(n_slots, min(args.warmup, 3)))
    barrier()
    t0 = time.perf_counter()
    pipeline(steps)
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    st = trig.stats(0)
    slot_bytes = [(20 * ((n + 3) // 4) if packed else 8 * n) + 4 * (E * L + 1) for n in nh]  # H2D bytes of a step on slot s
    h2d_bytes = sum(slot_bytes[i % n_slots] for i in range(steps)) // steps                   # mean over the timed steps
    h2d_copy_gbs = slot_bytes[0] / (float(st.h2d_ms) * 1e-3) / 1e9 if st.h2d_ms > 0 else None  # stats(0): last upload of slot 0
    trig.close()
    # parity, untimed: slot 0 holds `batch` (device-resident results: ref); the other chunks of a streaming run are
    # run device-resident here and compared
    parity = {"slots_checked": 0, "ok": True}
    for s in range(min(n_slots, steps)):
        b = chunks[s % len(chunks)]
        if b is batch:
            want = ref
        else:  # device-resident results of the other chunks, computed once per process
            if id(b) not in _OTHER_RESULTS:
                _OTHER_RESULTS[id(b)] = device_results(torch, K, cfg, b, local_rank)
            want = _OTHER_RESULTS[id(b)]
        ok = all(np.array_equal(a, w) for a, w in zip(out[s], want))
        parity["slots_checked"] += 1
        parity["ok"] = parity["ok"] and ok
    if not parity["ok"]:
        raise SystemExit("bench.py: results fetched through the slot pipeline differ from the device-resident results")
    return {"seconds": dt, "steps": steps, "slots": n_slots, "distinct": len(chunks), "h2d_bytes": h2d_bytes,
            "d2h_bytes": E * (4 * S + 5) + 64 + 4, "parity": parity, "h2d_copy_gbs": h2d_copy_gbs}


_OTHER_CHUNKS = {}
_OTHER_RESULTS = {}  # id(chunk) -> device-resident results (the chunks live in _OTHER_CHUNKS for the whole run)


def other_chunk(W, cfg, n_events, first_event):
    """A further chunk of the same workload (other events of the same generator), generated once per process."""
    key = (cfg.name, n_events, first_event)
    if key not in _OTHER_CHUNKS:
        _OTHER_CHUNKS[key] = W.generate(cfg, n_events=n_events, first_event=first_event)
    return _OTHER_CHUNKS[key]


def device_results(torch, K, cfg, b, local_rank):
    """(n_triplets, n_candidates, accept) of batch b from cbm_trigger_run_device (untimed; parity of the e2e legs)."""
    dev = torch.device("cuda", local_rank)
    E, S = b.n_events, cfg.n_stations
    dx, dy = to_device_padded(torch, b.x, dev), to_device_padded(torch, b.y, dev)
    doff = torch.from_numpy(b.off.view(np.int32)).to(dev)
    dnt = torch.zeros(E * S, dtype=torch.int32, device=dev)
    dnc = torch.zeros(E, dtype=torch.int32, device=dev)
    dac = torch.zeros(E, dtype=torch.uint8, device=dev)
    with K.Trigger(cfg.layer_z, E, b.n_hits, win_in=cfg.win_in, win_link=cfg.win_link, min_candidates=cfg.min_candidates,
                   max_hits_per_layer=cfg.max_hits_per_layer, n_slots=0, device=local_rank) as trig:
        trig.run_device(E, b.n_hits, dx, dy, doff, dnt, dnc, dac)
        torch.cuda.synchronize()
    return (dnt.cpu().numpy().view(np.uint32).reshape(E, S), dnc.cpu().numpy().view(np.uint32), dac.cpu().numpy())


# ---------------------------------------------------------------------------------------------- the paper-literal mode
def run_msd(args):
    """--mode msd: cbm_trigger_msd_device (literally) on the workload of the paper's Table 1
    (one station, about 15 hits per layer), device-resident, with its own roofline and the
    paper's numbers beside it as context."""
    from paper_1810_11966_b200 import binding as K
    from paper_1810_11966_b200 import workloads as W
    torch, rank, world, local_rank, dev, dist, barrier = setup_rank()
    cfg = W.PAPER_TABLE1
    E = args.events or 1_000_000
    batch = W.generate(cfg, n_events=E, first_event=rank_event_range(rank, E)[0])
    n_hits, S, L = batch.n_hits, cfg.n_stations, cfg.n_layers
    dx, dy = to_device_padded(torch, batch.x, dev), to_device_padded(torch, batch.y, dev)
    doff = torch.from_numpy(batch.off.view(np.int32)).to(dev)
    dnp = torch.zeros(E, dtype=torch.int32, device=dev)
    dac = torch.zeros(E, dtype=torch.uint8, device=dev)
    par = K.make_msd_params()
    trig = K.Trigger(cfg.layer_z, E, n_hits, n_slots=0, device=local_rank)
    sampler = ClockSampler(local_rank)
    sampler.start()
    ms_total, n_warm, clocks = timed_device_loop(
        torch, args, sampler, barrier, lambda: trig.msd_device(par, E, n_hits, dx, dy, doff, dnp, dac))
    trig.close()
    (ms_total_max,), (events_all, hits_all) = reduce_over_ranks(dist, dev, [ms_total], [E, n_hits])
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    if rank != 0:
        return
    ms_per_step = ms_total_max / args.steps
    value = whole_job_rate(events_all, args.steps, ms_total_max * 1e-3)
    peak, peak_src = measured_peaks()
    B_alg = 8 * n_hits + 4 * (E * L + 1) + 5 * E  # hits, offsets, n_passing + accept
    gbs = B_alg / (ms_per_step * 1e-3) / 1e9
    msd_traffic = ncu_traffic(cfg.name, "msd_kernel")
    out = {
        "metric": METRIC, "value": value, "value_kind": "hbm_resident", "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "int128", "data": "synthetic",
        "config": {"workload": cfg.name, "mode": "msd (PAPER.md:71-88)", "events_per_batch": E, "hits_per_batch": n_hits,
                   "stations": S, "bytes_per_batch": B_alg, "l2": "inputs larger than L2 (no flush needed)" if B_alg > 200e6
                   else "inputs smaller than L2: L2-resident between steps", "parallelism": f"replicas x{world}"},
        "hits_per_second": hits_all * args.steps / (ms_total_max * 1e-3), "vs_10MHz": value / CBM_INTERACTION_RATE_HZ,
        "gpu_launches": args.steps, "accepted_events": int(dac.sum().item()),
        "roofline": {"bound": "hbm", "kernel": "msd_kernel", "achieved": gbs, "peak": peak, "unit": "GB/s", "frac": gbs / peak,
                     "traffic": msd_traffic["bytes"] if msd_traffic and not msd_traffic["stale"] else None,
                     "traffic_source": msd_traffic, "peak_source": peak_src, "algorithmic_bytes_per_launch": B_alg, "ms_per_launch": ms_per_step},
        "paper_context": {"gpu_events_per_s": 2.84e5, "gpu": "Tesla C2075, 40 000 events (PAPER.md:220, Table 1)",
                          "cpu_events_per_s_1_thread": 6.25e4, "cpu": "Xeon 2.8 GHz, one core (PAPER.md:213-221)",
                          "note": "other hardware, the paper's own data sample: context, not a baseline"},
        "clocks": clocks, "warmup_steps_run": n_warm,
    }
    if world == 1 and not args.no_cpu_baseline:
        import oracle
        mp = oracle.msd_params(cfg.layer_z)
        out["cpu_baseline"] = cpu_baseline_block(cfg, 1, batch, msd_params=mp, what="oracle/msd_oracle.c")
        n_chk = min(E, 200_000)  # parity of this run's outputs on a sample (the tests hold the full checks)
        want = oracle.run_msd(mp, batch.x, batch.y, batch.off, 0, n_chk)
        ok = np.array_equal(dnp.cpu().numpy().view(np.uint32)[:n_chk], want[0]) and np.array_equal(dac.cpu().numpy()[:n_chk], want[1])
        out["parity"] = {"events_checked": n_chk, "ok": bool(ok)}
        if not ok:
            raise SystemExit("bench.py --mode msd: device results differ from oracle/msd_oracle.c")
    print(json.dumps(out))


def self_launch_command(argv, n_gpus, port):
    """`python bench.py --gpus N ...` started without a launcher: the command that starts the N ranks (one per GPU of this
    node, rendezvous on 127.0.0.1), each of which runs this script again with the same arguments.  Events are
    independent, so the ranks are replicas with their own event ranges; NCCL carries the barrier and the max-reduction of
    the times only."""
    return [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n_gpus}",
            "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + list(argv)


def free_port():
    import socket
    with socket.socket() as sock:
        sock.bind(("127.0.0.1", 0))
        return sock.getsockname()[1]


def main():
    args = parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and args.impl == "ours":
        import subprocess
        raise SystemExit(subprocess.call(self_launch_command(sys.argv[1:], args.gpus, free_port())))
    from paper_1810_11966_b200 import workloads as W
    cfg = W.CONFIGS[args.config]
    if args.impl == "reference":
        run_reference(args, cfg, args.config)
    elif args.mode == "msd":
        run_msd(args)
    else:
        out = run_ours(args, cfg, args.config)
        if out is None:  # not rank 0
            return
        if args.config == 3 and out["n_gpus"] == 1 and not args.no_streaming_leg and not args.no_e2e:
            out["config4_streaming"] = streaming_leg()
        print(json.dumps(out))


def streaming_leg():
    """BASELINE.json configs[4] beside the default line (config 3 carries the roofline target, config 4 the sustained
    rate against 10 MHz): this script again with --config 4 in a process of its own -- a ring of three distinct
    10^6-event chunks of seed 5, ten chunk-iterations, int32 and packed wire format, results of every slot compared
    with device-resident results -- and the key figures of its line."""
    import subprocess
    cmd = [sys.executable, os.path.abspath(__file__), "--config", "4", "--steps", "10", "--warmup", "3", "--no-cpu-baseline",
           "--no-ubench", "--no-caller-memory"]
    try:
        r = subprocess.run(cmd, capture_output=True, text=True, timeout=900)
        line = [l for l in r.stdout.strip().splitlines() if l.startswith("{")][-1]
        d = json.loads(line)
    except Exception as ex:  # the default line must survive a failure of the extra leg
        return {"error": f"{type(ex).__name__}: {ex}"}
    keep = {"workload": d["config"]["workload"], "events_per_chunk": d["config"]["events_per_batch"],
            "hits_per_chunk": d["config"]["hits_per_batch"], "value_hbm_resident": d["value"], "ms_per_step": d["ms_per_step"],
            "roofline_step_frac": d["roofline_step"]["frac"], "kernels_ms": {k: v["ms"] for k, v in d["kernels"].items()},
            "clocks": d.get("clocks")}
    for k in ("e2e", "e2e_packed_xy20"):
        if k in d:
            keep[k] = d[k]
    if "e2e" in d:
        keep["sustained_value"] = d["e2e"]["value"]
        keep["sustained_vs_10MHz"] = d["e2e"]["vs_10MHz"]
    if "e2e_packed_xy20" in d:
        keep["sustained_packed_vs_10MHz"] = d["e2e_packed_xy20"]["vs_10MHz"]
    return keep


if __name__ == "__main__":
    main()
