"""N > 1 bookkeeping of bench.py on CPU: two gloo ranks (replicas only).

Events are independent, so the path shards into contiguous event ranges with no
exchange step.  What has to be right with more than one rank is host logic only: every rank generates its
own range of the one synthetic event stream, the timed value is the MAX over ranks, the processed units are
the SUM over ranks.  The CPU oracle stands in for the kernels here (this is a tests/ file).
"""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

WORLD = 2
EVENTS_PER_RANK = 300


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, port, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=WORLD)
    try:
        import bench
        import oracle
        from paper_1810_11966_b200 import workloads as W
        cfg = W.CONFIGS[0]
        lo, hi = bench.rank_event_range(rank, EVENTS_PER_RANK)
        b = W.generate(cfg, n_events=hi - lo, first_event=lo)
        g = oracle.geometry(cfg.layer_z, cfg.win_in, cfg.win_link, cfg.min_candidates)
        nt, nc, ac = oracle.run(g, b.x, b.y, b.off)
        # per-rank "device time": rank 1 is the slow one
        times, counts = bench.reduce_over_ranks(dist, torch.device("cpu"), [10.0 + 5.0 * rank, 1.0 + rank],
                                                [b.n_events, b.n_hits])
        np.savez(os.path.join(out_dir, f"rank{rank}.npz"), x=b.x, y=b.y, off=b.off, nt=nt, nc=nc, ac=ac,
                 times=np.array(times), counts=np.array(counts), n_hits=b.n_hits)
        dist.barrier()
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(300)
def test_two_gloo_ranks_shard_the_event_stream(tmp_path):
    import oracle
    from paper_1810_11966_b200 import workloads as W
    W.build()
    oracle.build()
    port = _free_port()
    mp.spawn(_worker, args=(port, str(tmp_path)), nprocs=WORLD, join=True)
    r = [np.load(os.path.join(tmp_path, f"rank{k}.npz")) for k in range(WORLD)]

    # every rank saw the same reduced values: MAX of the times, SUM of the counts
    for k in range(WORLD):
        assert r[k]["times"].tolist() == [15.0, 2.0]
        assert r[k]["counts"].tolist() == [WORLD * EVENTS_PER_RANK, float(r[0]["n_hits"] + r[1]["n_hits"])]

    # the ranks' batches are the two halves of one stream: generating the whole range in one go gives the
    # concatenation of the ranks' hits, and the oracle's per-event results concatenate too (no event of one
    # rank depends on another rank's data)
    import bench
    cfg = W.CONFIGS[0]
    whole = W.generate(cfg, n_events=WORLD * EVENTS_PER_RANK, first_event=0)
    assert np.array_equal(whole.x, np.concatenate([r[0]["x"], r[1]["x"]]))
    assert np.array_equal(whole.y, np.concatenate([r[0]["y"], r[1]["y"]]))
    off1 = r[1]["off"].astype(np.uint64) + r[0]["off"][-1]
    assert np.array_equal(whole.off.astype(np.uint64), np.concatenate([r[0]["off"].astype(np.uint64), off1[1:]]))
    g = oracle.geometry(cfg.layer_z, cfg.win_in, cfg.win_link, cfg.min_candidates)
    nt, nc, ac = oracle.run(g, whole.x, whole.y, whole.off)
    assert np.array_equal(nt, np.concatenate([r[0]["nt"], r[1]["nt"]]))
    assert np.array_equal(nc, np.concatenate([r[0]["nc"], r[1]["nc"]]))
    assert np.array_equal(ac, np.concatenate([r[0]["ac"], r[1]["ac"]]))
    assert ac.sum() > 0  # config 0 plants signal pairs in 10 % of events

    # whole-job value = units of all ranks / time of the slowest rank
    assert bench.rank_event_range(1, EVENTS_PER_RANK) == (EVENTS_PER_RANK, 2 * EVENTS_PER_RANK)
    assert bench.whole_job_rate(r[0]["counts"][0], steps=4, seconds_max=15.0e-3) == pytest.approx(
        WORLD * EVENTS_PER_RANK * 4 / 15.0e-3)
