"""Host-side helpers of bench.py that need no GPU: the committed ncu figures the bench line quotes
(profiles/r3_traffic.csv, profiles/r3_inst.csv) parse, name existing captures, are not stale and are plausible against the
algorithmic bytes; the byte formula itself."""
import os

import bench

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_algorithmic_bytes_formula():
    # B_alg = 8 N + 4 (E L + 1) + E (4 S + 5): config 3's batch as DESIGN.md section 5 states it
    assert bench.algorithmic_bytes(1_000_000, 235_509_459, 4) == 1_953_075_676


def test_committed_ncu_figures_parse_and_name_their_captures():
    t = bench.ncu_traffic("cfg3_imbalance", "chain_kernel_H")
    assert t is not None and os.path.exists(os.path.join(ROOT, t["capture"]))
    alg = 1_430_529_244  # algorithmic bytes of class H on config 3 (profiles/r3_chain_kernel_H.md)
    assert alg <= t["bytes"] <= 1.5 * alg  # DRAM traffic: at least the algorithmic bytes, no large re-reads
    assert bench.ncu_traffic("cfg3_imbalance", "no_such_kernel") is None
    inst = bench.ncu_instructions("cfg3_imbalance")
    assert {"chain_kernel_H", "tile_kernel"} <= set(inst)
    for v in inst.values():
        assert v["warp_instructions"] > 0 and os.path.exists(os.path.join(ROOT, v["capture"]))
    assert bench.ncu_instructions("no_such_workload") == {}


def test_committed_ncu_figures_belong_to_the_kernel_sources_in_the_tree():
    """Every row of the two CSVs carries the hash of the kernel sources it was captured from; a row that no longer
    matches the tree is stale (bench.py then leaves its figure out of the line) and needs a fresh capture."""
    import csv
    for path, kernels in ((bench.TRAFFIC_CSV, 5), (bench.INST_CSV, 5)):
        with open(os.path.join(ROOT, path)) as f:
            rows = list(csv.DictReader(f))
        assert len(rows) >= kernels
        for row in rows:
            assert row["source_sha16"] == bench.kernel_source_sha(row["kernel"]), (path, row["kernel"], "stale capture")
            assert os.path.exists(os.path.join(ROOT, row["capture"]))
            for col in ("dram_bytes_read", "dram_bytes_write", "warp_instructions"):
                if col in row:
                    assert int(row[col]) > 0 and not row[col].endswith("0000000"), (row["kernel"], col, "rounded figure?")
    t = bench.ncu_traffic("paper_table1_trigger_station", "msd_kernel")
    assert t is not None and t["stale"] is False and t["kind"] == "committed_capture"


def test_stale_capture_is_flagged(monkeypatch):
    monkeypatch.setattr(bench, "kernel_source_sha", lambda kernel: "0" * 16)
    t = bench.ncu_traffic("cfg3_imbalance", "chain_kernel_H")
    assert t["stale"] is True
    assert all(v["stale"] for v in bench.ncu_instructions("cfg3_imbalance").values())


def test_gpus_n_without_a_launcher_starts_n_ranks(monkeypatch):
    """`python bench.py --gpus 4` with no WORLD_SIZE in the environment re-launches itself under torch.distributed.run
    with four ranks on 127.0.0.1; under a launcher (WORLD_SIZE set) it does not."""
    import subprocess
    import sys
    cmd = bench.self_launch_command(["--gpus", "4", "--steps", "5"], 4, 29511)
    assert cmd[1:4] == ["-m", "torch.distributed.run", "--nnodes=1"] and "--nproc-per-node=4" in cmd
    assert cmd[cmd.index("--master-addr") + 1] == "127.0.0.1" and cmd[cmd.index("--master-port") + 1] == "29511"
    assert cmd[-5:] == [os.path.join(ROOT, "bench.py"), "--gpus", "4", "--steps", "5"]
    calls = []
    monkeypatch.setattr(subprocess, "call", lambda c: calls.append(c) or 0)
    monkeypatch.setattr(sys, "argv", ["bench.py", "--gpus", "4", "--steps", "5"])
    monkeypatch.delenv("WORLD_SIZE", raising=False)
    try:
        bench.main()
    except SystemExit as ex:
        assert ex.code == 0
    assert len(calls) == 1 and calls[0][-4:] == ["--gpus", "4", "--steps", "5"] and "--nproc-per-node=4" in calls[0]
