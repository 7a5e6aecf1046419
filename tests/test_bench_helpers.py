"""Host-side helpers of bench.py that need no GPU: the committed ncu figures the bench line quotes
(profiles/r2_traffic.csv, profiles/r2_inst.csv) parse, name existing captures, and are plausible against the
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
    alg = 1_430_529_244  # algorithmic bytes of class H on config 3 (profiles/r2_chain_kernel_H.md)
    assert alg <= t["bytes"] <= 1.5 * alg  # DRAM traffic: at least the algorithmic bytes, no large re-reads
    assert bench.ncu_traffic("cfg3_imbalance", "no_such_kernel") is None
    inst = bench.ncu_instructions("cfg3_imbalance")
    assert {"chain_kernel_H", "tile_kernel"} <= set(inst)
    for v in inst.values():
        assert v["warp_instructions"] > 0 and os.path.exists(os.path.join(ROOT, v["capture"]))
    assert bench.ncu_instructions("no_such_workload") == {}
