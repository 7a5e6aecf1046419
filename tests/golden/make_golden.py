"""Writes tests/golden/*.txt.  Calls ONLY oracle/ and the seeded input generator -- never the CUDA path.

    python tests/golden/make_golden.py

The paper prints no worked example for this path, so these files are not "the paper's values":
they are regression fixtures of the pinned oracle on seeded inputs (config 0 in full, the first events of
configs 1-3), stored sparsely as the events with any non-zero output.  The GPU parity tests compare against
the live oracle AND against these files, so that a later change of the oracle's arithmetic is visible.
"""
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

import oracle  # noqa: E402
from paper_1810_11966_b200 import workloads as W  # noqa: E402

CASES = [(0, 1000), (1, 2000), (2, 1000), (3, 4000)]


def main():
    for cid, n in CASES:
        cfg = W.CONFIGS[cid]
        b = W.generate(cfg, n_events=n)
        g = oracle.geometry(cfg.layer_z, cfg.win_in, cfg.win_link, cfg.min_candidates)
        nt, nc, ac = oracle.run(g, b.x, b.y, b.off)
        path = os.path.join(HERE, f"cfg{cid}_first{n}.txt")
        with open(path, "w") as f:
            f.write(f"# oracle/cbm_oracle.c on workloads.CONFIGS[{cid}] (seed {cfg.seed}), events [0,{n}); "
                    f"n_hits={b.n_hits}\n")
            f.write("# selection: PAPER.md:73-88 (section 3.2) with north_star windows 1/100, 2/100, >=2 candidates\n")
            f.write(f"# totals: triplets={int(nt.sum())} candidates={int(nc.sum())} accepted={int(ac.sum())}\n")
            f.write("# event  n_triplets[0..S)  n_candidates  accept     (events with all-zero output omitted)\n")
            for e in range(n):
                if nt[e].any() or nc[e] or ac[e]:
                    f.write(f"{e} {' '.join(str(int(v)) for v in nt[e])} {int(nc[e])} {int(ac[e])}\n")
        print(path, int(nt.sum()), int(nc.sum()), int(ac.sum()))


if __name__ == "__main__":
    main()
