"""N_eval of SURVEY.md section 8(d): algorithmic window evaluations per event of the canonical slope-sorted
search (oracle/slope_sorted.c), the work term of the integer-pipe roofline.  TEST INFRASTRUCTURE (calls only
oracle/ and the input generator).

    python -m oracle.n_eval [config index] [events]        # prints one line; DESIGN.md section 6.5 quotes it
"""
import sys

import oracle
from paper_1810_11966_b200 import workloads as W


def main():
    cid = int(sys.argv[1]) if len(sys.argv) > 1 else 3
    n = int(sys.argv[2]) if len(sys.argv) > 2 else 20000
    cfg = W.CONFIGS[cid]
    b = W.generate(cfg, n_events=n)
    g = oracle.geometry(cfg.layer_z, cfg.win_in, cfg.win_link, cfg.min_candidates)
    nt, nc, ac, n_eval = oracle.run_slope_sorted(g, b.x, b.y, b.off)
    print(f"{cfg.name}: first {n} events, {b.n_hits / n:.1f} hits/event, N_eval = {n_eval / n:.1f} window evaluations/event, "
          f"{nt.sum() / n:.3f} triplets/event")


if __name__ == "__main__":
    main()
