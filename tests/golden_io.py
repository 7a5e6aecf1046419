"""Reader for tests/golden/cfg*_first*.txt (written by tests/golden/make_golden.py from the oracle)."""
import os
import re

import numpy as np

GOLDEN_DIR = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def golden_cases():
    out = []
    for name in sorted(os.listdir(GOLDEN_DIR)):
        m = re.match(r"cfg(\d+)_first(\d+)\.txt$", name)
        if m:
            out.append((int(m.group(1)), int(m.group(2)), os.path.join(GOLDEN_DIR, name)))
    return out


def read_golden(path, n_events, n_stations):
    nt = np.zeros((n_events, n_stations), dtype=np.uint32)
    nc = np.zeros(n_events, dtype=np.uint32)
    ac = np.zeros(n_events, dtype=np.uint8)
    with open(path) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            v = [int(t) for t in line.split()]
            e = v[0]
            nt[e] = v[1:1 + n_stations]
            nc[e] = v[1 + n_stations]
            ac[e] = v[2 + n_stations]
    return nt, nc, ac
