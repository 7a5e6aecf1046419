"""BRUTE-FORCE CHECKER -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

The definition of the selection with no shortcut at all, in pure Python with arbitrary-
precision integers, for tiny hand-built events only (cost n0*n1*n2 per station and
prod |T_s| per event).  It pins oracle/cbm_oracle.c:

* every (h0, h1, h2) of a station is visited and ALL THREE pair tests are evaluated
  (no (h0,h1) short-circuit)                        -- PAPER.md:73-76, section 3.2 steps 1-2
* candidates are counted by explicit enumeration of all S-tuples of triplets and
  checking every consecutive link (no chain-count recursion)   -- BASELINE.json north_star
* accept iff candidates >= min_candidates                        -- PAPER.md:88, step 3

The window is tested with exact rationals (fractions.Fraction), i.e. literally
|x_h/z_A - x_g/z_B| <= a/b, not in the cross-multiplied form the oracle uses.
"""
from fractions import Fraction
from itertools import product

SAT = 2**32 - 1


def compat(h, zA, g, zB, win):
    w = Fraction(win[0], win[1])
    return (abs(Fraction(h[0], zA) - Fraction(g[0], zB)) <= w) & (abs(Fraction(h[1], zA) - Fraction(g[1], zB)) <= w)


def brute_force_event(layer_z, layers, win_in, win_link, min_candidates=2):
    """layers: list of L lists of (x, y).  Returns (n_triplets[S], n_candidates, accept)."""
    S = len(layer_z) // 3
    T = []
    for s in range(S):
        z0, z1, z2 = layer_z[3 * s: 3 * s + 3]
        H0, H1, H2 = layers[3 * s: 3 * s + 3]
        ts = []
        for h0 in H0:
            for h1 in H1:
                for h2 in H2:
                    ok01 = compat(h0, z0, h1, z1, win_in)
                    ok02 = compat(h0, z0, h2, z2, win_in)
                    ok12 = compat(h1, z1, h2, z2, win_in)
                    if ok01 & ok02 & ok12:
                        ts.append((h0, h1, h2))
        T.append(ts)
    n_cand = 0
    for chain in product(*T):
        ok = True
        for s in range(S - 1):
            ok &= bool(compat(chain[s][1], layer_z[3 * s + 1], chain[s + 1][1], layer_z[3 * (s + 1) + 1], win_link))
        n_cand += 1 if ok else 0
    n_cand = min(SAT, n_cand)
    return [min(SAT, len(t)) for t in T], n_cand, 1 if n_cand >= min_candidates else 0
