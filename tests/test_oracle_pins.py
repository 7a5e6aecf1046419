"""Pins for the CPU oracle (oracle/cbm_oracle.c): the oracle is checked against what the paper's
algorithm statement (section 3.2) and the mathematics fix, never against itself.

The paper prints no worked example (no event with listed hits and a listed decision), so the pins are:
hand-computed boundary cases, closed forms of constructed events, brute force without any shortcut,
invariances, an independent sorted/multiplicity implementation, and a closed-form background rate.
"""
import math

import numpy as np
import pytest

import oracle
from oracle import brute_force
from paper_1810_11966_b200 import workloads as W
from tests import adversarial as A

Z4 = list(W.GEOMETRY_4)


def run_events(layer_z, events, win_in=(1, 100), win_link=(2, 100), min_candidates=2):
    x, y, off = W.batch_from_layers(layer_z, events)
    g = oracle.geometry(layer_z, win_in, win_link, min_candidates)
    return oracle.run(g, x, y, off)


# ---------------------------------------------------------------- compat(): inclusivity and exactness
def one_station_event(h0, h1, h2, layer_z=(60000, 70000, 80000)):
    return list(layer_z), [[[h0] if h0 else [], [h1] if h1 else [], [h2] if h2 else []]]


def test_boundary_equality_in_station_x():
    # z0 = 60000, z1 = 70000, z2 = 80000.  x0 = 0, x1 = 700: x1/z1 = 0.01 exactly => |dslope| = 0.01: PASS
    # (closed window, R3).  x2 = 0 is within 0.01 of both only if x1/z1 - 0 <= 0.01: yes (equal).
    z, ev = one_station_event((0, 0), (700, 0), (0, 0))
    nt, nc, ac = run_events(z, ev)
    assert nt.tolist() == [[1]] and nc.tolist() == [1] and ac.tolist() == [0]
    # one unit more: 701/70000 = 0.0100142... > 0.01: FAIL
    z, ev = one_station_event((0, 0), (701, 0), (0, 0))
    nt, nc, ac = run_events(z, ev)
    assert nt.tolist() == [[0]] and nc.tolist() == [0]
    # negative side, and the (h0,h2) and (h1,h2) pairs: x2 = 800 -> 0.01 from h0=0 exactly, h1 = 350 -> 0.005
    z, ev = one_station_event((0, 0), (350, 0), (800, 0))
    assert run_events(z, ev)[0].tolist() == [[1]]
    z, ev = one_station_event((0, 0), (350, 0), (801, 0))   # h0-h2 fails by one unit
    assert run_events(z, ev)[0].tolist() == [[0]]
    z, ev = one_station_event((0, 0), (-700, 0), (0, 0))
    assert run_events(z, ev)[0].tolist() == [[1]]
    z, ev = one_station_event((0, 0), (-701, 0), (0, 0))
    assert run_events(z, ev)[0].tolist() == [[0]]
    # h1-h2 pair alone fails: h0 = 300 (0.005), h1 = 0 (0), h2 = 801 (0.0100125): h0-h2 diff 0.0050125 ok,
    # h0-h1 ok (0.005), h1-h2 = 0.0100125 > 0.01 fails
    z, ev = one_station_event((300, 0), (0, 0), (801, 0))
    assert run_events(z, ev)[0].tolist() == [[0]]
    z, ev = one_station_event((300, 0), (0, 0), (800, 0))
    assert run_events(z, ev)[0].tolist() == [[1]]


def full_range_cases():
    """Hand-computed cases at the edge of the int32 coordinate range (reading B2): z0 = 8 000 000,
    z1 = 8 200 000, z2 = 8 388 608 = 2^23, window 4095/4096.  b*|D| reaches 2^67 here, beyond int64.
    Returns (layer_z, win_in, events, expected triplets per event)."""
    z = [8_000_000, 8_200_000, 8_388_608]
    X = 2**31 - 1
    ev, exp = [], []
    # far apart: slopes +268.4 and -261.9 differ by 530 >> 0.99976: no triplet.  D = X*(z0+z1) = 3.48e16,
    # b*D = 1.43e20 = 7*2^64 + 1.36e19: an int64 product would come out NEGATIVE and pass the window.
    ev.append([[(X, 0)], [(-X, 0)], [(X, 0)]]); exp.append(0)
    # h0 and h2 on the line of slope +250, h1 at slope -207.6: no triplet.  Here 4096*|D| of the pairs (h0,h1) and
    # (h1,h2) is 1.2297e20 and 1.2894e20: both wrap to a NEGATIVE int64 (D mod 2^52 >= 2^51), so a 64-bit evaluation
    # of b*|D| <= a*z_A*z_B accepts both pairs and counts one triplet.  (Checked with Python integers.)
    ev.append([[(2_000_000_000, 0)], [(-1_702_700_000, 0)], [(2_097_152_000, 0)]]); exp.append(0)
    # the same line: slopes 250 exactly in all three layers (x = 250*z): one triplet
    ev.append([[(2_000_000_000, 5)], [(2_050_000_000, 5)], [(2_097_152_000, 5)]]); exp.append(1)
    # boundary: h0 = (0,0); h1 at slope a/b exactly: x1 = 4095*z1/4096 = 8 197 998.046875 -> not an integer, so
    # x1 = 8 197 998 passes (below) and 8 197 999 fails (b*x1*z0 = 4096*8197999*z0 > 4095*z0*z1 <=> 4096*8197999 >
    # 4095*8200000 = 33 579 000 000: 33 579 003 904 > 33 579 000 000 yes).  h2 = (0,0) is within the window of h0,
    # and of h1 iff h1 is within the window of the origin direction (|x1/z1| <= a/b): the same condition.
    ev.append([[(0, 0)], [(8_197_998, 0)], [(0, 0)]]); exp.append(1)
    ev.append([[(0, 0)], [(8_197_999, 0)], [(0, 0)]]); exp.append(0)
    # large offsets with a small difference: x0 = -2 000 000 000 (slope -250), x1 = -250*z1 + d, d = 8 197 998 passes
    ev.append([[(-2_000_000_000, 0)], [(-2_050_000_000 + 8_197_998, 0)], [(-2_097_152_000, 0)]]); exp.append(1)
    ev.append([[(-2_000_000_000, 0)], [(-2_050_000_000 + 8_197_999, 0)], [(-2_097_152_000, 0)]]); exp.append(0)
    return z, (4095, 4096), ev, exp


def test_compat_over_the_full_int32_range():
    z, win, ev, exp = full_range_cases()
    nt, nc, ac = run_events(z, ev, win_in=win, win_link=win)
    assert nt[:, 0].tolist() == exp
    assert nc.tolist() == exp  # one station: candidates = triplets


def test_boundary_equality_in_station_y_and_nonzero_slopes():
    # same in y, on top of a common slope 0.2: y = 0.2*z + delta keeps differences unchanged
    z, ev = one_station_event((5, 12000), (5, 14000 + 700), (5, 16000))
    assert run_events(z, ev)[0].tolist() == [[1]]
    z, ev = one_station_event((5, 12000), (5, 14000 + 701), (5, 16000))
    assert run_events(z, ev)[0].tolist() == [[0]]
    # x passes but y fails and vice versa: both projections are required
    z, ev = one_station_event((0, 0), (0, 701), (0, 0))
    assert run_events(z, ev)[0].tolist() == [[0]]
    z, ev = one_station_event((0, 0), (700, 700), (0, 0))
    assert run_events(z, ev)[0].tolist() == [[1]]


def test_window_is_a_rational_not_a_float():
    # window 1/3: x1/z1 = 1/3 needs z1 divisible by 3: z1 = 60000 -> x1 = 20000 passes exactly, 20001 fails
    z = [30000, 60000, 90000]
    ev = [[[(0, 0)], [(20000, 0)], [(0, 0)]]]
    assert run_events(z, ev, win_in=(1, 3))[0].tolist() == [[1]]
    ev = [[[(0, 0)], [(20001, 0)], [(0, 0)]]]
    assert run_events(z, ev, win_in=(1, 3))[0].tolist() == [[0]]


def test_boundary_equality_link_window_uses_middle_hits():
    # two stations; exact lines in each; the link compares the MIDDLE-layer hits (z = 70000 and 110000)
    # with window 0.02 (closed).  Station 0 line slope 0; station 1 middle hit at slope 0.02 exactly:
    # x = 0.02 * 110000 = 2200.  Its own triplet must still pass the 0.01 in-station window, so the outer
    # layers of station 1 sit at slope 0.02 too.
    z = W.station_layers_z([60, 100])
    st0 = [[(0, 0)], [(0, 0)], [(0, 0)]]
    def st1(xm):
        return [[(2000, 0)], [(xm, 0)], [(2400, 0)]]
    nt, nc, ac = run_events(z, [st0 + st1(2200)], min_candidates=1)
    assert nt.tolist() == [[1, 1]] and nc.tolist() == [1] and ac.tolist() == [1]
    nt, nc, ac = run_events(z, [st0 + st1(2201)], min_candidates=1)   # 2201/110000 = 0.020009 > 0.02
    assert nt.tolist() == [[1, 1]] and nc.tolist() == [0] and ac.tolist() == [0]
    # the outer layers do NOT enter the link: move station-1 outer hits to slope 0.029 (still within 0.01 of
    # the middle hit at 0.02 -> triplet ok); link still passes because only the middle hit counts (R8)
    st1b = [[(2900, 0)], [(2200, 0)], [(3480, 0)]]
    nt, nc, ac = run_events(z, [st0 + st1b], min_candidates=1)
    assert nt.tolist() == [[1, 1]] and nc.tolist() == [1]
    # and an in-station-compatible triplet whose middle hit is beyond the link window is not linked even
    # though its first-layer hit is within it
    st1c = [[(2000, 0)], [(2310, 0)], [(2400, 0)]]   # middle 0.021, outer 0.02 / 0.02
    nt, nc, ac = run_events(z, [st0 + st1c], min_candidates=1)
    assert nt.tolist() == [[1, 1]] and nc.tolist() == [0]


def test_products_exceed_32_bits():
    # |x| ~ 130000 and z ~ 380000: x*z ~ 5e10 > 2^32.  A 32-bit product would wrap and mis-decide.
    z = [360000, 370000, 380000]
    # slope 0.35 exactly: x = 126000, 129500, 133000
    ev = [[[(126000, -126000)], [(129500, -129500)], [(133000, -133000)]]]
    assert run_events(z, ev)[0].tolist() == [[1]]
    # shift the middle hit by 0.01 * 370000 = 3700 exactly -> still inside; +1 -> outside
    ev = [[[(126000, -126000)], [(129500 + 3700, -129500)], [(133000, -133000)]]]
    assert run_events(z, ev)[0].tolist() == [[1]]
    ev = [[[(126000, -126000)], [(129500 + 3701, -129500)], [(133000, -133000)]]]
    assert run_events(z, ev)[0].tolist() == [[0]]


def test_abi_range_extremes_do_not_overflow():
    # |x| = 2^23, z = 2^23 and den = 4096: b*|D| < 2^59, a*zA*zB <= 2^58 (header's overflow argument)
    z = [2 ** 23 - 2, 2 ** 23 - 1, 2 ** 23]
    X = 2 ** 23
    ev = [[[(X, -X)], [(X, -X)], [(X, -X)]]]
    # slopes ~1.0000002, 1.0000001, 1.0: within 1/4096
    assert run_events(z, ev, win_in=(1, 4096))[0].tolist() == [[1]]
    ev = [[[(X, -X)], [(-X, X)], [(X, -X)]]]
    assert run_events(z, ev, win_in=(1, 4096))[0].tolist() == [[0]]


# ---------------------------------------------------------------- closed forms of constructed events
@pytest.mark.parametrize("case", [c for c in A.adversarial_suite() if c[3] is not None], ids=lambda c: c[0])
def test_closed_form_cases(case):
    name, layer_z, events, (exp_nt, exp_nc, exp_ac) = case
    nt, nc, ac = run_events(layer_z, events)
    assert nt.tolist() == exp_nt
    assert nc.tolist() == exp_nc
    assert ac.tolist() == exp_ac


def test_single_station_reduces_to_paper_step3():
    # S = 1: candidates == triplets of that station, accept iff >= 2 triplets
    z = [210000, 220000, 230000]   # the trigger station of the 4-station geometry
    rng = np.random.default_rng(7)
    events = [A.narrow_cone_event(z, [int(rng.integers(0, 4)) for _ in range(3)], rng) for _ in range(30)]
    nt, nc, ac = run_events(z, events)
    for e, ev in enumerate(events):
        n = len(ev[0]) * len(ev[1]) * len(ev[2])
        assert nt[e, 0] == n and nc[e] == n and ac[e] == (1 if n >= 2 else 0)


def test_candidate_saturation_is_min_of_cap_and_exact():
    z = list(W.GEOMETRY_6)
    rng = np.random.default_rng(3)
    # 6 stations x (6*6*6 = 216 triplets): 216^6 ~ 1e14 > 2^32 -> saturates; 216^... partial products do not
    ev = [A.narrow_cone_event(z, 6, rng)]
    nt, nc, ac = run_events(z, ev)
    assert nt.tolist() == [[216] * 6] and nc.tolist() == [2 ** 32 - 1] and ac.tolist() == [1]
    # just below the cap: 4 stations, 16*16*16 = 4096 = 2^12 per station -> 2^48 saturates; (3 stations 2^36
    # saturates); 2 stations of 2^12 and two of 2^4 (=16: 2*2*4): 2^32 saturates to 2^32-1, 2^31 does not
    z4 = Z4
    ev = [A.narrow_cone_event(z4, [16, 16, 16, 16, 16, 16, 2, 2, 4, 2, 2, 4], rng),
          A.narrow_cone_event(z4, [16, 16, 16, 16, 16, 16, 2, 2, 4, 2, 2, 2], rng)]
    nt, nc, ac = run_events(z4, ev)
    assert nc.tolist() == [2 ** 32 - 1, 2 ** 31]


# ---------------------------------------------------------------- brute force on tiny events
@pytest.mark.parametrize("case", [c for c in A.adversarial_suite() if c[3] is None], ids=lambda c: c[0])
def test_oracle_equals_brute_force_random(case):
    name, layer_z, events, _ = case
    nt, nc, ac = run_events(layer_z, events)
    nonzero = partial = 0
    for e, ev in enumerate(events):
        bt, bc, ba = brute_force.brute_force_event(layer_z, ev, (1, 100), (2, 100), 2)
        assert nt[e].tolist() == bt, (name, e)
        assert nc[e] == bc and ac[e] == ba, (name, e)
        nonzero += bc > 0
        partial += 0 < bc < int(np.prod(bt))
    assert nonzero >= 3, "the random tiny events must exercise the linking"
    if name == "random_clusters_S3":
        assert partial >= 5, "some events must have chains that are only partially linked"


def test_oracle_equals_brute_force_closed_form_cases_small():
    for name, layer_z, events, exp in A.adversarial_suite():
        if exp is None or name in ("narrow_cone", "duplicates"):
            continue   # 512^4 / 8^6 tuples are too many to enumerate explicitly
        for e, ev in enumerate(events):
            bt, bc, ba = brute_force.brute_force_event(layer_z, ev, (1, 100), (2, 100), 2)
            assert bt == exp[0][e] and bc == exp[1][e] and ba == exp[2][e], (name, e)


def test_brute_force_other_windows_and_thresholds():
    rng = np.random.default_rng(99)
    z3 = W.station_layers_z([60, 100, 150])
    events = [A.random_cluster_event(z3, rng, max_hits=4, n_dirs=1, jitter_slope=0.03) for _ in range(25)]
    for win_in, win_link, mc in [((3, 100), (1, 100), 1), ((1, 64), (5, 100), 3)]:
        nt, nc, ac = run_events(z3, events, win_in, win_link, mc)
        for e, ev in enumerate(events):
            bt, bc, ba = brute_force.brute_force_event(z3, ev, win_in, win_link, mc)
            assert nt[e].tolist() == bt and nc[e] == bc and ac[e] == ba


# ---------------------------------------------------------------- invariances
def test_permutation_invariance_and_batch_splitting():
    cfg = W.CONFIGS[0]
    b = W.generate(cfg, n_events=300)
    g = oracle.geometry(cfg.layer_z)
    nt, nc, ac = oracle.run(g, b.x, b.y, b.off)
    assert nc.sum() > 0
    # shuffle the hits inside every layer
    rng = np.random.default_rng(5)
    x2, y2 = b.x.copy(), b.y.copy()
    off = b.off.astype(np.int64)
    for i in range(off.size - 1):
        lo, hi = off[i], off[i + 1]
        if hi - lo > 1:
            p = rng.permutation(hi - lo)
            x2[lo:hi] = b.x[lo:hi][p]
            y2[lo:hi] = b.y[lo:hi][p]
    nt2, nc2, ac2 = oracle.run(g, x2, y2, b.off)
    assert (nt == nt2).all() and (nc == nc2).all() and (ac == ac2).all()
    # an event's result does not depend on the rest of the batch: split in two, and run a sub-range
    L = cfg.n_layers
    k = 117
    offa = b.off[: k * L + 1]
    offb = b.off[k * L:] - b.off[k * L]
    xa, ya = b.x[: offa[-1]], b.y[: offa[-1]]
    xb, yb = b.x[b.off[k * L]:], b.y[b.off[k * L]:]
    ra = oracle.run(g, xa, ya, offa)
    rb = oracle.run(g, xb, yb, offb)
    assert (np.concatenate([ra[0], rb[0]]) == nt).all()
    assert (np.concatenate([ra[1], rb[1]]) == nc).all()
    assert (np.concatenate([ra[2], rb[2]]) == ac).all()
    rr = oracle.run(g, b.x, b.y, b.off, 40, 90)
    assert (rr[0] == nt[40:90]).all() and (rr[1] == nc[40:90]).all()
    ids = [3, 299, 17, 17, 0]
    rl = oracle.run_list(g, b.x, b.y, b.off, ids)
    assert (rl[0] == nt[ids]).all() and (rl[1] == nc[ids]).all() and (rl[2] == ac[ids]).all()


# ---------------------------------------------------------------- independent second implementation
@pytest.mark.parametrize("cfg_id,n_events", [(0, 1000), (1, 3000), (2, 1500), (3, 12000)])
def test_slope_sorted_counter_agrees(cfg_id, n_events):
    cfg = W.CONFIGS[cfg_id]
    b = W.generate(cfg, n_events=n_events)
    g = oracle.geometry(cfg.layer_z)
    nt, nc, ac = oracle.run(g, b.x, b.y, b.off)
    st, sc, sa, n_eval = oracle.run_slope_sorted(g, b.x, b.y, b.off)
    assert (nt == st).all()
    assert (nc == sc).all()
    assert (ac == sa).all()
    assert nt.sum() > 0 and n_eval > 0


def test_slope_sorted_counter_agrees_on_adversarial():
    for name, layer_z, events, exp in A.adversarial_suite():
        x, y, off = W.batch_from_layers(layer_z, events)
        g = oracle.geometry(layer_z)
        nt, nc, ac = oracle.run(g, x, y, off)
        st, sc, sa, _ = oracle.run_slope_sorted(g, x, y, off)
        assert (nt == st).all() and (nc == sc).all() and (ac == sa).all(), name


# ---------------------------------------------------------------- closed-form background rate
def test_uniform_background_triplet_rate_closed_form():
    # Three independent Poisson(lam) layers, slopes uniform on [-0.35, 0.35]^2: the three slopes must lie
    # within w of each other in x and in y: P(range of 3 iid U(0,1) <= r) = 3r^2 - 2r^3, r = w/0.7.
    # E[triplets per station-event] = lam^3 (3r^2 - 2r^3)^2.
    lam = 60.0
    cfg = W.WorkloadConfig("bg_only", 6000, 77, tuple(W.GEOMETRY_4), 0, lam, signal_fraction=0.0)
    b = W.generate(cfg)
    g = oracle.geometry(cfg.layer_z)
    nt, nc, ac = oracle.run(g, b.x, b.y, b.off)
    r = 0.01 / 0.7
    expect = lam ** 3 * (3 * r * r - 2 * r ** 3) ** 2
    n = nt.size
    mean = nt.mean()
    # triplet counts are roughly Poisson with some clustering: allow 5 sigma of sqrt(expect/n)*1.5
    tol = 5 * 1.5 * math.sqrt(expect / n)
    assert abs(mean - expect) < tol, (mean, expect, tol)
    # and a wrong window convention would be far off: full-width (r/2) gives ~1/16 of it, 2w gives ~16x
    assert abs(mean - expect) < 0.2 * expect


def test_acceptance_follows_layer_efficiency():
    # accepted signal events need every layer of both tracks (no chain may skip a station, R9):
    # complete pairs are (almost) always accepted; window efficiency of a complete track is ~1
    cfg = W.CONFIGS[0]
    b = W.generate(cfg, n_events=4000, seed=11)
    g = oracle.geometry(cfg.layer_z)
    nt, nc, ac = oracle.run(g, b.x, b.y, b.off)
    complete = (b.truth & 2) > 0
    planted = (b.truth & 1) > 0
    assert complete.sum() > 50
    assert ac[complete].mean() > 0.97
    assert ac[~planted].mean() < 0.01          # pure background is essentially never accepted
    frac = complete.sum() / planted.sum()
    assert abs(frac - 0.95 ** 24) < 4 * math.sqrt(0.95 ** 24 * (1 - 0.95 ** 24) / planted.sum())


# ---------------------------------------------------------------- stored fixtures still match the oracle
def test_golden_files_match_live_oracle():
    from tests.golden_io import golden_cases, read_golden
    cases = golden_cases()
    assert len(cases) >= 4
    for cid, n, path in cases:
        cfg = W.CONFIGS[cid]
        b = W.generate(cfg, n_events=n)
        g = oracle.geometry(cfg.layer_z, cfg.win_in, cfg.win_link, cfg.min_candidates)
        nt, nc, ac = oracle.run(g, b.x, b.y, b.off)
        gt, gc, ga = read_golden(path, n, cfg.n_stations)
        assert (nt == gt).all() and (nc == gc).all() and (ac == ga).all(), path


# ---------------------------------------------------------------- N_eval of the slope-sorted counter
def test_n_eval_hand_counts():
    """oracle.run_slope_sorted's evaluation counter (the work term of the integer-pipe roofline)
    against hand counts.  Per middle hit h1: one y-evaluation for every h0 in its x-band; for every (h0,h1) that
    passes in y, two evaluations for every h2 in the x-band of both; per pair of consecutive stations two
    evaluations for every (middle hit with triplets of s-1) x (middle hit with triplets of s)."""
    z1 = [60000, 70000, 80000]
    g1 = oracle.geometry(z1, (1, 100), (2, 100), 2)

    def n_eval(layer_z, g, events):
        x, y, off = W.batch_from_layers(layer_z, events)
        return int(oracle.run_slope_sorted(g, x, y, off)[3])

    # (a) one exact line: 1 y-evaluation (h0,h1) + 2 for the single h2
    assert n_eval(z1, g1, [A.planted_lines_event(z1, [(100, -50)])]) == 3
    # (b) n0 = 2, n1 = 1, n2 = 2, all on the axis: 2 y-evaluations, both pass, 2 h2 each -> 2 + 2*2*2 = 10
    assert n_eval(z1, g1, [[[(0, 0), (1, 1)], [(0, 0)], [(0, 0), (2, -1)]]]) == 10
    # (c) an h0 outside the x-band of h1 (slope 0.02 vs 0) is never evaluated; one inside the x-band but outside
    #     in y costs its y-evaluation only: layer 0 = {far in x, in x-band but far in y}, one h1, one h2 -> 1
    assert n_eval(z1, g1, [[[(1200, 0), (0, 3000)], [(0, 0)], [(0, 0)]]]) == 1
    # (d) two stations, two separated exact lines: per station 2 middle hits x (1 + 2) = 6 (the other line's hits are
    #     outside every x-band); link: 2 x 2 middle hits x 2 = 8 -> 6 + 6 + 8 = 20
    z2 = list(W.GEOMETRY_4)[:6]
    g2 = oracle.geometry(z2, (1, 100), (2, 100), 2)
    assert n_eval(z2, g2, [A.planted_lines_event(z2, [(-200, 10), (150, 40)])]) == 20
    # (e) a station without a triplet stops the linking: station 0 has a line, station 1 misses layer 1 -> 3 + 0
    ev = A.planted_lines_event(z2, [(100, 100)])
    ev[4] = []
    assert n_eval(z2, g2, [ev]) == 3
