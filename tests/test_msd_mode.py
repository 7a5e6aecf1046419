"""The paper's own selection, literally (section 3.2).

CPU: oracle/msd_oracle.c (exact 128-bit evaluation of the MSD cut) is pinned against hand-computed residuals,
exact lines, an independent evaluation with Python fractions, float64 least squares away from the threshold,
closed-form counts and invariances.
GPU: cbm_trigger_msd_device against the oracle, bit-exact passing-triplet counts and decisions.
"""
from fractions import Fraction

import numpy as np
import pytest

import oracle
from paper_1810_11966_b200 import workloads as W

Z3 = [1000, 2000, 3000]  # one station, z = k, 2k, 3k


def one_event(layers_x, layers_y):
    x = np.concatenate([np.asarray(v, dtype=np.int32) for v in layers_x])
    y = np.concatenate([np.asarray(v, dtype=np.int32) for v in layers_y])
    off = np.concatenate([[0], np.cumsum([len(v) for v in layers_x])]).astype(np.uint32)
    return x, y, off


def fraction_count(layer_z, station, x, y, off, e, thr_x, thr_y, ndf):
    """Independent exact evaluation: fitted slope, residuals and MSD as rationals."""
    L = len(layer_z)
    z = [layer_z[3 * station + l] for l in range(3)]
    o = [int(off[e * L + 3 * station + l]) for l in range(4)]
    n = 0
    for i0 in range(o[0], o[1]):
        for i1 in range(o[1], o[2]):
            for i2 in range(o[2], o[3]):
                ok = True
                for v, thr in ((x, thr_x), (y, thr_y)):
                    pts = [int(v[i0]), int(v[i1]), int(v[i2])]
                    m = Fraction(sum(p * zz for p, zz in zip(pts, z)), sum(zz * zz for zz in z))  # least squares through 0
                    ssr = sum((p - m * zz) ** 2 for p, zz in zip(pts, z))
                    ok &= ssr / ndf <= Fraction(thr[0], thr[1]) * 10 ** 6  # cm^2 -> (10 um)^2
                n += ok
    return n


# ------------------------------------------------------------------------------------------------ CPU pins
@pytest.mark.parametrize("ndf,thr,axis,d_pass", [(2, (3, 100), "x", 409), (2, (25, 1000), "y", 374), (3, (3, 100), "x", 501)])
def test_hand_computed_residuals(ndf, thr, axis, d_pass):
    """z = k, 2k, 3k and v = 0, 0, d: m = 3d/(14k), SSR = d^2 - 9d^2/14 = 5 d^2 / 14, so MSD = 5 d^2 / (14 ndf)
    against thr * 10^6: ndf 2, 0.03 -> d <= 409.88; ndf 2, 0.025 -> d <= 374.17; ndf 3, 0.03 -> d <= 501.99."""
    for d, want in ((d_pass, 1), (d_pass + 1, 0), (-d_pass, 1), (-d_pass - 1, 0)):
        v, w = [[0], [0], [d]], [[0], [0], [0]]
        x, y, off = one_event(v, w) if axis == "x" else one_event(w, v)
        par = oracle.msd_params(Z3, thr_x=thr if axis == "x" else (3, 100), thr_y=thr if axis == "y" else (25, 1000),
                                ndf=ndf, min_triplets=1)
        npass, ac = oracle.run_msd(par, x, y, off)
        assert npass.tolist() == [want] and ac.tolist() == [want], (d, want)


def test_exact_lines_and_closed_form_count():
    # hits exactly on x = p z / 1000, y = q z / 1000: residuals 0; duplicates count separately: n0*n1*n2 triplets
    z = W.GEOMETRY_4
    zt = z[9:12]
    lx = [[37 * zz // 1000] * n for zz, n in zip(zt, (2, 3, 4))]
    ly = [[-91 * zz // 1000] * n for zz, n in zip(zt, (2, 3, 4))]
    pad = [[]] * 9
    x, y, off = one_event(pad + lx, pad + ly)
    npass, ac = oracle.run_msd(oracle.msd_params(z), x, y, off)
    assert npass.tolist() == [24] and ac.tolist() == [1]
    # a single triplet does not select the event (at least two)
    x, y, off = one_event(pad + [[v[0]] for v in lx], pad + [[v[0]] for v in ly])
    npass, ac = oracle.run_msd(oracle.msd_params(z), x, y, off)
    assert npass.tolist() == [1] and ac.tolist() == [0]


def test_against_fractions_on_small_events_near_the_threshold():
    rng = np.random.default_rng(3)
    z = W.GEOMETRY_4
    total = 0
    for trial in range(8):
        ndf = (2, 3)[trial % 2]
        layers_x, layers_y = [], []
        for l in range(12):
            n = int(rng.integers(2, 6)) if l >= 9 else int(rng.integers(0, 3))
            tx, ty = rng.uniform(-0.3, 0.3, n), rng.uniform(-0.3, 0.3, n)
            if l >= 9:  # a few common directions + noise of the size of the cut: about half of the triplets pass
                tx, ty = np.array([0.1, -0.2, 0.1, 0.05, -0.2])[:n], np.array([0.0, 0.15, 0.0, -0.1, 0.15])[:n]
            layers_x.append(np.rint(tx * z[l] + rng.normal(0, 120, n)).astype(np.int32))
            layers_y.append(np.rint(ty * z[l] + rng.normal(0, 120, n)).astype(np.int32))
        x, y, off = one_event(layers_x, layers_y)
        par = oracle.msd_params(z, ndf=ndf)
        npass, ac = oracle.run_msd(par, x, y, off)
        want = fraction_count(z, 3, x, y, off, 0, (3, 100), (25, 1000), ndf)
        assert npass[0] == want and ac[0] == (want >= 2)
        total += want
    assert total >= 4  # the construction does produce passing (and failing) triplets


def test_against_float64_least_squares_away_from_the_threshold():
    rng = np.random.default_rng(8)
    z = np.array(Z3, dtype=np.float64)
    checked = 0
    for _ in range(400):
        t = rng.uniform(-0.3, 0.3, 2)
        vx = np.rint(t[0] * z + rng.normal(0, 200, 3)).astype(np.int32)
        vy = np.rint(t[1] * z + rng.normal(0, 200, 3)).astype(np.int32)
        msd = []
        for v in (vx, vy):
            m, res, _, _ = np.linalg.lstsq(z[:, None], v.astype(np.float64), rcond=None)
            msd.append(float(((v - m[0] * z) ** 2).sum()) / 2 / 1e6)  # cm^2 per degree of freedom
        if abs(msd[0] / 0.03 - 1) < 1e-6 or abs(msd[1] / 0.025 - 1) < 1e-6:
            continue
        x, y, off = one_event([[vx[0]], [vx[1]], [vx[2]]], [[vy[0]], [vy[1]], [vy[2]]])
        npass, _ = oracle.run_msd(oracle.msd_params(Z3, min_triplets=1), x, y, off)
        assert int(npass[0]) == int(msd[0] <= 0.03 and msd[1] <= 0.025)
        checked += 1
    assert checked > 350


def test_only_the_trigger_station_and_no_hit_order_matter():
    cfg = W.CONFIGS[0]
    b = W.generate(cfg, n_events=200)
    par = oracle.msd_params(cfg.layer_z)
    npass, ac = oracle.run_msd(par, b.x, b.y, b.off)
    assert ac.sum() > 0  # planted muon pairs (smear 0.1 cm: MSD ~ 0.01 cm^2) are selected
    rng = np.random.default_rng(0)
    x2, y2 = b.x.copy(), b.y.copy()
    L = cfg.n_layers
    for e in range(200):
        for l in range(L):
            a, c = int(b.off[e * L + l]), int(b.off[e * L + l + 1])
            if l < L - 3:      # other stations: any content
                x2[a:c] = rng.integers(-1000, 1000, c - a)
            else:              # trigger station: permuted
                perm = rng.permutation(c - a)
                x2[a:c], y2[a:c] = b.x[a:c][perm], b.y[a:c][perm]
    n2, a2 = oracle.run_msd(par, x2, y2, b.off)
    assert np.array_equal(n2, npass) and np.array_equal(a2, ac)
    # another trigger station gives another answer, and event ranges concatenate
    n0, _ = oracle.run_msd(oracle.msd_params(cfg.layer_z, station=0), b.x, b.y, b.off)
    assert not np.array_equal(n0, npass)
    nA, _ = oracle.run_msd(par, b.x, b.y, b.off, 0, 77)
    nB, _ = oracle.run_msd(par, b.x, b.y, b.off, 77, 200)
    assert np.array_equal(np.concatenate([nA, nB]), npass)


# ------------------------------------------------------------------------------------------------ GPU parity
def _gpu_msd(cfg_layer_z, x, y, off, n_events, **kw):
    import torch
    from paper_1810_11966_b200 import binding as K
    with K.Trigger(cfg_layer_z, max(n_events, 1), max(int(off[-1]), 1), n_slots=0) as trig:
        dx = torch.from_numpy(np.ascontiguousarray(x, np.int32)).cuda()
        dy = torch.from_numpy(np.ascontiguousarray(y, np.int32)).cuda()
        do = torch.from_numpy(np.ascontiguousarray(off, np.uint32).view(np.int32)).cuda()
        dn = torch.full((max(n_events, 1),), -1, dtype=torch.int32, device="cuda")
        da = torch.full((max(n_events, 1),), 9, dtype=torch.uint8, device="cuda")
        trig.msd_device(K.make_msd_params(**kw), n_events, int(off[-1]), dx, dy, do, dn, da)
        torch.cuda.synchronize()
        return dn.cpu().numpy().view(np.uint32)[:n_events], da.cpu().numpy()[:n_events]


@pytest.mark.gpu
@pytest.mark.parametrize("cid,n", [(0, 1000), (1, 500), (3, 200), (2, 250)])
def test_msd_mode_matches_oracle_on_the_workloads(cid, n):
    cfg = W.CONFIGS[cid]
    b = W.generate(cfg, n_events=n)
    for kw in ({}, {"ndf": 3, "station": 0, "thr_x": (1, 10), "thr_y": (1, 20), "min_triplets": 1}):
        par = oracle.msd_params(cfg.layer_z, **kw)
        want_n, want_a = oracle.run_msd(par, b.x, b.y, b.off)
        got_n, got_a = _gpu_msd(cfg.layer_z, b.x, b.y, b.off, n, **kw)
        assert np.array_equal(got_n, want_n) and np.array_equal(got_a, want_a), (cfg.name, kw)


@pytest.mark.gpu
def test_msd_mode_near_the_threshold_and_edges():
    rng = np.random.default_rng(21)
    z = W.GEOMETRY_4
    n_events = 300
    xs, ys, counts = [], [], []
    for e in range(n_events):
        base = rng.uniform(-0.3, 0.3, 2)                # one direction per event; noise of the size of the cut
        for l in range(12):
            n = int(rng.integers(0, 9))
            if e % 50 == 0 and l == 10:
                n = 0                                   # an empty layer: nothing passes
            xs.append(np.rint(base[0] * z[l] * (l >= 9) + rng.normal(0, 170, n)).astype(np.int32))
            ys.append(np.rint(base[1] * z[l] * (l >= 9) + rng.normal(0, 170, n)).astype(np.int32))
            counts.append(n)
    x, y = np.concatenate(xs), np.concatenate(ys)
    off = np.concatenate([[0], np.cumsum(counts)]).astype(np.uint32)
    want_n, want_a = oracle.run_msd(oracle.msd_params(z), x, y, off)
    got_n, got_a = _gpu_msd(z, x, y, off, n_events)
    assert np.array_equal(got_n, want_n) and np.array_equal(got_a, want_a)
    assert 0.1 < (want_n > 0).mean() < 0.95           # the cut is exercised on both sides
    # hand case through the device: 409 passes, 410 fails
    for d, w in ((409, 1), (410, 0)):
        hx, hy, ho = one_event([[0], [0], [d]], [[0], [0], [0]])
        got_n, got_a = _gpu_msd(Z3, hx, hy, ho, 1, min_triplets=1)
        assert got_n.tolist() == [w] and got_a.tolist() == [w]


@pytest.mark.gpu
def test_msd_malformed_event_is_never_accepted():
    """include/cbm_trigger.h: an event with malformed offsets has n_passing = 0 and accept = 0, also with
    min_triplets = 0 (which accepts every well-formed event)."""
    import torch
    from paper_1810_11966_b200 import binding as K
    cfg = W.CONFIGS[0]
    n = 40
    b = W.generate(cfg, n_events=n)
    L = cfg.n_layers
    off = b.off.copy()
    off[7 * L + (L - 2)] = off[7 * L + (L - 1)] + 5   # trigger station of event 7: offsets not monotone
    par = K.make_msd_params(min_triplets=0)
    with K.Trigger(cfg.layer_z, n, b.n_hits, n_slots=0) as trig:
        dx = torch.from_numpy(np.concatenate([b.x, np.zeros(8, np.int32)])).cuda()
        dy = torch.from_numpy(np.concatenate([b.y, np.zeros(8, np.int32)])).cuda()
        do = torch.from_numpy(off.view(np.int32)).cuda()
        dnp = torch.full((n,), 9, dtype=torch.int32, device="cuda")
        dac = torch.full((n,), 9, dtype=torch.uint8, device="cuda")
        trig.msd_device(par, n, b.n_hits, dx, dy, do, dnp, dac)
        torch.cuda.synchronize()
        ac = dac.cpu().numpy()
        assert ac[7] == 0 and int(dnp[7].item()) == 0
        assert ac[np.arange(n) != 7].all()


@pytest.mark.gpu
def test_msd_paper_table1_workload_full_size():
    """The paper-literal mode at bench.py --mode msd size: 1,000,000 events of the Table-1-shaped workload
    (one station, about 15 hits per layer), every event against oracle/msd_oracle.c."""
    import torch
    from paper_1810_11966_b200 import binding as K
    from tests.helpers import oracle_msd_mt
    cfg = W.PAPER_TABLE1
    E = 1_000_000
    b = W.generate(cfg, n_events=E)
    assert 40 < b.n_hits / E < 50
    dx = torch.from_numpy(np.concatenate([b.x, np.zeros(8, np.int32)])).cuda()
    dy = torch.from_numpy(np.concatenate([b.y, np.zeros(8, np.int32)])).cuda()
    do = torch.from_numpy(b.off.view(np.int32)).cuda()
    dnp = torch.full((E,), -1, dtype=torch.int32, device="cuda")
    dac = torch.full((E,), 9, dtype=torch.uint8, device="cuda")
    with K.Trigger(cfg.layer_z, E, b.n_hits, n_slots=0) as trig:
        trig.msd_device(K.make_msd_params(), E, b.n_hits, dx, dy, do, dnp, dac)
        torch.cuda.synchronize()
    want = oracle_msd_mt(oracle.msd_params(cfg.layer_z), b.x, b.y, b.off)
    assert np.array_equal(dnp.cpu().numpy().view(np.uint32), want[0]) and np.array_equal(dac.cpu().numpy(), want[1])
    assert 0 < int(want[1].sum()) < E // 20
