"""Event building from a free-streaming, time-stamped hit stream (section 8 "Outlook"; DESIGN.md
reading B9: a gap of more than t_gap between consecutive records opens a new event): pins of the oracle
(oracle.build_events) and GPU parity of cbm_trigger_build_events_device, alone and in front of the input filter and
the selection."""
import numpy as np
import pytest

import oracle
from paper_1810_11966_b200 import workloads as W


def test_build_events_hand_cases():
    # gaps: 1, 4, 0, 6, 5, 1  with t_gap = 4: a new event where the gap is > 4, i.e. before records 4 and 5
    t = [10, 11, 15, 15, 21, 26, 27]
    assert oracle.build_events(t, 4).tolist() == [0, 4, 5, 7]
    assert oracle.build_events(t, 5).tolist() == [0, 4, 7]       # the gap of 5 no longer splits (closed: gap <= t_gap stays)
    assert oracle.build_events(t, 0).tolist() == [0, 1, 2, 4, 5, 6, 7]  # only simultaneous records stay together
    assert oracle.build_events(t, 100).tolist() == [0, 7]
    assert oracle.build_events([], 4).tolist() == [0]
    assert oracle.build_events([5], 4).tolist() == [0, 1]
    # a record that is earlier than its predecessor (negative gap) does not open an event: stream order rules
    assert oracle.build_events([10, 30, 12, 40], 5).tolist() == [0, 1, 3, 4]
    # int32 extremes: the difference is taken without overflow
    assert oracle.build_events([-2**31, 2**31 - 1], 2**31).tolist() == [0, 1, 2]


def test_build_events_closed_forms_and_invariants():
    rng = np.random.default_rng(3)
    # equidistant records, spacing d: one event if d <= gap, n events otherwise
    for d, gap, want in [(3, 3, 1), (3, 2, 50), (1, 0, 50), (0, 0, 1)]:
        assert oracle.build_events(np.arange(50) * d, gap).size - 1 == want
    t = np.cumsum(rng.integers(0, 12, size=5000))
    for gap in (0, 3, 7, 20):
        eo = oracle.build_events(t, gap).astype(np.int64)
        # the definition restated with numpy's own difference (not the oracle's loop)
        assert np.array_equal(eo[1:-1], np.flatnonzero(np.diff(t) > gap) + 1)
        assert eo[0] == 0 and eo[-1] == t.size and np.all(np.diff(eo) > 0)
        for k in range(eo.size - 1):  # no gap above t_gap inside an event; one above it in front of every later event
            seg = t[eo[k]:eo[k + 1]]
            assert seg.size == 1 or np.max(np.diff(seg)) <= gap
            assert k == 0 or t[eo[k]] - t[eo[k] - 1] > gap
    # a larger gap can only merge events: the boundaries of gap g2 >= g1 are a subset of those of g1
    b3, b7 = set(oracle.build_events(t, 3).tolist()), set(oracle.build_events(t, 7).tolist())
    assert b7 <= b3


def test_build_events_recovers_well_separated_interactions():
    # interactions further apart than spread + t_gap come back exactly; the filter then gives the batch back
    b = W.generate(W.CONFIGS[0], n_events=40)
    xyz, t, ev_off = W.timed_stream(b, other_hits_per_event=30, mean_dt=10_000, spread=8, seed=4)
    gaps = t[ev_off[1:-1].astype(np.int64)] - t[ev_off[1:-1].astype(np.int64) - 1]
    assert gaps.min() > 20
    eo = oracle.build_events(t, 20)
    assert np.array_equal(eo, ev_off)
    x, y, off = oracle.filter_layers(xyz, eo, b.cfg.layer_z)
    assert np.array_equal(x, b.x) and np.array_equal(y, b.y) and np.array_equal(off, b.off)


def timed_case(cid, n, other, mean_dt, spread, seed):
    cfg = W.CONFIGS[cid]
    b = W.generate(cfg, n_events=n)
    xyz, t, _ = W.timed_stream(b, other_hits_per_event=other, mean_dt=mean_dt, spread=spread, seed=seed)
    return cfg, xyz, t


@pytest.mark.gpu
@pytest.mark.parametrize("cid,n,other,mean_dt,spread,gap", [(0, 3000, 60, 100, 8, 12), (3, 3000, 20, 100, 10, 15), (0, 500, 10, 5, 3, 0),
                                                            (1, 400, 100, 1000, 20, 25)])
def test_timeslice_pipeline_matches_oracle(cid, n, other, mean_dt, spread, gap):
    """free-streaming records -> events (time gaps) -> MUCH hits by layer -> selection, all on the device, against the
    same chain on the oracle side.  At 100 ns mean distance many interactions pile up into one built event."""
    import torch
    from paper_1810_11966_b200 import binding as K
    cfg, xyz, t = timed_case(cid, n, other, mean_dt, spread, seed=cid + 7)
    eo = oracle.build_events(t, gap)
    E = eo.size - 1
    x, y, off = oracle.filter_layers(xyz, eo, cfg.layer_z)
    L, S = cfg.n_layers, cfg.n_stations
    per_layer = np.diff(off.astype(np.int64))
    keep = np.ones(E, dtype=bool)
    if per_layer.size:  # built events above the per-layer capacity are rejected by the selection, as documented
        keep = per_layer.reshape(E, L).max(axis=1) <= 4096
    g = oracle.geometry(cfg.layer_z, cfg.win_in, cfg.win_link, cfg.min_candidates)
    want = oracle.run(g, x, y, off)
    N = xyz.shape[0]
    with K.Trigger(cfg.layer_z, max(E, 1), max(N, 1), win_in=cfg.win_in, win_link=cfg.win_link, min_candidates=cfg.min_candidates,
                   n_slots=0) as trig:
        dxyz = torch.from_numpy(xyz.reshape(-1)).cuda()
        dt = torch.from_numpy(t).cuda()
        deo = torch.full((N + 1,), -1, dtype=torch.int32, device="cuda")
        n_built = trig.build_events_device(N, dt, gap, deo)
        assert n_built == E
        assert np.array_equal(deo.cpu().numpy().view(np.uint32)[:E + 1], eo)
        ox = torch.full((N + 8,), 77, dtype=torch.int32, device="cuda")
        oy = torch.full((N + 8,), 77, dtype=torch.int32, device="cuda")
        oo = torch.full((E * L + 1,), -1, dtype=torch.int32, device="cuda")
        trig.filter_device(E, N, dxyz, deo, ox, oy, oo)
        torch.cuda.synchronize()
        assert np.array_equal(oo.cpu().numpy().view(np.uint32), off)
        nh = int(off[-1])
        assert np.array_equal(ox.cpu().numpy()[:nh], x) and np.array_equal(oy.cpu().numpy()[:nh], y)
        dnt = torch.zeros(E * S, dtype=torch.int32, device="cuda")
        dnc = torch.zeros(E, dtype=torch.int32, device="cuda")
        dac = torch.zeros(E, dtype=torch.uint8, device="cuda")
        trig.run_device(E, nh, ox, oy, oo, dnt, dnc, dac)
        torch.cuda.synchronize()
    assert keep.all()
    assert np.array_equal(dnt.cpu().numpy().view(np.uint32).reshape(E, S), want[0])
    assert np.array_equal(dnc.cpu().numpy().view(np.uint32), want[1]) and np.array_equal(dac.cpu().numpy(), want[2])


@pytest.mark.gpu
def test_build_events_device_small_cases():
    import torch
    from paper_1810_11966_b200 import binding as K
    cases = [([10, 11, 15, 15, 21, 26, 27], 4), ([10, 11, 15, 15, 21, 26, 27], 0), ([], 4), ([5], 4), ([10, 30, 12, 40], 5),
             ([-2**31, 2**31 - 1], 2**31 - 1), (list(range(0, 30000, 3)), 2), (list(range(0, 30000, 3)), 3), ([7] * 5000, 0)]
    with K.Trigger([60000, 70000, 80000], 16, 16, n_slots=0) as trig:
        for t, gap in cases:
            want = oracle.build_events(t, gap)
            n = len(t)
            dt = torch.tensor(t if n else [0], dtype=torch.int32, device="cuda")
            deo = torch.full((n + 1,), -1, dtype=torch.int32, device="cuda")
            ne = trig.build_events_device(n, dt, gap, deo)
            assert ne == want.size - 1
            assert np.array_equal(deo.cpu().numpy().view(np.uint32)[:ne + 1], want)


@pytest.mark.gpu
def test_record_count_limit_is_checked_before_anything_runs():
    """include/cbm_trigger.h: n_records <= CBM_TRIGGER_MAX_INDEX = 2^32 - 8192 for the stream calls (above it the
    uint32 block arithmetic of the scans would wrap and truncate the output silently); refused with CBM_ERR_CAPACITY."""
    import torch
    from paper_1810_11966_b200 import binding as K
    small = torch.zeros(16, dtype=torch.int32, device="cuda")
    with K.Trigger([60000, 70000, 80000], 16, 16, n_slots=0) as trig:
        for n_records in (0xFFFFE000 + 1, 2**32 - 1, 2**32):
            with pytest.raises(K.CbmTriggerError) as ei:
                trig.build_events_device(n_records, small, 4, small)
            assert ei.value.code == K.CBM_ERR_CAPACITY
            with pytest.raises(K.CbmTriggerError) as ei:
                trig.filter_device(1, n_records, small, small, small, small, small)
            assert ei.value.code == K.CBM_ERR_CAPACITY
        # the handle is still usable
        t = torch.tensor([1, 2, 9], dtype=torch.int32, device="cuda")
        eo = torch.full((4,), -1, dtype=torch.int32, device="cuda")
        assert trig.build_events_device(3, t, 4, eo) == 2 and eo.cpu().tolist()[:3] == [0, 2, 3]
