"""The list of selected events.

CPU: oracle.selected is pinned against numpy's flatnonzero and hand-written cases.
GPU: cbm_trigger_fetch_selected / cbm_trigger_select_device against oracle.selected, bit-exact (index work).
"""
import numpy as np
import pytest

import oracle
from paper_1810_11966_b200 import workloads as W


# ------------------------------------------------------------------------------------------------ CPU pins
def test_oracle_selected_hand_cases():
    assert oracle.selected(np.zeros(0, dtype=np.uint8)).tolist() == []
    assert oracle.selected(np.array([0, 0, 0], dtype=np.uint8)).tolist() == []
    assert oracle.selected(np.array([1, 0, 1, 1, 0], dtype=np.uint8)).tolist() == [0, 2, 3]
    assert oracle.selected(np.array([0, 0, 0, 0, 7], dtype=np.uint8)).tolist() == [4]  # any non-zero byte counts
    assert oracle.selected(np.ones(5, dtype=np.uint8)).dtype == np.uint32


def test_oracle_selected_against_library_routine():
    rng = np.random.default_rng(11)
    for n, p in ((1, 0.5), (17, 0.3), (4096, 0.01), (4097, 0.5), (10000, 0.999)):
        a = (rng.random(n) < p).astype(np.uint8)
        got = oracle.selected(a)
        assert np.array_equal(got, np.flatnonzero(a).astype(np.uint32))
        assert np.all(np.diff(got.astype(np.int64)) > 0)  # ascending, no duplicates
        assert got.size == int(a.sum())


def test_oracle_selected_is_the_accept_flags_of_the_oracle():
    cfg = W.CONFIGS[0]
    b = W.generate(cfg, n_events=400)
    g = oracle.geometry(cfg.layer_z, cfg.win_in, cfg.win_link, cfg.min_candidates)
    _, nc, ac = oracle.run(g, b.x, b.y, b.off)
    ids = oracle.selected(ac)
    assert ids.size > 0
    assert np.all(nc[ids] >= cfg.min_candidates) and np.all(np.delete(nc, ids) < cfg.min_candidates)


# ------------------------------------------------------------------------------------------------ GPU parity
@pytest.mark.gpu
@pytest.mark.parametrize("cid,n", [(0, 1000), (1, 3000), (3, 20000), (2, 1500)])
def test_fetch_selected_matches_oracle(cid, n):
    from paper_1810_11966_b200 import binding as K
    from tests.helpers import oracle_mt
    cfg = W.CONFIGS[cid]
    b = W.generate(cfg, n_events=n)
    g = oracle.geometry(cfg.layer_z, cfg.win_in, cfg.win_link, cfg.min_candidates)
    _, _, oac = oracle_mt(g, b.x, b.y, b.off)
    with K.Trigger(cfg.layer_z, n, b.n_hits, win_in=cfg.win_in, win_link=cfg.win_link,
                   min_candidates=cfg.min_candidates, n_slots=1) as trig:
        trig.upload_events(0, b.x, b.y, b.off)
        trig.run(0)
        ids_before = trig.fetch_selected(0)            # before fetch_results
        _, _, ac = trig.fetch_results(0, n)
        ids_after = trig.fetch_selected(0)             # and after it
        assert np.array_equal(ac, oac)
        want = oracle.selected(oac)
        assert np.array_equal(ids_before, want) and np.array_equal(ids_after, want)
        # too little room: the count is still reported, nothing is written
        if want.size > 1:
            with pytest.raises(K.CbmTriggerError) as ei:
                trig.fetch_selected(0, capacity=want.size - 1)
            assert ei.value.code == K.CBM_ERR_CAPACITY
        # a new upload invalidates the list
        trig.upload_events(0, b.x, b.y, b.off)
        with pytest.raises(K.CbmTriggerError) as ei:
            trig.fetch_selected(0)
        assert ei.value.code == K.CBM_ERR_STATE


@pytest.mark.gpu
def test_fetch_selected_none_all_and_empty():
    from paper_1810_11966_b200 import binding as K
    cfg = W.CONFIGS[0]
    b = W.generate(cfg, n_events=300)
    # min_candidates = 0 accepts every event (B3); a huge threshold accepts none
    for minc, want in ((0, np.arange(300, dtype=np.uint32)), (0xFFFFFFFF, np.zeros(0, dtype=np.uint32))):
        with K.Trigger(cfg.layer_z, 300, b.n_hits, min_candidates=minc, n_slots=1) as trig:
            trig.upload_events(0, b.x, b.y, b.off)
            trig.run(0)
            assert np.array_equal(trig.fetch_selected(0), want)
    with K.Trigger(cfg.layer_z, 8, 8, n_slots=1) as trig:  # empty batch
        trig.upload_events(0, np.zeros(0, np.int32), np.zeros(0, np.int32), np.zeros(1, np.uint32), 0, 0)
        trig.run(0)
        assert trig.fetch_selected(0).size == 0


@pytest.mark.gpu
@pytest.mark.parametrize("n", [1, 15, 16, 4095, 4096, 4097, 70001])
def test_select_device_on_arbitrary_flags(n):
    """The compaction alone on device arrays: block boundaries (4096 events), ragged tails, unaligned start."""
    import torch
    from paper_1810_11966_b200 import binding as K
    rng = np.random.default_rng(n)
    cfg = W.CONFIGS[0]
    with K.Trigger(cfg.layer_z, 80000, 16, n_slots=0) as trig:
        for p, shift in ((0.02, 0), (0.5, 0), (1.0, 0), (0.3, 3)):
            a = (rng.random(n + shift) < p).astype(np.uint8)
            a[a != 0] = rng.integers(1, 256, size=int(a.sum()), dtype=np.uint8)  # any non-zero byte
            d_a = torch.from_numpy(a).cuda()
            d_ids = torch.full((n,), 0xFFFFFFF, dtype=torch.int32, device="cuda")
            d_n = torch.zeros(1, dtype=torch.int32, device="cuda")
            trig.select_device(n, d_a[shift:], d_ids, d_n)
            torch.cuda.synchronize()
            want = oracle.selected(a[shift:])
            assert int(d_n.item()) == want.size
            assert np.array_equal(d_ids.cpu().numpy().view(np.uint32)[:want.size], want)


# ------------------------------------------------------------------------------------------------ gather
def test_oracle_gather_hand_case_and_identity():
    # 2 layers per "event" for brevity (the routine only needs the layer count): event 0: [1,2 | 3], event 1: [ | 4,5],
    # event 2: [6 | ]
    x = np.array([1, 2, 3, 4, 5, 6], np.int32)
    y = -x
    off = np.array([0, 2, 3, 3, 5, 6, 6], np.uint32)
    gx, gy, go = oracle.gather(x, y, off, 2, [2, 0])
    assert gx.tolist() == [6, 1, 2, 3] and gy.tolist() == [-6, -1, -2, -3] and go.tolist() == [0, 1, 1, 3, 4]
    gx, gy, go = oracle.gather(x, y, off, 2, [])
    assert gx.size == 0 and go.tolist() == [0]
    # every event in order gives the batch back
    cfg = W.CONFIGS[0]
    b = W.generate(cfg, n_events=50)
    gx, gy, go = oracle.gather(b.x, b.y, b.off, cfg.n_layers, np.arange(50))
    assert np.array_equal(gx, b.x) and np.array_equal(gy, b.y) and np.array_equal(go, b.off)
    # the gathered batch of the selected events gives the selected events' results
    g = oracle.geometry(cfg.layer_z, cfg.win_in, cfg.win_link, cfg.min_candidates)
    nt, nc, ac = oracle.run(g, b.x, b.y, b.off)
    ids = oracle.selected(ac)
    gx, gy, go = oracle.gather(b.x, b.y, b.off, cfg.n_layers, ids)
    nt2, nc2, ac2 = oracle.run(g, gx, gy, go)
    assert np.array_equal(nt2, nt[ids]) and np.array_equal(nc2, nc[ids]) and ac2.all()


@pytest.mark.gpu
@pytest.mark.parametrize("cid,n,minc", [(0, 1000, 2), (3, 9000, 2), (1, 700, 0), (2, 600, 2), (0, 300, 0xFFFFFFFF)])
def test_gather_device_matches_oracle(cid, n, minc):
    """run_device -> select_device -> gather_device on device arrays, against oracle.selected / oracle.gather."""
    import torch
    from paper_1810_11966_b200 import binding as K
    from tests.helpers import oracle_mt
    cfg = W.CONFIGS[cid]
    b = W.generate(cfg, n_events=n)
    g = oracle.geometry(cfg.layer_z, cfg.win_in, cfg.win_link, minc)
    _, _, oac = oracle_mt(g, b.x, b.y, b.off)
    want_ids = oracle.selected(oac)
    wx, wy, wo = oracle.gather(b.x, b.y, b.off, cfg.n_layers, want_ids)
    S, L = cfg.n_stations, cfg.n_layers
    with K.Trigger(cfg.layer_z, n, b.n_hits, win_in=cfg.win_in, win_link=cfg.win_link, min_candidates=minc, n_slots=0) as trig:
        pad = lambda a: torch.from_numpy(np.concatenate([a.view(np.int32), np.zeros(8, np.int32)])).cuda()
        dx, dy = pad(b.x), pad(b.y)
        do = torch.from_numpy(b.off.view(np.int32)).cuda()
        dnt = torch.zeros(n * S, dtype=torch.int32, device="cuda")
        dnc = torch.zeros(n, dtype=torch.int32, device="cuda")
        dac = torch.zeros(n, dtype=torch.uint8, device="cuda")
        dids = torch.zeros(n, dtype=torch.int32, device="cuda")
        dn = torch.zeros(1, dtype=torch.int32, device="cuda")
        ox = torch.full((b.n_hits + 1,), 77, dtype=torch.int32, device="cuda")
        oy = torch.full((b.n_hits + 1,), 77, dtype=torch.int32, device="cuda")
        oo = torch.full((n * L + 1,), -1, dtype=torch.int32, device="cuda")
        on = torch.zeros(1, dtype=torch.int64, device="cuda")
        trig.run_device(n, b.n_hits, dx, dy, do, dnt, dnc, dac)
        trig.select_device(n, dac, dids, dn)
        trig.gather_device(n, b.n_hits, dx, dy, do, dids, dn, ox, oy, oo, on)
        torch.cuda.synchronize()
        ns, nh = int(dn.item()), int(on.item())
        assert ns == want_ids.size and nh == wx.size
        assert np.array_equal(dids.cpu().numpy().view(np.uint32)[:ns], want_ids)
        assert np.array_equal(oo.cpu().numpy().view(np.uint32)[:ns * L + 1], wo)
        assert np.array_equal(ox.cpu().numpy()[:nh], wx) and np.array_equal(oy.cpu().numpy()[:nh], wy)
        assert int(ox[nh].item()) == 77  # nothing written past the end


@pytest.mark.gpu
def test_gather_device_does_not_trust_the_list():
    """ids beyond the batch, a count beyond n_events and events with a malformed extent are gathered as empty events;
    nothing is read or written out of bounds (include/cbm_trigger.h)."""
    import torch
    from paper_1810_11966_b200 import binding as K
    cfg = W.CONFIGS[0]
    n = 64
    b = W.generate(cfg, n_events=n)
    L = cfg.n_layers
    off = b.off.copy()
    off[5 * L + 3] = off[5 * L + L] + 7          # event 5: an inner offset beyond its end
    off[9 * L + 1] = off[9 * L] - 1              # event 9: offsets decrease
    ids = np.array([3, 9, 1000, 5, 2**32 - 1, 7], dtype=np.uint32)
    with K.Trigger(cfg.layer_z, n, b.n_hits, n_slots=0) as trig:
        dx, dy = torch.from_numpy(np.concatenate([b.x, np.zeros(8, np.int32)])).cuda(), torch.from_numpy(np.concatenate([b.y, np.zeros(8, np.int32)])).cuda()
        do = torch.from_numpy(off.view(np.int32)).cuda()
        dids = torch.from_numpy(np.concatenate([ids, np.full(n - ids.size, 2**31 + 5, np.uint32)]).view(np.int32)).cuda()
        dn = torch.tensor([1_000_000], dtype=torch.int32, device="cuda")   # a count far beyond n_events
        ox = torch.full((b.n_hits + 1,), 77, dtype=torch.int32, device="cuda")
        oy = torch.full((b.n_hits + 1,), 77, dtype=torch.int32, device="cuda")
        oo = torch.full((n * L + 1,), -1, dtype=torch.int32, device="cuda")
        on = torch.zeros(1, dtype=torch.int64, device="cuda")
        trig.gather_device(n, b.n_hits, dx, dy, do, dids, dn, ox, oy, oo, on)
        torch.cuda.synchronize()
        o = oo.cpu().numpy().view(np.uint32)
        size = lambda e: int(b.off[e * L + L] - b.off[e * L])
        # entries: 3 ok, 9 malformed (empty), 1000 out of range (empty), 5 malformed (empty), 2^32-1 (empty), 7 ok, then ids
        # beyond the batch (empty)
        want_sizes = [size(3), 0, 0, 0, 0, size(7)] + [0] * (n - ids.size)
        got_sizes = [int(o[(i + 1) * L] - o[i * L]) for i in range(n)]
        assert got_sizes == want_sizes
        assert int(on.item()) == sum(want_sizes) and int(o[n * L]) == sum(want_sizes)
        assert (np.diff(o[:n * L + 1].astype(np.int64)) >= 0).all()           # offsets stay monotone
        x3 = ox.cpu().numpy()[:size(3)]
        assert np.array_equal(x3, b.x[b.off[3 * L]:b.off[3 * L + L]])
        assert int(ox[sum(want_sizes)].item()) == 77                            # nothing written past the end
        # a list that repeats events can gather more than the batch holds: the total is reported, nothing is copied
        sizes = np.array([size(e) if e not in (5, 9) else 0 for e in range(n)])
        big = np.argsort(sizes)[-4:].astype(np.uint32)                          # the four largest well-formed events, 16 times each
        total = 16 * int(sizes[big].sum())
        assert total > b.n_hits
        rep = torch.from_numpy(np.resize(big, n).view(np.int32)).cuda()
        dn.fill_(n)
        ox.fill_(77)
        trig.gather_device(n, b.n_hits, dx, dy, do, rep, dn, ox, oy, oo, on)
        torch.cuda.synchronize()
        assert int(on.item()) == total
        assert int((ox != 77).sum().item()) == 0


@pytest.mark.gpu
def test_gather_device_repeated_ids_total_of_exactly_two_to_the_32():
    """A list of 2^20 entries that all name one 4096-hit event gathers 2^32 hits.  The total is summed in 64 bits: a
    32-bit sum would wrap to 0, pass the "fits the output" test and copy to wrapped positions far outside the output
    arrays.  Required (include/cbm_trigger.h): *d_out_n_hits reports the true total and nothing else is written."""
    import torch
    from paper_1810_11966_b200 import binding as K
    cfg = W.CONFIGS[0]
    L = cfg.n_layers
    n, big, size = 1 << 20, 12345, 4096
    off = np.zeros(n * L + 1, dtype=np.uint32)
    off[big * L + 1:] = size                      # event `big` holds all 4096 hits in its first layer; every other event is empty
    rng = np.random.default_rng(5)
    x = rng.integers(-30000, 30000, size=size + 8, dtype=np.int32)
    with K.Trigger(cfg.layer_z, n, size, n_slots=0) as trig:
        dx, dy = torch.from_numpy(x).cuda(), torch.from_numpy(-x).cuda()
        do = torch.from_numpy(off.view(np.int32)).cuda()
        dids = torch.full((n,), big, dtype=torch.int32, device="cuda")
        dn = torch.tensor([n], dtype=torch.int32, device="cuda")
        ox = torch.full((size + 1,), 77, dtype=torch.int32, device="cuda")
        oy = torch.full((size + 1,), 77, dtype=torch.int32, device="cuda")
        oo = torch.full((n * L + 1,), -1, dtype=torch.int32, device="cuda")
        on = torch.zeros(1, dtype=torch.int64, device="cuda")
        trig.gather_device(n, size, dx, dy, do, dids, dn, ox, oy, oo, on)
        torch.cuda.synchronize()
        assert int(on.item()) == n * size == 1 << 32
        assert bool((ox == 77).all()) and bool((oy == 77).all()) and bool((oo == -1).all())
        # the same list cut to one entry fits and is gathered (the handle is still usable)
        dn.fill_(1)
        trig.gather_device(n, size, dx, dy, do, dids, dn, ox, oy, oo, on)
        torch.cuda.synchronize()
        assert int(on.item()) == size
        assert np.array_equal(ox.cpu().numpy()[:size], x[:size]) and int(ox[size].item()) == 77
        o = oo.cpu().numpy().view(np.uint32)
        assert o[:L + 1].tolist() == [0] + [size] * L
