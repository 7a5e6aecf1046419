"""The input filter of the paper's implementation "i3" (only the hits of the layers the selection
uses are kept out of the full-setup hit data): pins of the oracle (oracle.filter_layers) and GPU parity of
cbm_trigger_filter_device."""
import numpy as np
import pytest

import oracle
from paper_1810_11966_b200 import workloads as W

Z = [60000, 70000, 80000]


def test_filter_hand_case():
    # two events; records (x, y, z).  Layer z = 60000, 70000, 80000; 65000 and 10 are other planes.
    xyz = np.array([[1, -1, 70000], [2, -2, 65000], [3, -3, 60000], [4, -4, 70000], [5, -5, 10], [6, -6, 80000], [7, -7, 60000],
                    [8, -8, 80000], [9, -9, 80000]], dtype=np.int32)
    ev_off = [0, 7, 9]
    x, y, off = oracle.filter_layers(xyz, ev_off, Z)
    # event 0: layer 0 = records 2, 6 (stream order); layer 1 = records 0, 3; layer 2 = record 5.  event 1: layer 2 = 7, 8
    assert x.tolist() == [3, 7, 1, 4, 6, 8, 9]
    assert y.tolist() == [-3, -7, -1, -4, -6, -8, -9]
    assert off.tolist() == [0, 2, 4, 5, 5, 5, 7]


def test_filter_identities():
    rng = np.random.default_rng(1)
    # nothing kept: no record has a layer z
    xyz = np.stack([rng.integers(-9, 9, 40), rng.integers(-9, 9, 40), np.full(40, 12345)], axis=1).astype(np.int32)
    x, y, off = oracle.filter_layers(xyz, [0, 10, 40], Z)
    assert x.size == 0 and off.tolist() == [0] * 7
    # everything kept and already grouped by layer: the stream comes back unchanged
    b = W.generate(W.CONFIGS[0], n_events=20)
    L = b.cfg.n_layers
    lay = np.repeat(np.tile(np.arange(L), 20), np.diff(b.off.astype(np.int64)))
    xyz = np.stack([b.x, b.y, np.asarray(b.cfg.layer_z, dtype=np.int32)[lay]], axis=1)
    x, y, off = oracle.filter_layers(xyz, b.off[::L], b.cfg.layer_z)
    assert np.array_equal(x, b.x) and np.array_equal(y, b.y) and np.array_equal(off, b.off)
    # empty events and an empty stream
    x, y, off = oracle.filter_layers(np.zeros((0, 3), np.int32), [0, 0, 0], Z)
    assert x.size == 0 and off.tolist() == [0] * 7
    # the number of kept hits is the number of records with a layer z (checked with numpy, not with the oracle)
    xyz, eo = W.full_setup_stream(b, other_hits_per_event=50, seed=2)
    x, y, off = oracle.filter_layers(xyz, eo, b.cfg.layer_z)
    assert x.size == int(np.isin(xyz[:, 2], b.cfg.layer_z).sum()) == b.n_hits


def test_filter_recovers_the_batch_and_the_selection():
    # a mixed full-setup stream built around a generated batch: the filter gives the batch back, so the selection on the
    # filtered stream is the selection on the batch ("only hit data in the trigger station are transferred")
    b = W.generate(W.CONFIGS[0], n_events=60)
    xyz, eo = W.full_setup_stream(b, other_hits_per_event=200, seed=5)
    x, y, off = oracle.filter_layers(xyz, eo, b.cfg.layer_z)
    assert np.array_equal(x, b.x) and np.array_equal(y, b.y) and np.array_equal(off, b.off)


@pytest.mark.gpu
@pytest.mark.parametrize("cid,n,other", [(0, 300, 400), (3, 2000, 150), (2, 400, 4000)])
def test_filter_device_matches_oracle(cid, n, other):
    import torch
    from paper_1810_11966_b200 import binding as K
    cfg = W.CONFIGS[cid]
    b = W.generate(cfg, n_events=n)
    xyz, eo = W.full_setup_stream(b, other_hits_per_event=other, seed=cid + 1)
    L = cfg.n_layers
    with K.Trigger(cfg.layer_z, n, max(xyz.shape[0], 1), n_slots=0) as trig:
        dxyz = torch.from_numpy(xyz.reshape(-1)).cuda()
        deo = torch.from_numpy(eo.view(np.int32)).cuda()
        ox = torch.full((xyz.shape[0] + 8,), 77, dtype=torch.int32, device="cuda")
        oy = torch.full((xyz.shape[0] + 8,), 77, dtype=torch.int32, device="cuda")
        oo = torch.full((n * L + 1,), -1, dtype=torch.int32, device="cuda")
        trig.filter_device(n, xyz.shape[0], dxyz, deo, ox, oy, oo)
        torch.cuda.synchronize()
        off = oo.cpu().numpy().view(np.uint32)
        nh = int(off[-1])
        assert np.array_equal(off, b.off)
        assert np.array_equal(ox.cpu().numpy()[:nh], b.x) and np.array_equal(oy.cpu().numpy()[:nh], b.y)
        assert int(ox[nh].item()) == 77
        # the filtered batch goes straight into the selection (same device arrays)
        S = cfg.n_stations
        dnt = torch.zeros(n * S, dtype=torch.int32, device="cuda")
        dnc = torch.zeros(n, dtype=torch.int32, device="cuda")
        dac = torch.zeros(n, dtype=torch.uint8, device="cuda")
        trig.run_device(n, nh, ox, oy, oo, dnt, dnc, dac)
        torch.cuda.synchronize()
    g = oracle.geometry(cfg.layer_z, cfg.win_in, cfg.win_link, cfg.min_candidates)
    want = oracle.run(g, b.x, b.y, b.off)
    assert np.array_equal(dnt.cpu().numpy().view(np.uint32).reshape(n, S), want[0])
    assert np.array_equal(dnc.cpu().numpy().view(np.uint32), want[1]) and np.array_equal(dac.cpu().numpy(), want[2])


@pytest.mark.gpu
def test_filter_device_small_cases():
    import torch
    from paper_1810_11966_b200 import binding as K
    cases = [(np.array([[1, -1, 70000], [2, -2, 65000], [3, -3, 60000], [4, -4, 70000], [5, -5, 10], [6, -6, 80000], [7, -7, 60000],
                        [8, -8, 80000], [9, -9, 80000]], dtype=np.int32), [0, 7, 9]),
             (np.zeros((0, 3), np.int32), [0, 0, 0]),
             (np.array([[5, 5, 1]] * 700 + [[6, 6, 70000]] * 3, dtype=np.int32), [0, 0, 703])]
    for xyz, eo in cases:
        E = len(eo) - 1
        want = oracle.filter_layers(xyz, eo, Z)
        with K.Trigger(Z, max(E, 1), max(xyz.shape[0], 1), n_slots=0) as trig:
            dxyz = torch.from_numpy(np.ascontiguousarray(xyz).reshape(-1)).cuda() if xyz.size else torch.zeros(3, dtype=torch.int32, device="cuda")
            deo = torch.from_numpy(np.asarray(eo, dtype=np.uint32).view(np.int32)).cuda()
            ox = torch.full((xyz.shape[0] + 8,), 77, dtype=torch.int32, device="cuda")
            oy = torch.full((xyz.shape[0] + 8,), 77, dtype=torch.int32, device="cuda")
            oo = torch.full((E * 3 + 1,), -1, dtype=torch.int32, device="cuda")
            trig.filter_device(E, xyz.shape[0], dxyz, deo, ox, oy, oo)
            torch.cuda.synchronize()
            off = oo.cpu().numpy().view(np.uint32)
            assert np.array_equal(off, want[2])
            assert np.array_equal(ox.cpu().numpy()[:want[0].size], want[0]) and np.array_equal(oy.cpu().numpy()[:want[0].size], want[1])
