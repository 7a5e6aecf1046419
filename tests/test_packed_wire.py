"""The packed wire format XY20 (include/cbm_trigger.h).

CPU: oracle.unpack_xy20 (the format's definition, decoded hit by hit) is pinned against hand-written byte
strings and against the packer of the workloads module (round trip, range limits).
GPU: a batch uploaded packed gives bit-identical results to the oracle on the unpacked integers.
"""
import numpy as np
import pytest

import oracle
from paper_1810_11966_b200 import workloads as W


# ------------------------------------------------------------------------------------------------ CPU pins
def test_unpack_hand_written_bytes():
    # x = 1, y = 0 -> bit 0;  x = 0, y = 1 -> bit 20 = bit 4 of byte 2;  all ones -> (-1, -1)
    x, y = oracle.unpack_xy20(bytes([1, 0, 0, 0, 0, 0, 0, 0x10, 0, 0, 0xFF, 0xFF, 0xFF, 0xFF, 0xFF]))
    assert x.tolist() == [1, 0, -1] and y.tolist() == [0, 1, -1]
    # x = 0x7FFFF (largest), y = 0x80000 (smallest): v = 0x80000_7FFFF -> FF FF 07 00 80
    x, y = oracle.unpack_xy20(bytes([0xFF, 0xFF, 0x07, 0x00, 0x80]))
    assert x.tolist() == [524287] and y.tolist() == [-524288]
    # x = 0x12345, y = 0x0ABCD: v = 0x0ABCD_12345 = 0x0ABCD12345 -> 45 23 D1 BC 0A
    x, y = oracle.unpack_xy20(bytes([0x45, 0x23, 0xD1, 0xBC, 0x0A]))
    assert x.tolist() == [0x12345] and y.tolist() == [0x0ABCD]
    assert oracle.unpack_xy20(b"")[0].size == 0


def test_pack_unpack_round_trip_and_limits():
    rng = np.random.default_rng(5)
    for n in (1, 3, 4, 5, 1001):
        x = rng.integers(W.XY20_MIN, W.XY20_MAX + 1, size=n, dtype=np.int32)
        y = rng.integers(W.XY20_MIN, W.XY20_MAX + 1, size=n, dtype=np.int32)
        p = W.pack_xy20(x, y)
        assert p.dtype == np.uint8 and p.size == 5 * n
        ux, uy = oracle.unpack_xy20(p)
        assert np.array_equal(ux, x) and np.array_equal(uy, y)
    for bad in (W.XY20_MAX + 1, W.XY20_MIN - 1):
        with pytest.raises(ValueError):
            W.pack_xy20(np.array([bad], np.int32), np.array([0], np.int32))
        with pytest.raises(ValueError):
            W.pack_xy20(np.array([0], np.int32), np.array([bad], np.int32))


def test_library_packer_against_the_oracle_decoder_and_hand_written_bytes():
    """cbm_trigger_pack_xy20 (host code of the C library, no CUDA): hand-written byte strings, a round trip through
    oracle.unpack_xy20 (the format's definition), the range limits with the index of the first bad hit."""
    from paper_1810_11966_b200 import binding as K
    # the hand cases of test_unpack_hand_written_bytes, in the packing direction
    p = K.cbm_trigger_pack_xy20(np.array([1, 0, -1], np.int32), np.array([0, 1, -1], np.int32))
    assert bytes(p) == bytes([1, 0, 0, 0, 0, 0, 0, 0x10, 0, 0, 0xFF, 0xFF, 0xFF, 0xFF, 0xFF])
    assert bytes(K.cbm_trigger_pack_xy20(np.array([524287], np.int32), np.array([-524288], np.int32))) == bytes([0xFF, 0xFF, 0x07, 0x00, 0x80])
    assert bytes(K.cbm_trigger_pack_xy20(np.array([0x12345], np.int32), np.array([0x0ABCD], np.int32))) == bytes([0x45, 0x23, 0xD1, 0xBC, 0x0A])
    assert K.cbm_trigger_pack_xy20(np.zeros(0, np.int32), np.zeros(0, np.int32)).size == 0
    rng = np.random.default_rng(8)
    for n in (1, 3, 4, 5, 1001):
        x = rng.integers(W.XY20_MIN, W.XY20_MAX + 1, size=n, dtype=np.int32)
        y = rng.integers(W.XY20_MIN, W.XY20_MAX + 1, size=n, dtype=np.int32)
        out = np.full(5 * n + 3, 0xAB, dtype=np.uint8)
        p = K.cbm_trigger_pack_xy20(x, y, out)
        ux, uy = oracle.unpack_xy20(p)
        assert np.array_equal(ux, x) and np.array_equal(uy, y)
        assert (out[5 * n:] == 0xAB).all()  # nothing written past the end
    for bad in (W.XY20_MAX + 1, W.XY20_MIN - 1, 2**31 - 1, -2**31):
        for xs, ys in (([5, 6, bad, 7], [1, 2, 3, 4]), ([5, 6, 7, 8], [1, 2, bad, bad])):
            with pytest.raises(K.CbmTriggerError) as ei:
                K.cbm_trigger_pack_xy20(np.array(xs, np.int32), np.array(ys, np.int32))
            assert ei.value.code == K.CBM_ERR_RANGE and ei.value.first_bad == 2


def test_workload_coordinates_fit_the_format():
    for cid in (0, 1, 2, 3):
        b = W.generate(W.CONFIGS[cid], n_events=300)
        assert b.x.min() >= W.XY20_MIN and b.x.max() <= W.XY20_MAX
        assert b.y.min() >= W.XY20_MIN and b.y.max() <= W.XY20_MAX


# ------------------------------------------------------------------------------------------------ GPU parity
@pytest.mark.gpu
@pytest.mark.parametrize("cid,n", [(0, 1000), (1, 2001), (3, 20000), (2, 1203)])
def test_packed_upload_matches_oracle(cid, n):
    from paper_1810_11966_b200 import binding as K
    from tests.helpers import assert_same, oracle_mt
    cfg = W.CONFIGS[cid]
    b = W.generate(cfg, n_events=n)
    packed = W.pack_xy20(b.x, b.y)
    ux, uy = oracle.unpack_xy20(packed[:5 * 2000])  # the oracle's decoder agrees with the packer on this batch
    assert np.array_equal(ux, b.x[:2000]) and np.array_equal(uy, b.y[:2000])
    g = oracle.geometry(cfg.layer_z, cfg.win_in, cfg.win_link, cfg.min_candidates)
    want = oracle_mt(g, b.x, b.y, b.off)
    with K.Trigger(cfg.layer_z, n, b.n_hits, win_in=cfg.win_in, win_link=cfg.win_link,
                   min_candidates=cfg.min_candidates, n_slots=2, flags=K.CBM_FLAG_PACKED_INPUT) as trig:
        # slot 0: caller memory; slot 1: written straight into the slot's pinned staging
        trig.upload_events_packed(0, packed, b.off)
        hp, ho = trig.host_buffers_packed(1)
        hp[:packed.size] = packed
        ho[:b.off.size] = b.off
        trig.upload_events_packed(1, hp, ho, n, b.n_hits)
        trig.run(0)
        trig.run(1)
        for slot in (0, 1):
            got = trig.fetch_results(slot, n)
            assert_same(got, want, f"{cfg.name} packed slot {slot}")
            assert np.array_equal(trig.fetch_selected(slot), oracle.selected(want[2]))
        # the int32 calls are refused on a packed handle
        with pytest.raises(K.CbmTriggerError) as ei:
            trig.upload_events(0, b.x, b.y, b.off)
        assert ei.value.code == K.CBM_ERR_STATE


@pytest.mark.gpu
def test_packed_extreme_coordinates_and_ragged_tail():
    """Hits at the limits of the 20-bit range and hit counts that are not multiples of 4 (the expansion kernel
    works on groups of 4 hits = 20 bytes)."""
    from paper_1810_11966_b200 import binding as K
    from tests.helpers import assert_same
    z = W.GEOMETRY_4
    rng = np.random.default_rng(2)
    for n_per_layer in (1, 2, 3, 5):
        n_events = 7
        L = len(z)
        n_hits = n_events * L * n_per_layer
        x = rng.integers(W.XY20_MIN, W.XY20_MAX + 1, size=n_hits, dtype=np.int32)
        y = rng.integers(W.XY20_MIN, W.XY20_MAX + 1, size=n_hits, dtype=np.int32)
        x[::3] = W.XY20_MIN; y[1::3] = W.XY20_MAX
        # event 0: an exact straight line from the origin through every layer (one candidate ... twice -> accept)
        for l in range(L):
            x[l * n_per_layer] = z[l] // 10
            y[l * n_per_layer] = -(z[l] // 20)
        off = (np.arange(n_events * L + 1, dtype=np.uint32) * n_per_layer).astype(np.uint32)
        g = oracle.geometry(z)
        want = oracle.run(g, x, y, off)
        assert want[1][0] >= 1
        with K.Trigger(z, n_events, n_hits, n_slots=1, flags=K.CBM_FLAG_PACKED_INPUT) as trig:
            trig.upload_events_packed(0, W.pack_xy20(x, y), off)
            trig.run(0)
            assert_same(trig.fetch_results(0, n_events), want, f"n_per_layer {n_per_layer}")
        with K.Trigger(z, n_events, n_hits, n_slots=1) as trig:  # and without packing: the same
            assert_same(trig.select(x, y, off), want, "int32")
