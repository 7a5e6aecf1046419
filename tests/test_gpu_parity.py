"""Parity of the CUDA path (through the C ABI) against the CPU oracle: bit-exact n_triplets,
n_candidates and accept on the same seeded inputs (integer work: no tolerance).

Needs a B200: every test here is marked gpu."""
import numpy as np
import pytest

import oracle
from paper_1810_11966_b200 import binding as K
from paper_1810_11966_b200 import workloads as W
from tests import adversarial as A
from tests.golden_io import golden_cases, read_golden
from tests.helpers import assert_same, device_run, gpu_select, oracle_mt

pytestmark = pytest.mark.gpu

FLAG_SETS = [0, K.CBM_FLAG_NO_TINY_PATH]


def oracle_of(layer_z, x, y, off, **kw):
    g = oracle.geometry(layer_z, kw.get("win_in", (1, 100)), kw.get("win_link", (2, 100)), kw.get("min_candidates", 2))
    return oracle_mt(g, x, y, off)


# ------------------------------------------------------------------------------- hand-built events
@pytest.mark.parametrize("flags", FLAG_SETS)
@pytest.mark.parametrize("case", A.adversarial_suite(), ids=lambda c: c[0])
def test_adversarial_events(case, flags):
    name, layer_z, events, expected = case
    x, y, off = W.batch_from_layers(layer_z, events)
    got = gpu_select(layer_z, x, y, off, flags=flags)
    if expected is not None:  # closed form of the construction
        assert_same(got, (np.array(expected[0], dtype=np.uint32), np.array(expected[1], dtype=np.uint32),
                          np.array(expected[2], dtype=np.uint8)), name + " closed form")
    assert_same(got, oracle_of(layer_z, x, y, off), name + " oracle")


@pytest.mark.parametrize("flags", FLAG_SETS)
def test_boundary_equality(flags):
    # |dslope| = 0.01 exactly passes, one unit more fails (closed window, R3); same for the link window
    z = [60000, 70000, 80000]
    events = [[[(0, 0)], [(700, 0)], [(0, 0)]], [[(0, 0)], [(701, 0)], [(0, 0)]], [[(0, 0)], [(0, -700)], [(0, 0)]],
              [[(0, 0)], [(0, -701)], [(0, 0)]], [[(0, 0)], [(350, 0)], [(800, 0)]], [[(0, 0)], [(350, 0)], [(801, 0)]],
              [[(300, 0)], [(0, 0)], [(800, 0)]], [[(300, 0)], [(0, 0)], [(801, 0)]]]
    x, y, off = W.batch_from_layers(z, events)
    nt, nc, ac, _ = gpu_select(z, x, y, off, flags=flags)
    assert nt[:, 0].tolist() == [1, 0, 1, 0, 1, 0, 1, 0]
    assert nc.tolist() == [1, 0, 1, 0, 1, 0, 1, 0]
    # link window 0.02 between middle layers z = 70000 and 110000: x = 0 vs 2200 passes, 2201 fails
    z2 = list(W.GEOMETRY_4)[:6]
    ev = []
    for xm in (2200, 2201):
        ev.append([[(0, 0)], [(0, 0)], [(0, 0)], [(xm * 100 // 110, 0)], [(xm, 0)], [(xm * 120 // 110, 0)]])
    x, y, off = W.batch_from_layers(z2, ev)
    got = gpu_select(z2, x, y, off, flags=flags)
    want = oracle_of(z2, x, y, off)
    assert_same(got, want, "link boundary")
    assert got[1].tolist() == [1, 0]


@pytest.mark.parametrize("flags", FLAG_SETS)
def test_empty_batch_and_empty_events(flags):
    z = list(W.GEOMETRY_4)
    x, y, off = W.batch_from_layers(z, [])
    nt, nc, ac, st = gpu_select(z, x, y, off, flags=flags)
    assert nt.shape == (0, 4) and nc.size == 0 and ac.size == 0 and st["n_launches"] == 0
    x, y, off = W.batch_from_layers(z, [A.empty_event(z)] * 70)
    nt, nc, ac, _ = gpu_select(z, x, y, off, flags=flags)
    assert not nt.any() and not nc.any() and not ac.any()
    # min_candidates = 0 accepts everything, including empty events
    nt, nc, ac, _ = gpu_select(z, x, y, off, flags=flags, min_candidates=0)
    assert ac.all()


@pytest.mark.parametrize("flags", FLAG_SETS)
@pytest.mark.parametrize("seed", [1, 2, 3])
def test_random_geometries_and_windows(seed, flags):
    rng = np.random.default_rng(seed)
    for _ in range(6):
        S = int(rng.integers(1, 9))
        zs, zc = [], int(rng.integers(2000, 80000))
        for _s in range(S):
            for _l in range(3):
                zs.append(zc)
                zc += int(rng.integers(1000, 20000))
            zc += int(rng.integers(5000, 60000))
        win_in = [(1, 100), (1, 64), (3, 100), (1, 3), (0, 1), (7, 4096)][int(rng.integers(0, 6))]
        win_link = [(2, 100), (1, 10), (1, 1), (0, 5)][int(rng.integers(0, 4))]
        events = []
        for _e in range(40):
            k = rng.integers(0, 4)
            if k == 0:
                events.append(A.random_cluster_event(zs, rng, max_hits=6, n_dirs=2, jitter_slope=0.012, dir_spread=0.02))
            elif k == 1:
                events.append(A.two_direction_event(zs, rng, max_hits=3))
            elif k == 2:
                events.append(A.random_cluster_event(zs, rng, max_hits=40, n_dirs=3, jitter_slope=0.02, dir_spread=0.05))
            else:
                events.append(A.narrow_cone_event(zs, int(rng.integers(0, 4)), rng, spread_units=int(rng.integers(0, 400))))
        x, y, off = W.batch_from_layers(zs, events)
        mc = int(rng.integers(0, 4))
        got = gpu_select(zs, x, y, off, win_in=win_in, win_link=win_link, min_candidates=mc, flags=flags,
                         tiny_max_layer_hits=int(rng.choice([0, 4, 32])))
        want = oracle_of(zs, x, y, off, win_in=win_in, win_link=win_link, min_candidates=mc)
        assert_same(got, want, f"S={S} win_in={win_in} win_link={win_link}")


@pytest.mark.parametrize("flags", FLAG_SETS)
def test_full_int32_coordinate_range(flags):
    # include/cbm_trigger.h: exact for any int32 x, y and 0 < z <= 2^23.  Hand-computed expectations:
    # tests/test_oracle_pins.py::full_range_cases
    from tests.test_oracle_pins import full_range_cases
    z, win, ev, exp = full_range_cases()
    x, y, off = W.batch_from_layers(z, ev)
    got = gpu_select(z, x, y, off, win_in=win, win_link=win, flags=flags)
    assert got[0][:, 0].tolist() == exp and got[1].tolist() == exp
    assert_same(got, oracle_of(z, x, y, off, win_in=win, win_link=win), "full int32 range")
    # the same hits inside fuller layers (class M / H kernels): 200 background hits per layer far away in y
    rng = np.random.default_rng(5)
    big = []
    for e in ev:
        big.append([lay + [(int(rng.integers(-2**31, 2**31)), int(rng.integers(2_000_000_000, 2**31))) for _ in range(n)]
                    for lay, n in zip(e, (200, 40, 130))])
    x, y, off = W.batch_from_layers(z, big)
    got = gpu_select(z, x, y, off, win_in=win, win_link=win, flags=flags)
    assert_same(got, oracle_of(z, x, y, off, win_in=win, win_link=win), "full int32 range, full layers")


def test_saturation_closed_forms():
    # narrow cone: every combination passes => |T_s| = n0*n1*n2, candidates = prod |T_s|
    rng = np.random.default_rng(7)
    z = list(W.GEOMETRY_4)
    ev = [A.narrow_cone_event(z, 50, rng), A.narrow_cone_event(z, 200, rng, spread_units=3)]
    x, y, off = W.batch_from_layers(z, ev)
    nt, nc, ac, st = gpu_select(z, x, y, off)
    assert nt.tolist() == [[125000] * 4, [8000000] * 4]
    assert nc.tolist() == [2**32 - 1, 2**32 - 1] and ac.tolist() == [1, 1]
    # triplet-count saturation: 1626^3 = 4298942376 > 2^32 - 1, one station
    z1 = [60000, 70000, 80000]
    x, y, off = W.batch_from_layers(z1, [A.narrow_cone_event(z1, 1626, rng)])
    nt, nc, ac, st = gpu_select(z1, x, y, off)
    assert nt.tolist() == [[2**32 - 1]] and nc.tolist() == [2**32 - 1] and st["n_class"][3] == 1
    # just below: 1625^3 = 4291015625 < 2^32 - 1
    x, y, off = W.batch_from_layers(z1, [A.narrow_cone_event(z1, 1625, rng)])
    nt, nc, ac, st = gpu_select(z1, x, y, off)
    assert nt.tolist() == [[1625**3]] and nc.tolist() == [1625**3]


def big_uniform_event(layer_z, counts, rng, half=0.35):
    layers = []
    for z, n in zip(layer_z, counts):
        xs = rng.integers(-int(half * z), int(half * z) + 1, size=n)
        ys = rng.integers(-int(half * z), int(half * z) + 1, size=n)
        layers.append(list(zip(xs.tolist(), ys.tolist())))
    return layers


def test_layers_up_to_max_hits_per_layer():
    rng = np.random.default_rng(11)
    z = list(W.GEOMETRY_4)
    ev = [big_uniform_event(z, [4096, 700, 900, 300, 4096, 300, 600, 600, 4096, 1500, 1500, 1500], rng),
          big_uniform_event(z, [129] * 12, rng), big_uniform_event(z, [128] * 12, rng),
          big_uniform_event(z, [449] + [40] * 11, rng), big_uniform_event(z, [448] * 12, rng),
          big_uniform_event(z, [25] * 12, rng), big_uniform_event(z, [24] * 12, rng)]
    x, y, off = W.batch_from_layers(z, ev)
    got = gpu_select(z, x, y, off)
    assert_same(got, oracle_of(z, x, y, off), "big layers")
    assert got[3]["n_class"] == [0, 3, 2, 2]  # 24/layer is 288 hits > tile budget: class M
    # planted tracks inside a full layer are still found
    lay = big_uniform_event(z, [3000] * 12, rng)
    for l, h in enumerate(A.exact_line_hits(z, 123, -77)):
        lay[l][17] = h
    for l, h in enumerate(A.exact_line_hits(z, -200, 31)):
        lay[l][2999] = h
    x, y, off = W.batch_from_layers(z, [lay])
    got = gpu_select(z, x, y, off)
    assert_same(got, oracle_of(z, x, y, off), "planted in 3000/layer")
    assert got[1][0] >= 2 and got[2][0] == 1


def test_invalid_offsets_are_rejected_on_the_device():
    rng = np.random.default_rng(5)
    z = list(W.GEOMETRY_4)
    ev = [A.random_cluster_event(z, rng, max_hits=5) for _ in range(100)]
    ev[40] = big_uniform_event(z, [10, 10, 60, 10, 10, 10, 10, 10, 10, 10, 10, 10], rng)
    x, y, off = W.batch_from_layers(z, ev)
    want = oracle_of(z, x, y, off)
    # (a) a layer above max_hits_per_layer = 50: event 40 is rejected, all others are right
    nt, nc, ac, st, rc, msg = gpu_select(z, x, y, off, max_hits_per_layer=50, check=False)
    assert rc == K.CBM_ERR_RANGE and st["n_invalid"] == 1 and st["first_invalid"] == 40 and "event 40" in msg
    keep = np.arange(100) != 40
    assert_same((nt[keep], nc[keep], ac[keep]), (want[0][keep], want[1][keep], want[2][keep]), "others")
    assert not nt[40].any() and nc[40] == 0 and ac[40] == 0
    # (b) non-monotone offsets inside events 7 and 63
    bad = off.copy()
    bad[7 * 12 + 5] = bad[7 * 12 + 6] + 3
    bad[63 * 12 + 1] = 0xFFFFFFF0
    nt, nc, ac, st, rc, msg = gpu_select(z, x, y, bad, check=False)
    assert rc == K.CBM_ERR_RANGE and st["n_invalid"] == 2 and st["first_invalid"] == 7
    keep = ~np.isin(np.arange(100), [7, 63])
    assert_same((nt[keep], nc[keep], ac[keep]), (want[0][keep], want[1][keep], want[2][keep]), "others")


def test_host_side_errors():
    z = list(W.GEOMETRY_4)
    trig = K.Trigger(z, 10, 100, n_slots=1)
    try:
        x, y, off = W.batch_from_layers(z, [A.empty_event(z)] * 11)
        with pytest.raises(K.CbmTriggerError) as ei:
            trig.upload_events(0, x, y, off)
        assert ei.value.code == K.CBM_ERR_CAPACITY
        with pytest.raises(K.CbmTriggerError) as ei:
            trig.run(0)
        assert ei.value.code == K.CBM_ERR_STATE
        with pytest.raises(K.CbmTriggerError) as ei:
            trig.fetch_results(0, 1)
        assert ei.value.code == K.CBM_ERR_STATE
        with pytest.raises(K.CbmTriggerError) as ei:
            trig.run(3)
        assert ei.value.code == K.CBM_ERR_STATE
        x, y, off = W.batch_from_layers(z, [A.empty_event(z)] * 3)
        off2 = off.copy()
        off2[-1] = 5
        with pytest.raises(K.CbmTriggerError) as ei:
            K.cbm_trigger_upload_events(trig.handle, 0, 3, 0, x, y, off2)
        assert ei.value.code == K.CBM_ERR_RANGE
        # the handle stays usable
        trig.upload_events(0, x, y, off)
        trig.run(0)
        nt, nc, ac = trig.fetch_results(0, 3)
        assert not nc.any()
    finally:
        trig.close()


# ------------------------------------------------------------------------------- the configs
CONFIG_SLICES = [(0, 1000), (1, 20000), (2, 12000), (3, 60000)]


@pytest.mark.parametrize("flags", FLAG_SETS)
@pytest.mark.parametrize("cid,n", CONFIG_SLICES)
def test_configs_against_oracle(cid, n, flags):
    cfg = W.CONFIGS[cid]
    b = W.generate(cfg, n_events=n)
    got = gpu_select(cfg.layer_z, b.x, b.y, b.off, win_in=cfg.win_in, win_link=cfg.win_link,
                     min_candidates=cfg.min_candidates, flags=flags)
    g = oracle.geometry(cfg.layer_z, cfg.win_in, cfg.win_link, cfg.min_candidates)
    assert_same(got, oracle_mt(g, b.x, b.y, b.off), cfg.name)
    st = got[3]
    assert sum(st["n_class"]) >= n and st["n_invalid"] == 0
    if flags & K.CBM_FLAG_NO_TINY_PATH:
        assert st["n_class"][0] == 0


@pytest.mark.parametrize("cid,n,path", golden_cases())
def test_configs_against_golden_files(cid, n, path):
    cfg = W.CONFIGS[cid]
    b = W.generate(cfg, n_events=n)
    got = gpu_select(cfg.layer_z, b.x, b.y, b.off)
    assert_same(got, read_golden(path, n, cfg.n_stations), f"golden cfg{cid}")


def test_permutation_and_batch_split_invariance():
    cfg = W.CONFIGS[3]
    b = W.generate(cfg, n_events=3000)
    base = gpu_select(cfg.layer_z, b.x, b.y, b.off)
    rng = np.random.default_rng(3)
    x2, y2 = b.x.copy(), b.y.copy()
    for i in range(b.off.size - 1):
        a, e = int(b.off[i]), int(b.off[i + 1])
        if e - a > 1:
            perm = rng.permutation(e - a)
            x2[a:e] = b.x[a:e][perm]
            y2[a:e] = b.y[a:e][perm]
    assert_same(gpu_select(cfg.layer_z, x2, y2, b.off), base, "permutation")
    L = cfg.n_layers
    cut = 1234
    o1 = b.off[:cut * L + 1].copy()
    o2 = (b.off[cut * L:] - b.off[cut * L]).astype(np.uint32)
    h = int(b.off[cut * L])
    r1 = gpu_select(cfg.layer_z, b.x[:h], b.y[:h], o1)
    r2 = gpu_select(cfg.layer_z, b.x[h:], b.y[h:], o2)
    assert_same((np.concatenate([r1[0], r2[0]]), np.concatenate([r1[1], r2[1]]), np.concatenate([r1[2], r2[2]])),
                base, "split")


# ------------------------------------------------------------------------------- pipeline and device path
def test_two_slot_pipeline_matches_per_batch():
    cfg = W.CONFIGS[3]
    batches = [W.generate(cfg, n_events=5000, first_event=i * 5000) for i in range(5)]
    g = oracle.geometry(cfg.layer_z, cfg.win_in, cfg.win_link, cfg.min_candidates)
    want = [oracle_mt(g, b.x, b.y, b.off) for b in batches]
    mh = max(b.n_hits for b in batches)
    with K.Trigger(cfg.layer_z, 5000, mh, n_slots=2, flags=K.CBM_FLAG_PROFILE) as trig:
        bufs = [trig.host_buffers(s) for s in (0, 1)]
        got = [None] * len(batches)
        for i, b in enumerate(batches + [None]):
            s = i & 1
            if b is not None:
                if i >= 2:
                    got[i - 2] = trig.fetch_results(s, 5000)
                if i % 2 == 0:  # zero-copy staging: the producer fills the pinned buffers
                    hx, hy, ho = bufs[s]
                    hx[:b.n_hits] = b.x
                    hy[:b.n_hits] = b.y
                    ho[:b.off.size] = b.off
                    trig.upload_events(s, hx, hy, ho, 5000, b.n_hits)
                else:           # caller memory: staged through the pinned buffers by the library
                    trig.upload_events(s, b.x, b.y, b.off)
                trig.run(s)
        for i in (len(batches) - 2, len(batches) - 1):
            got[i] = trig.fetch_results(i & 1, 5000)
        st = trig.stats(0)
        assert st.n_launches == 8 and st.kernel_ms[0] > 0 and st.h2d_ms > 0  # 6 selection + 2 list kernels
    for i in range(len(batches)):
        assert_same(got[i], want[i], f"batch {i}")


def test_device_resident_entry_point():
    import torch
    cfg = W.CONFIGS[3]
    b = W.generate(cfg, n_events=20000)
    host = gpu_select(cfg.layer_z, b.x, b.y, b.off)
    dev = torch.device("cuda:0")
    pad = (-b.n_hits) % 4 + 4
    dx = torch.zeros(b.n_hits + pad, dtype=torch.int32, device=dev)
    dy = torch.zeros(b.n_hits + pad, dtype=torch.int32, device=dev)
    dx[:b.n_hits] = torch.from_numpy(b.x).to(dev)
    dy[:b.n_hits] = torch.from_numpy(b.y).to(dev)
    doff = torch.from_numpy(b.off.view(np.int32)).to(dev)  # same 32 bits as uint32
    S = cfg.n_stations
    dnt = torch.full((20000 * S,), -1, dtype=torch.int32, device=dev)
    dnc = torch.full((20000,), -1, dtype=torch.int32, device=dev)
    dac = torch.full((20000,), 255, dtype=torch.uint8, device=dev)
    with K.Trigger(cfg.layer_z, 20000, b.n_hits, n_slots=0) as trig:
        stream = torch.cuda.Stream()
        with torch.cuda.stream(stream):
            trig.run_device(20000, b.n_hits, dx, dy, doff, dnt, dnc, dac)
            rc, st = trig.device_status()
        assert rc == K.CBM_OK and st.n_invalid == 0
    got = (dnt.cpu().numpy().view(np.uint32).reshape(-1, S), dnc.cpu().numpy().view(np.uint32), dac.cpu().numpy())
    assert_same(got, host, "run_device vs upload/run/fetch")


# ------------------------------------------------------------------------------- every config at bench size
@pytest.mark.parametrize("cid", [0, 1, 3])
def test_full_size_every_event(cid):
    """BASELINE.json configs 0, 1 and 3 at full size in bench.py's launch configuration (device-resident, kernels
    side by side): EVERY event against the oracle (north_star: bit-exact for every config)."""
    cfg = W.CONFIGS[cid]
    b = W.generate(cfg)
    nt, nc, ac, st = device_run(cfg, b)
    g = oracle.geometry(cfg.layer_z, cfg.win_in, cfg.win_link, cfg.min_candidates)
    assert_same((nt, nc, ac), oracle_mt(g, b.x, b.y, b.off), f"{cfg.name}, all {cfg.n_events} events")
    assert sum(st["n_class"]) == cfg.n_events and st["n_invalid"] == 0
    # the serial launch sequence gives the same results
    assert_same(device_run(cfg, b, flags=K.CBM_FLAG_SERIAL), (nt, nc, ac), f"{cfg.name} serial launch")


def test_full_size_config2_every_event():
    """Config 2 (1,000,000 events of six stations, log-normal occupancy) at full size in bench.py's launch
    configuration: EVERY event against the oracle (north_star: bit-exact for every config), plus invariants."""
    cfg = W.CONFIGS[2]
    b = W.generate(cfg)
    nt, nc, ac, st = device_run(cfg, b)
    assert ac.max() <= 1 and not nc[(nt == 0).any(axis=1)].any()
    assert np.array_equal(ac, (nc >= cfg.min_candidates).astype(np.uint8))
    assert st["n_class"][3] > 1000 and st["n_class"][1] > 800_000   # the scheduler's classes are all exercised
    g = oracle.geometry(cfg.layer_z, cfg.win_in, cfg.win_link, cfg.min_candidates)
    assert_same((nt, nc, ac), oracle_mt(g, b.x, b.y, b.off), f"{cfg.name}, all {cfg.n_events} events")


def test_config4_two_chunks_every_event_through_both_pipelines():
    """Config 4 (streaming, seed 5): two 1,000,000-event chunks of the stream with first_event != 0 through the
    two-slot upload / run / fetch pipeline in the int32 format AND in the packed wire format: both bit-identical on
    every event, and EVERY event of both chunks (2,000,000 events) against the oracle."""
    cfg = W.CONFIGS[4]
    E = cfg.chunk_events
    chunks = [W.generate(cfg, n_events=E, first_event=k * E) for k in (3, 7)]
    mh = max(b.n_hits for b in chunks)
    S, L = cfg.n_stations, cfg.n_layers
    results = {}
    for packed in (False, True):
        with K.Trigger(cfg.layer_z, E, mh, win_in=cfg.win_in, win_link=cfg.win_link, min_candidates=cfg.min_candidates,
                       n_slots=2, flags=K.CBM_FLAG_PACKED_INPUT if packed else 0) as trig:
            for s, b in enumerate(chunks):
                if packed:
                    hp, ho = trig.host_buffers_packed(s)
                    hp[:5 * b.n_hits] = W.pack_xy20(b.x, b.y)
                    ho[:b.off.size] = b.off
                    trig.upload_events_packed(s, hp, ho, E, b.n_hits)
                else:
                    hx, hy, ho = trig.host_buffers(s)
                    hx[:b.n_hits], hy[:b.n_hits], ho[:b.off.size] = b.x, b.y, b.off
                    trig.upload_events(s, hx, hy, ho, E, b.n_hits)
                trig.run(s)
            results[packed] = [trig.fetch_results(s, E) for s in range(2)]
    g = oracle.geometry(cfg.layer_z, cfg.win_in, cfg.win_link, cfg.min_candidates)
    for s, b in enumerate(chunks):
        nt, nc, ac = results[False][s]
        assert_same(results[True][s], (nt, nc, ac), f"cfg4 chunk {s}: packed vs int32 pipeline")
        assert_same((nt, nc, ac), oracle_mt(g, b.x, b.y, b.off), f"cfg4 chunk {s}: all {E} events")
