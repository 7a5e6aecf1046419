"""The seeded workload generator (paper_1810_11966_b200/workloads): determinism and moments.
Shapes follow BASELINE.json configs and SURVEY.md section 8(c) R13-R18."""
import math

import numpy as np

from paper_1810_11966_b200 import workloads as W


def counts(b):
    return np.diff(b.off.astype(np.int64)).reshape(b.n_events, b.cfg.n_layers)


def test_deterministic_across_threads_and_chunks():
    cfg = W.CONFIGS[3]
    a = W.generate(cfg, n_events=5000, n_threads=1)
    b = W.generate(cfg, n_events=5000, n_threads=7)
    assert (a.off == b.off).all() and (a.x == b.x).all() and (a.y == b.y).all() and (a.truth == b.truth).all()
    # chunk [2000, 3500) generated on its own equals the slice of the big batch
    c = W.generate(cfg, n_events=1500, first_event=2000, n_threads=3)
    L = cfg.n_layers
    lo, hi = int(a.off[2000 * L]), int(a.off[3500 * L])
    assert (c.x == a.x[lo:hi]).all() and (c.y == a.y[lo:hi]).all()
    assert (c.off.astype(np.int64) + lo == a.off[2000 * L: 3500 * L + 1].astype(np.int64)).all()
    # another seed gives other data
    d = W.generate(cfg, n_events=5000, seed=99)
    assert d.n_hits != a.n_hits or not (d.x[:100] == a.x[:100]).all()


def test_offsets_well_formed_and_coordinates_in_range():
    for cid in (0, 1, 2, 3):
        cfg = W.CONFIGS[cid]
        b = W.generate(cfg, n_events=3000)
        assert b.off[0] == 0 and (np.diff(b.off.astype(np.int64)) >= 0).all() and b.off[-1] == b.x.size == b.y.size
        n = counts(b)
        assert n.max() <= cfg.max_hits_per_layer
        zmax = max(cfg.layer_z)
        # background within 0.35 z; signal within 0.3 z + smear: well inside the ABI range 2^23
        assert np.abs(b.x).max() <= 0.36 * zmax and np.abs(b.y).max() <= 0.36 * zmax
        layer_of_hit = np.repeat(np.tile(np.arange(cfg.n_layers), b.n_events), n.reshape(-1))
        z = np.asarray(cfg.layer_z)[layer_of_hit]
        assert (np.abs(b.x) <= 0.35 * z + 1000).all()      # signal smear/vertex can exceed 0.35 z only slightly


def test_moments_fixed_and_mixture():
    b = W.generate(W.CONFIGS[1], n_events=4000)
    n = counts(b)
    lam = 60.0
    assert abs(n.mean() - lam) < 5 * math.sqrt(lam / n.size) + 0.02 * 2   # + planted hits (1% x 2 tracks)
    assert abs(n.var() - lam) < 0.05 * lam
    planted = (b.truth & 1) > 0
    assert abs(planted.mean() - 0.01) < 5 * math.sqrt(0.01 * 0.99 / b.n_events)
    b = W.generate(W.CONFIGS[3], n_events=40000)
    n = counts(b)
    central = (b.truth & 4) > 0
    assert abs(central.mean() - 0.05) < 5 * math.sqrt(0.05 * 0.95 / b.n_events)
    assert abs(n[central].mean() - 300) < 1.0 and abs(n[~central].mean() - 5) < 0.1
    # uniform background: x/z uniform on [-0.35, 0.35] -> variance 0.35^2/3
    L = W.CONFIGS[3].n_layers
    layer_of_hit = np.repeat(np.tile(np.arange(L), b.n_events), n.reshape(-1))
    z = np.asarray(W.CONFIGS[3].layer_z, dtype=np.float64)[layer_of_hit]
    sx, sy = b.x / z, b.y / z
    assert abs(sx.mean()) < 1e-3 and abs(sy.mean()) < 1e-3
    assert abs(sx.var() - 0.35 ** 2 / 3) < 1e-3 and abs(sy.var() - 0.35 ** 2 / 3) < 1e-3
    assert abs(np.corrcoef(sx[:200000], sy[:200000])[0, 1]) < 0.01


def test_moments_lognormal():
    cfg = W.CONFIGS[2]
    b = W.generate(cfg, n_events=60000)
    n = counts(b).astype(np.float64)
    per_event = n.mean(axis=1)
    # median of the per-event mean ~ 40; E[lambda] = 40 exp(0.32) = 55.1
    assert abs(np.median(per_event) - 40) < 1.5
    assert abs(per_event.mean() - 40 * math.exp(0.32)) < 1.5
    assert n.max() <= 4096
    # one lambda per event shared by all 18 layers: layers of one event are strongly correlated
    assert np.corrcoef(n[:, 0], n[:, 17])[0, 1] > 0.9


def test_batch_from_layers_roundtrip():
    z = W.GEOMETRY_4
    ev = [[[(1, 2)] * (l % 3) for l in range(12)], [[] for _ in range(12)]]
    x, y, off = W.batch_from_layers(z, ev)
    assert off.size == 2 * 12 + 1 and off[-1] == x.size == sum(l % 3 for l in range(12))
    assert off[12] == off[-1]
