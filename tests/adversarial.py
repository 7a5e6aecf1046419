"""Hand-built adversarial events shared by the oracle pins and the GPU parity tests.

Input construction only (no window test, no counting): each builder returns
(layer_z, events) where events is a list of events, each a list of L layers of (x, y).
Expected values, where a closed form exists, are returned alongside and are derived
from the construction, not from any implementation.
"""
import numpy as np

from paper_1810_11966_b200.workloads import GEOMETRY_4, GEOMETRY_6, station_layers_z


def exact_line_hits(layer_z, p, q):
    """Hits of the straight line x = (p/1000) z, y = (q/1000) z: integers because z % 1000 == 0."""
    assert all(z % 1000 == 0 for z in layer_z)
    return [(p * z // 1000, q * z // 1000) for z in layer_z]


def planted_lines_event(layer_z, slopes):
    """One event holding one exact line per (p, q) in slopes (units of 1e-3)."""
    L = len(layer_z)
    layers = [[] for _ in range(L)]
    for (p, q) in slopes:
        for l, h in enumerate(exact_line_hits(layer_z, p, q)):
            layers[l].append(h)
    return layers


def narrow_cone_event(layer_z, n_per_layer, rng, spread_units=2):
    """Every hit within +-spread_units of the beam axis: every pair of hits is compatible
    (|x/z| <= 2/60000 << 0.01), so |T_s| = n0*n1*n2 and candidates = prod_s |T_s|."""
    L = len(layer_z)
    layers = []
    for l in range(L):
        n = n_per_layer[l] if hasattr(n_per_layer, "__len__") else n_per_layer
        layers.append([(int(rng.integers(-spread_units, spread_units + 1)),
                        int(rng.integers(-spread_units, spread_units + 1))) for _ in range(n)])
    return layers


def lattice_noise_event(layer_z, n_per_layer):
    """Constructed non-collinear noise: in layer l of a station every hit has x-slope on the lattice
    0.05*k + 0.0125*(l+1) ... so slopes of different layers of a station differ by >= 0.0125 > 0.01
    in x, and hits of one layer never pair with another layer's.  => 0 triplets everywhere."""
    layers = []
    for li, z in enumerate(layer_z):
        l = li % 3
        hits = []
        for k in range(n_per_layer):
            sx = 0.05 * (k - n_per_layer // 2) + 0.0125 * (l + 1)   # lattice spacing 0.05, layer shift 0.0125
            sy = 0.03 * ((k * 7) % 11 - 5)
            hits.append((int(round(sx * z)), int(round(sy * z))))
        layers.append(hits)
    return layers


def empty_event(layer_z):
    return [[] for _ in layer_z]


def random_cluster_event(layer_z, rng, max_hits=5, n_dirs=2, jitter_slope=0.012, min_hits=0, dir_spread=0.3):
    """Tiny random event with hits clustered around a few directions so that pairs fall on both
    sides of the windows (for brute-force comparison)."""
    cx, cy = rng.uniform(-0.3 + dir_spread, 0.3 - dir_spread + 1e-9), rng.uniform(-0.3 + dir_spread, 0.3 - dir_spread + 1e-9)
    dirs = [(cx + rng.uniform(-dir_spread, dir_spread), cy + rng.uniform(-dir_spread, dir_spread))
            for _ in range(n_dirs)]
    layers = []
    for z in layer_z:
        n = int(rng.integers(min_hits, max_hits + 1))
        hits = []
        for _ in range(n):
            d = dirs[int(rng.integers(0, n_dirs))]
            sx = d[0] + rng.uniform(-jitter_slope, jitter_slope)
            sy = d[1] + rng.uniform(-jitter_slope, jitter_slope)
            hits.append((int(round(sx * z)), int(round(sy * z))))
        layers.append(hits)
    return layers


def two_direction_event(layer_z, rng, max_hits=2, jitter_slope=0.003):
    """Two directions 0.017-0.023 apart in x: triplets are pure-direction (in-station window 0.01), while
    links between the two directions straddle the 0.02 link window => partially linked chains."""
    cx, cy = rng.uniform(-0.25, 0.25), rng.uniform(-0.25, 0.25)
    dirs = [(cx, cy), (cx + rng.uniform(0.017, 0.023), cy + rng.uniform(-0.004, 0.004))]
    layers = []
    for z in layer_z:
        hits = []
        for d in dirs:
            for _ in range(int(rng.integers(1, max_hits + 1))):
                hits.append((int(round((d[0] + rng.uniform(-jitter_slope, jitter_slope)) * z)),
                             int(round((d[1] + rng.uniform(-jitter_slope, jitter_slope)) * z))))
        layers.append(hits)
    return layers


def adversarial_suite(seed=1234):
    """(name, layer_z, events, expected or None).  expected = (n_triplets[E][S], n_candidates[E], accept[E])."""
    rng = np.random.default_rng(seed)
    out = []
    z4 = list(GEOMETRY_4)
    # 1. planted exact lines, pairwise separated by >= 0.05 in slope: k triplets per station, k candidates
    slopes = [(-250, 100), (-100, -200), (0, 0), (120, 250), (300, -50)]
    ev = [planted_lines_event(z4, slopes[:k]) for k in range(0, 6)]
    exp = ([[k] * 4 for k in range(0, 6)], list(range(0, 6)), [1 if k >= 2 else 0 for k in range(0, 6)])
    out.append(("planted_lines", z4, ev, exp))
    # 2. narrow cone: closed form and saturation (8*8*8 = 512 per station, 512^4 > 2^32)
    ev = [narrow_cone_event(z4, 2, rng), narrow_cone_event(z4, [1, 2, 3, 2, 1, 2, 3, 1, 1, 1, 2, 2], rng),
          narrow_cone_event(z4, 8, rng)]
    exp = ([[8, 8, 8, 8], [6, 4, 3, 4], [512] * 4], [8 ** 4, 6 * 4 * 3 * 4, 2 ** 32 - 1], [1, 1, 1])
    out.append(("narrow_cone", z4, ev, exp))
    # 3. constructed non-collinear noise + empties
    ev = [lattice_noise_event(z4, 9), empty_event(z4), lattice_noise_event(z4, 14)]
    exp = ([[0] * 4] * 3, [0] * 3, [0] * 3)
    out.append(("lattice_noise_and_empty", z4, ev, exp))
    # 4. one station missing a layer: triplets elsewhere, zero candidates
    layers = planted_lines_event(z4, [(10, 20), (200, -100)])
    layers[7] = []
    out.append(("missing_layer", z4, [layers], ([[2, 2, 0, 2]], [0], [0])))
    # 5. duplicates count separately: the same exact line twice => 2*2*2 triplets per station, 8^S chains
    z6 = list(GEOMETRY_6)
    layers = planted_lines_event(z6, [(50, 50), (50, 50)])
    out.append(("duplicates", z6, [layers], ([[8] * 6], [8 ** 6], [1])))
    # 6. random clustered tiny events (no closed form; compared against brute force / oracle)
    z3 = station_layers_z([60, 100, 150])
    ev = [random_cluster_event(z3, rng, max_hits=3, n_dirs=2, jitter_slope=0.007, min_hits=1, dir_spread=0.012)
          for _ in range(30)]
    ev += [random_cluster_event(z3, rng, max_hits=4, n_dirs=3, jitter_slope=0.012) for _ in range(20)]
    ev += [two_direction_event(z3, rng) for _ in range(25)]
    out.append(("random_clusters_S3", z3, ev, None))
    ev = [random_cluster_event(z4, rng, max_hits=2, n_dirs=2, jitter_slope=0.006, min_hits=1, dir_spread=0.01)
          for _ in range(20)]
    out.append(("random_clusters_S4", z4, ev, None))
    return out
