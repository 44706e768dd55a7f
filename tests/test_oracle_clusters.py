"""Pins for oracle steps O1 (decode), O2 (clustering), O4 (sort) — DESIGN.md §4.

The oracle's flood fill is checked against things that are not the oracle: the generator's pixel truth, two other
formulations of connected components written here (union-find, transitive closure), scipy.ndimage.label with a
3x3 structuring element, hand-worked cases, and the invariants that define a maximal 8-connected component.
"""
import numpy as np
import pytest
from scipy import ndimage

import oracle
from paper_1912_09161_b200 import workload
from tests.helpers import ccl_closure, ccl_union_find

N_COLS = 768


def run_pixels(geometry, events, shuffle_seed=0):
    raw, off = workload.pack_events(geometry, events, shuffle_seed=shuffle_seed)
    return oracle.reconstruct(geometry, raw, off, with_pixels=True)


def clusters_as_sets(res, e=0):
    """{sensor: frozenset of frozenset((col,row))} for event e from the oracle's pixel membership."""
    out = {}
    sel = res.pix_event == e
    for k, c in zip(res.pix_key[sel], res.pix_cluster[sel]):
        s, idx = int(k) >> 18, int(k) & 0x3FFFF
        out.setdefault((s, int(c)), set()).add((idx % N_COLS, idx // N_COLS))
    per_sensor = {}
    for (s, _), pix in out.items():
        per_sensor.setdefault(s, set()).add(frozenset(pix))
    return {s: frozenset(v) for s, v in per_sensor.items()}


# ---------------------------------------------------------------- O1
def test_decode_roundtrip_against_generator_truth(oracle_of):
    batch, res = oracle_of(1, 40)
    px = batch.pixels
    truth = set(zip(px["event"].tolist(), ((px["sensor"].astype(np.uint32) << 18)
                                            | (px["row"].astype(np.uint32) * N_COLS + px["col"])).tolist()))
    decoded = list(zip(res.pix_event.tolist(), res.pix_key.tolist()))
    assert len(decoded) == len(set(decoded)), "a pixel was decoded twice"
    assert set(decoded) == truth


def test_decode_bit_layout(geometry):
    # bit 4*dc+dr <-> pixel (col = 2*sp_col+dc, row = 4*sp_row+dr): one word per bit, hand-assembled.
    for bit in range(8):
        sp_col, sp_row = 383, 63
        word = (sp_col << 14) | (sp_row << 8) | (1 << bit)
        words = [0x56454C4F, geometry.n_sensors, 1, 0] + [0] * 5 + [1] * (geometry.n_sensors - 4)
        while len(words) % 4:
            words.append(0)
        words += [word, 0, 0, 0]
        raw = np.array(words, np.uint32).view(np.uint8)
        res = oracle.reconstruct(geometry, raw, np.array([0, raw.size], np.uint32), with_pixels=True)
        assert res.clusters.status[0] == 0
        col, row = 2 * sp_col + (bit >> 2), 4 * sp_row + (bit & 3)
        assert res.pix_key.tolist() == [(4 << 18) | (row * N_COLS + col)]  # bank 4 holds the word


def test_bad_header_and_bad_sp(geometry):
    raw, off = workload.pack_events(geometry, [[(0, 5, 5)], [(1, 9, 9)]])
    bad = raw.copy()
    bad[0] ^= 0xFF  # magic of event 0
    res = oracle.reconstruct(geometry, bad, off)
    assert res.clusters.status[0] & oracle.STATUS_BAD_HEADER and res.clusters.status[1] == 0
    assert res.clusters.event_offsets.tolist() == [0, 0, 1]
    # SP column address 384 (beyond the 768-column sensor) is ignored and flagged
    w = raw.view(np.uint32).copy()
    first_sp = int(off[0]) // 4 + 4 + (geometry.n_sensors + 1 + 3) // 4 * 4
    w[first_sp] = (384 << 14) | (1 << 8) | 1
    res = oracle.reconstruct(geometry, w.view(np.uint8), off)
    assert res.clusters.status[0] == oracle.STATUS_BAD_SP
    assert res.clusters.event_offsets.tolist() == [0, 0, 1]


# ---------------------------------------------------------------- O2
HAND_CASES = [
    # (pixels (col,row) on one sensor, expected clusters)
    ([(10, 10)], [[(10, 10)]]),
    # 2x2 block straddling four super-pixels (SP = 2 cols x 4 rows): cols 1|2, rows 3|4
    ([(1, 3), (2, 3), (1, 4), (2, 4)], [[(1, 3), (2, 3), (1, 4), (2, 4)]]),
    # diagonal chain across sp_col and sp_row boundaries
    ([(0, 0), (1, 1), (2, 2), (3, 3), (4, 4), (5, 5)], [[(0, 0), (1, 1), (2, 2), (3, 3), (4, 4), (5, 5)]]),
    # anti-diagonal across an SP corner: (1,4) and (2,3) touch only by a corner
    ([(1, 4), (2, 3)], [[(1, 4), (2, 3)]]),
    # two pixels in ONE super-pixel separated by an empty row are two clusters
    ([(0, 0), (0, 2)], [[(0, 0)], [(0, 2)]]),
    ([(0, 0), (1, 3)], [[(0, 0)], [(1, 3)]]),
    # ... but a neighbouring super-pixel can bridge them
    ([(0, 0), (0, 2), (2, 1)], [[(0, 0)], [(0, 2)], [(2, 1)]]),
    ([(1, 0), (1, 2), (2, 1)], [[(1, 0), (1, 2), (2, 1)]]),
    # sensor corners and edges
    ([(0, 0), (767, 0), (0, 255), (767, 255)], [[(0, 0)], [(767, 0)], [(0, 255)], [(767, 255)]]),
    ([(766, 254), (767, 255)], [[(766, 254), (767, 255)]]),
    # gap of one pixel is not connected
    ([(100, 100), (102, 100), (100, 102)], [[(100, 100)], [(102, 100)], [(100, 102)]]),
    # U shape joined only at the bottom, spanning several SPs
    ([(20, r) for r in range(8, 17)] + [(24, r) for r in range(8, 17)] + [(c, 17) for c in range(20, 25)],
     [[(20, r) for r in range(8, 17)] + [(24, r) for r in range(8, 17)] + [(c, 17) for c in range(20, 25)]]),
]


@pytest.mark.parametrize("pixels,expected", HAND_CASES)
def test_ccl_hand_cases(geometry, pixels, expected):
    for sensor in (0, 57, 103):
        res = run_pixels(geometry, [[(sensor, c, r) for c, r in pixels]])
        got = clusters_as_sets(res)[sensor]
        assert got == frozenset(frozenset(c) for c in expected)


def test_same_address_in_two_sensors_stays_two_clusters(geometry):
    res = run_pixels(geometry, [[(8, 50, 60), (9, 50, 60), (9, 51, 61)]])
    got = clusters_as_sets(res)
    assert got[8] == frozenset([frozenset([(50, 60)])])
    assert got[9] == frozenset([frozenset([(50, 60), (51, 61)])])


def test_cluster_statistics_hand_case(geometry):
    # L-shaped 3-pixel cluster: n, sums, seed pixel and key by hand
    res = run_pixels(geometry, [[(5, 301, 77), (5, 302, 77), (5, 301, 78)]])
    c = res.clusters
    assert c.event_offsets.tolist() == [0, 1]
    assert (c.n_pixels[0], c.sum_col[0], c.sum_row[0]) == (3, 301 + 302 + 301, 77 + 77 + 78)
    assert c.key[0] == (5 << 18) | (77 * N_COLS + 301)
    want = sum(oracle.mix32(r * N_COLS + col) for col, r in [(301, 77), (302, 77), (301, 78)]) & 0xFFFFFFFF
    assert c.checksum[0] == want


def test_mix32_reference_values():
    # mix32 written out with Python integers (reading R2)
    def mix(v):
        m = ((v + 1) * 2654435761) & 0xFFFFFFFF
        m ^= m >> 15
        m = (m * 2246822519) & 0xFFFFFFFF
        m ^= m >> 13
        return m

    for v in [0, 1, 2, 767, 768, 196607, 0xFFFFFFFF, 123456789]:
        assert oracle.mix32(v) == mix(v)
    # distinct pixels of one sensor never collide in the low 32 bits often enough to matter: injective on a sample
    vals = [mix(v) for v in range(0, 196608, 7)]
    assert len(set(vals)) == len(vals)


@pytest.mark.parametrize("seed", range(6))
def test_ccl_three_formulations_and_scipy_on_random_grids(geometry, seed):
    rng = np.random.default_rng(1000 + seed)
    h, w = 24, 20  # rows x cols, offset so that the patch straddles SP boundaries and the sensor edge
    density = [0.08, 0.2, 0.35, 0.5, 0.65, 0.9][seed]
    events, grids, origins = [], [], []
    for _ in range(4):
        grid = rng.random((h, w)) < density
        c0 = int(rng.choice([0, 3, 377, N_COLS - w]))
        r0 = int(rng.choice([0, 2, 117, 256 - h]))
        sensor = int(rng.integers(0, geometry.n_sensors))
        rows, cols = np.nonzero(grid)
        events.append([(sensor, int(c) + c0, int(r) + r0) for r, c in zip(rows, cols)])
        grids.append(grid)
        origins.append((sensor, c0, r0))
    res = run_pixels(geometry, events, shuffle_seed=seed)
    for e, (grid, (sensor, c0, r0)) in enumerate(zip(grids, origins)):
        pixels = [(c, r) for _, c, r in events[e]]
        got = clusters_as_sets(res, e).get(sensor, frozenset())
        assert got == ccl_union_find(pixels)
        assert got == ccl_closure(pixels)
        labels, n = ndimage.label(grid, structure=np.ones((3, 3)))
        scipy_sets = frozenset(
            frozenset((int(c) + c0, int(r) + r0) for r, c in zip(*np.nonzero(labels == k))) for k in range(1, n + 1))
        assert got == scipy_sets
        assert res.clusters.event_offsets[e + 1] - res.clusters.event_offsets[e] == n


def test_ccl_invariants_on_generated_events(oracle_of):
    batch, res = oracle_of(1, 40)
    c = res.clusters
    # every fired pixel in exactly one cluster; sum of n = number of distinct fired pixels
    assert len(res.pix_key) == int(c.n_pixels.sum())
    for e in range(0, batch.n_events, 7):
        sel = res.pix_event == e
        keys, cl = res.pix_key[sel], res.pix_cluster[sel]
        sensor, idx = keys >> 18, keys & 0x3FFFF
        col, row = (idx % N_COLS).astype(np.int64), (idx // N_COLS).astype(np.int64)
        base = int(c.event_offsets[e])
        # statistics follow from membership
        n_cl = int(c.event_offsets[e + 1]) - base
        assert np.array_equal(np.bincount(cl, minlength=n_cl), c.n_pixels[base:base + n_cl])
        assert np.array_equal(np.bincount(cl, weights=col, minlength=n_cl).astype(np.uint32), c.sum_col[base:base + n_cl])
        assert np.array_equal(np.bincount(cl, weights=row, minlength=n_cl).astype(np.uint32), c.sum_row[base:base + n_cl])
        seed = np.full(n_cl, 0xFFFFFFFF, np.uint32)
        np.minimum.at(seed, cl, keys)
        assert np.array_equal(seed, c.key[base:base + n_cl])
        # no two different clusters of a sensor are 8-adjacent (maximality) — all pixel pairs of the event
        same_sensor = sensor[:, None] == sensor[None, :]
        adjacent = same_sensor & (np.abs(col[:, None] - col[None, :]) <= 1) & (np.abs(row[:, None] - row[None, :]) <= 1)
        assert np.all(cl[:, None][adjacent.any(axis=1)] >= 0)
        ii, jj = np.nonzero(adjacent)
        assert np.all(cl[ii] == cl[jj])
        # each cluster connected: union-find over the adjacency edges gives exactly the oracle's partition
        parent = np.arange(len(cl))
        for i, j in zip(ii, jj):
            while parent[i] != i:
                i = parent[i]
            while parent[j] != j:
                j = parent[j]
            if i != j:
                parent[max(i, j)] = min(i, j)
        roots = np.array([_root(parent, i) for i in range(len(cl))])
        assert len(set(roots.tolist())) == n_cl
        assert len(set(zip(roots.tolist(), cl.tolist()))) == n_cl


def _root(parent, i):
    while parent[i] != i:
        i = parent[i]
    return i


def test_sp_word_order_inside_bank_is_irrelevant(geometry):
    rng = np.random.default_rng(5)
    pix = [(int(s), int(c), int(r)) for s, c, r in zip(rng.integers(0, 104, 400), rng.integers(0, 40, 400),
                                                       rng.integers(0, 40, 400))]
    a = run_pixels(geometry, [pix], shuffle_seed=None)
    b = run_pixels(geometry, [pix], shuffle_seed=99)
    for name in ("key", "n_pixels", "sum_col", "sum_row", "checksum", "phi16", "x", "y", "z"):
        assert np.array_equal(getattr(a.clusters, name), getattr(b.clusters, name))


# ---------------------------------------------------------------- O4
def test_sort_order_and_layer_offsets(oracle_of, geometry):
    batch, res = oracle_of(1, 40)
    c = res.clusters
    L = geometry.n_layers
    sensor_layer = geometry.sensor_layer()
    assert c.layer_offsets[0] == 0 and c.layer_offsets[-1] == len(c.key)
    assert np.array_equal(c.layer_offsets[::L], c.event_offsets)
    assert np.all(np.diff(c.layer_offsets.astype(np.int64)) >= 0)
    layer_of_cluster = sensor_layer[c.key >> 18]
    for e in range(batch.n_events):
        for l in range(L):
            a, b = int(c.layer_offsets[e * L + l]), int(c.layer_offsets[e * L + l + 1])
            assert np.all(layer_of_cluster[a:b] == l)
            sk = (c.phi16[a:b].astype(np.int64) + 32768) * (1 << 32) + c.key[a:b]
            assert np.all(np.diff(sk) > 0), "not strictly ascending in (phi16, key)"


def test_sort_tie_rule_equal_phi(geometry):
    # Many isolated single-pixel clusters on one layer: several share a phi16 value; among those the order must
    # follow the key, and the whole layer must be strictly ascending in (phi16, key).
    rng = np.random.default_rng(11)
    cells = rng.choice(250 * 80, size=4000, replace=False)
    pix = [(int(s), 3 * int(k % 250) + 1, 3 * int(k // 250) + 1) for s, k in zip(rng.integers(0, 4, 4000), cells)]
    res = run_pixels(geometry, [pix])
    c = res.clusters
    assert len(c.key) == 4000 and np.all(c.n_pixels == 1)
    phi, key = c.phi16.astype(np.int64), c.key.astype(np.int64)
    ties = phi[1:] == phi[:-1]
    assert ties.sum() > 20, "test needs ties to be meaningful"
    assert np.all(key[1:][ties] > key[:-1][ties])
    assert np.all((phi[1:] > phi[:-1]) | ties)
