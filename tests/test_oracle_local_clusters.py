"""Pins of the oracle's local clustering variant (O2-local; R11; "a clustering algorithm employing bit
masks, which searches for clusters locally in small regions. Every region can be treated independently").

Definition under test: with regions of sp_cols x sp_rows super-pixels switched on, a cluster is a maximal 8-connected
set of fired pixels inside one region; (0, 0) = exact connected components.  Pinned to things other than the oracle:
scipy.ndimage.label applied region by region, hand cases, invariants, and the limit of one region per sensor."""
import numpy as np
import pytest

import oracle
from paper_1912_09161_b200 import workload


def clusters_of(geometry, pixels, regions):
    raw, off = workload.pack_events(geometry, [pixels])
    return oracle.reconstruct(geometry, raw, off, with_pixels=True, cluster_regions=regions)


def test_hand_cases(geometry):
    # a 2x2 pixel block straddling four super-pixels: SP columns 5|6 meet at pixel columns 11|12, SP rows 2|3 at pixel rows 11|12
    block = [(3, 11, 11), (3, 12, 11), (3, 11, 12), (3, 12, 12)]
    assert clusters_of(geometry, block, (0, 0)).clusters.n_pixels.tolist() == [4]
    assert sorted(clusters_of(geometry, block, (1, 1)).clusters.n_pixels.tolist()) == [1, 1, 1, 1]
    # regions of 2x2 super-pixels: columns 10..13 and rows 8..15 are one region (SP col 5 -> region 2 with SP col 4: no!)
    # SP col 5 = region 2 (SP cols 4,5), SP col 6 = region 3: still split in columns, joined in rows (SP rows 2,3 = region 1)
    assert sorted(clusters_of(geometry, block, (2, 2)).clusters.n_pixels.tolist()) == [2, 2]
    # regions of 2 x 1: split in rows as well
    assert sorted(clusters_of(geometry, block, (2, 1)).clusters.n_pixels.tolist()) == [1, 1, 1, 1]
    # a horizontal run of 10 pixels from column 0: regions of 2 SP columns = 4 pixel columns -> 4 + 4 + 2
    run = [(7, c, 100) for c in range(10)]
    assert sorted(clusters_of(geometry, run, (2, 64)).clusters.n_pixels.tolist()) == [2, 4, 4]
    # the sums of the pieces add up to the sums of the whole
    whole = clusters_of(geometry, run, (0, 0)).clusters
    parts = clusters_of(geometry, run, (2, 64)).clusters
    assert int(parts.sum_col.sum()) == int(whole.sum_col.sum()) and int(parts.sum_row.sum()) == int(whole.sum_row.sum())


def test_one_region_per_sensor_is_the_exact_definition(geometry):
    batch = workload.generate(2, n_events=6)
    exact = oracle.reconstruct(geometry, batch.raw, batch.event_offsets)
    big = oracle.reconstruct(geometry, batch.raw, batch.event_offsets, cluster_regions=(512, 64))
    for name in ("event_offsets", "layer_offsets", "key", "n_pixels", "sum_col", "sum_row", "phi16", "checksum"):
        assert np.array_equal(getattr(exact.clusters, name), getattr(big.clusters, name)), name
    assert np.array_equal(exact.tracks.hits, big.tracks.hits)
    # and the switch does not stick: the next default run is exact again
    again = oracle.reconstruct(geometry, batch.raw, batch.event_offsets)
    assert np.array_equal(exact.clusters.key, again.clusters.key)


@pytest.mark.parametrize("regions", [(1, 1), (2, 2), (4, 2), (8, 8)])
def test_against_scipy_label_region_by_region(geometry, regions):
    ndimage = pytest.importorskip("scipy.ndimage")
    rng = np.random.default_rng(17 + regions[0])
    w, h = 64, 48  # pixels; a corner of sensor 5
    for density in (0.05, 0.2, 0.45):
        grid = rng.random((h, w)) < density
        pixels = [(5, int(c), int(r)) for r, c in zip(*np.nonzero(grid))]
        res = clusters_of(geometry, pixels, regions)
        pw, ph = 2 * regions[0], 4 * regions[1]
        want = []  # (n, sum_col, sum_row) of every component of every region, by scipy on the region's own tile
        for r0 in range(0, h, ph):
            for c0 in range(0, w, pw):
                lab, n = ndimage.label(grid[r0:r0 + ph, c0:c0 + pw], structure=np.ones((3, 3)))
                for k in range(1, n + 1):
                    rr, cc = np.nonzero(lab == k)
                    want.append((len(rr), int(cc.sum()) + c0 * len(rr), int(rr.sum()) + r0 * len(rr)))
        got = sorted(zip(res.clusters.n_pixels.tolist(), res.clusters.sum_col.tolist(), res.clusters.sum_row.tolist()))
        assert got == sorted(want), (regions, density)


def test_invariants_and_deviation_on_physics_like_events(geometry):
    """Every fired pixel in exactly one cluster, no cluster crosses a region border; the deviation from the exact
    components (clusters whose pixel set differs) is counted: this is the number DESIGN.md R11 quotes."""
    batch = workload.generate(2, n_events=40)
    exact = oracle.reconstruct(geometry, batch.raw, batch.event_offsets, with_pixels=True)
    for regions in ((1, 1), (2, 2), (8, 8)):
        loc = oracle.reconstruct(geometry, batch.raw, batch.event_offsets, with_pixels=True, cluster_regions=regions)
        assert len(loc.pix_key) == len(exact.pix_key) == int(exact.clusters.n_pixels.sum()) == int(loc.clusters.n_pixels.sum())
        # pixels of one cluster share sensor and region
        px = loc.pix_key & 0x3FFFF
        col, row = px % geometry.n_cols, px // geometry.n_cols
        reg = ((loc.pix_key >> 18).astype(np.int64) << 40) | ((col // 2 // regions[0]).astype(np.int64) << 20) | (row // 4 // regions[1])
        order = np.lexsort((loc.pix_cluster, loc.pix_event))
        same = (loc.pix_event[order][1:] == loc.pix_event[order][:-1]) & (loc.pix_cluster[order][1:] == loc.pix_cluster[order][:-1])
        assert np.all(reg[order][1:][same] == reg[order][:-1][same])
        # deviation: exact clusters that were split
        n_exact, n_loc = len(exact.clusters.key), len(loc.clusters.key)
        assert n_loc >= n_exact
        split = n_loc - n_exact
        multi = int((exact.clusters.n_pixels > 1).sum())
        print(f"regions {regions}: {n_exact} exact clusters ({multi} with > 1 pixel), {n_loc} local clusters, +{split} "
              f"({100.0 * split / n_exact:.2f} %)")
        if regions == (8, 8):
            assert split < 0.02 * n_exact
