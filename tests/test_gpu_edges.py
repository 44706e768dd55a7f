"""Edge cases of the CUDA path against the oracle: inputs and capacities the seeded batches never reach."""
import time

import numpy as np
import pytest

from tests.test_gpu_parity import as_oracle_types

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def velo(geometry):
    import torch

    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1912_09161_b200 import binding

    v = binding.AllenVelo(geometry)
    yield v
    v.destroy()


def test_repeated_sp_address_and_zero_hitmap(velo, geometry):
    """R1: a repeated SP address inside a bank ORs its hit maps (set semantics), a zero hit map fires no pixel.  The raw
    words are assembled by hand (pack_events de-duplicates addresses and never writes an empty hit map)."""
    import oracle
    from paper_1912_09161_b200 import binding
    from tests.helpers import compare_clusters, raw_from_sp_words, sp_word

    ev0 = {
        5: [sp_word(10, 7, 0x01), sp_word(10, 7, 0x10), sp_word(11, 7, 0x00),      # same address twice; an empty word
            sp_word(40, 3, 0x81), sp_word(40, 3, 0x81), sp_word(40, 3, 0x18)],     # three times, overlapping maps
        6: [sp_word(0, 0, 0x00)],                                                 # a bank with only an empty word
        9: [sp_word(100, 20, 0x0F), sp_word(100, 21, 0x01), sp_word(100, 20, 0xF0), sp_word(101, 20, 0x00)],
    }
    # the same address on two sensors stays two clusters; duplicates that bridge two neighbours into one cluster
    ev1 = {7: [sp_word(5, 5, 0x08), sp_word(5, 6, 0x01), sp_word(5, 5, 0x08)], 8: [sp_word(5, 5, 0x08)],
           12: [sp_word(30, 9, 0x80), sp_word(31, 10, 0x01), sp_word(30, 9, 0x00), sp_word(30, 9, 0x80)]}
    raw, off = raw_from_sp_words(geometry.n_sensors, [ev0, ev1, {}])
    ref = oracle.reconstruct(geometry, raw, off)
    clusters, tracks = binding.reconstruct_batch(velo, raw, off)
    c, _ = as_oracle_types(clusters, tracks)
    assert not compare_clusters(c, ref.clusters)
    # pinned by hand, not only against the oracle: event 0 = 2 pixels in one SP of sensor 5 (columns 0 and 1 of row 0: one
    # cluster), 4 pixels of SP (40, 3) (rows 0 and 3 of both columns: two clusters), sensor 9: 8 + 1 pixels in one cluster
    n0 = int(ref.clusters.event_offsets[1])
    assert sorted(clusters["n_pixels"][:n0].tolist()) == [2, 2, 2, 9]
    assert clusters["status"].tolist() == [0, 0, 0]


def test_track_capacity_is_respected(velo, oracle_of):
    """out_tracks too small: events whose tracks do not fit are flagged TRACK_CAPACITY and not written, the offsets and
    the total at hit_offsets[capacity_tracks] still report the true sizes, the events that fit are exact."""
    import torch

    from paper_1912_09161_b200 import binding

    batch, ref = oracle_of(1, 64)
    rt = ref.tracks
    nt = int(rt.event_offsets[-1])
    tcap = nt // 2
    raw_bytes = int(batch.raw.size)
    oc, ot = binding.alloc_outputs(batch.n_events, velo.n_layers, raw_bytes // 2 + 16, tcap, raw_bytes // 2, "cuda:0", True, False)
    ws = torch.empty(velo.workspace_bytes(batch.n_events, raw_bytes), dtype=torch.uint8, device="cuda:0")
    velo.set_workspace(ws)
    d_raw = torch.from_numpy(batch.raw).to("cuda:0")
    d_off = torch.from_numpy(batch.event_offsets.view(np.int32)).to("cuda:0")
    assert velo.reconstruct(d_raw, d_off, batch.n_events, None, oc, ot) == 0, velo.last_error()
    torch.cuda.synchronize()
    te = ot.event_offsets.cpu().numpy().view(np.uint32)
    ho = ot.hit_offsets.cpu().numpy().view(np.uint32)
    status = oc.status.cpu().numpy().view(np.uint32)
    assert np.array_equal(te, rt.event_offsets)                       # true totals
    assert int(ho[tcap]) == int(rt.hit_offsets[-1])                   # total hits at the fixed place, also on overflow
    over = rt.event_offsets[1:] > tcap
    assert over.any() and not over.all()
    assert np.array_equal((status & binding.STATUS_TRACK_CAPACITY) != 0, over & (np.diff(rt.event_offsets) > 0))
    n_ok = int(rt.event_offsets[:-1][over][0])                        # tracks of the events before the first that overflows
    assert np.array_equal(ho[:n_ok + 1], rt.hit_offsets[:n_ok + 1])
    hits = ot.hits.cpu().numpy().view(np.uint16)
    assert np.array_equal(hits[:int(ho[n_ok])], rt.hits[:int(rt.hit_offsets[n_ok])])
    assert np.array_equal(ot.tx.cpu().numpy()[:n_ok].view(np.uint32), rt.tx[:n_ok].view(np.uint32))


def hot_sensor_event(rng, sensor, n_sp):
    """n_sp super-pixels on one sensor with 1-3 pixels each (some touching their neighbours)."""
    px = set()
    while len({(c >> 1, r >> 2) for _, c, r in px}) < n_sp:
        c, r = int(rng.integers(768)), int(rng.integers(256))
        px.add((sensor, c, r))
        if rng.random() < 0.4:
            px.add((sensor, min(767, c + 1), r))
        if rng.random() < 0.2:
            px.add((sensor, c, min(255, r + 1)))
    return sorted(px)


def test_more_oversize_layers_than_pool_slots(velo, geometry):
    """Every event has one sensor with > 512 SP words: such a layer runs in a slot of the BIG pool (16 slots for a batch
    this size).  The slots are given back after each item, so 48 of them all finish: no STAGE_OVERFLOW, clusters exact
    (the pool used to be a bump counter that a batch like this exhausted)."""
    import oracle
    from paper_1912_09161_b200 import binding, workload
    from tests.helpers import compare_clusters

    rng = np.random.default_rng(5)
    events = [hot_sensor_event(rng, 4 * (e % 20) + 1, 560 + 5 * (e % 7)) + [(60, 10 + e, 10)] for e in range(48)]
    raw, off = workload.pack_events(geometry, events, shuffle_seed=9)
    ref = oracle.reconstruct(geometry, raw, off, n_threads=8)
    a = binding.reconstruct_batch(velo, raw, off)
    b = binding.reconstruct_batch(velo, raw, off)
    assert not a[0]["status"].any()
    c, _ = as_oracle_types(*a)
    assert not compare_clusters(c, ref.clusters)
    for k in ("key", "x", "phi16", "layer_offsets"):  # bit-identical from call to call under this load
        assert np.array_equal(a[0][k], b[0][k])


def test_a_snake_that_fills_the_largest_slot_is_fast(velo, geometry):
    """One serpentine cluster of ~8000 SP words on one sensor (label propagation took one pass per hop of
    the component's diameter, thousands of passes over global memory; with pointer jumping it is O(log diameter))."""
    import oracle
    import torch

    from paper_1912_09161_b200 import binding, workload
    from tests.helpers import compare_clusters

    snake = []
    for k in range(62):                     # runs along the columns on every fourth row, joined alternately left / right
        r = 4 * k
        snake += [(9, c, r) for c in range(0, 256)]
        if k < 61:
            edge = 255 if k % 2 == 0 else 0
            snake += [(9, edge, r + 1), (9, edge, r + 2), (9, edge, r + 3)]
    raw, off = workload.pack_events(geometry, [snake, [(3, 5, 5)]], shuffle_seed=2)
    ref = oracle.reconstruct(geometry, raw, off)
    assert int(ref.clusters.n_pixels.max()) == len(snake)   # one cluster
    binding.reconstruct_batch(velo, raw, off)                # warm-up (allocations, first launch)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    clusters, tracks = binding.reconstruct_batch(velo, raw, off)
    dt = time.perf_counter() - t0
    c, _ = as_oracle_types(clusters, tracks)
    assert not compare_clusters(c, ref.clusters)
    assert not clusters["status"].any()
    assert dt < 0.25, f"{dt:.3f} s for one call (allocation and copies included)"


@pytest.mark.parametrize("params", [dict(s_seed=4.0, s_fwd=4.0, w_seed_phi16=1500), dict(s_seed=0.5, max_slope=2.0, max_skipped=3)])
def test_loose_cuts_overflow_the_candidate_lists_and_track_slots(geometry, batch_of, params):
    """With very loose seeding cuts nearly every (a, b, c) in the windows passes: the candidate lists of velo_seed.cu
    outgrow their regions and events run out of active-track slots in velo_follow.cu; those events are redone by the
    CTA-per-event kernel.  Results still equal the oracle's."""
    import oracle
    from paper_1912_09161_b200 import binding
    from tests.helpers import compare_clusters, compare_tracks

    batch = batch_of(2, 48)
    ref = oracle.reconstruct(geometry, batch.raw, batch.event_offsets, params=params, n_threads=8)
    v = binding.AllenVelo(geometry, params=params)
    try:
        clusters, tracks = binding.reconstruct_batch(v, batch.raw, batch.event_offsets)
        counters = v.track_counters()
    finally:
        v.destroy()
    assert sum(counters["follow"]) == batch.n_events and sum(counters["second_pass"]) > 0, counters
    c, t = as_oracle_types(clusters, tracks)
    assert not compare_clusters(c, ref.clusters)
    rep = compare_tracks(t, ref.tracks, ref)
    assert rep["n_got"] == rep["n_ref"] and rep["mismatched_tracks"] == 0 and rep["bad_fits"] == 0, rep
    assert np.array_equal(t.hits, ref.tracks.hits)
    assert not clusters["status"].any()


@pytest.mark.parametrize("regions", [(1, 1), (2, 2), (8, 8), (4, 1)])
def test_local_clustering_variant_against_the_oracle(geometry, batch_of, regions):
    """SURVEY 8(f4) / DESIGN.md R11 ("searches for clusters locally in small regions"): clusters confined to regions
    of sp_cols x sp_rows super-pixels.  Everything (clusters bit for bit, tracks, fit) equals the oracle run with the same
    regions; the deviation from the exact components is what the oracle counts (tests/test_oracle_local_clusters.py)."""
    import oracle
    from paper_1912_09161_b200 import binding
    from tests.helpers import compare_clusters, compare_tracks

    batch = batch_of(2, 64)
    ref = oracle.reconstruct(geometry, batch.raw, batch.event_offsets, cluster_regions=regions, n_threads=8)
    exact = oracle.reconstruct(geometry, batch.raw, batch.event_offsets, n_threads=8)
    assert len(ref.clusters.key) > len(exact.clusters.key)  # the variant does split clusters on this batch
    v = binding.AllenVelo(geometry)
    try:
        v.set_cluster_regions(*regions)
        clusters, tracks = binding.reconstruct_batch(v, batch.raw, batch.event_offsets)
        v.set_cluster_regions(0, 0)
        back = binding.reconstruct_batch(v, batch.raw, batch.event_offsets)
    finally:
        v.destroy()
    c, t = as_oracle_types(clusters, tracks)
    assert not compare_clusters(c, ref.clusters)
    rep = compare_tracks(t, ref.tracks, ref)
    assert rep["n_got"] == rep["n_ref"] and rep["mismatched_tracks"] == 0 and rep["bad_fits"] == 0, rep
    assert np.array_equal(t.hits, ref.tracks.hits)
    c0, _ = as_oracle_types(*back)
    assert not compare_clusters(c0, exact.clusters)  # switched off again: exact components


def test_more_than_65535_clusters_in_one_event(velo, geometry):
    """R8: hit indices are 16 bit, so an event with more than 65535 clusters gets its clusters (all exact) but no tracks,
    and is flagged TOO_MANY_CLUSTERS; the oracle does the same.  The other event of the batch is untouched."""
    import oracle
    from paper_1912_09161_b200 import binding, workload
    from tests.helpers import compare_clusters

    # isolated pixels on a 3 x 3 grid over all 104 sensors: 256 x 85 per sensor would be too many; 700 per sensor = 72 800
    big = [(s, 3 * (k % 256), 3 * (k // 256)) for s in range(geometry.n_sensors) for k in range(700)]
    small = workload.generate(1, n_events=1)
    m = small.pixels["event"] == 0
    other = sorted(set(zip(small.pixels["sensor"][m].tolist(), small.pixels["col"][m].tolist(), small.pixels["row"][m].tolist())))
    raw, off = workload.pack_events(geometry, [big, other], shuffle_seed=1)
    ref = oracle.reconstruct(geometry, raw, off)
    assert int(ref.clusters.event_offsets[1]) == len(big) > 65535
    assert ref.clusters.status.tolist() == [oracle.STATUS_TOO_MANY_CLUSTERS, 0]
    clusters, tracks = binding.reconstruct_batch(velo, raw, off)
    c, t = as_oracle_types(clusters, tracks)
    assert not compare_clusters(c, ref.clusters)
    assert np.array_equal(t.event_offsets, ref.tracks.event_offsets) and t.event_offsets[1] == 0
    assert np.array_equal(t.hits, ref.tracks.hits) and len(t.hits) > 0
