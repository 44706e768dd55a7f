"""Parity of the CUDA path (through the C ABI) against the oracle, element by element, on the same seeded inputs.

Bar (BASELINE.json north_star): clusters bit-exact (incl. fp32 positions, phi16 and the membership checksum); track
hit lists exact as canonically sorted sets (near-cut mismatches counted, must stay < 0.1 % of tracks — expected 0
because both sides decide in the same fp32 arithmetic, R3/R5/R7); fit parameters within 1e-5 (R6).
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def velo(geometry):
    import torch

    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1912_09161_b200 import binding

    v = binding.AllenVelo(geometry)
    yield v
    v.destroy()


def as_oracle_types(clusters, tracks):
    import oracle

    c = oracle.Clusters(clusters["event_offsets"], clusters["layer_offsets"], clusters["key"], clusters["n_pixels"],
                        clusters["sum_col"], clusters["sum_row"], clusters["x"], clusters["y"], clusters["z"],
                        clusters["phi16"], clusters["checksum"], clusters["status"])
    t = oracle.Tracks(tracks["event_offsets"], tracks["hit_offsets"], tracks["hits"], tracks["x0"], tracks["y0"],
                      tracks["tx"], tracks["ty"])
    return c, t


def check_parity(velo, batch, ref, **kw):
    from paper_1912_09161_b200 import binding
    from tests.helpers import compare_clusters, compare_tracks

    clusters, tracks = binding.reconstruct_batch(velo, batch.raw, batch.event_offsets, **kw)
    c, t = as_oracle_types(clusters, tracks)
    diffs = compare_clusters(c, ref.clusters)
    assert not diffs, diffs
    rep = compare_tracks(t, ref.tracks, ref)
    assert rep["n_got"] == rep["n_ref"], rep
    assert rep["hard_mismatched_tracks"] == 0, rep
    assert rep["near_cut_mismatched_tracks"] <= 1e-3 * max(1, rep["n_ref"]), rep
    assert rep["mismatched_tracks"] == 0, rep  # expected: exactly equal
    assert rep["bad_fits"] == 0, rep
    # identical order of tracks and hits (order of creation / addition), not only identical sets
    assert np.array_equal(t.hit_offsets, ref.tracks.hit_offsets)
    assert np.array_equal(t.hits, ref.tracks.hits)
    return clusters, tracks


@pytest.mark.parametrize("config,n_events", [(0, None), (1, 64), (2, 200), (3, 48)])
def test_parity_on_seeded_configs(velo, oracle_of, config, n_events):
    batch, ref = oracle_of(config, n_events)
    check_parity(velo, batch, ref)


def test_parity_without_checksum_array(velo, oracle_of):
    batch, ref = oracle_of(2, 200)
    from paper_1912_09161_b200 import binding
    from tests.helpers import compare_clusters

    clusters, tracks = binding.reconstruct_batch(velo, batch.raw, batch.event_offsets, with_checksum=False)
    clusters["checksum"] = ref.clusters.checksum
    c, t = as_oracle_types(clusters, tracks)
    assert not compare_clusters(c, ref.clusters, check_checksum=False)
    assert np.array_equal(t.hits, ref.tracks.hits)


def test_empty_batch_and_empty_events(velo, geometry):
    import oracle
    from paper_1912_09161_b200 import binding, workload

    clusters, tracks = binding.reconstruct_batch(velo, np.zeros(0, np.uint8), np.zeros(1, np.uint32))
    assert clusters["n"] == 0 and tracks["n"] == 0
    raw, off = workload.pack_events(geometry, [[], [(3, 5, 5)], []])
    ref = oracle.reconstruct(geometry, raw, off)
    clusters, tracks = binding.reconstruct_batch(velo, raw, off)
    assert clusters["event_offsets"].tolist() == [0, 0, 1, 1] == ref.clusters.event_offsets.tolist()
    assert tracks["n"] == 0


def test_malformed_events(velo, geometry):
    import oracle
    from paper_1912_09161_b200 import workload
    from tests.helpers import compare_clusters

    b = workload.generate(1, n_events=6)
    raw = b.raw.copy()
    w = raw.view(np.uint32)
    w[b.event_offsets[1] // 4] ^= 0xFF                       # bad magic in event 1
    w[b.event_offsets[2] // 4 + 2] += 4                      # n_sp_total inconsistent with the size in event 2
    table = (geometry.n_sensors + 1 + 3) // 4 * 4
    w[b.event_offsets[3] // 4 + 4 + table] |= 400 << 14     # SP column out of range in event 3
    w[b.event_offsets[4] // 4 + 4 + 7] = 0x7FFFFFF0            # bank offsets no longer monotone in event 4
    ref = oracle.reconstruct(geometry, raw, b.event_offsets)
    assert ref.clusters.status.tolist()[:6] == [0, 1, 1, 2, 1, 0]
    from paper_1912_09161_b200 import binding

    clusters, tracks = binding.reconstruct_batch(velo, raw, b.event_offsets)
    c, t = as_oracle_types(clusters, tracks)
    assert not compare_clusters(c, ref.clusters)
    assert np.array_equal(t.hits, ref.tracks.hits)


def test_adversarial_cluster_shapes(velo, geometry):
    """Large and awkward clusters: full rows, a long snake, a dense block, checkerboards, duplicates of addresses."""
    import oracle
    from paper_1912_09161_b200 import workload
    from tests.helpers import compare_clusters

    snake = []
    for k in range(40):  # serpentine: long horizontal runs joined alternately left and right
        r = 2 * k
        snake += [(7, c, r) for c in range(10, 60)]
        snake.append((7, 59 if k % 2 == 0 else 10, r + 1))
    block = [(20, c, r) for c in range(100, 124) for r in range(50, 70)]
    checker = [(33, c, r) for c in range(200, 232) for r in range(100, 132) if (c + r) % 2 == 0]
    sparse = [(41, c, r) for c in range(0, 64, 2) for r in range(0, 64, 2)]  # isolated pixels, 2 per SP
    rows = [(55, c, 128) for c in range(0, 768)] + [(55, c, 131) for c in range(0, 768, 3)]
    events = [snake, block, checker, sparse, rows, snake + block + checker + sparse + rows]
    raw, off = workload.pack_events(geometry, events, shuffle_seed=3)
    ref = oracle.reconstruct(geometry, raw, off)
    from paper_1912_09161_b200 import binding

    clusters, tracks = binding.reconstruct_batch(velo, raw, off)
    c, t = as_oracle_types(clusters, tracks)
    assert not compare_clusters(c, ref.clusters)
    assert ref.clusters.n_pixels.max() >= 2000


def test_output_capacity_is_respected(velo, oracle_of):
    from paper_1912_09161_b200 import binding

    batch, ref = oracle_of(1, 64)
    total = int(ref.clusters.event_offsets[-1])
    cap = total // 2
    clusters, tracks = binding.reconstruct_batch(velo, batch.raw, batch.event_offsets, cluster_capacity=cap)
    # offsets still report true totals; events beyond the capacity are flagged and not written
    assert np.array_equal(clusters["event_offsets"], ref.clusters.event_offsets)
    over = ref.clusters.event_offsets[1:] > cap
    assert np.all((clusters["status"] & binding.STATUS_CLUSTER_CAPACITY != 0) == over)
    n_ok = int(ref.clusters.event_offsets[:-1][~over].max())
    assert np.array_equal(clusters["key"][:n_ok], ref.clusters.key[:n_ok])
    # tracks of the events that fit are still exact
    first_bad = int(np.argmax(over))
    assert tracks["event_offsets"][first_bad] == ref.tracks.event_offsets[first_bad]


def test_deterministic_across_runs(velo, oracle_of):
    from paper_1912_09161_b200 import binding

    batch, _ = oracle_of(2, 200)
    a = binding.reconstruct_batch(velo, batch.raw, batch.event_offsets)
    b = binding.reconstruct_batch(velo, batch.raw, batch.event_offsets)
    for d0, d1 in zip(a, b):
        for k in d0:
            if isinstance(d0[k], np.ndarray):
                assert np.array_equal(d0[k], d1[k]), k


@pytest.mark.parametrize("params", [
    # very loose cuts: hundreds of (fake) tracks per event -> the first instance runs out of track slots and the
    # second pass (larger instances, reading the already compacted clusters) redoes those events
    dict(w_seed_phi16=3000, w_fwd_phi16=3000, s_seed=4.0, s_fwd=4.0, s_weak=4.0, max_slope=2.0),
    # tracks may skip two layers: their last hit leaves the three-layer ring of the search
    dict(max_skipped=2),
    dict(max_skipped=4, w_fwd_phi16=1500, s_fwd=0.5),
    # tight windows, no weak tracks
    dict(w_seed_phi16=100, w_fwd_phi16=60, s_weak=0.0),
    # the widest forwarding window the ABI admits (half the circle: more than 63 hits, so velo_follow searches the layer
    # itself instead of using the packed window), with the default and with the widest seeding window
    dict(w_fwd_phi16=16383),
    dict(w_seed_phi16=16383, w_fwd_phi16=16383),
    # no window at all: only hits at exactly the same phi16
    dict(w_seed_phi16=0, w_fwd_phi16=0),
])
def test_parity_with_other_cuts(geometry, batch_of, params):
    import oracle
    from paper_1912_09161_b200 import binding
    from tests.helpers import compare_clusters, compare_tracks

    batch = batch_of(2, 96)
    ref = oracle.reconstruct(geometry, batch.raw, batch.event_offsets, params=params, n_threads=8)
    v = binding.AllenVelo(geometry, params=params)
    try:
        clusters, tracks = binding.reconstruct_batch(v, batch.raw, batch.event_offsets)
    finally:
        v.destroy()
    c, t = as_oracle_types(clusters, tracks)
    assert not compare_clusters(c, ref.clusters)
    rep = compare_tracks(t, ref.tracks, ref)
    assert rep["n_got"] == rep["n_ref"] and rep["mismatched_tracks"] == 0 and rep["bad_fits"] == 0, rep
    assert np.array_equal(t.hits, ref.tracks.hits)
    assert not clusters["status"].any()


def test_parity_on_a_larger_batch(velo, oracle_of):
    """2000 nu=6 events: several waves of CTAs per SM, events of every size class in one batch."""
    batch, ref = oracle_of(2, 2000)
    check_parity(velo, batch, ref)


@pytest.mark.parametrize("config,n_events,hint", [(3, 48, 0), (1, 64, 1000), (2, 200, 1000)])
def test_results_do_not_depend_on_the_occupancy_hint(velo, oracle_of, config, n_events, hint):
    """Both cluster-kernel instances (256 / 512 entries per layer in shared memory) and the pool paths behind them."""
    from paper_1912_09161_b200 import binding
    from tests.helpers import compare_clusters

    batch, ref = oracle_of(config, n_events)
    orig = velo.set_occupancy_hint
    velo.set_occupancy_hint = lambda n, b: orig(1, 4 * hint * velo.n_layers)  # reconstruct_batch sets its own otherwise
    try:
        clusters, tracks = binding.reconstruct_batch(velo, batch.raw, batch.event_offsets)
    finally:
        velo.set_occupancy_hint = orig
    c, t = as_oracle_types(clusters, tracks)
    assert not compare_clusters(c, ref.clusters)
    assert np.array_equal(t.hits, ref.tracks.hits)


def test_streamed_host_to_host_reconstruction(geometry, oracle_of):
    """binding.StreamedVelo: chunks on several streams give the oracle's tracks, chunk by chunk, in host memory."""
    import torch

    from paper_1912_09161_b200 import binding

    batch, ref = oracle_of(2, 200)
    h_raw = torch.from_numpy(batch.raw).pin_memory()
    got = {}

    def on_chunk(info, slot):
        slot["stream"].synchronize()
        nt, nh, n = info["n_tracks"], info["n_hits"], info["n_events"]
        got[info["first_event"]] = dict(
            te=slot["h_te"][:n + 1].numpy().view(np.uint32).copy(), ho=slot["h_ho"][:nt + 1].numpy().view(np.uint32).copy(),
            hits=slot["h_hits"][:nh].numpy().view(np.uint16).copy(), tx=slot["h_fit"][2][:nt].numpy().copy(),
            status=slot["h_st"][:n].numpy().copy())

    sv = binding.StreamedVelo(geometry, 64, int(batch.raw.size), n_streams=3)
    try:
        infos = sv.reconstruct(h_raw, batch.event_offsets.astype(np.int64), on_chunk=on_chunk)
        assert [i["first_event"] for i in infos] == [0, 64, 128, 192]
        check_chunks(got, ref.tracks, infos)
        got.clear()
        # a short first chunk (bench.py's e2e does this), then a 40-event one, the rest in chunks of 64
        infos = sv.reconstruct(h_raw, batch.event_offsets.astype(np.int64), on_chunk=on_chunk, chunk_sizes=[8, 40])
        assert [(i["first_event"], i["n_events"]) for i in infos] == [(0, 8), (8, 40), (48, 64), (112, 64), (176, 24)]
        check_chunks(got, ref.tracks, infos)
        with pytest.raises(ValueError):
            sv.reconstruct(h_raw, batch.event_offsets.astype(np.int64), chunk_sizes=[65])
    finally:
        sv.destroy()


def check_chunks(got, rt, infos):
    for first, g in got.items():
        n = len(g["te"]) - 1
        t0, t1 = int(rt.event_offsets[first]), int(rt.event_offsets[first + n])
        assert np.array_equal(g["te"], rt.event_offsets[first:first + n + 1] - t0)
        h0, h1 = int(rt.hit_offsets[t0]), int(rt.hit_offsets[t1])
        assert np.array_equal(g["ho"], rt.hit_offsets[t0:t1 + 1] - h0)
        assert np.array_equal(g["hits"], rt.hits[h0:h1])
        assert np.allclose(g["tx"], rt.tx[t0:t1], rtol=1e-5, atol=1e-8)
        assert not g["status"].any()
    assert sum(i["n_tracks"] for i in infos) == int(rt.event_offsets[-1])


def run_in_the_bench_configuration(geometry, batch, calls=2):
    """The launch configuration bench.py times: buffers sized from the SP word count, no checksum array, workspace and
    outputs reused from call to call.  Returns host copies (dicts as binding.reconstruct_batch) of the last call."""
    import torch

    from paper_1912_09161_b200 import binding

    n_events, L = batch.n_events, geometry.n_layers
    raw_bytes, n_sp = int(batch.raw.size), batch.n_sp_words()
    velo = binding.AllenVelo(geometry)
    ccap = int(1.15 * n_sp) + 4096
    oc, ot = binding.alloc_outputs(n_events, L, ccap, ccap // 3, ccap // 2, "cuda:0", with_checksum=False)
    ws = torch.empty(velo.workspace_bytes(n_events, raw_bytes), dtype=torch.uint8, device="cuda:0")
    velo.set_workspace(ws)
    velo.set_occupancy_hint(n_events, raw_bytes)
    d_raw = torch.from_numpy(batch.raw).to("cuda:0")
    d_off = torch.from_numpy(batch.event_offsets.view(np.int32)).to("cuda:0")
    first = None
    for _ in range(calls):  # the later calls reuse workspace and outputs, as the timed steps do
        assert velo.reconstruct(d_raw, d_off, n_events, None, oc, ot) == 0, velo.last_error()
        torch.cuda.synchronize()
        snap = [t.clone() for t in (oc.layer_offsets, oc.key, oc.x, oc.phi16, ot.event_offsets, ot.hit_offsets, ot.hits, ot.tx)]
        if first is not None:  # bit-identical from call to call, whatever the thread schedule
            assert all(torch.equal(a, b) for a, b in zip(first, snap))
        first = snap
    del first, snap
    u32 = lambda t: t.cpu().numpy().view(np.uint32)
    ce, te = u32(oc.event_offsets), u32(ot.event_offsets)
    nc, nt = int(ce[n_events]), int(te[n_events])
    clusters = dict(event_offsets=ce, layer_offsets=u32(oc.layer_offsets), status=u32(oc.status)[:n_events], n=nc)
    for name in ("key", "n_pixels", "sum_col", "sum_row"):
        clusters[name] = u32(getattr(oc, name))[:nc]
    for name in ("x", "y", "z", "phi16"):
        clusters[name] = getattr(oc, name).cpu().numpy()[:nc]
    ho = u32(ot.hit_offsets)
    assert int(ho[ot.capacity_tracks]) == int(ho[nt])  # the total number of hits is also at the fixed place
    tracks = dict(event_offsets=te, hit_offsets=ho[:nt + 1], hits=ot.hits.cpu().numpy().view(np.uint16)[:int(ho[nt])], n=nt)
    for name in ("x0", "y0", "tx", "ty"):
        tracks[name] = getattr(ot, name).cpu().numpy()[:nt]
    velo.destroy()
    return clusters, tracks


@pytest.mark.parametrize("config,n_events", [(2, 10000), (3, 10000), (2, 50000)])
def test_full_size_batches_in_the_bench_configuration(geometry, config, n_events):
    """BASELINE.json configs[2] (the headline batch), configs[3] (nu = 12) and the largest point of configs[4] (50 000
    events) at full size, in the launch configuration bench.py times: EVERY event of the batch against the oracle, whole
    arrays, element by element (the oracle does ~6 k events/s on the box's cores); plus properties that hold at any size."""
    import os

    import oracle
    from paper_1912_09161_b200 import workload

    batch = workload.generate(config, n_events=n_events)
    L = geometry.n_layers
    clusters, tracks = run_in_the_bench_configuration(geometry, batch)
    ref = oracle.reconstruct(geometry, batch.raw, batch.event_offsets, n_threads=os.cpu_count() or 1)
    rc, rt = ref.clusters, ref.tracks
    assert not clusters["status"].any() and not rc.status.any()
    # -- clusters: offsets and every per-cluster array, bit for bit (the checksum array is off in this configuration)
    assert np.array_equal(clusters["event_offsets"], rc.event_offsets)
    assert np.array_equal(clusters["layer_offsets"], rc.layer_offsets)
    for name in ("key", "n_pixels", "sum_col", "sum_row", "phi16"):
        assert np.array_equal(clusters[name], getattr(rc, name)), name
    for name in ("x", "y", "z"):
        assert np.array_equal(clusters[name].view(np.uint32), getattr(rc, name).view(np.uint32)), name
    # -- tracks: same tracks in the same order with the same hits in the same order; fit within 1e-5 (R6)
    assert np.array_equal(tracks["event_offsets"], rt.event_offsets)
    assert np.array_equal(tracks["hit_offsets"], rt.hit_offsets)
    assert np.array_equal(tracks["hits"], rt.hits)
    from tests.helpers import fit_close

    ok = fit_close([tracks[k] for k in ("x0", "y0", "tx", "ty")], [rt.x0, rt.y0, rt.tx, rt.ty])
    assert ok.all(), int((~ok).sum())
    # -- properties that hold at any size: layers sorted by (phi16, key); every hit in at most one track
    ce, lo, te, ho = (clusters["event_offsets"], clusters["layer_offsets"], tracks["event_offsets"], tracks["hit_offsets"])
    layer_of = np.repeat(np.arange(n_events * L), np.diff(lo))
    same = layer_of[1:] == layer_of[:-1]
    k64 = ((clusters["phi16"].astype(np.int64) + 32768) << 32) | clusters["key"]
    assert np.all(k64[1:][same] > k64[:-1][same])
    ev_of_hit = np.repeat(np.repeat(np.arange(n_events), np.diff(te)), np.diff(ho))
    glob = ce[ev_of_hit].astype(np.int64) + tracks["hits"]
    assert len(np.unique(glob)) == len(glob)
    print(f"config {config}, {n_events} events: {clusters['n']} clusters, {tracks['n']} tracks identical to the oracle; "
          f"near-cut decisions logged by the oracle: {int(ref.near_cut_per_event.sum())}")



@pytest.mark.parametrize("config,n_events", [(0, None), (2, 200), (3, 48)])
def test_kalman_fit_against_the_oracle(velo, geometry, oracle_of, config, n_events):
    """Optional output of the track stage: simple Kalman fit (R9), fp32 on the GPU against the fp64
    oracle.  Tolerances (R9): positions 1e-5 (1 mm + |value|), slopes 1e-5 |slope| + 1e-7, covariances 2e-4
    relative (fp32 recursion over <= 26 hits); chi2 2e-3 relative + 1e-3: its residuals (~0.01 mm) are differences of
    fp32 coordinates of up to ~50 mm (ulp 4e-6 mm), so every term carries ~1e-3 relative error."""
    import oracle
    from paper_1912_09161_b200 import binding

    batch, ref = oracle_of(config, n_events)
    clusters, tracks = binding.reconstruct_batch(velo, batch.raw, batch.event_offsets, with_kalman=True)
    assert np.array_equal(tracks["hits"], ref.tracks.hits)
    want = oracle.kalman_of(ref, geometry.pitch_mm)
    got = tracks["kalman"].astype(np.float64)
    assert got.shape == want.shape and len(want) > 0
    dev = dict(pos=np.abs(got[:, 0:2] - want[:, 0:2]).max(), slope=(np.abs(got[:, 2:4] - want[:, 2:4]) / (np.abs(want[:, 2:4]) + 1e-3)).max(),
               chi2=(np.abs(got[:, 5] - want[:, 5]) / (want[:, 5] + 1e-3)).max(),
               cov=(np.abs(got[:, 6:] - want[:, 6:]) / np.abs(want[:, 6:])).max())
    print("max deviations", dev)
    assert np.all(np.abs(got[:, 0:2] - want[:, 0:2]) <= 1e-5 * (1 + np.abs(want[:, 0:2])))
    assert np.all(np.abs(got[:, 2:4] - want[:, 2:4]) <= 1e-5 * np.abs(want[:, 2:4]) + 1e-7)
    assert np.array_equal(got[:, 4], want[:, 4])
    assert np.all(np.abs(got[:, 5] - want[:, 5]) <= 2e-3 * want[:, 5] + 1e-3)
    assert np.all(np.abs(got[:, 6:] - want[:, 6:]) <= 2e-4 * np.abs(want[:, 6:]))


def _pv_step4_is_near_a_cut(cand, seed, rel=1e-3):
    """True if step 4 of R10 for the oracle's candidate with this seed involves a decision within `rel` of a cut:
    its own sum w against 3, or — for another candidate that is (nearly) accepted — the 1 mm distance, the 0.1 % band of
    the sums, or that candidate's own acceptance."""
    i = int(np.argmin(np.abs(cand[:, 0] - seed)))
    if abs(cand[i, 0] - seed) > 2e-3:
        return False
    zi, swi = cand[i, 3], cand[i, 4]
    if abs(swi - 3.0) <= 3.0 * rel:
        return True
    for j in range(len(cand)):
        zj, swj = cand[j, 3], cand[j, 4]
        if j == i or swj < 3.0 * (1 - rel) or abs(zj - zi) > 1.0 + rel:
            continue
        if abs(abs(zj - zi) - 1.0) <= rel or abs(swj - 3.0) <= 3.0 * rel:
            return True
        if abs(swj / swi - 1.001) <= rel or abs(swi / swj - 1.001) <= rel:
            return True
    return False


@pytest.mark.parametrize("config,n_events", [(0, None), (2, 200), (3, 48)])
def test_primary_vertices_against_the_oracle(velo, geometry, oracle_of, config, n_events):
    """Optional output: primary vertices (R10), oracle-pure: the oracle runs on its OWN tracks, fit values
    and Kalman states.  The histogram seeds are integer decisions on fp32 values both sides compute with the same operations
    from bit-identical inputs (asserted): the candidates must be identical.  The fits (fp32 on the GPU, fp64 in the oracle)
    are compared vertex by vertex, matched by their seed; acceptance (sum w >= 3) and duplicate removal (1 mm, 0.1 % band)
    are cuts on fitted floats: a vertex found on one side only must have an oracle value within 1e-3 of one of those cuts,
    and such vertices must stay below 0.1 % of all."""
    import math

    import oracle
    from paper_1912_09161_b200 import binding

    batch, ref = oracle_of(config, n_events)
    clusters, tracks = binding.reconstruct_batch(velo, batch.raw, batch.event_offsets, with_kalman=True,
                                                 with_vertices=True)
    assert np.array_equal(tracks["hits"], ref.tracks.hits)
    t = ref.tracks
    # the straight-line fit feeds the histogram: both sides round an fp64 result to fp32 -> bit-identical
    for k in ("x0", "y0", "tx", "ty"):
        assert np.array_equal(tracks[k].view(np.uint32), getattr(t, k).view(np.uint32)), k
    kal = oracle.kalman_of(ref, geometry.pitch_mm)
    want, n_want, _ = oracle.find_pvs(t.event_offsets, t.x0, t.y0, t.tx, t.ty, kal)
    got, n_got = tracks["vertices"].astype(np.float64), tracks["n_vertices"]
    n_total = n_one_sided = 0
    worst = dict(xy=0.0, z=0.0, sw=0.0)
    for e in range(batch.n_events):
        w, g = want[e, :n_want[e]], got[e, :n_got[e]]
        n_total += len(w)
        # match by the histogram seed (candidates are at least one bin apart; the GPU computes the seed in fp32)
        pairs = [(a, b) for b in w for a in g if abs(a[6] - b[6]) < 2e-3]
        lonely = [b[6] for b in w if not any(abs(a[6] - b[6]) < 2e-3 for a in g)] + \
                 [a[6] for a in g if not any(abs(a[6] - b[6]) < 2e-3 for b in w)]
        if lonely:   # accepted on one side only: must be a near-cut case of step 4
            t0, t1 = int(t.event_offsets[e]), int(t.event_offsets[e + 1])
            _, cand = oracle.pv_candidates(t.x0[t0:t1], t.y0[t0:t1], t.tx[t0:t1], t.ty[t0:t1], kal[t0:t1])
            for seed in lonely:
                assert _pv_step4_is_near_a_cut(cand, seed), (e, seed, cand)
            n_one_sided += len(lonely)
        for a, b in pairs:
            worst["xy"] = max(worst["xy"], abs(a[0] - b[0]), abs(a[1] - b[1]))
            worst["z"] = max(worst["z"], abs(a[2] - b[2]))
            worst["sw"] = max(worst["sw"], abs(a[3] - b[3]) / b[3])
            # a vertex far from its seed is still moving after 8 passes: rounding differences are amplified there
            loose = 10.0 if abs(b[2] - b[6]) > 2.0 else 1.0
            assert abs(a[0] - b[0]) < 2e-4 * loose and abs(a[1] - b[1]) < 2e-4 * loose and abs(a[2] - b[2]) < 2e-3 * loose, (e, a, b)
            assert abs(a[3] - b[3]) <= 2e-3 * loose * b[3] and abs(a[5] - b[5]) <= 5e-3 * loose * b[5] + 1e-2, (e, a, b)
            assert abs(a[4] - b[4]) <= 1, (e, a, b)   # a track exactly at the Tukey cut-off may flip
    print("vertices", n_total, "one-sided near-cut vertices", n_one_sided, "worst", worst)
    assert n_total > 0 and n_one_sided <= math.ceil(1e-3 * n_total)


def test_layer_beyond_the_largest_staging_capacity_is_flagged_not_wrong(velo, geometry):
    """Documented limit: more than 1024 hits in one layer -> the event is flagged STAGE_OVERFLOW and
    gets no tracks; its clusters are still complete and exact, and the other events of the batch are untouched."""
    import oracle
    from paper_1912_09161_b200 import binding, workload
    from tests.helpers import compare_clusters

    rng = np.random.default_rng(11)
    busy = set()
    while len(busy) < 1300:   # isolated pixels (every third column / row) on the four sensors of layer 6
        busy.add((24 + int(rng.integers(4)), 3 * int(rng.integers(256)), 3 * int(rng.integers(85))))
    normal = workload.generate(1, n_events=3)
    ev = []
    for e in range(3):   # re-pack three generated events through pack_events, with the busy layer added to the second
        m = normal.pixels["event"] == e
        px = sorted(set(zip(normal.pixels["sensor"][m].tolist(), normal.pixels["col"][m].tolist(), normal.pixels["row"][m].tolist())))
        ev.append(px + (sorted(busy) if e == 1 else []))
    raw, off = workload.pack_events(geometry, ev, shuffle_seed=5)
    ref = oracle.reconstruct(geometry, raw, off)
    clusters, tracks = binding.reconstruct_batch(velo, raw, off)
    assert clusters["status"].tolist() == [0, binding.STATUS_STAGE_OVERFLOW, 0]
    clusters["status"] = ref.clusters.status   # compare everything but the flag
    c, t = as_oracle_types(clusters, tracks)
    assert not compare_clusters(c, ref.clusters)
    rt = ref.tracks
    assert int(np.diff(rt.event_offsets)[1]) > 0   # the oracle, without the limit, does find tracks there
    assert np.diff(tracks["event_offsets"]).tolist() == [int(np.diff(rt.event_offsets)[0]), 0, int(np.diff(rt.event_offsets)[2])]
    # events 0 and 2: identical hit lists
    h0 = rt.hits[:rt.hit_offsets[rt.event_offsets[1]]]
    h2 = rt.hits[rt.hit_offsets[rt.event_offsets[2]]:]
    assert np.array_equal(tracks["hits"], np.concatenate([h0, h2]))
