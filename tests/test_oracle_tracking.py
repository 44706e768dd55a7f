"""Pins for oracle step O5 (search by triplet, reading R5) — BASELINE.json self-checks:

* noiseless straight-line events with full hit efficiency -> 100 % efficiency, 0 ghosts (config 0);
* a brute-force enumeration of all compatible hit triplets on tiny events agrees with the seeding;
* every hit is used by at most one track;
* results conserved under event permutation (and SP-word permutation inside a bank);
* structural invariants re-evaluated from the outputs.
"""
import numpy as np
import pytest

import oracle
from paper_1912_09161_b200 import workload
from tests.helpers import brute_force_tracking, dphi16, physics_report

P = oracle.DEFAULT_PARAMS


def test_config0_full_efficiency_no_ghosts(oracle_of):
    batch, res = oracle_of(0)
    rep = physics_report(batch, res)
    assert rep["n_particles"] == 16 * 20
    assert rep["eff_consecutive"] == 1.0, rep["missed_consecutive"]
    assert rep["ghost_rate"] == 0.0
    # A particle may only come out as two tracks where the acceptance leaves a hole of >= 2 consecutive layers in
    # its hit pattern (more than max_skipped = 1 missed layers closes a track by definition, reading R5 T2).
    mp = rep["matched_particle"]
    sensor_layer = batch.geometry.sensor_layer()
    particles, counts = np.unique(mp, return_counts=True)
    for p in particles[counts > 1]:
        layers = np.unique(sensor_layer[batch.pixels["sensor"][batch.pixels["particle"] == p]])
        assert np.max(np.diff(layers)) >= 3, (p, layers)
    assert rep["n_tracks"] - rep["n_reconstructible_consecutive"] == int((counts - 1).sum())


def test_physics_rates_on_minimum_bias_like_events_are_sane(oracle_of):
    # Reported, not graded against the paper (no Velo-only number in its text): loose sanity bounds only.
    batch, res = oracle_of(2, 60)
    rep = physics_report(batch, res)
    assert rep["eff_consecutive"] > 0.95
    assert rep["ghost_rate"] < 0.05
    assert rep["clone_rate"] < 0.05


def test_every_hit_used_at_most_once(oracle_of):
    for cfg, n in ((0, None), (2, 60), (3, 20)):
        batch, res = oracle_of(cfg, n)
        t = res.tracks
        for e in range(batch.n_events):
            h = t.hits[t.hit_offsets[t.event_offsets[e]]:t.hit_offsets[t.event_offsets[e + 1]]]
            assert len(h) == len(set(h.tolist()))
            n_cl = int(res.clusters.event_offsets[e + 1] - res.clusters.event_offsets[e])
            assert len(h) == 0 or int(h.max()) < n_cl


def test_structural_invariants(oracle_of, geometry):
    batch, res = oracle_of(2, 60)
    c, t = res.clusters, res.tracks
    L = geometry.n_layers
    for e in range(batch.n_events):
        base = int(c.event_offsets[e])
        lo = c.layer_offsets[e * L:(e + 1) * L + 1].astype(np.int64) - base
        x, y, z, phi = (a[base:int(c.event_offsets[e + 1])] for a in (c.x, c.y, c.z, c.phi16))
        for k in range(int(t.event_offsets[e]), int(t.event_offsets[e + 1])):
            hits = t.hits[t.hit_offsets[k]:t.hit_offsets[k + 1]].astype(np.int64)
            layers = np.searchsorted(lo, hits, side="right") - 1
            assert len(hits) >= 3
            assert np.all(np.diff(layers) < 0), "hits must lie on strictly decreasing layers"
            assert np.all(-np.diff(layers) - 1 <= P["max_skipped"]), "too many skipped layers in a row"
            assert np.all(layers[:3] == layers[0] - np.arange(3)), "seed must sit on three consecutive layers"
            a, b, cc = hits[:3]
            S = oracle.scatter((x[a], y[a], z[a]), (x[b], y[b], z[b]), (x[cc], y[cc], z[cc]))
            assert S <= P["s_seed"]
            assert abs(dphi16(phi[a], phi[b])) <= P["w_seed_phi16"] and abs(dphi16(phi[cc], phi[b])) <= P["w_seed_phi16"]
            tx = (np.float32(x[b]) - np.float32(x[a])) / (np.float32(z[b]) - np.float32(z[a]))
            ty = (np.float32(y[b]) - np.float32(y[a])) / (np.float32(z[b]) - np.float32(z[a]))
            assert abs(tx) <= np.float32(P["max_slope"]) and abs(ty) <= np.float32(P["max_slope"])
            if len(hits) == 3:
                assert S <= P["s_weak"]
            for j in range(3, len(hits)):
                p_, q_, n_ = hits[j - 2], hits[j - 1], hits[j]
                Sf = oracle.scatter((x[p_], y[p_], z[p_]), (x[q_], y[q_], z[q_]), (x[n_], y[n_], z[n_]))
                assert Sf <= P["s_fwd"]
                assert abs(dphi16(phi[n_], phi[q_])) <= P["w_fwd_phi16"]


def test_event_permutation_invariance(oracle_of):
    batch, res = oracle_of(2, 60)
    rng = np.random.default_rng(0)
    perm = rng.permutation(batch.n_events)
    shuffled = batch.select(perm)
    res2 = oracle.reconstruct(shuffled.geometry, shuffled.raw, shuffled.event_offsets)
    assert res2.tracks.event_offsets[-1] == res.tracks.event_offsets[-1]  # track count conserved
    for new_e, old_e in enumerate(perm):
        assert res2.tracks.hit_sets(new_e) == res.tracks.hit_sets(int(old_e))
        a0, a1 = res.clusters.event_offsets[old_e], res.clusters.event_offsets[old_e + 1]
        b0, b1 = res2.clusters.event_offsets[new_e], res2.clusters.event_offsets[new_e + 1]
        assert np.array_equal(res.clusters.key[a0:a1], res2.clusters.key[b0:b1])


def test_sp_permutation_invariance_and_determinism(geometry):
    a = workload.generate(2, n_events=12, shuffle_sp=True)
    b = workload.generate(2, n_events=12, shuffle_sp=False)
    assert not np.array_equal(a.raw, b.raw) and len(a.raw) == len(b.raw)
    ra = oracle.reconstruct(geometry, a.raw, a.event_offsets)
    rb = oracle.reconstruct(geometry, b.raw, b.event_offsets)
    ra2 = oracle.reconstruct(geometry, a.raw, a.event_offsets, n_threads=3)
    for r in (rb, ra2):
        assert np.array_equal(ra.clusters.key, r.clusters.key)
        assert np.array_equal(ra.tracks.hits, r.tracks.hits)
        assert np.array_equal(ra.tracks.x0.view(np.uint32), r.tracks.x0.view(np.uint32))


def _tiny_event(rng, n_layers=8, n_tracks=5, n_noise=25, spread=0.012):
    """Hits of a tiny synthetic event straight in the oracle's hit format (normative order)."""
    z_layers = np.linspace(100.0, 100.0 + 25.0 * (n_layers - 1), n_layers)
    rows = []
    for _ in range(n_tracks):
        tx, ty = rng.uniform(-0.15, 0.15, 2)
        x0, y0 = rng.normal(0, 0.05, 2)
        for l in range(n_layers):
            if rng.random() < 0.9:
                zz = z_layers[l] + (12.5 if rng.random() < 0.5 else 0.0)
                rows.append((l, x0 + tx * zz + rng.normal(0, spread), y0 + ty * zz + rng.normal(0, spread), zz))
    for _ in range(n_noise):
        l = int(rng.integers(0, n_layers))
        rows.append((l, rng.uniform(-25, 25), rng.uniform(-25, 25), z_layers[l]))
    lay = np.array([r[0] for r in rows])
    x, y, z = (np.array([r[k] for r in rows], np.float32) for k in (1, 2, 3))
    phi = np.array([oracle.phi16(a, b) for a, b in zip(x, y)], np.int16)
    key = rng.permutation(len(rows))
    order = np.lexsort((key, phi.astype(np.int64), lay))
    lay, x, y, z, phi = lay[order], x[order], y[order], z[order], phi[order]
    lo = np.searchsorted(lay, np.arange(n_layers + 1)).astype(np.uint32)
    return x, y, z, phi, lo


@pytest.mark.parametrize("seed", range(12))
def test_brute_force_enumeration_agrees_on_tiny_events(seed):
    rng = np.random.default_rng(500 + seed)
    # wide windows and loose cuts force many competing triplets and conflicts on a handful of hits
    params = dict(P)
    if seed % 3 == 1:
        params.update(w_seed_phi16=4000, w_fwd_phi16=4000, s_seed=4.0, s_fwd=8.0, s_weak=1.0)
    if seed % 3 == 2:
        params.update(w_seed_phi16=32767 // 2, w_fwd_phi16=32767 // 2, s_seed=100.0, s_fwd=100.0, s_weak=100.0,
                      max_skipped=2)
    x, y, z, phi, lo = _tiny_event(rng, n_tracks=3 + seed % 4, n_noise=10 + 3 * seed)
    res = oracle.search_hits(x, y, z, phi, lo, params)

    def scat(a, b, c):
        return oracle.scatter((x[a], y[a], z[a]), (x[b], y[b], z[b]), (x[c], y[c], z[c]))

    want = brute_force_tracking(x, y, z, phi, lo, params, scat)
    assert res.tracks.hit_sets(0) == want
    if seed % 3:
        assert len(want) > 0


def test_phi_window_wraps_around_pi():
    # a straight track along phi = pi (x < 0, y ~ 0) has hits whose phi16 jump between +32767 and -32768
    z = np.array([300.0, 275.0, 250.0, 225.0, 200.0], np.float32)[::-1].copy()
    x = (-0.05 * z).astype(np.float32)
    y = np.array([1e-3, -1e-3, 1e-3, -1e-3, 1e-3], np.float32)
    phi = np.array([oracle.phi16(a, b) for a, b in zip(x, y)], np.int16)
    assert phi.max() > 32000 and phi.min() < -32000
    lo = np.arange(6, dtype=np.uint32)
    res = oracle.search_hits(x, y, z, phi, lo)
    assert res.tracks.hit_sets(0) == [(0, 1, 2, 3, 4)]


def test_conflict_rules_hand_case():
    # Two parallel tracks 0.3 mm apart share the same candidate region; a single extra hit between them on the
    # last layer can only be taken by the track with the smaller scatter.  Layers 0..4 at z = 0, 25, ..., 100.
    z5 = np.array([0.0, 25.0, 50.0, 75.0, 100.0], np.float32)
    rows = []
    for l in range(1, 5):
        rows.append((l, 10.0, 10.0, z5[l]))        # track U: x = 10, y = 10
        rows.append((l, 10.0, 10.3, z5[l]))        # track V: x = 10, y = 10.3
    rows.append((0, 10.0, 10.1, z5[0]))            # lone hit on layer 0: closer to U (0.1) than to V (0.2)
    lay = np.array([r[0] for r in rows])
    x, y, zz = (np.array([r[k] for r in rows], np.float32) for k in (1, 2, 3))
    phi = np.array([oracle.phi16(a, b) for a, b in zip(x, y)], np.int16)
    order = np.lexsort((phi.astype(np.int64), lay))
    lay, x, y, zz, phi = lay[order], x[order], y[order], zz[order], phi[order]
    lo = np.searchsorted(lay, np.arange(6)).astype(np.uint32)
    res = oracle.search_hits(x, y, zz, phi, lo, dict(P, s_fwd=1.0))
    sets = res.tracks.hit_sets(0)
    lone = 0
    assert len(sets) == 2
    with_lone = [s for s in sets if lone in s]
    assert len(with_lone) == 1 and len(with_lone[0]) == 5
    ys = y[list(with_lone[0])]
    assert np.allclose(ys[1:], 10.0), "the lone hit must go to the nearer track U"


def test_weak_three_hit_tracks_are_dropped_and_missed_layers_close_tracks():
    # three collinear hits with a little scatter: S between s_weak and s_seed -> seeded but dropped at T5
    z = np.array([50.0, 25.0, 0.0], np.float32)[::-1].copy()  # layers 0,1,2 -> z 0,25,50
    x = np.array([10.0, 10.0, 10.0], np.float32)
    y = np.array([10.0, 10.0, 10.1], np.float32)  # S = 0.01 mm^2: s_weak = 2^-7 = 0.0078 < S < s_seed = 0.0156
    phi = np.array([oracle.phi16(a, b) for a, b in zip(x, y)], np.int16)
    lo = np.arange(4, dtype=np.uint32)
    assert oracle.search_hits(x, y, z, phi, lo).tracks.hit_sets(0) == []
    assert oracle.search_hits(x, y, z, phi, lo, dict(P, s_weak=0.011)).tracks.hit_sets(0) == [(0, 1, 2)]
    # a 7-layer track with a 2-layer hole (layers 2,3 missing) is split: max_skipped = 1 closes it
    zs = np.array([0, 25, 100, 125, 150], np.float32)  # layers 0,1,4,5,6
    lo = np.array([0, 1, 2, 2, 2, 3, 4, 5], np.uint32)
    x = (5.0 + 0.01 * (zs + 400)).astype(np.float32)  # points back to the beamline: constant phi
    y = (10.0 + 0.02 * (zs + 400)).astype(np.float32)
    phi = np.array([oracle.phi16(a, b) for a, b in zip(x, y)], np.int16)
    assert oracle.search_hits(x, y, zs, phi, lo).tracks.hit_sets(0) == [(2, 3, 4)]
    assert oracle.search_hits(x, y, zs, phi, lo, dict(P, max_skipped=2)).tracks.hit_sets(0) == [(0, 1, 2, 3, 4)]


# ------------------------------------------------------------------------------------------------
# Near-cut accounting (R7; BASELINE.json: "decisions falling within 1e-4 of a window cut ... are counted and
# reported").  Hand cases: one a (layer 2), one b (layer 1), one or two c (layer 0); the expected counts follow from
# R7's three rules: a value within relative 1e-4 of its cut, |dphi| in {w, w + 1}, a runner-up within 1e-4 of the winner.
# ------------------------------------------------------------------------------------------------
def _abc(yc=0.02, phi_a=0, phi_c=(0,), xc=(0.0,)):
    """a = (10, 5, 50), b = (9, 4.5, 25) -> slopes 0.04, 0.02; prediction at z = 0: (8, 4); c = (8 + xc, 4 + yc, 0)."""
    n_c = len(xc)
    x = np.array([8.0 + v for v in xc] + [9.0, 10.0], np.float32)
    y = np.array([4.0 + yc] * n_c + [4.5, 5.0], np.float32)
    z = np.array([0.0] * n_c + [25.0, 50.0], np.float32)
    phi = np.array(list(phi_c) + [0, phi_a], np.int16)
    lo = np.array([0, n_c, n_c + 1, n_c + 2], np.uint32)
    return x, y, z, phi, lo


def _near(args, params=None):
    res = oracle.search_hits(*args, dict(P, **(params or {})))
    return int(res.near_cut_per_event[0]), sorted(res.near_cut_hit_index.tolist()), res.tracks.hit_sets(0)


def test_near_cut_counter_far_from_every_cut_is_zero():
    # S = 0.02^2 = 4e-4: far below s_weak = 7.8e-3; slopes 0.04 / 0.02 against 0.4; all dphi = 0
    assert _near(_abc()) == (0, [], [(0, 1, 2)])


@pytest.mark.parametrize("d,count,found", [(511, 0, True), (512, 1, True), (513, 1, False), (514, 0, False),
                                           (-512, 1, True), (-513, 1, False)])
def test_near_cut_counts_phi_differences_at_the_window_edge(d, count, found):
    # |dphi(a, b)| = w and w + 1 are the two values "within 1e-4 rad of the window cut" (1 LSB = 9.6e-5 rad)
    n, hits, tracks = _near(_abc(phi_a=d))
    assert (n, hits, tracks) == (count, [2] * count, [(0, 1, 2)] if found else [])
    n, hits, tracks = _near(_abc(phi_c=(d,)))
    assert (n, hits, tracks) == (count, [0] * count, [(0, 1, 2)] if found else [])


@pytest.mark.parametrize("rel,count,found", [(5e-5, 1, False), (-5e-5, 1, True), (3e-4, 0, False), (-3e-4, 0, True)])
def test_near_cut_counts_values_within_1e_4_of_a_cut(rel, count, found):
    args = _abc()
    x, y, z = args[:3]
    S = oracle.scatter((x[2], y[2], z[2]), (x[1], y[1], z[1]), (x[0], y[0], z[0]))
    assert S == pytest.approx(4e-4, rel=1e-3)
    # scatter against s_seed: the cut sits at S / (1 + rel), i.e. S exceeds it by `rel` (relative)
    n, hits, tracks = _near(args, dict(s_seed=S / (1 + rel), s_weak=1.0))
    assert (n, hits, tracks) == (count, [1] * count, [(0, 1, 2)] if found else [])
    # three-hit track against s_weak at T5 (seed accepted far from s_seed)
    n, hits, tracks = _near(args, dict(s_weak=S / (1 + rel)))
    assert (n, hits, tracks) == (count, [1] * count, [(0, 1, 2)] if found else [])
    # slope of a -> b against max_slope: tx = 0.04 exactly at the cut, ty = 0.02 far from it
    tx = (np.float32(9.0) - np.float32(10.0)) / (np.float32(25.0) - np.float32(50.0))
    n, hits, tracks = _near(args, dict(max_slope=float(tx) / (1 + rel)))
    assert (n, hits, tracks) == (count, [2] * count, [(0, 1, 2)] if found else [])


def test_near_cut_counts_a_runner_up_within_1e_4():
    # two candidates c at mirror positions about the prediction: equal scatter -> one tie, logged on b; the lower index wins
    n, hits, tracks = _near(_abc(yc=0.0, xc=(-0.01, 0.01), phi_c=(0, 0)))
    assert (n, hits) == (1, [2]) and tracks == [(0, 2, 3)]
    # 2 % apart in distance (4 % in scatter): no tie
    n, hits, tracks = _near(_abc(yc=0.0, xc=(-0.0102, 0.01), phi_c=(0, 0)))
    assert (n, hits) == (0, []) and tracks == [(1, 2, 3)]


def test_near_cut_counts_forwarding_decisions():
    # four layers: seed on layers 3, 2, 1 (exact line), forwarding to a hit on layer 0 that is 0.1 mm off in y
    x = np.array([7.0, 8.0, 9.0, 10.0], np.float32)
    y = np.array([3.6, 4.0, 4.5, 5.0], np.float32)
    z = np.array([-25.0, 0.0, 25.0, 50.0], np.float32)
    lo = np.arange(5, dtype=np.uint32)
    S = oracle.scatter((x[2], y[2], z[2]), (x[1], y[1], z[1]), (x[0], y[0], z[0]))
    assert S == pytest.approx(0.01, rel=1e-3)
    phi0 = np.zeros(4, np.int16)
    assert _near((x, y, z, phi0, lo)) == (0, [], [(0, 1, 2, 3)])
    assert _near((x, y, z, phi0, lo), dict(s_fwd=S / (1 - 5e-5))) == (1, [0], [(0, 1, 2, 3)])
    n, hits, tracks = _near((x, y, z, phi0, lo), dict(s_fwd=S / (1 + 5e-5)))
    assert (n, hits, tracks) == (1, [0], [(1, 2, 3)])
    for d, count, found in ((512, 1, True), (513, 1, False), (520, 0, False)):
        phi = np.array([d, 0, 0, 0], np.int16)
        n, hits, tracks = _near((x, y, z, phi, lo))
        assert (n, hits) == (count, [0] * count) and tracks == ([(0, 1, 2, 3)] if found else [(1, 2, 3)])
