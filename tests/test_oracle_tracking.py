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
