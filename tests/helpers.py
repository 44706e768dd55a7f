"""Test-side utilities: truth matching (PAPER.md:236 definitions), result comparison (BASELINE.json tolerance
rules) and independent brute-force restatements used to pin the oracle.  Nothing here is used by the product."""
from __future__ import annotations

from collections import defaultdict

import numpy as np


# ------------------------------------------------------------------------------------------------
# Truth matching.  P:236: a track is correctly reconstructed if >= 70 % of its hits belong to one MC particle;
# a particle is reconstructible in the Velo if it has >= 1 hit in >= 3 different modules.
# ------------------------------------------------------------------------------------------------
def physics_report(batch, res):
    """res: an oracle.Result with pixel membership (pix_*).  Returns a dict of rates vs generator truth."""
    geo = batch.geometry
    px = batch.pixels
    n_cols = geo.n_cols
    truth_key = (px["sensor"].astype(np.uint32) << 18) | (px["row"].astype(np.uint32) * n_cols + px["col"])
    # (event, pixel key) -> particles (>= 0) firing that pixel
    pix_particles = defaultdict(set)
    for e, k, p in zip(px["event"], truth_key, px["particle"]):
        if p >= 0:
            pix_particles[(int(e), int(k))].add(int(p))
    # (event, cluster) -> particles
    cl_particles = defaultdict(set)
    for e, k, c in zip(res.pix_event, res.pix_key, res.pix_cluster):
        s = pix_particles.get((int(e), int(k)))
        if s:
            cl_particles[(int(e), int(c))] |= s
    # particle -> layers / modules with a main-pixel hit
    sensor_layer = geo.sensor_layer()
    p_layers, p_modules = defaultdict(set), defaultdict(set)
    main = (px["particle"] >= 0) & (px["main"] == 1)
    for p, s in zip(px["particle"][main], px["sensor"][main]):
        p_layers[int(p)].add(int(sensor_layer[s]))
        p_modules[int(p)].add(int(geo.sensor_module[s]))

    def has_3_consecutive(layers):
        return any(l + 1 in layers and l + 2 in layers for l in layers)

    n_particles = len(batch.particles["event"])
    recible_consec = {p for p in range(n_particles) if has_3_consecutive(p_layers[p])}
    recible_p236 = {p for p in range(n_particles) if len(p_modules[p]) >= 3}

    tr = res.tracks
    n_tracks = len(tr.x0)
    matched_particle = -np.ones(n_tracks, np.int64)
    for e in range(batch.n_events):
        for t in range(int(tr.event_offsets[e]), int(tr.event_offsets[e + 1])):
            hits = tr.hits[tr.hit_offsets[t]:tr.hit_offsets[t + 1]]
            votes = defaultdict(int)
            for h in hits:
                for p in cl_particles.get((e, int(h)), ()):
                    votes[p] += 1
            if votes:
                p, v = max(votes.items(), key=lambda kv: (kv[1], -kv[0]))
                if v >= 0.7 * len(hits):
                    matched_particle[t] = p
    found = set(int(p) for p in matched_particle if p >= 0)
    n_ghost = int((matched_particle < 0).sum())
    n_clone = int((matched_particle >= 0).sum()) - len(found)
    return dict(
        n_particles=n_particles,
        n_tracks=n_tracks,
        n_reconstructible_consecutive=len(recible_consec),
        n_reconstructible_p236=len(recible_p236),
        eff_consecutive=len(found & recible_consec) / max(1, len(recible_consec)),
        eff_p236=len(found & recible_p236) / max(1, len(recible_p236)),
        ghost_rate=n_ghost / max(1, n_tracks),
        clone_rate=n_clone / max(1, n_tracks),
        missed_consecutive=sorted(recible_consec - found),
        matched_particle=matched_particle,
    )


# ------------------------------------------------------------------------------------------------
# Comparator for the parity tests (BASELINE.json north_star):
#   clusters bit-exact; track hit sets exact (near-cut mismatches counted, < 0.1 % of tracks);
#   fit parameters within 1e-5 (reading R6 in DESIGN.md for near-zero components).
# ------------------------------------------------------------------------------------------------
CLUSTER_FIELDS = ("key", "n_pixels", "sum_col", "sum_row", "x", "y", "z", "phi16", "checksum")


def compare_clusters(got, ref, check_checksum=True):
    """Bit-exact comparison of two Clusters objects; returns a list of human-readable differences."""
    diffs = []
    for name in ("event_offsets", "layer_offsets", "status"):
        a, b = getattr(got, name), getattr(ref, name)
        if a.shape != b.shape or not np.array_equal(a, b):
            diffs.append(f"{name} differs")
    n = int(ref.event_offsets[-1])
    for name in CLUSTER_FIELDS:
        if name == "checksum" and not check_checksum:
            continue
        a, b = getattr(got, name)[:n], getattr(ref, name)[:n]
        if a.dtype.kind == "f":
            a, b = a.view(np.uint32), b.view(np.uint32)
        if a.shape != b.shape or not np.array_equal(a, b):
            bad = int(np.sum(a != b)) if a.shape == b.shape else -1
            diffs.append(f"{name}: {bad} of {n} differ")
    return diffs


def fit_close(got4, ref4, rel=1e-5):
    """|dx0|,|dy0| <= rel*max(1 mm, hypot(x0,y0)); |dtx|,|dty| <= rel*hypot(tx,ty) (tiny floor for tx=ty=0)."""
    x0, y0, tx, ty = (np.asarray(v, np.float64) for v in ref4)
    gx0, gy0, gtx, gty = (np.asarray(v, np.float64) for v in got4)
    pos_tol = rel * np.maximum(1.0, np.hypot(x0, y0))
    slope_tol = rel * np.maximum(np.hypot(tx, ty), 1e-3)
    return (np.abs(gx0 - x0) <= pos_tol) & (np.abs(gy0 - y0) <= pos_tol) & (np.abs(gtx - tx) <= slope_tol) & (
        np.abs(gty - ty) <= slope_tol)


def compare_tracks(got, ref, near_cut=None):
    """Compare Tracks as canonically sorted hit sets per event, then fit parameters of identical tracks.

    `near_cut`: the oracle.Result of the reference (its near-cut log, R7) or None.  A mismatching track counts as
    "near-cut" only if the oracle logged a decision within 1e-4 of a cut that touches one of the hits on which the two
    track sets of that event differ, or a hit of an EARLIER iteration of the same event (iterations run from the last
    layer down, hit indices grow with the layer: a logged hit with an index above the lowest differing hit), from which
    the difference can cascade; every other mismatch is a hard failure.

    Returns dict(n_ref, n_got, mismatched_tracks, near_cut_mismatched_tracks, hard_mismatched_tracks, bad_fits,
    near_cut_decisions).
    """
    n_events = len(ref.event_offsets) - 1
    logged = [()] * n_events
    n_decisions = 0
    if near_cut is not None:
        n_decisions = int(near_cut.near_cut_per_event.sum())
        order = np.argsort(near_cut.near_cut_hit_event, kind="stable")
        ev, idx = near_cut.near_cut_hit_event[order], near_cut.near_cut_hit_index[order]
        first = np.searchsorted(ev, np.arange(n_events + 1))
        logged = [idx[first[e]:first[e + 1]] for e in range(n_events)]
    mism = near = bad_fit = 0
    for e in range(n_events):
        def table(t):
            out = {}
            for i in range(int(t.event_offsets[e]), int(t.event_offsets[e + 1])):
                hs = tuple(sorted(int(h) for h in t.hits[t.hit_offsets[i]:t.hit_offsets[i + 1]]))
                out[hs] = i
            return out

        tg, tr = table(got), table(ref)
        diff = set(tg) ^ set(tr)
        if diff:
            mism += len(diff)
            differing = set(h for hs in diff for h in hs)
            if len(logged[e]) and (differing & set(int(h) for h in logged[e]) or int(max(logged[e])) > min(differing)):
                near += len(diff)
        for hs in set(tg) & set(tr):
            i, j = tg[hs], tr[hs]
            ok = fit_close((got.x0[i], got.y0[i], got.tx[i], got.ty[i]), (ref.x0[j], ref.y0[j], ref.tx[j], ref.ty[j]))
            bad_fit += int(not ok)
    return dict(n_ref=len(ref.x0), n_got=len(got.x0), mismatched_tracks=mism, near_cut_mismatched_tracks=near,
                hard_mismatched_tracks=mism - near, bad_fits=bad_fit, near_cut_decisions=n_decisions)


# ------------------------------------------------------------------------------------------------
# Independent restatements used as pins
# ------------------------------------------------------------------------------------------------
def ccl_union_find(pixels):
    """8-connected components of a set of (col,row) by union-find; returns frozenset of frozensets."""
    pixels = list(set(pixels))
    index = {p: i for i, p in enumerate(pixels)}
    parent = list(range(len(pixels)))

    def find(i):
        while parent[i] != i:
            parent[i] = parent[parent[i]]
            i = parent[i]
        return i

    for (c, r), i in index.items():
        for dc in (-1, 0, 1):
            for dr in (-1, 0, 1):
                j = index.get((c + dc, r + dr))
                if j is not None:
                    a, b = find(i), find(j)
                    if a != b:
                        parent[a] = b
    groups = defaultdict(set)
    for p, i in index.items():
        groups[find(i)].add(p)
    return frozenset(frozenset(g) for g in groups.values())


def ccl_closure(pixels):
    """8-connected components by transitive closure of the adjacency matrix (boolean matrix squaring)."""
    pixels = sorted(set(pixels))
    n = len(pixels)
    if n == 0:
        return frozenset()
    c = np.array([p[0] for p in pixels])
    r = np.array([p[1] for p in pixels])
    adj = (np.abs(c[:, None] - c[None, :]) <= 1) & (np.abs(r[:, None] - r[None, :]) <= 1)
    reach = adj.copy()
    while True:
        nxt = (reach.astype(np.int32) @ reach.astype(np.int32)) > 0
        if np.array_equal(nxt, reach):
            break
        reach = nxt
    comps = set()
    for i in range(n):
        comps.add(frozenset(pixels[j] for j in np.nonzero(reach[i])[0]))
    return frozenset(comps)


def dphi16(a, b):
    return int(np.int16(np.uint16((int(a) - int(b)) & 0xFFFF)))


def fbits(s):
    return int(np.float32(s).view(np.uint32))


def brute_force_tracking(x, y, z, phi, layer_offsets, P, scatter):
    """Exhaustive restatement of the search (reading R5) for tiny events.

    Seeding enumerates ALL triplets A x B x C and filters afterwards; forwarding enumerates all (track, hit)
    pairs.  `scatter(a_idx, b_idx, c_idx)` supplies S (the fp32 value is pinned separately).  Returns the sorted
    list of sorted hit tuples of accepted tracks.
    """
    L = len(layer_offsets) - 1
    used = set()
    tracks = []  # dicts: hits, seed_b, s_seed, missed, active
    layer = lambda i: range(int(layer_offsets[i]), int(layer_offsets[i + 1]))
    for i in range(L - 1, 1, -1):
        A, B, C = layer(i), layer(i - 1), layer(i - 2)
        # forward: all (track, c) pairs
        pairs = []
        for ti, t in enumerate(tracks):
            if not t["active"]:
                continue
            p, q = t["hits"][-2], t["hits"][-1]
            for c in C:
                if c in used or abs(dphi16(phi[c], phi[q])) > P["w_fwd_phi16"]:
                    continue
                S = scatter(p, q, c)
                if S <= P["s_fwd"]:
                    pairs.append((ti, c, S))
        choice = {}
        for ti, c, S in pairs:
            k = (fbits(S), c)
            if ti not in choice or k < choice[ti][0]:
                choice[ti] = (k, c, S)
        winners = {}
        for ti, (_, c, S) in choice.items():
            k = (fbits(S), tracks[ti]["seed_b"])
            if c not in winners or k < winners[c][0]:
                winners[c] = (k, ti)
        extended = set()
        for c, (_, ti) in winners.items():
            tracks[ti]["hits"].append(c)
            used.add(c)
            extended.add(ti)
        for ti, t in enumerate(tracks):
            if not t["active"]:
                continue
            if ti in extended:
                t["missed"] = 0
            else:
                t["missed"] += 1
                if t["missed"] > P["max_skipped"]:
                    t["active"] = False
        # seeding: all triplets, then filter
        compatible = []
        for a in A:
            for b in B:
                for c in C:
                    if a in used or b in used or c in used:
                        continue
                    if abs(dphi16(phi[a], phi[b])) > P["w_seed_phi16"] or abs(dphi16(phi[c], phi[b])) > P["w_seed_phi16"]:
                        continue
                    dz = np.float32(z[b]) - np.float32(z[a])
                    tx = (np.float32(x[b]) - np.float32(x[a])) / dz
                    ty = (np.float32(y[b]) - np.float32(y[a])) / dz
                    if not (abs(tx) <= np.float32(P["max_slope"]) and abs(ty) <= np.float32(P["max_slope"])):
                        continue
                    S = scatter(a, b, c)
                    if S <= P["s_seed"]:
                        compatible.append((fbits(S), a, c, b, S))
        best_of_b = {}
        for k in compatible:
            b = k[3]
            if b not in best_of_b or k[:3] < best_of_b[b][:3]:
                best_of_b[b] = k
        trip = list(best_of_b.values())
        for (sb, a, c, b, S) in trip:
            key = (sb, b)
            ok = all(not ((o[1] == a or o[2] == c) and o[3] != b and (o[0], o[3]) < key) for o in trip)
            if ok:
                tracks.append(dict(hits=[a, b, c], seed_b=b, s_seed=S, missed=0, active=True))
        for t in tracks:
            if len(t["hits"]) == 3 and t["seed_b"] in B:
                used.update(t["hits"])
    out = []
    for t in tracks:
        if len(t["hits"]) >= 4 or t["s_seed"] <= P["s_weak"]:
            out.append(tuple(sorted(t["hits"])))
    return sorted(out)


# ------------------------------------------------------------------------------------------------
# Raw format v1 assembled from explicit SP words (R1): for inputs that pack_events cannot make (a repeated
# SP address inside a bank, a zero hit map).  Format assembly only; no arithmetic of the method.
# ------------------------------------------------------------------------------------------------
def sp_word(sp_col: int, sp_row: int, hitmap: int) -> int:
    return (sp_col << 14) | (sp_row << 8) | (hitmap & 0xFF)


def raw_from_sp_words(n_sensors: int, events: list[dict[int, list[int]]]):
    """events: per event {sensor: [sp words in bank order]}.  Returns (raw u8 array, event_offsets u32 array)."""
    chunks, offsets = [], [0]
    for banks in events:
        words = [0x56454C4F, n_sensors, sum(len(v) for v in banks.values()), 0]
        off = 0
        for s in range(n_sensors):
            words.append(off)
            off += len(banks.get(s, ()))
        words.append(off)
        while len(words) % 4:
            words.append(0)
        for s in range(n_sensors):
            words.extend(int(w) for w in banks.get(s, ()))
        while len(words) % 4:
            words.append(0)
        a = np.array(words, dtype=np.uint32)
        chunks.append(a.view(np.uint8))
        offsets.append(offsets[-1] + a.nbytes)
    raw = np.concatenate(chunks) if chunks else np.zeros(0, np.uint8)
    return raw, np.array(offsets, dtype=np.uint32)
