"""The seeded input generator: determinism, raw-format structure, and the workload statistics DESIGN.md quotes."""
import numpy as np

from paper_1912_09161_b200 import workload


def test_geometry_g0(geometry):
    g = geometry
    assert (g.n_sensors, g.n_modules, g.n_layers, g.n_cols, g.n_rows) == (104, 52, 26, 768, 256)
    z = g.sensor_ltg[:, 8]
    zm = np.array([z[g.sensor_module == m][0] for m in range(52)])
    assert np.all(np.diff(zm) > 0) and zm[0] == -290.0 and zm[-1] == 750.0
    assert np.array_equal(g.module_layer, np.arange(52) // 2)
    # the four sensors of a station leave the 8 mm square beam hole free and do not overlap
    p = g.pitch_mm
    corners = []
    for s in range(4):
        M = g.sensor_ltg[s].reshape(3, 3).astype(np.float64)
        c = [(M @ np.array([u, v, 1.0]))[:2] for u in (0, 768 * p) for v in (0, 256 * p)]
        corners.append(np.array(c))
        lo, hi = np.min(c, axis=0), np.max(c, axis=0)
        assert not (lo[0] < 4 and hi[0] > -4 and lo[1] < 4 and hi[1] > -4) or (
            max(lo[0], -4) >= min(hi[0], 4) or max(lo[1], -4) >= min(hi[1], 4))
    boxes = [(c.min(axis=0), c.max(axis=0)) for c in corners]
    for i in range(4):
        for j in range(i + 1, 4):
            (alo, ahi), (blo, bhi) = boxes[i], boxes[j]
            ox = min(ahi[0], bhi[0]) - max(alo[0], blo[0])
            oy = min(ahi[1], bhi[1]) - max(alo[1], blo[1])
            assert ox <= 1e-9 or oy <= 1e-9


def test_deterministic_and_event_streams_independent_of_batch():
    a = workload.generate(2, n_events=20)
    b = workload.generate(2, n_events=20)
    assert a.sha() == b.sha()
    c = workload.generate(2, n_events=5, first_event=10)
    assert np.array_equal(c.raw, a.raw[a.event_offsets[10]:a.event_offsets[15]])
    d = workload.generate(2, n_events=20, batch_index=1)
    assert d.sha() != a.sha()


def test_raw_format_structure(batch_of, geometry):
    b = batch_of(1, 40)
    w = b.raw.view(np.uint32)
    assert np.all(b.event_offsets % 16 == 0)
    for e in range(b.n_events):
        ev = w[b.event_offsets[e] // 4:b.event_offsets[e + 1] // 4]
        assert ev[0] == 0x56454C4F and ev[1] == geometry.n_sensors and ev[3] == 0
        n_sp = int(ev[2])
        off = ev[4:4 + geometry.n_sensors + 1]
        assert off[0] == 0 and off[-1] == n_sp and np.all(np.diff(off.astype(np.int64)) >= 0)
        table = (geometry.n_sensors + 1 + 3) // 4 * 4
        sp = ev[4 + table:4 + table + n_sp]
        assert len(ev) == 4 + table + (n_sp + 3) // 4 * 4
        assert np.all(sp & 0xFF), "hitmap must be non-zero"
        assert np.all(sp >> 23 == 0) and np.all(((sp >> 14) & 0x1FF) < 384)
        for s in range(geometry.n_sensors):
            addr = sp[off[s]:off[s + 1]] >> 8
            assert len(np.unique(addr)) == len(addr), "an SP address occurs at most once per bank"


def test_config0_recipe(batch_of):
    b = batch_of(0)
    assert b.n_events == 16
    assert np.all(np.bincount(b.particles["event"]) == 20)
    assert np.all(b.pixels["particle"] >= 0) and np.all(b.pixels["main"] == 1)
    assert np.all(b.particles["n_hits"] == b.particles["n_crossings"])
    assert len(b.pvs["event"]) == 16
    # isolation: no two pixels of different particles 8-touch
    px = b.pixels
    for e in range(16):
        sel = px["event"] == e
        s, c, r, p = (px[k][sel].astype(np.int64) for k in ("sensor", "col", "row", "particle"))
        touch = (s[:, None] == s[None, :]) & (np.abs(c[:, None] - c[None, :]) <= 1) & (np.abs(r[:, None] - r[None, :]) <= 1)
        assert np.all(p[:, None][touch.any(1)] >= 0)
        ii, jj = np.nonzero(touch)
        assert np.all(p[ii] == p[jj])


def test_workload_statistics_match_design_md(batch_of):
    b = batch_of(2, 300)
    n = b.n_events
    assert 135 < len(b.particles["event"]) / n < 165  # ~ 6 x 25
    assert 3200 < b.n_sp_words() / n < 3700
    assert 13500 < len(b.raw) / n < 15000
    noise = (b.pixels["particle"] < 0).sum() / n
    assert 1950 < noise < 2150  # 104 x 196608 x 1e-4 = 2044.7
    eta_ok = np.hypot(b.particles["tx"], b.particles["ty"])
    assert eta_ok.max() <= np.tan(2 * np.arctan(np.exp(-2.0))) + 1e-12
    assert 0.07 < b.particles["displaced"].mean() < 0.13
    eff = b.particles["n_hits"].sum() / b.particles["n_crossings"].sum()
    assert 0.985 < eff < 0.995
    # charge sharing: 1 / 2 / 3 pixel clusters in 36 / 48 / 16 %
    sig = b.pixels["particle"] >= 0
    per_hit = sig.sum() / b.particles["n_hits"].sum()
    assert 1.75 < per_hit < 1.85  # 0.36 + 2*0.48 + 3*0.16 = 1.8 (minus edge losses)


def test_select_reindexes_truth(batch_of):
    b = batch_of(1, 40)
    s = b.select([5, 3])
    assert s.n_events == 2
    assert np.array_equal(s.raw[:s.event_offsets[1]], b.raw[b.event_offsets[5]:b.event_offsets[6]])
    assert set(np.unique(s.pixels["event"])) <= {0, 1}
    p = s.pixels["particle"]
    assert p.max() < len(s.particles["event"])
    assert np.all(s.particles["event"][p[p >= 0]] == s.pixels["event"][p >= 0])


def test_pack_events_matches_generator_packer(geometry):
    # the pure-Python packer used for hand-made test events produces the same words as the C++ packer
    b = workload.generate(1, n_events=3, shuffle_sp=False)
    events = [[] for _ in range(3)]
    for e, s, c, r in zip(b.pixels["event"], b.pixels["sensor"], b.pixels["col"], b.pixels["row"]):
        events[e].append((int(s), int(c), int(r)))
    raw, off = workload.pack_events(geometry, events)
    assert np.array_equal(off, b.event_offsets) and np.array_equal(raw, b.raw)


def test_geometry_variants():
    """The other detector descriptions of tests/test_gpu_geometries.py: inside what include/allen_velo.h admits, layers
    numbered by increasing z, and the oracle finds the generated tracks on each of them."""
    import oracle

    for kind, layers, per_layer in (("g52", 52, 4), ("g13", 13, 8), ("coarse", 26, 4), ("shuffled", 26, 4)):
        g = workload.geometry_variant(kind)
        assert g.n_layers == layers and 3 <= g.n_layers <= 64
        lay = g.sensor_layer()
        assert np.array_equal(np.bincount(lay, minlength=layers), np.full(layers, per_layer))
        z = g.sensor_ltg[:, 8]
        zmin = np.array([z[lay == l].min() for l in range(layers)])
        assert np.all(np.diff(zmin) > 0)
        assert g.n_cols % 2 == 0 and g.n_rows % 4 == 0 and g.n_cols * g.n_rows <= 1 << 18
        b = workload.generate(2, n_events=8, geometry=g)
        r = oracle.reconstruct(g, b.raw, b.event_offsets)
        assert len(r.tracks.x0) > 8 * 80 and not r.clusters.status.any()
        if kind == "shuffled":  # the sensors of a layer are no longer neighbours in the bank order
            assert max(np.ptp(np.nonzero(lay == l)[0]) for l in range(layers)) > 50
