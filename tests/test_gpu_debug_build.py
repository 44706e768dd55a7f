"""The library built with -DVELO_DEBUG (bounds checks on every shared-memory / workspace capacity where an index is
formed; compute-sanitizer is closed on this pool): the seeded configs and the stress inputs run through it without a
single failed check, and give the oracle's results."""
import numpy as np
import pytest

from tests.test_gpu_parity import as_oracle_types

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def velo_debug(geometry):
    from paper_1912_09161_b200 import binding, build

    build.build(debug=True)
    v = binding.AllenVelo(geometry, debug=True)
    assert v.checks_compiled()
    yield v
    v.destroy()


def test_the_default_library_has_no_checks(geometry):
    from paper_1912_09161_b200 import binding

    v = binding.AllenVelo(geometry)
    try:
        assert not v.checks_compiled() and v.debug_fault() == 0
    finally:
        v.destroy()


@pytest.mark.parametrize("config,n_events", [(0, None), (1, 64), (2, 300), (3, 64)])
def test_seeded_configs_under_bounds_checks(velo_debug, oracle_of, config, n_events):
    from paper_1912_09161_b200 import binding
    from tests.helpers import compare_clusters

    batch, ref = oracle_of(config, n_events)
    clusters, tracks = binding.reconstruct_batch(velo_debug, batch.raw, batch.event_offsets)
    assert velo_debug.debug_fault() == 0
    c, t = as_oracle_types(clusters, tracks)
    assert not compare_clusters(c, ref.clusters)
    assert np.array_equal(t.hits, ref.tracks.hits)


def test_stress_inputs_under_bounds_checks(geometry):
    """Oversize layers (pool paths), a layer beyond the staging capacity, loose cuts (candidate lists and track slots
    overflow, second pass): no check fails."""
    import oracle
    from paper_1912_09161_b200 import binding, workload
    from tests.test_gpu_edges import hot_sensor_event

    rng = np.random.default_rng(3)
    events = [hot_sensor_event(rng, 4 * (e % 20) + 1, 300 + 60 * (e % 6)) for e in range(24)]
    busy = set()
    while len(busy) < 1300:
        busy.add((24 + int(rng.integers(4)), 3 * int(rng.integers(256)), 3 * int(rng.integers(85))))
    events.append(sorted(busy))
    raw, off = workload.pack_events(geometry, events, shuffle_seed=4)
    ref = oracle.reconstruct(geometry, raw, off, n_threads=8)
    v = binding.AllenVelo(geometry, debug=True)
    try:
        clusters, _ = binding.reconstruct_batch(v, raw, off)
        assert v.debug_fault() == 0
        assert np.array_equal(clusters["key"], ref.clusters.key)
    finally:
        v.destroy()
    params = dict(s_seed=4.0, s_fwd=4.0, w_seed_phi16=1500)
    batch = workload.generate(2, n_events=32)
    ref = oracle.reconstruct(geometry, batch.raw, batch.event_offsets, params=params, n_threads=8)
    v = binding.AllenVelo(geometry, params=params, debug=True)
    try:
        _, tracks = binding.reconstruct_batch(v, batch.raw, batch.event_offsets)
        assert v.debug_fault() == 0
        assert sum(v.track_counters()["second_pass"]) > 0
        assert np.array_equal(tracks["hits"], ref.tracks.hits)
    finally:
        v.destroy()


@pytest.mark.parametrize("kind", ["g52", "g13", "coarse", "shuffled"])
def test_other_geometries_under_bounds_checks(kind):
    """52 layers (two layer offsets per lane), 8 sensors per layer, a coarser pixel matrix: no check fails."""
    import oracle
    from paper_1912_09161_b200 import binding, build, workload

    build.build(debug=True)
    geo = workload.geometry_variant(kind)
    batch = workload.generate(2, n_events=64, geometry=geo)
    ref = oracle.reconstruct(geo, batch.raw, batch.event_offsets, n_threads=8)
    v = binding.AllenVelo(geo, debug=True)
    try:
        clusters, tracks = binding.reconstruct_batch(v, batch.raw, batch.event_offsets)
        assert v.debug_fault() == 0
        assert np.array_equal(clusters["key"], ref.clusters.key) and np.array_equal(tracks["hits"], ref.tracks.hits)
    finally:
        v.destroy()


@pytest.mark.parametrize("params", [dict(w_fwd_phi16=16383), dict(w_seed_phi16=16383, w_fwd_phi16=16383),
                                    dict(max_skipped=4, w_fwd_phi16=1500, s_fwd=0.5)])
def test_extreme_windows_under_bounds_checks(geometry, params):
    """Windows of half the circle (velo_follow searches the layer itself), tracks that skip four layers: no check fails."""
    import oracle
    from paper_1912_09161_b200 import binding, build, workload

    build.build(debug=True)
    batch = workload.generate(2, n_events=64, batch_index=2)
    ref = oracle.reconstruct(geometry, batch.raw, batch.event_offsets, params=params, n_threads=8)
    v = binding.AllenVelo(geometry, params=params, debug=True)
    try:
        _, tracks = binding.reconstruct_batch(v, batch.raw, batch.event_offsets)
        assert v.debug_fault() == 0
        assert np.array_equal(tracks["hits"], ref.tracks.hits)
    finally:
        v.destroy()
