"""Parity on detector descriptions other than G0 (include/allen_velo.h, allen_velo_geometry_t: "3 <= n_layers <= 64; at
most 8 sensors per layer", other sensor sizes).  The benchmarks use G0 only; the boundary promises more, so the kernels'
per-layer tables (sensors of a layer, occupancy cells, phi tables, layer offsets held by lane) are exercised here with
52 layers (two offsets per lane), 8 sensors per layer at four z, a coarser pixel matrix, and sensors numbered in random
order (the banks of a layer are then not contiguous in the raw event).  Same bar as
test_gpu_parity.py: clusters bit-exact, tracks and hit lists identical and in the same order, fit within 1e-5."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("kind,params", [
    ("g52", None),
    ("g52", dict(max_skipped=3)),
    ("g13", None),
    ("coarse", None),
    ("coarse", dict(w_seed_phi16=1500, w_fwd_phi16=1500, max_skipped=2)),
    # the banks of a layer's sensors are scattered over the raw event: the cluster kernel stages word by word instead
    # of one contiguous range with 128-bit loads
    ("shuffled", None),
])
def test_parity_on_other_geometries(kind, params):
    import oracle
    from paper_1912_09161_b200 import binding, workload
    from tests.test_gpu_parity import check_parity

    geo = workload.geometry_variant(kind)
    batch = workload.generate(2, n_events=160, geometry=geo)
    ref = oracle.reconstruct(geo, batch.raw, batch.event_offsets, params=params, n_threads=8)
    assert len(ref.tracks.x0) > 100 * 160 and not ref.clusters.status.any()
    velo = binding.AllenVelo(geo, params=params)
    try:
        clusters, tracks = check_parity(velo, batch, ref)
    finally:
        velo.destroy()
    assert not clusters["status"].any()
    print(f"{kind} {params}: {geo.n_layers} layers, {clusters['n'] / 160:.0f} clusters and {tracks['n'] / 160:.0f} tracks per "
          f"event, {np.diff(tracks['hit_offsets']).mean():.1f} hits per track: identical to the oracle")


def test_local_clustering_on_another_geometry():
    """R11 regions on the coarse matrix (192 x 32 super-pixels per sensor): region borders at other places than in G0."""
    import oracle
    from paper_1912_09161_b200 import binding, workload
    from tests.test_gpu_parity import check_parity

    geo = workload.geometry_variant("coarse")
    batch = workload.generate(2, n_events=96, geometry=geo)
    for regions in ((2, 2), (8, 4)):
        ref = oracle.reconstruct(geo, batch.raw, batch.event_offsets, n_threads=8, cluster_regions=regions)
        velo = binding.AllenVelo(geo)
        try:
            velo.set_cluster_regions(*regions)
            check_parity(velo, batch, ref)
        finally:
            velo.destroy()
