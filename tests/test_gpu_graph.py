"""allen_velo_reconstruct inside a CUDA graph.  The call enqueues kernels and memsets only (no host synchronisation, no
allocation, no attribute calls: those happen in allen_velo_create; the side streams of the larger search instances
fork from and join the caller's stream through events), so it can be captured once and replayed: same bytes out as the
direct call, and the replay follows new contents of the same input buffers."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def test_reconstruct_is_capturable_in_a_cuda_graph(geometry):
    import torch

    import oracle
    from paper_1912_09161_b200 import binding, workload

    n_events, L = 300, geometry.n_layers
    first = workload.generate(2, n_events=n_events)
    second = workload.generate(2, n_events=n_events, batch_index=5)
    raw_cap = max(first.raw.size, second.raw.size)
    ccap = int(1.15 * max(first.n_sp_words(), second.n_sp_words())) + 4096
    velo = binding.AllenVelo(geometry)
    try:
        oc, ot = binding.alloc_outputs(n_events, L, ccap, ccap // 3, ccap // 2, "cuda:0", with_checksum=False)
        ws = torch.empty(velo.workspace_bytes(n_events, raw_cap), dtype=torch.uint8, device="cuda:0")
        velo.set_workspace(ws)
        d_raw = torch.zeros(raw_cap, dtype=torch.uint8, device="cuda:0")
        d_off = torch.zeros(n_events + 1, dtype=torch.int32, device="cuda:0")

        def load(batch):
            d_raw[:batch.raw.size].copy_(torch.from_numpy(batch.raw))
            d_off.copy_(torch.from_numpy(batch.event_offsets.view(np.int32)))

        load(first)
        s = torch.cuda.Stream()
        with torch.cuda.stream(s):
            assert velo.reconstruct(d_raw, d_off, n_events, s, oc, ot) == 0, velo.last_error()
        s.synchronize()
        direct = [t.clone() for t in (oc.layer_offsets, oc.key, oc.x, ot.event_offsets, ot.hit_offsets, ot.hits, ot.tx)]
        for t in (oc.layer_offsets, oc.key, oc.x, ot.event_offsets, ot.hit_offsets, ot.hits, ot.tx):
            t.zero_()
        torch.cuda.synchronize()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=s):
            assert velo.reconstruct(d_raw, d_off, n_events, s, oc, ot) == 0, velo.last_error()
        graph.replay()
        torch.cuda.synchronize()
        replayed = (oc.layer_offsets, oc.key, oc.x, ot.event_offsets, ot.hit_offsets, ot.hits, ot.tx)
        assert all(torch.equal(a, b) for a, b in zip(direct, replayed))
        # new events in the same buffers: the replay reconstructs those
        load(second)
        graph.replay()
        torch.cuda.synchronize()
        ref = oracle.reconstruct(geometry, second.raw, second.event_offsets, n_threads=8)
        nc, nt = len(ref.clusters.key), len(ref.tracks.x0)
        assert np.array_equal(oc.event_offsets.cpu().numpy().view(np.uint32), ref.clusters.event_offsets)
        assert np.array_equal(oc.key.cpu().numpy().view(np.uint32)[:nc], ref.clusters.key)
        assert np.array_equal(ot.event_offsets.cpu().numpy().view(np.uint32), ref.tracks.event_offsets)
        nh = int(ref.tracks.hit_offsets[nt])
        assert np.array_equal(ot.hits.cpu().numpy().view(np.uint16)[:nh], ref.tracks.hits)
        assert not oc.status.cpu().numpy().any()
    finally:
        velo.destroy()
