"""allen_velo_offsets_noalloc (include/allen_velo_noalloc.h): the path's output-compaction scan with its scratch in a
static device array of the library — no handle, no workspace, no allocation — against the existing path.

The existing path computes layer_offsets = exclusive prefix sum of the clusters per (event, layer) inside
allen_velo_reconstruct (scan_kernel of csrc/velo_scan.cu, scratch in the caller's workspace).  Here the counts are taken
back from those offsets (differences), handed to the new entry point, and the result must be the existing path's
layer_offsets bit for bit (integer work: the tolerance of every offset comparison in tests/test_gpu_parity.py) — on two
calls in a row that share the static array: a large batch, then a smaller one whose tiles find the first call's status
words if the clear were missing, then the large one again.

Collected last on purpose (the suite runs with pytest -x); passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def existing_path_layer_offsets(geometry, config, n_events, batch_index):
    """layer_offsets [n_events * n_layers + 1] of allen_velo_reconstruct, as a device tensor (int32 view of u32)."""
    import torch

    from paper_1912_09161_b200 import binding, workload

    batch = workload.generate(config, n_events=n_events, batch_index=batch_index)
    L = geometry.n_layers
    raw_bytes = int(batch.raw.size)
    ccap = int(1.15 * batch.n_sp_words()) + 4096
    velo = binding.AllenVelo(geometry)
    try:
        oc, ot = binding.alloc_outputs(n_events, L, ccap, ccap // 3, ccap // 2, "cuda:0", with_checksum=False)
        ws = torch.empty(velo.workspace_bytes(n_events, raw_bytes), dtype=torch.uint8, device="cuda:0")
        velo.set_workspace(ws)
        d_raw = torch.from_numpy(batch.raw).to("cuda:0")
        d_off = torch.from_numpy(batch.event_offsets.view(np.int32)).to("cuda:0")
        assert velo.reconstruct(d_raw, d_off, n_events, None, oc, ot) == 0, velo.last_error()
        torch.cuda.synchronize()
        assert not oc.status.cpu().numpy().any()
        return oc.layer_offsets[:n_events * L + 1].clone()
    finally:
        velo.destroy()


def test_offsets_noalloc_matches_the_existing_path_on_calls_in_a_row(geometry):
    import torch

    from paper_1912_09161_b200 import binding

    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    large = existing_path_layer_offsets(geometry, 2, 700, 3)   # 18 200 counts: 9 tiles of the scan, ragged tail
    small = existing_path_layer_offsets(geometry, 3, 150, 4)   # 3 900 counts: 2 tiles
    stream = torch.cuda.Stream()
    for want in (large, small, large):  # calls in a row on one stream: they share the static scratch array
        n = want.numel() - 1
        counts = (want[1:] - want[:-1]).contiguous()  # u32 differences in int32 arithmetic: exact modulo 2^32
        got = torch.full((n + 1,), -1, dtype=torch.int32, device="cuda:0")
        stream.wait_stream(torch.cuda.current_stream())
        before = torch.cuda.memory_allocated()
        rc, text = binding.offsets_noalloc(counts, n, got, stream)
        assert rc == binding.OK, text
        assert torch.cuda.memory_allocated() == before  # (torch's allocator saw nothing; the library has no other)
        stream.synchronize()
        assert torch.equal(got, want), int((got != want).sum())
        assert int(got[-1]) == int(counts.sum())
    # the numpy definition on one of them, so that "equal to the existing path" is not all there is
    host = np.concatenate([[0], np.cumsum((large[1:] - large[:-1]).cpu().numpy().view(np.uint32), dtype=np.uint64)])
    assert np.array_equal(large.cpu().numpy().view(np.uint32), host.astype(np.uint32))


def test_offsets_noalloc_edges():
    import torch

    from paper_1912_09161_b200 import binding

    # n = 0: offsets[0] = 0
    got = torch.full((1,), 7, dtype=torch.int32, device="cuda:0")
    rc, text = binding.offsets_noalloc(None, 0, got)
    torch.cuda.synchronize()
    assert rc == binding.OK and int(got[0]) == 0, text
    # beyond the maximum: rejected with a clear message, nothing enqueued, the output untouched
    n = binding.NOALLOC_MAX_COUNTS + 1
    counts = torch.ones(n, dtype=torch.int32, device="cuda:0")
    out = torch.full((n + 1,), -1, dtype=torch.int32, device="cuda:0")
    rc, text = binding.offsets_noalloc(counts, n, out)
    torch.cuda.synchronize()
    assert rc == binding.ERR_TOO_LARGE and "exceeds ALLEN_VELO_NOALLOC_MAX_COUNTS" in text
    assert int(out[0]) == -1 and int(out[-1]) == -1
    # exactly the maximum (2048 tiles: the whole array), all ones, then a ragged size right after it
    for m in (binding.NOALLOC_MAX_COUNTS, 2048 * 3 + 1, 1):
        rc, text = binding.offsets_noalloc(counts, m, out)
        assert rc == binding.OK, text
        torch.cuda.synchronize()
        assert torch.equal(out[:m + 1], torch.arange(m + 1, dtype=torch.int32, device="cuda:0"))
