"""N > 1 path on CPU: two gloo ranks, each with its own batch, whole-job value = all events / slowest rank."""
import os
import socket

import pytest


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    import torch.distributed as dist

    from paper_1912_09161_b200 import replicas, workload

    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        batch = workload.generate(1, n_events=8 + rank, batch_index=replicas.batch_index_of(rank))
        red = replicas.Reducer()
        red.barrier()
        value, ms = replicas.whole_job_value(red, batch.n_events, 10.0 * (rank + 1))
        out.put((rank, batch.sha(), batch.n_events, value, ms))
    finally:
        dist.destroy_process_group()


def test_two_ranks_reconstruct_disjoint_batches_and_aggregate():
    import torch.multiprocessing as mp

    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (_, sha0, n0, v0, ms0), (_, sha1, n1, v1, ms1) = res
    assert sha0 != sha1 and (n0, n1) == (8, 9)          # every rank has its own events
    assert ms0 == ms1 == 20.0                           # the slowest rank sets the step time
    assert v0 == v1 == pytest.approx(17 / 20e-3)        # whole-job events/s


def test_event_ranges_partition_a_batch():
    from paper_1912_09161_b200 import replicas

    for n in (0, 1, 7, 10000):
        for world in (1, 2, 3, 8):
            r = [replicas.event_range_of(k, world, n) for k in range(world)]
            assert r[0][0] == 0 and r[-1][1] == n
            assert all(a[1] == b[0] for a, b in zip(r, r[1:]))
            assert max(b - a for a, b in r) - min(b - a for a, b in r) <= 1


def test_reducer_is_identity_without_process_group():
    from paper_1912_09161_b200 import replicas

    red = replicas.Reducer()
    assert red.max(3.5) == 3.5 and red.sum(2.0) == 2.0
    red.barrier()
