"""N > 1 path of bench.py (T-parallel replicas, no data-path collective), on CPU with gloo, world_size 2."""
import os
import socket

import pytest
import torch.multiprocessing as mp

from paper_1604_07983_b200 import replicas


def test_rank_slices_partition_the_time_extent():
    for world in (1, 2, 3, 8):
        seen = []
        for r in range(world):
            own = replicas.rank_slices(r, world, 64)
            assert own == sorted(own) and all(t % world == r for t in own)
            seen += own
        assert sorted(seen) == list(range(64))
    assert replicas.rank_slices(1, 2, 64, count=4) == [1, 3, 5, 7]
    assert replicas.rank_slices(5, 8, 4, count=3) == [1, 1, 1]  # more ranks than slices: reuse a slice
    with pytest.raises(ValueError):
        replicas.rank_slices(2, 2, 64)


def _worker(rank, world, port, out):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    own = replicas.rank_slices(rank, world, 8)
    # every rank reports its own (fake) device time; the job time is the maximum
    ms, ms_e2e = replicas.max_over_ranks([100.0 + 10.0 * rank, 200.0 - 5.0 * rank])
    dist.barrier()
    out.put((rank, own, ms, ms_e2e, replicas.aggregate_throughput(4, world, ms)))
    dist.destroy_process_group()


def test_two_gloo_ranks_disjoint_slices_and_max_timing():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, own0, ms0, e0, v0), (r1, own1, ms1, e1, v1) = res
    assert own0 == [0, 2, 4, 6] and own1 == [1, 3, 5, 7]
    assert ms0 == ms1 == 110.0 and e0 == e1 == 200.0
    assert v0 == v1 == pytest.approx(2 * 4 / 0.110)


def test_single_process_is_identity():
    assert replicas.max_over_ranks([1.5, 2.5]) == [1.5, 2.5]
