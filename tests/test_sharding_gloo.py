"""N > 1 host logic on CPU: plane sharding of the depth stack and the max-over-ranks timing that
bench.py uses, run as a world_size-2 gloo job.  No GPU, no field arithmetic."""
import os
import socket

import pytest

torch = pytest.importorskip("torch")
import torch.multiprocessing as mp  # noqa: E402

from paper_1107_5578_b200 import sharding as S  # noqa: E402


@pytest.mark.parametrize("n,world", [(64, 1), (64, 2), (64, 8), (7, 2), (3, 8), (0, 4), (1, 2)])
def test_plane_shard_is_a_contiguous_partition(n, world):
    spans = [S.plane_shard(n, world, r) for r in range(world)]
    assert spans[0][0] == 0 and spans[-1][1] == n
    for (a0, b0), (a1, b1) in zip(spans, spans[1:]):
        assert b0 == a1 and a0 <= b0
    sizes = [b - a for a, b in spans]
    assert max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)


def test_plane_shard_rejects_bad_ranks():
    for args in [(4, 0, 0), (4, 2, 2), (4, 2, -1), (-1, 2, 0)]:
        with pytest.raises(ValueError):
            S.plane_shard(*args)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        zs = [0.001 * k for k in range(1, 8)]            # 7 planes over 2 ranks: 4 + 3
        mine, first = S.shard_zs(zs, world, rank)
        # every rank's (first, count) gathered: together they cover 0..n exactly once
        got = [None] * world
        dist.all_gather_object(got, (first, len(mine), mine))
        ms = S.max_over_ranks(10.0 + 5.0 * rank)          # the slowest rank defines the job time
        dist.barrier()
        q.put((rank, got, ms))
    finally:
        dist.destroy_process_group()


def test_two_rank_gloo_stack_sharding_and_timing():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = [q.get(timeout=120) for _ in range(world)]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    zs = [0.001 * k for k in range(1, 8)]
    for rank, got, ms in res:
        assert ms == 15.0
        cover = []
        for first, cnt, mine in got:
            assert mine == zs[first:first + cnt]
            cover += list(range(first, first + cnt))
        assert cover == list(range(len(zs)))
    assert S.whole_job_rate([300, 300], 15.0) == pytest.approx(600 / 0.015)
