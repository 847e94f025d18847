"""Host-side logic of the N>1 path on CPU: world_size 2, gloo backend (no data-path collective exists)."""
import os

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2606_09377_b200 import multi


def test_shard_range_partitions_exactly():
    for n in (0, 1, 7, 64, 192, 1001):
        for world in (1, 2, 3, 8):
            seen = []
            for r in range(world):
                lo, hi = multi.shard_range(n, r, world)
                assert 0 <= lo <= hi <= n
                seen += list(range(lo, hi))
            assert seen == list(range(n))
            sizes = [multi.shard_range(n, r, world)[1] - multi.shard_range(n, r, world)[0] for r in range(world)]
            assert max(sizes) - min(sizes) <= 1


def test_shard_rows_tile_aligned():
    for n in (100, 256, 16384, 16385):
        for world in (2, 4, 8):
            cuts = [multi.shard_rows(n, r, world) for r in range(world)]
            assert cuts[0][0] == 0 and cuts[-1][1] == n
            for a, b in zip(cuts[:-1], cuts[1:]):
                assert a[1] == b[0] and (a[1] % 128 == 0 or a[1] == n)


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        n_total = 9
        lo, hi = multi.shard_range(n_total, rank, world)
        step_ms = 10.0 + 5.0 * rank                       # rank 1 is the slow replica
        verified = torch.tensor([(i % 2) for i in range(lo, hi)], dtype=torch.uint8)
        q.put((rank, multi.max_over_ranks(step_ms), multi.sum_over_ranks(hi - lo),
               multi.gather_verdicts(verified, n_total, rank, world)))
    finally:
        dist.destroy_process_group()


def test_two_rank_gloo_bookkeeping():
    world, port = 2, 29500 + (os.getpid() % 2000)
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, tmax, tot, verdicts in res:
        assert tmax == 15.0            # max over ranks, not this rank's own time
        assert tot == 9.0              # every property owned exactly once
        assert verdicts == [i % 2 for i in range(9)]
