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


# ---- NEXT-4: row-sharded intermediate bounds; the compute of a rank is stood in by the oracle -------
class _OracleCtx:
    """Duck-typed stand-in for CrownContext on CPU: the same calls, answered by the float64 oracle (test
    infrastructure; the GPU path is covered by tests/test_gpu_sharded.py).  Exercises the sharding / gather logic."""

    def __init__(self, net, chunk):
        import numpy as np
        self.net = net
        self.relu_ids = net.relu_ids()
        self.sizes = [int(np.prod(n.shape)) for n in net.nodes]
        self.device = torch.device("cpu")
        self._chunk = chunk
        self.calls = []

    def row_chunk(self):
        return self._chunk

    def ibp_forward(self, x_lo, x_hi, Cmat=None, nodes=None):
        from oracle import crown_oracle as O
        out = {}
        for i in nodes:
            ls, us = [], []
            for p in range(x_lo.shape[0]):
                iv = O.ibp(self.net, x_lo[p].numpy(), x_hi[p].numpy())
                ls.append(torch.from_numpy(iv[i][0].reshape(-1))); us.append(torch.from_numpy(iv[i][1].reshape(-1)))
            out[i] = (torch.stack(ls), torch.stack(us))
        return out, None

    def crown_backward(self, B, start, pre, Cmat=None, row0=0, rows=None, alpha_lo=None, alpha_up=None, box=None,
                       want_A=True):
        import numpy as np
        from oracle import crown_oracle as O
        self.calls.append((start, row0, rows))
        lbs, ubs = [], []
        for p in range(B):
            if Cmat is None:
                C0 = np.zeros((rows, self.sizes[start])); C0[np.arange(rows), row0 + np.arange(rows)] = 1.0
            else:
                C0 = Cmat[p].numpy()
            pp = {i: (l[p].numpy(), u[p].numpy()) for i, (l, u) in pre.items()}
            al = None if alpha_lo is None else {i: a[p].numpy() for i, a in alpha_lo.items()}
            A_lo, A_up, d_lo, d_up = O.backward(self.net, start, C0, pp, al, al)
            lb, ub = O.concretize(A_lo, A_up, d_lo, d_up, box[0][p].numpy(), box[1][p].numpy())
            lbs.append(torch.from_numpy(lb)); ubs.append(torch.from_numpy(ub))
        return {"A": None, "d": None, "lb": torch.stack(lbs), "ub": torch.stack(ubs)}


def _sharded_case():
    import numpy as np
    import workloads as W
    wl = W.small_mlp([5, 11, 9, 10, 3], seed=21, B=2, eps=0.15)
    lo, hi = wl.box()
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64))
    alpha = {i: t(a) for i, a in zip(wl.net.relu_ids(), wl.alpha)}
    return wl, t(lo), t(hi), t(wl.C), alpha


def _sharded_worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        wl, lo, hi, C, alpha = _sharded_case()
        ctx = _OracleCtx(wl.net, chunk=3)
        r = multi.crown_run_row_sharded(ctx, lo, hi, C, alpha, rank, world, multiple=4)
        q.put((rank, {i: (l.numpy(), u.numpy()) for i, (l, u) in r["pre"].items()}, r["lb"].numpy(), r["ub"].numpy(),
               ctx.calls))
    finally:
        dist.destroy_process_group()


def test_row_sharded_run_two_ranks_equals_unsharded():
    """world_size 2 over gloo: every rank ends with the full (l_k, u_k) of every layer and the same final bounds as the
    unsharded float64 run; each rank propagated only its own rows (in chunks of the context's row chunk)."""
    import numpy as np
    from oracle import crown_oracle as O
    world, port = 2, 31500 + (os.getpid() % 2000)
    mpx = mp.get_context("spawn")
    q = mpx.Queue()
    procs = [mpx.Process(target=_sharded_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted((q.get(timeout=300) for _ in range(world)), key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    wl, lo, hi, C, alpha = _sharded_case()
    for rank, pre, lb, ub, calls in res:
        for p in range(wl.B):
            ref = O.crown_bounds(wl.net, lo[p].numpy(), hi[p].numpy())
            for i in wl.net.relu_ids():
                np.testing.assert_allclose(pre[i][0][p], ref[i][0], rtol=0, atol=1e-12)
                np.testing.assert_allclose(pre[i][1][p], ref[i][1], rtol=0, atol=1e-12)
            al = {i: a[p].numpy() for i, a in alpha.items()}
            olb, oub, _ = O.final_bounds(wl.net, lo[p].numpy(), hi[p].numpy(), C[p].numpy(), ref, al, al)
            np.testing.assert_allclose(lb[p], olb, rtol=0, atol=1e-10)
            np.testing.assert_allclose(ub[p], oub, rtol=0, atol=1e-10)
        # identity passes: only this rank's rows, in chunks of <= 3; node 2 (9 rows): rank 0 owns [0,8), rank 1 [8,9)
        ident = [(s, a, n) for (s, a, n) in calls if s != len(wl.net.nodes) - 1]
        for s, a, n in ident:
            r0, r1 = multi.shard_rows(wl.net.nodes[s].size, rank, world, 4)
            assert r0 <= a and a + n <= r1 and n <= 3
        covered = {s: sum(n for (s2, _, n) in ident if s2 == s) for s in {c[0] for c in ident}}
        for s, tot in covered.items():
            r0, r1 = multi.shard_rows(wl.net.nodes[s].size, rank, world, 4)
            assert tot == r1 - r0
    assert res[0][1].keys() == res[1][1].keys()


def test_allgather_rows_single_process_is_identity():
    l, u = torch.arange(6.).reshape(2, 3), torch.arange(6.).reshape(2, 3) + 1
    a, b = multi.allgather_rows(l, u, 3, 0, 1)
    assert a is l and b is u
