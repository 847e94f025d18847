"""NEXT-4 on one GPU: the row-sharded run (paper_2606_09377_b200.multi.crown_run_row_sharded) against the unsharded
crown_run.  A box has one GPU, so ranks are emulated ONE AFTER ANOTHER on it (no kernel waits on another): the gather
callback computes the other ranks' row shards with the same `local_rows` the ranks would run.  Rows are independent
linear bounds, so sharded == unsharded bitwise whenever the shard cuts are multiples of 32 rows (the
fused relaxation epilogue needs R % 32 == 0; a ragged tail shard takes the unfused kernels: same bound within tolerance).
The world_size-2 exchange itself is covered on CPU by tests/test_multi_gloo.py."""
import numpy as np
import pytest
import torch

import workloads as W
from oracle import crown_oracle as O

pytestmark = pytest.mark.gpu


def _emulated_gather(ctx, pre_ref, box, B, src_of, world, rank):
    from paper_2606_09377_b200 import multi

    def gather(l_loc, u_loc, n_rows, rk, wd, multiple):
        # which layer is this?  the one whose pre-activations are being produced: found by row count + order of calls
        src = src_of.pop(0)
        ls, us = [], []
        for r in range(wd):
            r0, r1 = multi.shard_rows(n_rows, r, wd, multiple)
            if r == rk:
                assert l_loc.shape[1] == r1 - r0
                ls.append(l_loc); us.append(u_loc)
            else:
                l, u = multi.local_rows(ctx, B, src, pre_ref(), box, r0, r1)
                ls.append(l); us.append(u)
        return torch.cat(ls, dim=1).contiguous(), torch.cat(us, dim=1).contiguous()
    return gather


@pytest.mark.parametrize("world,multiple,exact", [(1, 128, True), (2, 128, True), (4, 128, True), (3, 100, False)])
def test_row_sharded_equals_unsharded(world, multiple, exact):
    from paper_2606_09377_b200 import CrownContext, multi
    wl = W.make(3, scale=16, B=3)            # 256-1024-1024-1024-10
    lo, hi = wl.box()
    ctx = CrownContext(wl.net, wl.B, wl.S, mem_cap_bytes=96 << 20)     # forces row chunks inside a shard
    assert ctx.row_chunk() < 1024
    ref = ctx.run(lo, hi, wl.C, None, wl.intermediate)
    xlo, xhi, Cd = ctx._dev(lo), ctx._dev(hi), ctx._dev(wl.C)
    for rank in range(world):
        state = {}
        srcs = [wl.net.nodes[i].in0 for i in ctx.relu_ids if wl.net.nodes[wl.net.nodes[i].in0].in0 >= 0]
        # the gather emulation needs the bounds of the earlier layers: they are what the sharded run has so far
        holder = {}
        g = _emulated_gather(ctx, lambda: holder["pre"], (xlo, xhi), wl.B, list(srcs), world, rank)

        def gather(l_loc, u_loc, n_rows, rk, wd, mult, _g=g):
            return _g(l_loc, u_loc, n_rows, rk, wd, mult)

        # crown_run_row_sharded fills `pre` as it goes; expose the dict to the emulation through a small subclass
        class Ctx2:
            def __getattr__(self, k):
                return getattr(ctx, k)

            def crown_backward(self, B, start, pre, *a, **kw):
                holder["pre"] = pre
                return ctx.crown_backward(B, start, pre, *a, **kw)
        out = multi.crown_run_row_sharded(Ctx2(), xlo, xhi, Cd, None, rank, world, gather=gather, multiple=multiple)
        ctx.stream.synchronize()
        for i in ctx.relu_ids:
            for k in (0, 1):
                a, b = out["pre"][i][k], ref["pre"][i][k]
                if exact:
                    assert torch.equal(a, b), f"world {world} rank {rank} relu {i}"
                else:
                    torch.testing.assert_close(a, b, rtol=1e-4, atol=1e-5)
        if exact:
            assert torch.equal(out["lb"], ref["lb"]) and torch.equal(out["ub"], ref["ub"])
        else:
            torch.testing.assert_close(out["lb"], ref["lb"], rtol=1e-4, atol=1e-5)
    # and against the oracle (forced protocol on the final bound of property 0)
    p = 0
    forced = {i: (l[p].cpu().numpy().astype(np.float64), u[p].cpu().numpy().astype(np.float64)) for i, (l, u) in out["pre"].items()}
    olb, oub, _ = O.final_bounds(wl.net, lo[p], hi[p], wl.C[p], forced, None, None)
    err = np.abs(out["lb"][p].cpu().numpy() - olb) - (1e-5 + 1e-4 * np.abs(olb))
    assert np.all(err <= 0)
    ctx.close()
