"""Multi-GPU plumbing for the hot path: one process per GPU.

Default ("replicas only" in DESIGN.md; weak scaling): properties are independent problems (each row of Eq. 1 is its own
linear bound), so N GPUs run N batches side by side with NO data-path collective; the only exchanges are
host-side bookkeeping (which properties a rank owns, the max-over-ranks step time, the sum of verified counts).

NEXT-4 (opt-in; strong scaling of ONE batch): `crown_run_row_sharded` shards the identity rows of
every intermediate-bound pass across the ranks -- inside a property every start-spec row is an independent linear bound
-- with the weights replicated; the one exchange per layer is an AllGather of that layer's (l_k, u_k) ([B, n_k] each:
kilobytes to a megabyte).  This is neither of the paper's designs: TP shards W and A with an AllReduce per Col-Row pair
and loses tightness, FSDP shards only W with an AllGather of every full weight.
Works with the `nccl` backend on GPUs and `gloo` on CPU.
"""
from __future__ import annotations

from typing import Callable, Dict, List, Optional, Tuple

import torch
import torch.distributed as dist


def shard_range(n_units: int, rank: int, world: int) -> Tuple[int, int]:
    """Contiguous block [lo, hi) of `n_units` owned by `rank`; sizes differ by at most one, earlier ranks get
    the extra unit, every unit is owned exactly once."""
    if world <= 0 or not (0 <= rank < world) or n_units < 0:
        raise ValueError("bad shard arguments")
    base, extra = divmod(n_units, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def shard_rows(n_rows: int, rank: int, world: int, multiple: int = 128) -> Tuple[int, int]:
    """Row shard of an identity start spec aligned to `multiple` rows (one GEMM tile) except at the tail: the
    partition SURVEY.md 8(e) records for a future row-sharded pass (rows are independent, so no exchange is
    needed inside a pass)."""
    tiles = (n_rows + multiple - 1) // multiple
    lo, hi = shard_range(tiles, rank, world)
    return min(lo * multiple, n_rows), min(hi * multiple, n_rows)


def _device_for_backend() -> torch.device:
    if dist.get_backend() == "nccl":
        return torch.device("cuda", torch.cuda.current_device())
    return torch.device("cpu")


def max_over_ranks(value: float) -> float:
    """Slowest rank's value (step time): the job is as slow as its slowest replica."""
    if not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=_device_for_backend())
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float) -> float:
    if not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=_device_for_backend())
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def gather_verdicts(verified: torch.Tensor, n_total: int, rank: int, world: int) -> List[int]:
    """All ranks' verdict bytes in property order (rank r owns shard_range(n_total, r, world)); bookkeeping only."""
    lo, hi = shard_range(n_total, rank, world)
    assert verified.numel() == hi - lo
    if not dist.is_initialized() or world == 1:
        return [int(v) for v in verified.cpu().tolist()]
    out = [None] * world
    dist.all_gather_object(out, [int(v) for v in verified.cpu().tolist()])
    return [v for part in out for v in part]


# ------------------------------------------------------------------------------------------------------------------
# NEXT-4 -- row-sharded intermediate bounds (strong scaling of one batch)
# ------------------------------------------------------------------------------------------------------------------
def local_rows(ctx, B: int, src: int, pre: Dict[int, tuple], box, r0: int, r1: int) -> Tuple[torch.Tensor, torch.Tensor]:
    """Pre-activation bounds of rows [r0, r1) of node `src` (an identity-start CROWN pass per row chunk through the
    C-ABI, concretised inside): (l, u) [B, r1 - r0] on ctx.device."""
    rc = max(1, int(ctx.row_chunk()))
    ls, us = [], []
    for a in range(r0, r1, rc):
        rows = min(rc, r1 - a)
        out = ctx.crown_backward(B, src, pre, None, row0=a, rows=rows, box=box, want_A=False)
        ls.append(out["lb"]); us.append(out["ub"])
    if not ls:
        z = torch.empty(B, 0, device=ctx.device)
        return z, z.clone()
    return torch.cat(ls, dim=1), torch.cat(us, dim=1)


def allgather_rows(l_loc: torch.Tensor, u_loc: torch.Tensor, n_rows: int, rank: int, world: int,
                   multiple: int = 128) -> Tuple[torch.Tensor, torch.Tensor]:
    """The exchange of SURVEY.md 8(e): every rank contributes its row shard of (l_k, u_k) [B, rows_r] and receives the
    full [B, n_rows] pair.  One all_gather of equal-size padded buffers (shards differ by at most one tile)."""
    if world == 1 or not dist.is_initialized():
        return l_loc, u_loc
    B = l_loc.shape[0]
    cuts = [shard_rows(n_rows, r, world, multiple) for r in range(world)]
    width = max(hi - lo for lo, hi in cuts)
    mine = torch.zeros(2, B, width, dtype=l_loc.dtype, device=l_loc.device)
    mine[0, :, :l_loc.shape[1]] = l_loc
    mine[1, :, :u_loc.shape[1]] = u_loc
    parts = [torch.empty_like(mine) for _ in range(world)]
    dist.all_gather(parts, mine)
    l = torch.cat([parts[r][0, :, :hi - lo] for r, (lo, hi) in enumerate(cuts)], dim=1)
    u = torch.cat([parts[r][1, :, :hi - lo] for r, (lo, hi) in enumerate(cuts)], dim=1)
    return l.contiguous(), u.contiguous()


def crown_run_row_sharded(ctx, x_lo, x_hi, Cmat, alpha: Optional[Dict[int, torch.Tensor]], rank: int, world: int,
                          gather: Optional[Callable] = None, multiple: int = 128):
    """O4 + O5 for ONE batch with the identity rows of every intermediate pass sharded over `world` ranks.

    ctx: a CrownContext (or anything with its .net / .relu_ids / .sizes / .ibp_forward / .crown_backward / .row_chunk);
    weights are replicated, every rank passes the same inputs.  Per ReLU in topological order: first layer by IBP
    (closed form, every rank); otherwise this rank's rows by `local_rows`, then `gather` (default `allgather_rows`)
    -- the only data-path collective.  The final pass (S rows) is tiny and runs on every rank.
    Returns dict pre {relu id: (l, u)}, lb, ub [B, S], verified [B]."""
    gather = gather or allgather_rows
    net = ctx.net
    B = x_lo.shape[0]
    box = (x_lo, x_hi)
    pre: Dict[int, tuple] = {}
    first = [net.nodes[i].in0 for i in ctx.relu_ids if net.nodes[net.nodes[i].in0].in0 < 0]
    ib, _ = ctx.ibp_forward(x_lo, x_hi, nodes=first) if first else ({}, None)
    for i in ctx.relu_ids:
        src = net.nodes[i].in0
        if src in ib:
            pre[i] = ib[src]
            continue
        if net.nodes[src].op != "linear":
            raise ValueError("row-sharded CROWN intermediate bounds need Linear pre-activations")
        n = ctx.sizes[src]
        r0, r1 = shard_rows(n, rank, world, multiple)
        l_loc, u_loc = local_rows(ctx, B, src, pre, box, r0, r1)
        pre[i] = gather(l_loc, u_loc, n, rank, world, multiple)
    out = ctx.crown_backward(B, len(net.nodes) - 1, pre, Cmat, alpha_lo=alpha, alpha_up=alpha, box=box, want_A=False)
    ver = ctx.verdict(out["lb"]) if hasattr(ctx, "verdict") else None
    return {"pre": pre, "lb": out["lb"], "ub": out["ub"], "verified": ver}
