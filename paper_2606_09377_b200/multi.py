"""Multi-GPU plumbing for the hot path: one process per GPU, NO data-path collective.

Properties are independent problems (each row of Eq. 1 is its own linear bound), so N GPUs run N
batches side by side ("replicas only" in DESIGN.md; weak scaling).  The only exchanges are host-side bookkeeping:
which properties a rank owns, the max-over-ranks step time, and the sum of verified counts.  The paper's TP/FSDP
sharding is prior art and is not built.  Works with the `nccl` backend on GPUs and `gloo` on CPU.
"""
from __future__ import annotations

from typing import List, Tuple

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
