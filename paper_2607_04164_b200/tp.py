"""Tensor parallelism over F for the grouped MoE layer (PAPER.md:289-295 scales with TP).

Plumbing only: the shard slicing and the all-reduce around the C-ABI calls.  Every rank holds the rows of W1 / W3
and the columns of W2 that belong to its slice of the F hidden features, runs the replicated routing and
bm_moe_forward_f32 on its shard, and the fp32 partial layer outputs are summed across ranks with
torch.distributed (NCCL on GPUs) before one rounding to bf16.
"""
from __future__ import annotations

import torch


def shard_bounds(F: int, rank: int, world: int, multiple: int = 8):
    """[lo, hi) of rank's slice of the F features: contiguous, multiples of `multiple` (16-byte rows), sizes differ
    by at most `multiple`."""
    units = F // multiple
    assert units * multiple == F and world >= 1 and 0 <= rank < world and units >= world
    lo = (units * rank) // world * multiple
    hi = (units * (rank + 1)) // world * multiple
    return lo, hi


def shard_f(W1, W3, W2, rank: int, world: int):
    """Rank's shard: W1, W3 [N, F, D] -> [N, F_r, D] (rows), W2 [N, D, F] -> [N, D, F_r] (columns), contiguous."""
    lo, hi = shard_bounds(W1.shape[1], rank, world)
    return W1[:, lo:hi, :].contiguous(), W3[:, lo:hi, :].contiguous(), W2[:, :, lo:hi].contiguous()


def tp_moe_forward(x, routing, W1_r, W3_r, W2_r, out, workspace, S: int = 0, group=None, partial=None):
    """One tensor-parallel layer call on this rank: fp32 partial on the shard, all-reduce (sum), round to bf16.
    `workspace` is sized for the shard (F_r).  Returns `out` [T, D] bf16, identical on every rank."""
    from . import binding as bm
    import torch.distributed as dist
    T, D = x.shape
    if partial is None:
        partial = torch.empty((T, D), dtype=torch.float32, device=x.device)
    bm.bm_moe_forward_f32(x, routing, W1_r, W3_r, W2_r, partial, workspace, S=S)
    if dist.is_available() and dist.is_initialized():        # (also with one rank: the same call path)
        dist.all_reduce(partial, op=dist.ReduceOp.SUM, group=group)
    return bm.bm_round_bf16(partial, out)
