"""Flattened Ulysses context parallelism around the attention-JVP call.

PAPER.md:318: before attention every rank holds the sequence shard `[B, H, N/P, d]`; one all-to-all turns it into the
head shard `[B, H/P, N, d]`; attention runs locally on full sequences (the mask descriptor is unchanged); a second
all-to-all brings the outputs back.  PAPER.md:358-360: with the JVP the tangents ride along, so six tensors go in
(Q, K, V, tQ, tK, tV) and two come out (O, tO).  Here the six (two) tensors are packed into ONE buffer and exchanged
with ONE `all_to_all_single` per direction (NCCL over NVLink / NVSwitch on GPUs; gloo in the CPU tests).

Only plumbing lives here (packing, the collective, unpacking): the attention itself is the `local_op` the caller
passes, in production `local_attn_jvp(plan)` = the C-ABI call on this rank's `H/P` heads.
"""
from __future__ import annotations

from typing import Callable, Optional, Sequence, Tuple

import torch
import torch.distributed as dist


def _exchange(buf: torch.Tensor, group) -> torch.Tensor:
    """buf [P, ...]: chunk j goes to rank j; returns [P, ...] with chunk i received from rank i."""
    out = torch.empty_like(buf)
    dist.all_to_all_single(out, buf, group=group)
    return out


def seq_to_head_shard(xs: Sequence[torch.Tensor], group=None) -> Tuple[torch.Tensor, ...]:
    """T tensors `[B, H, N/P, d]` (this rank's tokens, all heads) -> T tensors `[B, H/P, N, d]` (all tokens, this rank's
    heads), one collective.  Rank r owns tokens [r N/P, (r+1) N/P) and heads [r H/P, (r+1) H/P)."""
    P = dist.get_world_size(group)
    B, H, n, d = xs[0].shape
    if H % P:
        raise ValueError(f"H = {H} is not divisible by the context-parallel size {P}")
    T = len(xs)
    # [T, B, P, H/P, n, d] -> [P, T, B, H/P, n, d]: chunk j = the heads of rank j
    send = torch.stack(list(xs)).view(T, B, P, H // P, n, d).permute(2, 0, 1, 3, 4, 5).contiguous()
    recv = _exchange(send, group)                       # chunk i = rank i's tokens of my heads
    full = recv.permute(1, 2, 3, 0, 4, 5).reshape(T, B, H // P, P * n, d)
    return tuple(full[t] for t in range(T))


def head_to_seq_shard(ys: Sequence[torch.Tensor], group=None) -> Tuple[torch.Tensor, ...]:
    """The inverse: T tensors `[B, H/P, N, d]` -> T tensors `[B, H, N/P, d]`, one collective."""
    P = dist.get_world_size(group)
    B, h, N, d = ys[0].shape
    if N % P:
        raise ValueError(f"N = {N} is not divisible by the context-parallel size {P}")
    T = len(ys)
    # [T, B, h, P, n, d] -> [P, T, B, h, n, d]: chunk j = the tokens of rank j
    send = torch.stack(list(ys)).view(T, B, h, P, N // P, d).permute(3, 0, 1, 2, 4, 5).contiguous()
    recv = _exchange(send, group)                       # chunk i = my tokens of rank i's heads
    local = recv.permute(1, 2, 0, 3, 4, 5).reshape(T, B, P * h, N // P, d)
    return tuple(local[t] for t in range(T))


LocalOp = Callable[[torch.Tensor, torch.Tensor, torch.Tensor, torch.Tensor, torch.Tensor, torch.Tensor],
                   Tuple[torch.Tensor, torch.Tensor, Optional[torch.Tensor]]]


def ulysses_attn_jvp(local_op: LocalOp, q, k, v, tq, tk, tv, group=None):
    """q, k, v, tq, tk, tv: this rank's `[B, H, N/P, d]` shards.  -> (o, to) `[B, H, N/P, d]`, lse `[B, H/P, N]` or None
    (lse stays head-sharded: it is consumed by the primal backward on the same rank)."""
    hq, hk, hv, htq, htk, htv = seq_to_head_shard((q, k, v, tq, tk, tv), group)
    o, to, lse = local_op(hq, hk, hv, htq, htk, htv)
    o_l, to_l = head_to_seq_shard((o, to), group)
    return o_l, to_l, lse


def local_attn_jvp(plan, stream: int = 0) -> LocalOp:
    """The production local op: `attn_jvp_fwd` of a plan created for (B, H/P heads, N, N) on this rank's GPU."""
    from . import binding as aj

    def op(q, k, v, tq, tk, tv):
        o, to = torch.empty_like(q), torch.empty_like(q)
        lse = torch.empty(q.shape[:3], dtype=torch.float32, device=q.device)
        aj.attn_jvp_fwd(plan, q, k, v, tq, tk, tv, o, to, lse, stream)
        return o, to, lse
    return op
