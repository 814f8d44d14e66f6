"""Flattened Ulysses context parallelism around the attention-JVP call.

PAPER.md:318: before attention every rank holds the sequence shard `[B, H, N/P, d]`; one all-to-all turns it into the
head shard `[B, H/P, N, d]`; attention runs locally on full sequences (the mask descriptor is unchanged); a second
all-to-all brings the outputs back.  PAPER.md:358-360: with the JVP the tangents ride along, so six tensors go in
(Q, K, V, tQ, tK, tV) and two come out (O, tO).  The primal backward sends dO in and dQ, dK, dV out;
Q, K, V, O and lse stay head-sharded on the rank between the two calls.

How the exchange is organised here
  * The rank's H/P heads are cut into `head_groups` groups.  Per group and direction ALL tensors travel in ONE group of
    point-to-point transfers (`mode="p2p"`, the default: `dist.batch_isend_irecv` = one ncclGroupStart / End on GPUs) whose
    chunks are the `[n, d]` blocks themselves -- sent from the `[B, H, n, d]` shard in place and received at rows
    `[i n, (i + 1) n)` of the `[B, hg, N, d]` tensor the kernel reads (and back: sent from the kernel's output in place,
    received in the `[B, H, n, d]` result).  No send buffer, no receive buffer, no pack or unpack pass; the rank's own chunk
    is one strided copy.  `mode="packed"` is the earlier form: ONE `all_to_all_single` per group and direction around
    `pack_*` / `unpack_*` copies (four extra passes over the data).
  * The groups are pipelined: the collective of group g + 1 is issued (async) before the kernel of group g is enqueued, and
    the outputs of group g go back while group g + 1 computes, so that the exchange hides under the kernel except for the
    first group's way in and the last group's way out.
  * Packing is one strided copy per tensor into the send buffer and one per tensor out of the receive buffer (no stacked
    intermediate), with the index arithmetic in `pack_*` / `unpack_*` below -- the same functions the single-process
    emulation of the tests drives, so that what the tests check is what production runs.

Only plumbing lives here (packing, the collective, stream ordering): the attention itself is the `local_op` the caller
passes, in production `local_attn_jvp(plan)` / `local_attn_bwd(plan)` = the C-ABI calls on one head group.
"""
from __future__ import annotations

from typing import Callable, List, Optional, Sequence, Tuple

import torch
import torch.distributed as dist


# ---------------------------------------------------------------------------------------------- index arithmetic
def pack_seq_shard(xs: Sequence[torch.Tensor], P: int, g: int, G: int) -> torch.Tensor:
    """This rank's T tensors `[B, H, n, d]` (its n = N/P tokens, all H heads) -> the send buffer of head group g:
    `[P, T, B, hg, n, d]`, chunk j = heads `[j H/P + g hg, j H/P + (g + 1) hg)` (rank j's group g), hg = H/(P G)."""
    B, H, n, d = xs[0].shape
    if H % (P * G):
        raise ValueError(f"H = {H} is not divisible by context-parallel size {P} x head groups {G}")
    h, hg = H // P, H // (P * G)
    send = xs[0].new_empty((P, len(xs), B, hg, n, d))
    for t, x in enumerate(xs):
        send[:, t].copy_(x.unflatten(1, (P, h))[:, :, g * hg:(g + 1) * hg].permute(1, 0, 2, 3, 4))
    return send


def unpack_head_shard(recv: torch.Tensor) -> Tuple[torch.Tensor, ...]:
    """The receive buffer `[P, T, B, hg, n, d]` (chunk i = rank i's tokens of my heads) -> T tensors `[B, hg, P n, d]`
    (all tokens; rank i owns tokens `[i n, (i + 1) n)`)."""
    P, T, B, hg, n, d = recv.shape
    outs = []
    for t in range(T):
        full = recv.new_empty((B, hg, P * n, d))
        full.view(B, hg, P, n, d).copy_(recv[:, t].permute(1, 2, 0, 3, 4))
        outs.append(full)
    return tuple(outs)


def pack_head_shard(ys: Sequence[torch.Tensor], P: int) -> torch.Tensor:
    """T tensors `[B, hg, N, d]` (all tokens of my heads) -> the send buffer `[P, T, B, hg, n, d]`, chunk j = rank j's tokens."""
    B, hg, N, d = ys[0].shape
    if N % P:
        raise ValueError(f"N = {N} is not divisible by the context-parallel size {P}")
    n = N // P
    send = ys[0].new_empty((P, len(ys), B, hg, n, d))
    for t, y in enumerate(ys):
        send[:, t].copy_(y.unflatten(2, (P, n)).permute(2, 0, 1, 3, 4))
    return send


def unpack_seq_shard(recv: torch.Tensor, outs: Sequence[torch.Tensor], g: int, G: int) -> None:
    """The receive buffer `[P, T, B, hg, n, d]` (chunk i = my tokens of rank i's head group g) -> written into head group g
    of the T output tensors `[B, H, n, d]`."""
    P, T, B, hg, n, d = recv.shape
    h = hg * G
    for t, out in enumerate(outs):
        out.unflatten(1, (P, h))[:, :, g * hg:(g + 1) * hg].copy_(recv[:, t].permute(1, 0, 2, 3, 4))


# ---------------------------------------------------------------------------------------------- the collective
class _Done:
    def wait(self):
        return True


def _exchange(send: torch.Tensor, group, async_op: bool):
    """send [P, ...]: chunk j goes to rank j.  -> (recv [P, ...] with chunk i from rank i, work handle)."""
    recv = torch.empty_like(send)
    work = dist.all_to_all_single(recv, send, group=group, async_op=async_op)
    return recv, (work if async_op and work is not None else _Done())


# ---------------------------------------------------------------------------------------------- zero-copy point-to-point exchange
def p2p_chunks_in(ins: Sequence[torch.Tensor], heads: Sequence[torch.Tensor], P: int, r: int, g: int, G: int):
    """The way in for head group g on rank r.  ins: T tensors `[B, H, n, d]` (my tokens, all heads); heads: T tensors
    `[B, hg, P n, d]` (all tokens of my group-g heads).  -> [(peer, send_view, recv_view)] in the order both ends enumerate:
    send_view = my tokens of peer's head (a contiguous `[n, d]` block of `ins`), recv_view = peer's tokens of my head (rows
    `[peer n, (peer + 1) n)` of `heads`, contiguous).  peer == r: the same two views, to be copied locally."""
    B, H, n, d = ins[0].shape
    if H % (P * G):
        raise ValueError(f"H = {H} is not divisible by context-parallel size {P} x head groups {G}")
    h, hg = H // P, H // (P * G)
    out = []
    for j in range(P):
        for t in range(len(ins)):
            for b in range(B):
                for i in range(hg):
                    out.append((j, ins[t][b, j * h + g * hg + i], heads[t][b, i, j * n:(j + 1) * n]))
    return out


def p2p_chunks_out(res: Sequence[torch.Tensor], outs: Sequence[torch.Tensor], P: int, r: int, g: int, G: int):
    """The way back: res = T tensors `[B, hg, P n, d]` (the local op's results on my group-g heads), outs = T tensors
    `[B, H, n, d]` (my tokens, all heads).  send_view = peer's tokens of my head, recv_view = my tokens of peer's head."""
    B, hg, N, d = res[0].shape
    n, h = N // P, hg * G
    out = []
    for j in range(P):
        for t in range(len(res)):
            for b in range(B):
                for i in range(hg):
                    out.append((j, res[t][b, i, j * n:(j + 1) * n], outs[t][b, j * h + g * hg + i]))
    return out


class _Works:
    def __init__(self, works):
        self.works = works

    def wait(self):
        for w in self.works:
            w.wait()
        return True


def _exchange_p2p(chunks, r: int, group):
    """Issues every transfer of `chunks` as one batch (async); the rank's own chunks are copied in place.  -> work handle."""
    ops = []
    seq = {}                               # per peer: position of the chunk in that peer's sub-list (the same number at both ends)
    for peer, send, recv in chunks:
        if peer == r:
            recv.copy_(send)
        else:
            k = seq[peer] = seq.get(peer, -1) + 1
            dst = peer if group is None else dist.get_global_rank(group, peer)
            ops.append(dist.P2POp(dist.isend, send, dst, group=group, tag=k))
            ops.append(dist.P2POp(dist.irecv, recv, dst, group=group, tag=k))
    return _Works(dist.batch_isend_irecv(ops)) if ops else _Done()


LocalOp = Callable[..., Tuple[torch.Tensor, ...]]


def _pipeline_p2p(ins: Sequence[torch.Tensor], n_out: int, local_op: LocalOp, group, head_groups: int, out_like: Sequence[int]):
    """`_pipeline` with the zero-copy exchange: the transfers of group g + 1 are in flight under the kernel of group g, the
    results of group g travel back under the kernel of group g + 1.  The head-sharded tensors are fresh allocations per call
    (no pass over memory): the forward hands them to the caller as `saved`, which must outlive later calls."""
    P, r, G = dist.get_world_size(group), dist.get_rank(group), head_groups
    ins = [x if x.is_contiguous() else x.contiguous() for x in ins]
    B, H, n, d = ins[0].shape
    hg = H // (P * G)
    outs = [torch.empty(ins[i].shape, dtype=ins[i].dtype, device=ins[i].device) for i in out_like]
    extras: List = [None] * G

    def way_in(g):
        heads = [x.new_empty((B, hg, P * n, d)) for x in ins]
        return heads, _exchange_p2p(p2p_chunks_in(ins, heads, P, r, g, G), r, group)

    heads, work_in = way_in(0)
    pending = []                                            # way-back transfers in flight (their source tensors kept alive)
    for g in range(G):
        nxt = way_in(g + 1) if g + 1 < G else None
        work_in.wait()
        res = local_op(g, *heads)
        extras[g] = res[n_out:]
        back = [t if t.is_contiguous() else t.contiguous() for t in res[:n_out]]
        for wk, _ in pending:
            wk.wait()
        pending = [(_exchange_p2p(p2p_chunks_out(back, outs, P, r, g, G), r, group), back)]
        if nxt is not None:
            heads, work_in = nxt
    for wk, _ in pending:
        wk.wait()
    return outs, extras


def _pipeline(ins: Sequence[torch.Tensor], n_out: int, local_op: LocalOp, group, head_groups: int, out_like: Sequence[int],
              mode: str = "p2p"):
    """Shared by the forward and the backward: `ins` = this rank's `[B, H, n, d]` tensors; per head group: exchange in,
    `local_op(g, *head_sharded_inputs)` -> n_out head-sharded `[B, hg, N, d]` tensors (+ anything it wants to keep, which
    is returned per group), exchange out.  out_like[i] = index of the input whose shape output i has.
    -> (outs `[B, H, n, d]`, [extras of group g])."""
    if mode == "p2p":
        return _pipeline_p2p(ins, n_out, local_op, group, head_groups, out_like)
    if mode != "packed":
        raise ValueError(f"unknown exchange mode {mode!r}")
    P = dist.get_world_size(group)
    G = head_groups
    outs = [torch.empty(ins[i].shape, dtype=ins[i].dtype, device=ins[i].device) for i in out_like]
    extras: List = [None] * G
    recv_in, work_in = _exchange(pack_seq_shard(ins, P, 0, G), group, True)
    pending_out = None                                    # (recv, work, g) of the previous group's way back
    for g in range(G):
        nxt = _exchange(pack_seq_shard(ins, P, g + 1, G), group, True) if g + 1 < G else None   # in flight under kernel g
        work_in.wait()
        res = local_op(g, *unpack_head_shard(recv_in))
        extras[g] = res[n_out:]
        back = _exchange(pack_head_shard(res[:n_out], P), group, True)                            # in flight under kernel g + 1
        if pending_out is not None:
            pending_out[1].wait()
            unpack_seq_shard(pending_out[0], outs, pending_out[2], G)
        pending_out = (back[0], back[1], g)
        if nxt is not None:
            recv_in, work_in = nxt
    pending_out[1].wait()
    unpack_seq_shard(pending_out[0], outs, pending_out[2], G)
    return outs, extras


def ulysses_attn_jvp(local_op: LocalOp, q, k, v, tq, tk, tv, group=None, head_groups: int = 1, mode: str = "p2p"):
    """q, k, v, tq, tk, tv: this rank's `[B, H, N/P, d]` shards.  local_op(g, q, k, v, tq, tk, tv) -> (o, to, lse) on the
    head shard of group g.  -> (o, to) `[B, H, N/P, d]`, and `saved` = per head group (q, k, v, o, lse) head-sharded, which
    is what the primal backward on this rank consumes (lse never leaves the rank)."""
    def op(g, hq, hk, hv, htq, htk, htv):
        o, to, lse = local_op(g, hq, hk, hv, htq, htk, htv)
        return o, to, (hq, hk, hv, o, lse)
    (o_l, to_l), extras = _pipeline((q, k, v, tq, tk, tv), 2, op, group, head_groups, (0, 0), mode)
    return o_l, to_l, [e[0] for e in extras]


def ulysses_attn_bwd(local_bwd: LocalOp, saved, dout, group=None, head_groups: int = 1, mode: str = "p2p"):
    """dout: this rank's `[B, H, N/P, d]` shard of dO; `saved` from ulysses_attn_jvp (same head_groups).
    local_bwd(g, q, k, v, o, lse, dout) -> (dq, dk, dv) on the head shard.  -> dq, dk, dv `[B, H, N/P, d]`."""
    def op(g, hdo):
        hq, hk, hv, o, lse = saved[g]
        return local_bwd(g, hq, hk, hv, o, lse, hdo)
    (dq, dk, dv), _ = _pipeline((dout,), 3, op, group, head_groups, (0, 0, 0), mode)
    return dq, dk, dv


# ---------------------------------------------------------------------------------------------- production local ops
def _launch_stream(stream: Optional[int], device) -> int:
    """The cudaStream_t the kernel goes on.  None = torch's CURRENT stream of `device` at the moment of the call: the packing
    copies, the allocations and the collective's wait() in `_pipeline` are all ordered on that stream, so the kernel must be
    too (under `with torch.cuda.stream(s)` the legacy default stream 0 is ordered against none of them)."""
    return torch.cuda.current_stream(device).cuda_stream if stream is None else stream


def local_attn_jvp(plan, stream: Optional[int] = None) -> LocalOp:
    """`attn_jvp_fwd` of a plan created for (B, H / (P G) heads, N, N) on this rank's GPU; every head group reuses it.
    stream: a cudaStream_t handle, or None for torch's current stream when the op runs."""
    from . import binding as aj

    def op(g, q, k, v, tq, tk, tv):
        o, to = torch.empty_like(q), torch.empty_like(q)
        lse = torch.empty(q.shape[:3], dtype=torch.float32, device=q.device)
        aj.attn_jvp_fwd(plan, q, k, v, tq, tk, tv, o, to, lse, _launch_stream(stream, q.device))
        return o, to, lse
    return op


def local_attn_bwd(plan, stream: Optional[int] = None) -> LocalOp:
    """`attn_bwd` of the same plan (stream as in local_attn_jvp)."""
    from . import binding as aj

    def op(g, q, k, v, o, lse, dout):
        dq, dk, dv = torch.empty_like(q), torch.empty_like(k), torch.empty_like(k)
        aj.attn_bwd(plan, q, k, v, o, lse, dout, dq, dk, dv, _launch_stream(stream, q.device))
        return dq, dk, dv
    return op


# ---------------------------------------------------------------------------------------------- single-process emulation
def _deliver(plans):
    """plans[r] = rank r's chunk list: the k-th chunk rank i sends to rank j lands in the k-th chunk rank j receives from rank i."""
    P = len(plans)
    for i in range(P):
        for j in range(P):
            sends = [c[1] for c in plans[i] if c[0] == j]
            recvs = [c[2] for c in plans[j] if c[0] == i]
            assert len(sends) == len(recvs)
            for s_, r_ in zip(sends, recvs):
                r_.copy_(s_)


def emulate_ranks(P: int, shards: Sequence[Sequence[torch.Tensor]], n_out: int, local_op: LocalOp, head_groups: int = 1,
                  out_like: Optional[Sequence[int]] = None, mode: str = "p2p"):
    """P virtual ranks in ONE process (tests; one GPU): shards[r] = rank r's `[B, H, n, d]` tensors.  Runs the same index
    arithmetic as `_pipeline` (`p2p_chunks_*`, or `pack_*` / `unpack_*` for mode="packed"), with the transfers replaced by
    their definition.  -> outs[r] = rank r's n_out output shards."""
    G = head_groups
    out_like = out_like or [0] * n_out
    outs = [[torch.empty(shards[r][i].shape, dtype=shards[r][i].dtype, device=shards[r][i].device) for i in out_like] for r in range(P)]
    if mode == "p2p":
        B, H, n, d = shards[0][0].shape
        hg = H // (P * G)
        for g in range(G):
            heads = [[x.new_empty((B, hg, P * n, d)) for x in shards[r]] for r in range(P)]
            _deliver([p2p_chunks_in(shards[r], heads[r], P, r, g, G) for r in range(P)])
            res = [local_op(r, g, *heads[r])[:n_out] for r in range(P)]
            _deliver([p2p_chunks_out([t.contiguous() for t in res[r]], outs[r], P, r, g, G) for r in range(P)])
        return outs
    for g in range(G):
        sends = [pack_seq_shard(shards[r], P, g, G) for r in range(P)]
        backs = []
        for r in range(P):
            recv = torch.stack([sends[i][r] for i in range(P)])
            res = local_op(r, g, *unpack_head_shard(recv))
            backs.append(pack_head_shard(res[:n_out], P))
        for r in range(P):
            unpack_seq_shard(torch.stack([backs[i][r] for i in range(P)]), outs[r], g, G)
    return outs
