"""Sequence-parallel attention around the block-sparse kernel (appendix A): Ulysses
all-to-all with the heads re-partitioned by the greedy schedule.

Rank r of `group` (P ranks) holds the tokens [bounds[r], bounds[r+1]) of every head ([1][n_r][H][d];
`shard_bounds` cuts N as evenly as possible, the shards need not be equal).  seq_to_heads gathers the heads in
schedule order (chorus_gather_heads), exchanges the chunks with one all-to-all and returns [1][N][H/P][d]: all
tokens of this rank's heads, which is the layout chorus_block_sparse_attn_fwd takes.  heads_to_seq is the way
back for O.  The schedule (`order`, from chorus_schedule_heads on the per-head costs of the layer's index) is the
same on every rank because the masks are known before the attention call.  H must be a multiple of P (the
all-to-all gives every rank the same number of head slots, R24); pad the head axis otherwise.

The two local copies are this library's kernels; the exchange itself (`exchange_to_heads`, `exchange_to_seq`) is
torch.distributed (NCCL over NVLink / NVSwitch on CUDA tensors; the functions are device-agnostic so that the
multi-rank plumbing is also exercised over gloo on CPU).
"""
from __future__ import annotations

import torch
import torch.distributed as dist

from . import binding as B


def _world(group):
    return dist.get_world_size(group) if dist.is_available() and dist.is_initialized() else 1


def _rank(group):
    return dist.get_rank(group) if dist.is_available() and dist.is_initialized() else 0


def shard_bounds(N: int, P: int):
    """Token range of every rank: rank r holds [b[r], b[r+1]); sizes differ by at most one."""
    return [(N * r) // P for r in range(P + 1)]


def exchange_to_heads(packed, bounds, group=None):
    """packed: [P][n_r][slots][d] contiguous (chunk p = this rank's tokens of rank p's heads) ->
    [N][slots][d]: every rank's tokens (in rank order) of THIS rank's heads."""
    P = _world(group)
    assert packed.dim() == 4 and packed.is_contiguous() and packed.shape[0] == P == len(bounds) - 1
    _, n_r, slots, d = packed.shape
    r = _rank(group)
    assert n_r == bounds[r + 1] - bounds[r], (n_r, bounds, r)
    if P == 1:
        return packed[0]
    row = slots * d
    recv = torch.empty((bounds[-1], slots, d), dtype=packed.dtype, device=packed.device)
    dist.all_to_all_single(recv.view(-1), packed.view(-1),
                           output_split_sizes=[(bounds[p + 1] - bounds[p]) * row for p in range(P)],
                           input_split_sizes=[n_r * row] * P, group=group)
    return recv


def exchange_to_seq(o_heads, bounds, group=None):
    """o_heads: [N][slots][d] contiguous (all tokens of this rank's heads) -> [P][n_r][slots][d]: this rank's
    tokens of every rank's heads (chunk p = the heads rank p computed)."""
    P = _world(group)
    assert o_heads.dim() == 3 and o_heads.is_contiguous() and o_heads.shape[0] == bounds[-1]
    _, slots, d = o_heads.shape
    r = _rank(group)
    n_r = bounds[r + 1] - bounds[r]
    if P == 1:
        return o_heads[None]
    row = slots * d
    recv = torch.empty((P, n_r, slots, d), dtype=o_heads.dtype, device=o_heads.device)
    dist.all_to_all_single(recv.view(-1), o_heads.view(-1),
                           output_split_sizes=[n_r * row] * P,
                           input_split_sizes=[(bounds[p + 1] - bounds[p]) * row for p in range(P)], group=group)
    return recv


def seq_to_heads(x_loc, order, N: int, group=None):
    """x_loc: cuda [1][n_r][H][d] (this rank's tokens) -> cuda [1][N][H / P][d] (tokens in rank order)."""
    assert x_loc.is_cuda and x_loc.dim() == 4 and x_loc.shape[0] == 1, "cuda tensor, batch 1"
    P = _world(group)
    H = x_loc.shape[2]
    assert H % P == 0, f"H = {H} is not a multiple of the {P} ranks: pad the head axis"
    packed = B.chorus_gather_heads(x_loc[0], order, P)
    return exchange_to_heads(packed, shard_bounds(N, P), group)[None]


def heads_to_seq(o_heads, order, group=None, out=None):
    """o_heads: cuda [1][N][H / P][d] contiguous -> cuda [1][n_r][H][d] (this rank's tokens, all heads)."""
    assert o_heads.is_cuda and o_heads.dim() == 4 and o_heads.shape[0] == 1 and o_heads.is_contiguous()
    P = _world(group)
    _, N, slots, d = o_heads.shape
    chunks = exchange_to_seq(o_heads[0], shard_bounds(N, P), group)
    n_r = chunks.shape[1]
    if out is None:
        out = torch.empty((1, n_r, P * slots, d), dtype=o_heads.dtype, device=o_heads.device)
    B.chorus_scatter_heads(chunks.contiguous(), order, out[0])
    return out


def rank_rows(order, rank: int, n_ranks: int, nq_blk: int):
    """This rank's heads in schedule order as (head, first row, last row + 1) triples into the layer's row_ptr
    (rows of head h are h * nq_blk .. (h + 1) * nq_blk).  After seq_to_heads the rank's tensors hold these heads
    in this order, so either the mask rows are gathered the same way before the decode (the masks follow their
    heads) or the attention call is made per head with row_ptr[first : last + 1]."""
    H = len(order)
    slots = H // n_ranks
    return [(int(h), int(h) * nq_blk, (int(h) + 1) * nq_blk) for h in order[rank * slots:(rank + 1) * slots]]


def imbalance(cost, order, n_ranks: int) -> float:
    """max / mean of the per-rank loads when rank p takes the heads order[p*slots:(p+1)*slots] (appendix A,
    PAPER.md:L266: 1.34 before the schedule, 1.12 after it at 8 GPUs)."""
    H = len(order)
    slots = H // n_ranks
    loads = [sum(float(cost[int(h)]) for h in order[p * slots:(p + 1) * slots]) for p in range(n_ranks)]
    mean = sum(loads) / n_ranks
    return max(loads) / mean if mean > 0 else 1.0
