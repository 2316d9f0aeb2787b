"""Sequence-parallel attention around the block-sparse kernel (appendix A): Ulysses
all-to-all with the heads re-partitioned by the greedy schedule.

Each rank of `group` holds n_loc = N / P consecutive tokens of every head ([1][n_loc][H][d]).  seq_to_heads
gathers the heads in schedule order (chorus_gather_heads), exchanges equal chunks with one NCCL all-to-all and
returns [1][N][H/P][d]: all tokens of this rank's heads, which is the layout chorus_block_sparse_attn_fwd takes.
heads_to_seq is the way back for O.  The schedule (`order`, from chorus_schedule_heads on the per-head costs of
the layer's index) is the same on every rank because the masks are known before the attention call.

Only the two local copies are this library's kernels; the exchange is torch.distributed (NCCL over NVLink /
NVSwitch).  This container and the GPU pool have one GPU: the multi-rank path is covered by construction and by
the one-rank round trip in tests/test_gpu_head_exchange.py.  No CPU fallback: the tensors
must be CUDA tensors.
"""
from __future__ import annotations

import torch
import torch.distributed as dist

from . import binding as B


def _world(group):
    return dist.get_world_size(group) if dist.is_available() and dist.is_initialized() else 1


def seq_to_heads(x_loc, order, group=None, _gather=None):
    """x_loc: cuda [1][n_loc][H][d] -> cuda [1][P * n_loc][H / P][d] (tokens in rank order).
    _gather: test seam (the gloo tests on CPU pass the oracle's copy); the product path uses the CUDA kernel."""
    assert x_loc.dim() == 4 and x_loc.shape[0] == 1, "batch 1 (the token axis of the result must be one stride)"
    P = _world(group)
    _, n_loc, H, d = x_loc.shape
    packed = (_gather or B.chorus_gather_heads)(x_loc[0], order, P)
    if P > 1:
        recv = torch.empty_like(packed)
        dist.all_to_all_single(recv, packed, group=group)
        packed = recv
    return packed.view(1, P * n_loc, H // P, d)


def heads_to_seq(o_heads, order, group=None, out=None, _scatter=None):
    """o_heads: cuda [1][P * n_loc][H / P][d] contiguous -> cuda [1][n_loc][H][d].  _scatter: test seam."""
    assert o_heads.dim() == 4 and o_heads.shape[0] == 1 and o_heads.is_contiguous()
    P = _world(group)
    _, N, slots, d = o_heads.shape
    n_loc = N // P
    chunks = o_heads.view(P, n_loc, slots, d)
    if P > 1:
        recv = torch.empty_like(chunks)
        dist.all_to_all_single(recv, chunks, group=group)
        chunks = recv
    if out is None:
        out = torch.empty((1, n_loc, P * slots, d), dtype=o_heads.dtype, device=o_heads.device)
    (_scatter or B.chorus_scatter_heads)(chunks, order, out[0])
    return out


def rank_rows(order, rank: int, n_ranks: int, nq_blk: int):
    """This rank's heads in schedule order as (head, first row, last row + 1) triples into the layer's row_ptr
    (rows of head h are h * nq_blk .. (h + 1) * nq_blk).  After seq_to_heads the rank's tensors hold these heads
    in this order, so either the mask rows are gathered the same way before the decode (the masks follow their
    heads) or the attention call is made per head with row_ptr[first : last + 1]."""
    H = len(order)
    slots = H // n_ranks
    return [(int(h), int(h) * nq_blk, (int(h) + 1) * nq_blk) for h in order[rank * slots:(rank + 1) * slots]]
