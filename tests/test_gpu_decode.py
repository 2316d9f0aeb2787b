"""GPU parity: chorus_mask_to_index / chorus_visit_refresh vs the oracle, bit-exact."""
import numpy as np
import pytest
import torch

import oracle
from gpu_common import dev, dmask
from paper_2606_25040_b200 import binding as B
from paper_2606_25040_b200 import workloads as W

pytestmark = pytest.mark.gpu


def check(bm, nk):
    rp_o, ci_o = oracle.mask_to_index(bm, nk)
    rp, ci = B.chorus_mask_to_index(dmask(bm), nk)
    torch.cuda.synchronize()
    assert np.array_equal(rp.cpu().numpy(), rp_o)
    assert np.array_equal(ci.cpu().numpy()[: len(ci_o)], ci_o)
    return rp, ci


@pytest.mark.parametrize("L,H,nq,nk,rho", [
    (1, 2, 32, 64, 0.5), (2, 3, 7, 33, 0.3), (1, 2, 5, 1182, 0.15), (3, 2, 9, 512, 0.25),
    (1, 1, 1, 1, 1.0), (2, 2, 130, 31, 0.5), (1, 1, 300, 32, 0.02), (1, 3, 129, 1025, 0.1)])
def test_random_masks_with_garbage_pad_bits(L, H, nq, nk, rho):
    g = np.random.default_rng(nk * 7 + nq)
    bm = W.pack_bits(g.random((L, H, nq, nk)) < rho)
    if nk % 32:
        bm[..., -1] |= np.uint32((0xFFFFFFFF << (nk % 32)) & 0xFFFFFFFF)
    check(bm, nk)


def test_adversarial_rows():
    nk, nq = 100, 260
    keep = np.zeros((1, 1, nq, nk), bool)
    keep[0, 0, 1] = True                 # full row
    keep[0, 0, 2, 99] = True             # single bit in the last (partial) word
    keep[0, 0, 3, 0] = True
    keep[0, 0, 127:130, ::3] = True      # rows straddling a 128-row block boundary
    keep[0, 0, 259, 31:34] = True
    check(W.pack_bits(keep), nk)
    check(np.zeros((1, 2, 5, 4), np.uint32), nk)           # empty mask: all row_ptr = 0
    check(np.full((1, 2, 5, 4), 0xFFFFFFFF, np.uint32), nk)  # full mask with garbage pad bits


def test_full_size_layer_masks_cfg2_cfg4():
    for cfg in (W.CFG2, W.CFG4):
        bm = W.layer_mask(cfg)[None]
        rp, ci = check(bm, cfg.nk)
        per_row = 128 if cfg is W.CFG2 else 177
        assert int(rp[-1].item()) == cfg.H * cfg.nq * per_row


def test_multi_layer_mask_set_and_count_only_and_capacity():
    cfg = W.scaled(W.CFG2, H=4)
    bm = np.stack([W.layer_mask(cfg, seed=77 + 100 * l, density=0.1 + 0.1 * l) for l in range(3)])
    rp_o, ci_o = oracle.mask_to_index(bm, cfg.nk)
    d = dmask(bm)
    rp, none = B.chorus_mask_to_index(d, cfg.nk, count_only=True)
    torch.cuda.synchronize()
    assert none is None and np.array_equal(rp.cpu().numpy(), rp_o)
    # col_cap smaller than nnz: nothing beyond col_cap is written
    cap = len(ci_o) // 2
    buf = torch.full((len(ci_o),), -7, dtype=torch.int32, device=dev())
    B.chorus_mask_to_index(d, cfg.nk, col_idx=buf[:cap])
    torch.cuda.synchronize()
    got = buf.cpu().numpy()
    assert np.array_equal(got[:cap], ci_o[:cap]) and np.all(got[cap:] == -7)


def test_large_mask_set_four_words_per_thread():
    """>= 2^20 words selects the 4-words-per-thread instantiation; row densities from 0 to 1 in
    runs of uneven length put sparse (single pass) and full (four rounds) tiles next to each other, nk = 1182
    leaves a 30-bit last word with garbage above it, and the word count is no multiple of the tile."""
    L, H, nq, nk = 8, 8, 513, 1182
    g = np.random.default_rng(20260)
    rows = L * H * nq
    rho = np.empty(rows)
    i = 0
    while i < rows:
        n = int(g.integers(1, 90))
        rho[i:i + n] = g.choice([0.0, 0.03, 0.25, 0.27, 0.6, 1.0])
        i += n
    bm = W.pack_bits((g.random((rows, nk)) < rho[:, None]).reshape(L, H, nq, nk))
    bm[..., -1] |= np.uint32((0xFFFFFFFF << (nk % 32)) & 0xFFFFFFFF)
    assert bm.size >= 1 << 20 and bm.size % 1024 != 0
    rp, ci = check(bm, nk)
    # capacity guard on the same path
    rp_o, ci_o = oracle.mask_to_index(bm, nk)
    cap = len(ci_o) - 12345
    buf = torch.full((len(ci_o),), -7, dtype=torch.int32, device=dev())
    B.chorus_mask_to_index(dmask(bm), nk, col_idx=buf[:cap])
    torch.cuda.synchronize()
    got = buf.cpu().numpy()
    assert np.array_equal(got[:cap], ci_o[:cap]) and np.all(got[cap:] == -7)


@pytest.mark.parametrize("nq", [40, 500])
def test_more_than_65536_key_blocks_take_32_bit_staging_slots(nq):
    """nk > 65536: the entries do not fit the 16-bit staging slots of the usual path, so the kernel instantiation
    with 32-bit slots runs, one word per thread (nq = 40) and four (nq = 500: >= 2^20 words); row
    densities from 0 to 0.6 cover its sorted walk, its per-thread walk and its rounds."""
    nk = 70001
    g = np.random.default_rng(nq)
    rho = g.choice([0.0, 0.02, 0.2, 0.3, 0.6], size=nq)
    bm = W.pack_bits((g.random((nq, nk)) < rho[:, None]).reshape(1, 1, nq, nk))
    bm[..., -1] |= np.uint32((0xFFFFFFFF << (nk % 32)) & 0xFFFFFFFF)
    assert (bm.size >= 1 << 20) == (nq == 500)
    rp, ci = check(bm, nk)
    assert int(ci.max().item()) > 65536


def test_visit_refresh_matches_oracle():
    nk, nq, H, L = 45, 3, 2, 19
    g = np.random.default_rng(3)
    bm = W.pack_bits(g.random((L, H, nq, nk)) < 0.2)
    bm[..., -1] |= np.uint32(0xFFFFE000)          # garbage pad bits must be left as they are
    ref = oracle.visit_refresh(bm, nk, group=8)
    d = dmask(bm)
    B.chorus_visit_refresh(d, nk, group=8)
    torch.cuda.synchronize()
    assert np.array_equal(d.cpu().numpy().view(np.uint32), ref)


def test_head_costs_from_row_ptr():
    # PAPER.md:L95 / appendix A: the per-head cost is known from the reused mask before attention runs
    cfg = W.scaled(W.CFG2, H=6)
    bm = np.stack([W.layer_mask(cfg, seed=5, density=0.05 + 0.1 * 0)] )[0]
    for h in range(cfg.H):                           # different density per head
        bm[h] = W.layer_mask(W.scaled(cfg, H=1), seed=40 + h, density=0.05 + 0.07 * h)[0]
    rp, _ = B.chorus_mask_to_index(dmask(bm[None]), cfg.nk)
    cost = B.chorus_head_costs(rp, cfg.H, cfg.nq)
    torch.cuda.synchronize()
    want = W.unpack_bits(bm, cfg.nk).reshape(cfg.H, -1).sum(axis=1)
    assert np.array_equal(cost.cpu().numpy(), want)
    order, load = B.chorus_schedule_heads(cost.cpu(), 3)
    mine, load_o = oracle.schedule_heads(want, 3)
    assert [[h for h in r.tolist() if h >= 0] for r in order] == mine and load.tolist() == load_o
