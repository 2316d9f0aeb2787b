"""GPU parity of the full mask-reuse step (BASELINE.json configs[4]) at the 480p shape:
retrieve the stored mask set of the most similar request -> visit refresh -> decode the whole
40 x 40 set -> block-sparse attention of selected layers, every stage against the oracle.

The bank has the stated size: 1024 unit-norm 4096-d embeddings and 1024 full-size mask sets (40 layers x 40 heads
x 256 x 512 blocks each, 26.8 GB on the device, drawn there in chunks).  Decoy entries are unstructured ~25 %
Bernoulli rows; the target entry carries structured masks at 10-40 % density in the layers whose attention is
checked (layer 0 and the last layer of every 8-layer group, i.e. every layer the visit refresh changes) and seeded
unstructured rows elsewhere.  On a device with less than 48 GB free the mask bank shrinks to
64 sets (entry e lives in slot e mod 64); the embedding bank keeps its 1024 entries."""
import numpy as np
import pytest
import torch

import oracle
from gpu_common import (BF16_MAX, BF16_MAX_TIGHT, BF16_MEAN, BF16_RELFRO, dbf16, dev, err_stats,
                        gather_items, oracle_items, sample_items)
from paper_2606_25040_b200 import binding as B
from paper_2606_25040_b200 import workloads as W

pytestmark = pytest.mark.gpu

ENTRIES, TARGET = 1024, 617
STRUCTURED_LAYERS = (0, 7, 15, 23, 31, 39)      # 8g + 7 = last layer of group g: changed by the refresh


def _target_set(bcfg):
    a = bcfg.attn
    rho = W.bank_entry_densities(bcfg, TARGET)
    out = np.zeros((bcfg.layers, a.H, a.nq, a.words), dtype=np.uint32)
    for l in range(bcfg.layers):
        if l in STRUCTURED_LAYERS:
            for h in range(a.H):
                keep = W.head_mask(a.nq, a.nk, a.tokens_per_frame, float(rho[l, h]),
                                   bcfg.bank_seed * 1_000_003 + TARGET * 4099 + l * 64 + h, a.band)
                out[l, h] = W.pack_bits(keep)
        else:
            out[l] = W.hash_fill_masks(a.H * a.nq, a.words, a.nk, float(rho[l].mean()),
                                       seed=9000 + l).reshape(a.H, a.nq, a.words)
    return out


def test_reuse_step_480p():
    bcfg = W.BankConfig(entries=ENTRIES)
    a = bcfg.attn
    d = dev()
    # ---- the bank on the device: embeddings + mask sets --------------------------------------
    emb = W.embeddings(bcfg)
    demb = torch.from_numpy(emb).to(d)
    g = torch.Generator(device=d)
    g.manual_seed(11)
    set_shape = (bcfg.layers, a.H, a.nq, a.words)
    slots = ENTRIES if torch.cuda.mem_get_info(d)[0] >= 48 << 30 else 64
    bank = torch.empty((slots, *set_shape), dtype=torch.int32, device=d)
    for c in range(0, slots, 32):                       # 32 sets = 0.84 GB per draw
        n = min(32, slots - c)
        bank[c:c + n] = torch.randint(-2 ** 31, 2 ** 31 - 1, (n, *set_shape), dtype=torch.int32, device=d, generator=g)
        bank[c:c + n] &= torch.randint(-2 ** 31, 2 ** 31 - 1, (n, *set_shape), dtype=torch.int32, device=d, generator=g)  # ~25 %
    target = _target_set(bcfg)
    bank[TARGET % slots] = torch.from_numpy(target.view(np.int32)).to(d)
    print(f"mask bank: {slots} sets, {bank.numel() * 4 / 2 ** 30:.1f} GiB on the device")

    # ---- a-0 retrieve: hit on the planted entry, miss for an unrelated request ---------------
    q_hit = W.query_embedding(bcfg, emb, TARGET)
    idx, sim, hit = B.chorus_retrieve_top1(demb, torch.from_numpy(q_hit).to(d), bcfg.tau)
    ref_idx, ref_sim, ref_hit = oracle.retrieve_top1(emb, q_hit, bcfg.tau)
    assert (idx.item(), bool(hit.item())) == (ref_idx, ref_hit) == (TARGET, True)
    assert abs(sim.item() - ref_sim) <= 1e-5
    q_miss = W.query_embedding(bcfg, emb, None)
    _, _, hit2 = B.chorus_retrieve_top1(demb, torch.from_numpy(q_miss).to(d), bcfg.tau)
    assert not bool(hit2.item()) and not oracle.retrieve_top1(emb, q_miss, bcfg.tau)[2]

    # ---- f-1 visit refresh + a-1 decode of the whole selected set, bit-exact ------------------
    sel = bank[idx.item() % slots].clone()             # the request works on its own copy
    B.chorus_visit_refresh(sel, a.nk, group=8)
    refreshed = oracle.visit_refresh(target, a.nk, group=8)
    assert np.array_equal(sel.cpu().numpy().view(np.uint32), refreshed)
    rp, ci = B.chorus_mask_to_index(sel, a.nk)
    torch.cuda.synchronize()
    rp_o, ci_o = oracle.mask_to_index(refreshed, a.nk)
    assert np.array_equal(rp.cpu().numpy(), rp_o)
    assert np.array_equal(ci.cpu().numpy()[: len(ci_o)], ci_o)

    del bank
    # ---- a-2 attention of layer 0 and of every refreshed layer, from slices of the set's CSR ----
    Q, K, V = W.qkv_bits(a)
    tq, tk, tv = dbf16(Q), dbf16(K), dbf16(V)
    rows = a.H * a.nq
    for l in STRUCTURED_LAYERS:
        O = B.chorus_block_sparse_attn_fwd(tq, tk, tv, rp[l * rows: (l + 1) * rows + 1], ci, a.scale)
        torch.cuda.synchronize()
        O = O.float().cpu().numpy().astype(np.float64)
        items = sample_items(a.H, a.nq, 6, seed=50 + l, always=[(0, a.H - 1, a.nq - 1)])
        ref = oracle_items(Q, K, V, refreshed[l], a.scale, items)
        mx, mean, relfro, _ = err_stats(gather_items(O, items, a.N), ref)
        assert mx <= BF16_MAX and mean <= BF16_MEAN, (l, mx, mean)
        assert mx <= BF16_MAX_TIGHT and relfro <= BF16_RELFRO, (l, mx, relfro)
