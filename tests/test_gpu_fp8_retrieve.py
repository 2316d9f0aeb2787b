"""GPU parity: chorus_quantize_fp8 (bit-exact codes and scales) and chorus_retrieve_top1."""
import numpy as np
import pytest
import torch

import oracle
from gpu_common import dbf16, dev
from paper_2606_25040_b200 import binding as B
from paper_2606_25040_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("hp,wp,H", [(10, 33, 3), (16, 64, 2), (1, 100, 1)])
def test_quantize_bit_exact(hp, wp, H):
    cfg = W.AttnConfig("q", H=H, frames=1, hp=hp, wp=wp, density=0.5, data_seed=3, mask_seed=1,
                       stress_rows=0.01)
    Q, K, V = W.qkv_bits(cfg)
    ref = oracle.quantize_fp8(Q, K, V)
    got = B.chorus_quantize_fp8(dbf16(Q), dbf16(K), dbf16(V))
    torch.cuda.synchronize()
    for name, a, b in zip(("q8", "k8", "v8", "q_scale", "k_scale", "v_scale"), got, ref):
        assert np.array_equal(a.cpu().numpy(), b), name


def test_quantize_all_zero_block():
    cfg = W.AttnConfig("z", H=1, frames=1, hp=4, wp=64, density=0.5, data_seed=3, mask_seed=1)
    Q, K, V = W.qkv_bits(cfg)
    Q[0, :128] = 0
    ref = oracle.quantize_fp8(Q, K, V)
    got = B.chorus_quantize_fp8(dbf16(Q), dbf16(K), dbf16(V))
    torch.cuda.synchronize()
    assert np.array_equal(got[0].cpu().numpy(), ref[0]) and np.array_equal(got[3].cpu().numpy(), ref[3])


def test_retrieve_top1_hit_and_miss():
    cfg = W.CFG5
    bank = W.embeddings(cfg)
    dbank = torch.from_numpy(bank).to(dev())
    for target in (0, 517, 1023, None):
        q = W.query_embedding(cfg, bank, target)
        idx, sim, hit = B.chorus_retrieve_top1(dbank, torch.from_numpy(q).to(dev()), cfg.tau)
        torch.cuda.synchronize()
        o_idx, o_sim, o_hit = oracle.retrieve_top1(bank, q, cfg.tau)
        assert idx.item() == o_idx and bool(hit.item()) == o_hit
        assert abs(sim.item() - o_sim) <= 1e-5
        if target is not None:
            assert o_idx == target and o_hit


def test_retrieve_ties_lowest_index():
    cfg = W.BankConfig(entries=300, dim=512)
    bank = W.embeddings(cfg)
    bank[200] = bank[7]
    bank[100] = bank[7]
    idx, sim, hit = B.chorus_retrieve_top1(torch.from_numpy(bank).to(dev()),
                                           torch.from_numpy(bank[7].copy()).to(dev()), 0.4)
    torch.cuda.synchronize()
    assert idx.item() == 7 and hit.item() == 1
