"""Generator determinism and structure."""
import numpy as np

from paper_2606_25040_b200 import workloads as W


def test_shapes_match_baseline_configs():
    assert (W.CFG1.N, W.CFG1.nq, W.CFG1.nk) == (4096, 32, 64)
    assert (W.CFG2.N, W.CFG2.nq, W.CFG2.nk, W.CFG2.words) == (32760, 256, 512, 16)
    assert (W.CFG4.N, W.CFG4.nq, W.CFG4.nk, W.CFG4.words) == (75600, 591, 1182, 37)
    assert W.CFG2.N % 128 == 120 and W.CFG2.N % 64 == 56 and W.CFG4.N % 128 == 80 and W.CFG4.N % 64 == 16


def test_bf16_round_trip_and_rne():
    x = np.array([1.0, 1.00390625, 1.01171875, -2.5, 0.0, 3.0e38], np.float32)
    b = W.bf16_bits_from_f32(x)
    import torch
    ref = torch.from_numpy(x).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
    assert np.array_equal(b, ref)
    g = np.random.default_rng(0).standard_normal(10000).astype(np.float32)
    ref = torch.from_numpy(g).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
    assert np.array_equal(W.bf16_bits_from_f32(g), ref)


def test_masks_deterministic_exact_density_and_structure():
    for cfg, per_row in ((W.CFG1, 32), (W.scaled(W.CFG2, H=3), 128), (W.scaled(W.CFG4, H=2), 177)):
        m1, m2 = W.layer_mask(cfg), W.layer_mask(cfg)
        assert np.array_equal(m1, m2)
        keep = W.unpack_bits(m1, cfg.nk)
        assert np.all(keep.sum(-1) == per_row)
        n_f0 = (cfg.tokens_per_frame + 63) // 64
        assert keep[:, :, :n_f0].all()                       # all frame-0 key blocks kept
        qb = np.arange(cfg.nq)
        for off in (0, 1):
            ok = 2 * qb + off < cfg.nk
            assert keep[:, qb[ok], 2 * qb[ok] + off].all()   # diagonal => >= 1 block per row
        assert not np.array_equal(keep[0], keep[1])          # pattern differs across heads
    keep1 = W.unpack_bits(W.layer_mask(W.CFG1), W.CFG1.nk)
    for q in range(W.CFG1.nq):                               # cfg1: whole width-8 band kept
        lo, hi = max(0, 2 * q - 3), min(W.CFG1.nk - 1, 2 * q + 4)
        assert keep1[:, q, lo:hi + 1].all()


def test_density_sweep_and_full():
    cfg = W.scaled(W.CFG2, H=1)
    for rho in (0.05, 0.10, 0.50):
        keep = W.unpack_bits(W.layer_mask(cfg, density=rho), cfg.nk)
        assert abs(keep.mean() - rho) < 2e-3 and keep.sum(-1).min() >= 2
    assert W.unpack_bits(W.layer_mask(cfg, density=1.0), cfg.nk).all()


def test_qkv_deterministic_and_stress_rows():
    a = W.qkv_bits(W.CFG1)
    b = W.qkv_bits(W.CFG1)
    assert all(np.array_equal(x, y) for x, y in zip(a, b))
    assert not np.array_equal(a[0], a[1])
    cfg = W.scaled(W.CFG4, H=2, frames=1)
    q, _, _ = W.qkv_bits(cfg)
    rms = np.sqrt((W.f32_from_bf16_bits(q).astype(np.float64) ** 2).mean(-1))
    frac = (rms > 4).mean()
    assert 0.004 < frac < 0.02
