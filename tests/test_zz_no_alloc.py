"""chorus_mask_to_index_static: the mask decode with its scratch in a fixed device array of the library (no
workspace, no allocation inside the call; include/chorus.h).  Checked bit for bit (the decode's result is unique,
so the tolerance of the decode tests is exact equality) against the existing path, chorus_mask_to_index, on two calls
in a row: the array keeps the first call's status words, which the second call has to clear.

Collected last on purpose (pytest -x): a failure here hides nothing behind it."""
import numpy as np
import pytest
import torch

from gpu_common import dev, dmask
from paper_2606_25040_b200 import binding as B
from paper_2606_25040_b200 import workloads as W

pytestmark = pytest.mark.gpu


def random_mask(L, H, nq, nk, rho, seed):
    g = np.random.default_rng(seed)
    bm = W.pack_bits(g.random((L, H, nq, nk)) < rho)
    if nk % 32:                          # garbage in the pad bits of every row's last word
        bm[..., -1] |= np.uint32((0xFFFFFFFF << (nk % 32)) & 0xFFFFFFFF)
    return bm


def existing_path(bm, nk):
    rp, ci = B.chorus_mask_to_index(dmask(bm), nk)
    torch.cuda.synchronize()
    return rp, ci


def static_path(bm, nk, nnz):
    L, H, nq, _ = bm.shape
    rp = torch.full((L * H * nq + 1,), -7, dtype=torch.int32, device=dev())
    ci = torch.full((max(nnz, 1),), -7, dtype=torch.int32, device=dev())
    B.chorus_mask_to_index_static(dmask(bm), nk, rp, ci)
    torch.cuda.synchronize()
    return rp, ci


def test_static_decode_matches_the_workspace_path_on_two_calls_in_a_row():
    # first a mask of many tiles (2 x 3 x 300 rows x 17 words = 30 600 words = 120 tiles of 256 words), then a
    # smaller one with another density: the second call finds the first call's status words in the scratch array
    cases = [((2, 3, 300, 520, 0.25), 11), ((1, 2, 130, 70, 0.6), 12)]
    for (L, H, nq, nk, rho), seed in cases:
        bm = random_mask(L, H, nq, nk, rho, seed)
        rp_ref, ci_ref = existing_path(bm, nk)
        nnz = int(rp_ref[-1].item())
        rp, ci = static_path(bm, nk, nnz)
        assert torch.equal(rp, rp_ref)
        assert torch.equal(ci[:nnz], ci_ref[:nnz])
    # and the first mask once more, after the smaller one
    (L, H, nq, nk, rho), seed = cases[0]
    bm = random_mask(L, H, nq, nk, rho, seed)
    rp_ref, ci_ref = existing_path(bm, nk)
    nnz = int(rp_ref[-1].item())
    rp, ci = static_path(bm, nk, nnz)
    assert torch.equal(rp, rp_ref) and torch.equal(ci[:nnz], ci_ref[:nnz])


def test_static_decode_same_mask_twice_and_count_only():
    cfg = W.CFG1
    bm = W.layer_mask(cfg)[None]
    rp_ref, ci_ref = existing_path(bm, cfg.nk)
    nnz = int(rp_ref[-1].item())
    for _ in range(2):
        rp, ci = static_path(bm, cfg.nk, nnz)
        assert torch.equal(rp, rp_ref) and torch.equal(ci[:nnz], ci_ref[:nnz])
    rp = torch.empty_like(rp_ref)
    B.chorus_mask_to_index_static(dmask(bm), cfg.nk, rp)          # col_idx = NULL: counts only
    torch.cuda.synchronize()
    assert torch.equal(rp, rp_ref)


def test_static_decode_rejects_masks_beyond_its_scratch():
    # 20 000 rows x 1024 words = 20.5 M words > 2^24: refused before anything is launched (the tensors are dummies)
    tiny = torch.zeros(4, dtype=torch.int32, device=dev())
    with pytest.raises(B.ChorusError) as e:
        B._check(B.lib().chorus_mask_to_index_static(B._ptr(tiny), 1, 1, 20000, 32768, B._ptr(tiny), None, 0, None))
    assert "static scratch" in str(e.value) and f"status {B.CHORUS_ERR_CAPACITY}" in str(e.value)
    # the largest size it takes is accepted as a size (2^24 words; not run: 64 MiB of mask)
    assert B.STATIC_DECODE_MAX_WORDS == 1 << 24
