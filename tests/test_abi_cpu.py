"""CPU-only checks of the C-ABI library: it loads, exports every symbol include/chorus.h declares,
and rejects bad arguments on the host before anything is launched (no compute calls here)."""
import ctypes as C
import os
import re

import pytest

from paper_2606_25040_b200 import binding as B
from paper_2606_25040_b200 import build as libbuild

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    libbuild.build()
    return B.lib()


def test_exports_every_declared_symbol(lib):
    header = open(os.path.join(ROOT, "include", "chorus.h")).read()
    declared = set(re.findall(r"\b(chorus_[a-z0-9_]+)\s*\(", header))
    declared -= {"chorus_status", "chorus_dtype"}
    assert set(B.EXPORTS) == declared, (sorted(declared), sorted(B.EXPORTS))
    for name in declared:
        assert hasattr(lib, name), name
    assert "sm_100a" in B.chorus_version()


def test_workspace_queries_need_no_gpu(lib):
    assert B.mask_to_index_workspace_bytes(40, 40, 256, 512) > 0
    assert B.retrieve_workspace_bytes(1024, 4096) == 4096


def test_argument_validation_on_host(lib):
    n = C.c_size_t(0)
    st = lib.chorus_mask_to_index(None, 0, 1, 1, 1, None, None, 0, None, C.byref(n), None)
    assert st == B.CHORUS_ERR_INVALID_ARG and b"positive" in lib.chorus_last_error()
    st = lib.chorus_mask_to_index(None, 40, 40, 591, 1182 * 4, None, None, 0, None, C.byref(n), None)
    assert st == B.CHORUS_ERR_CAPACITY
    st = lib.chorus_mask_to_index(None, 1, 1, 1, 1, None, None, 0, None, None, None)
    assert st == B.CHORUS_ERR_INVALID_ARG
    # attention: head_dim != 128 is UNSUPPORTED, null pointers INVALID_ARG, fp8 mismatch INVALID_ARG
    shp = B.AttnShape(B=1, H=1, N=128, d=64)
    fake = C.c_void_p(4096)
    st = lib.chorus_block_sparse_attn_fwd(fake, fake, fake, fake, fake, C.c_float(1.0), B.CHORUS_BF16,
                                          fake, C.byref(shp), None, None)
    assert st == B.CHORUS_ERR_UNSUPPORTED
    st = lib.chorus_block_sparse_attn_fwd(None, fake, fake, fake, fake, C.c_float(1.0), B.CHORUS_BF16,
                                          fake, C.byref(shp), None, None)
    assert st == B.CHORUS_ERR_INVALID_ARG
    st = lib.chorus_block_sparse_attn_fwd(fake, fake, fake, fake, fake, C.c_float(1.0),
                                          B.CHORUS_FP8_E4M3, fake, C.byref(shp), None, None)
    assert st == B.CHORUS_ERR_INVALID_ARG
    st = lib.chorus_block_sparse_attn_fwd(C.c_void_p(4100), fake, fake, fake, fake, C.c_float(1.0),
                                          B.CHORUS_BF16, fake, C.byref(shp), None, None)
    assert st == B.CHORUS_ERR_INVALID_ARG and b"aligned" in lib.chorus_last_error()
    st = lib.chorus_block_sparse_attn_fwd(fake, fake, fake, fake, fake, C.c_float(1.0), 7, fake,
                                          C.byref(shp), None, None)
    assert st == B.CHORUS_ERR_UNSUPPORTED
    shp = B.AttnShape(B=1, H=2, N=128, d=128, q_stride_n=257, q_stride_h=128)
    st = lib.chorus_block_sparse_attn_fwd(fake, fake, fake, fake, fake, C.c_float(1.0), B.CHORUS_BF16,
                                          fake, C.byref(shp), None, None)
    assert st == B.CHORUS_ERR_INVALID_ARG and b"stride" in lib.chorus_last_error()
    st = lib.chorus_retrieve_top1(None, 10, 6, None, C.c_float(0.4), None, None, None, None,
                                  C.byref(n), None)
    assert st == B.CHORUS_ERR_INVALID_ARG
    st = lib.chorus_visit_refresh(None, 8, 1, 1, 1, 8, None)
    assert st == B.CHORUS_ERR_INVALID_ARG
    # mask construction, LSE variant, head scheduling
    shp = B.AttnShape(B=1, H=1, N=128, d=128)
    assert lib.chorus_block_mass(None, fake, C.c_float(1.0), C.byref(shp), None, fake, None) == B.CHORUS_ERR_INVALID_ARG
    shp64 = B.AttnShape(B=1, H=1, N=128, d=64)
    assert lib.chorus_block_mass(fake, fake, C.c_float(1.0), C.byref(shp64), None, fake, None) == B.CHORUS_ERR_UNSUPPORTED
    assert lib.chorus_mask_from_mass(fake, 4, 4096, C.c_double(0.9), C.c_double(0.1), fake, None, None) == B.CHORUS_ERR_UNSUPPORTED
    assert lib.chorus_mask_from_mass(fake, 4, 64, C.c_double(1.5), C.c_double(0.1), fake, None, None) == B.CHORUS_ERR_INVALID_ARG
    assert lib.chorus_mask_from_mass(fake, 0, 64, C.c_double(0.9), C.c_double(0.1), fake, None, None) == B.CHORUS_ERR_INVALID_ARG
    assert lib.chorus_mask_from_mass(None, 4, 64, C.c_double(0.9), C.c_double(0.1), fake, None, None) == B.CHORUS_ERR_INVALID_ARG
    assert lib.chorus_mask_coverage(fake, fake, 0, 1, 1, fake, None) == B.CHORUS_ERR_INVALID_ARG
    assert lib.chorus_head_costs(None, 4, 4, fake, None) == B.CHORUS_ERR_INVALID_ARG
    assert lib.chorus_schedule_heads(None, 4, 2, fake, None) == B.CHORUS_ERR_INVALID_ARG
    st = lib.chorus_block_sparse_attn_fwd_lse(fake, fake, fake, fake, fake, C.c_float(1.0), B.CHORUS_FP16,
                                              fake, C.byref(shp64), None, fake, None)
    assert st == B.CHORUS_ERR_UNSUPPORTED          # FP16 is a known dtype; d = 64 is what is refused
    assert b"head_dim" in lib.chorus_last_error()
    # scale must be positive and finite (the row maximum is taken on the raw scores)
    for bad in (0.0, -0.088, float("nan"), float("inf")):
        st = lib.chorus_block_sparse_attn_fwd(fake, fake, fake, fake, fake, C.c_float(bad), B.CHORUS_BF16,
                                              fake, C.byref(shp), None, None)
        assert st == B.CHORUS_ERR_INVALID_ARG and b"scale" in lib.chorus_last_error(), bad
        assert lib.chorus_block_mass(fake, fake, C.c_float(bad), C.byref(shp), None, fake, None) == B.CHORUS_ERR_INVALID_ARG


def test_product_path_does_not_touch_the_oracle():
    # neither side imports the other; the binding has no CPU fallback
    pkg = os.path.join(ROOT, "paper_2606_25040_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", src, re.M), f
                assert "chorus_oracle" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(import|from)\s+paper_2606_25040_b200", src, re.M), f
            for inc in re.findall(r'#include\s+"([^"]+)"', src):
                assert "csrc" not in inc and "chorus.h" not in inc, (f, inc)
