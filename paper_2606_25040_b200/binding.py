"""ctypes binding over libchorus.so — same names as include/chorus.h, argument marshalling only.

Every step of the path runs in the library's CUDA kernels; torch is used for device memory and the
current stream.  There is no CPU fallback: if the library is missing or a call fails, a
ChorusError is raised.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libchorus.so")

CHORUS_OK, CHORUS_ERR_INVALID_ARG, CHORUS_ERR_UNSUPPORTED, CHORUS_ERR_CAPACITY, CHORUS_ERR_CUDA = range(5)
CHORUS_BF16, CHORUS_FP8_E4M3, CHORUS_FP16 = 0, 1, 2
BLOCK_Q, BLOCK_K, HEAD_DIM = 128, 64, 128

EXPORTS = ["chorus_mask_to_index", "chorus_visit_refresh", "chorus_block_sparse_attn_fwd",
           "chorus_block_sparse_attn_fwd_lse", "chorus_block_sparse_attn_fwd_first_frame",
           "chorus_mask_to_index_64x128", "chorus_block_sparse_attn_fwd_64x128", "chorus_block_mass_64x128",
           "chorus_mask_to_index_u16", "chorus_mask_to_index_64x128_u16", "chorus_block_sparse_attn_fwd_idx16",
           "chorus_mask_to_index_static",
           "chorus_quantize_fp8", "chorus_retrieve_top1", "chorus_block_mass",
           "chorus_mask_from_mass", "chorus_mask_coverage", "chorus_head_costs", "chorus_schedule_heads", "chorus_gather_heads", "chorus_scatter_heads", "chorus_last_error", "chorus_version",
           "chorus_launch_count", "chorus_reset_launch_count", "chorus_tensor_map_encodes"]


class ChorusError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"libchorus status {status}: {msg}")
        self.status = status


class AttnShape(C.Structure):
    _fields_ = [("B", C.c_int), ("H", C.c_int), ("N", C.c_int), ("d", C.c_int)] + [
        (f"{t}_stride_{a}", C.c_int64) for t in "qkvo" for a in "bnh"]


class Fp8Scales(C.Structure):
    _fields_ = [("q_scale", C.c_void_p), ("k_scale", C.c_void_p), ("v_scale", C.c_void_p)]


_lib = None


def lib() -> C.CDLL:
    """Load libchorus.so (built in-tree by `python -m paper_2606_25040_b200.build`)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ChorusError(CHORUS_ERR_CUDA, f"{LIB_PATH} not found: build it with "
                              "`python -m paper_2606_25040_b200.build` (there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        L.chorus_last_error.restype = C.c_char_p
        L.chorus_version.restype = C.c_char_p
        L.chorus_launch_count.restype = C.c_int64
        L.chorus_tensor_map_encodes.restype = C.c_int64
        L.chorus_mask_to_index.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_void_p,
                                           C.c_void_p, C.c_int64, C.c_void_p,
                                           C.POINTER(C.c_size_t), C.c_void_p]
        L.chorus_visit_refresh.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int,
                                           C.c_void_p]
        L.chorus_block_sparse_attn_fwd.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                                   C.c_void_p, C.c_float, C.c_int, C.c_void_p,
                                                   C.POINTER(AttnShape), C.POINTER(Fp8Scales),
                                                   C.c_void_p]
        L.chorus_quantize_fp8.argtypes = [C.c_void_p] * 3 + [C.POINTER(AttnShape)] + [C.c_void_p] * 7
        L.chorus_retrieve_top1.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_float,
                                           C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                           C.POINTER(C.c_size_t), C.c_void_p]
        L.chorus_block_mass.argtypes = [C.c_void_p, C.c_void_p, C.c_float, C.POINTER(AttnShape),
                                        C.c_void_p, C.c_void_p, C.c_void_p]
        L.chorus_block_mass_64x128.argtypes = L.chorus_block_mass.argtypes
        L.chorus_block_sparse_attn_fwd_lse.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                                       C.c_void_p, C.c_float, C.c_int, C.c_void_p,
                                                       C.POINTER(AttnShape), C.POINTER(Fp8Scales),
                                                       C.c_void_p, C.c_void_p]
        L.chorus_block_sparse_attn_fwd_first_frame.argtypes = (
            L.chorus_block_sparse_attn_fwd_lse.argtypes[:-1] + [C.c_int, C.c_float, C.c_void_p])
        L.chorus_block_sparse_attn_fwd_64x128.argtypes = L.chorus_block_sparse_attn_fwd_first_frame.argtypes
        L.chorus_mask_to_index_64x128.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_void_p, C.c_void_p,
                                                  C.c_int64, C.c_void_p, C.POINTER(C.c_size_t), C.c_void_p]
        L.chorus_mask_to_index_u16.argtypes = L.chorus_mask_to_index.argtypes
        L.chorus_mask_to_index_static.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_void_p,
                                                  C.c_void_p, C.c_int64, C.c_void_p]
        L.chorus_mask_to_index_64x128_u16.argtypes = L.chorus_mask_to_index_64x128.argtypes
        L.chorus_block_sparse_attn_fwd_idx16.argtypes = (
            L.chorus_block_sparse_attn_fwd_first_frame.argtypes[:-1] + [C.c_int, C.c_void_p])
        L.chorus_mask_from_mass.argtypes = [C.c_void_p, C.c_int64, C.c_int, C.c_double, C.c_double,
                                            C.c_void_p, C.c_void_p, C.c_void_p]
        L.chorus_mask_coverage.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_int,
                                           C.c_void_p, C.c_void_p]
        L.chorus_gather_heads.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int64, C.c_int64,
                                          C.c_void_p, C.c_int, C.c_void_p, C.c_void_p]
        L.chorus_scatter_heads.argtypes = L.chorus_gather_heads.argtypes
        L.chorus_head_costs.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_void_p]
        L.chorus_schedule_heads.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_void_p]
        _lib = L
    return _lib


def _check(status: int):
    if status != CHORUS_OK:
        raise ChorusError(status, lib().chorus_last_error().decode())


def _stream(stream=None):
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def _ptr(t):
    return C.c_void_p(0 if t is None else t.data_ptr())


def chorus_version() -> str:
    return lib().chorus_version().decode()


def chorus_launch_count() -> int:
    return int(lib().chorus_launch_count())


def chorus_tensor_map_encodes() -> int:
    return int(lib().chorus_tensor_map_encodes())


def chorus_reset_launch_count() -> None:
    lib().chorus_reset_launch_count()


def mask_to_index_workspace_bytes(L: int, H: int, nq_blk: int, nk_blk: int) -> int:
    n = C.c_size_t(0)
    _check(lib().chorus_mask_to_index(None, L, H, nq_blk, nk_blk, None, None, 0, None, C.byref(n), None))
    return int(n.value)


def chorus_mask_to_index(bitmask, nk_blk: int, row_ptr=None, col_idx=None, workspace=None,
                         stream=None, count_only=False, idx16=False):
    """bitmask: cuda int32/uint32-bits tensor [L][H][nq][words].  Returns (row_ptr, col_idx).
    idx16 (or a 2-byte col_idx tensor): 16-bit entries (chorus_mask_to_index_u16).

    If col_idx is not given: count-only pass, one 4-byte read of nnz, allocation, second pass
    (the protocol include/chorus.h describes)."""
    L, H, nq, words = bitmask.shape
    assert bitmask.is_cuda and bitmask.is_contiguous() and bitmask.element_size() == 4
    assert words == (nk_blk + 31) // 32
    rows = L * H * nq
    dev = bitmask.device
    if row_ptr is None:
        row_ptr = torch.empty(rows + 1, dtype=torch.int32, device=dev)
    if workspace is None:
        workspace = torch.empty(max(mask_to_index_workspace_bytes(L, H, nq, nk_blk), 4),
                                dtype=torch.uint8, device=dev)
    wsb = C.c_size_t(workspace.numel())
    idx16 = idx16 or (col_idx is not None and col_idx.element_size() == 2)
    fn = lib().chorus_mask_to_index_u16 if idx16 else lib().chorus_mask_to_index
    if col_idx is None:
        _check(fn(_ptr(bitmask), L, H, nq, nk_blk, _ptr(row_ptr), None, 0,
                  _ptr(workspace), C.byref(wsb), _stream(stream)))
        if count_only:
            return row_ptr, None
        nnz = int(row_ptr[-1].item())
        col_idx = torch.empty(max(nnz, 1), dtype=torch.uint16 if idx16 else torch.int32, device=dev)
    assert col_idx.element_size() == (2 if idx16 else 4)
    _check(fn(_ptr(bitmask), L, H, nq, nk_blk, _ptr(row_ptr), _ptr(col_idx),
              col_idx.numel(), _ptr(workspace), C.byref(wsb), _stream(stream)))
    return row_ptr, col_idx


STATIC_DECODE_MAX_WORDS = 1 << 24


def chorus_mask_to_index_static(bitmask, nk_blk: int, row_ptr, col_idx=None, stream=None):
    """chorus_mask_to_index without a workspace and without any allocation inside the call (the kernel's scratch
    is a fixed device array of the library; at most STATIC_DECODE_MAX_WORDS mask words; calls that overlap on the
    GPU race).  row_ptr (and col_idx, unless only the counts are wanted) are the caller's tensors."""
    L, H, nq, words = bitmask.shape
    assert bitmask.is_cuda and bitmask.is_contiguous() and bitmask.element_size() == 4
    assert words == (nk_blk + 31) // 32
    assert row_ptr.is_cuda and row_ptr.dtype == torch.int32 and row_ptr.numel() >= L * H * nq + 1
    assert col_idx is None or (col_idx.is_cuda and col_idx.dtype == torch.int32)
    _check(lib().chorus_mask_to_index_static(_ptr(bitmask), L, H, nq, nk_blk, _ptr(row_ptr),
                                             None if col_idx is None else _ptr(col_idx),
                                             0 if col_idx is None else col_idx.numel(), _stream(stream)))
    return row_ptr, col_idx


def chorus_mask_to_index_64x128(bitmask, N: int, row_ptr=None, col_idx=None, workspace=None, stream=None,
                                count_only=False, idx16=False):
    """bitmask: cuda 4-byte tensor [L][H][ceil(N/64)][words] in the paper's 64 x 128 geometry.  Returns
    (row_ptr [L*H*ceil(N/128)+1], col_idx with the per-half flag bits) for chorus_block_sparse_attn_fwd(...,
    geometry_64x128=True).  Same two-pass protocol as chorus_mask_to_index."""
    L, H, nq64, words = bitmask.shape
    assert bitmask.is_cuda and bitmask.is_contiguous() and bitmask.element_size() == 4
    assert nq64 == (N + 63) // 64 and words == ((N + 127) // 128 + 31) // 32
    dev = bitmask.device
    if row_ptr is None:
        row_ptr = torch.empty(L * H * ((N + 127) // 128) + 1, dtype=torch.int32, device=dev)
    if workspace is None:
        need = C.c_size_t(0)
        _check(lib().chorus_mask_to_index_64x128(None, L, H, N, None, None, 0, None, C.byref(need), None))
        workspace = torch.empty(max(need.value, 16), dtype=torch.uint8, device=dev)
    wsb = C.c_size_t(workspace.numel())
    idx16 = idx16 or (col_idx is not None and col_idx.element_size() == 2)
    fn = lib().chorus_mask_to_index_64x128_u16 if idx16 else lib().chorus_mask_to_index_64x128
    if col_idx is None:
        _check(fn(_ptr(bitmask), L, H, N, _ptr(row_ptr), None, 0, _ptr(workspace), C.byref(wsb), _stream(stream)))
        if count_only:
            return row_ptr, None
        col_idx = torch.empty(max(int(row_ptr[-1].item()), 1), dtype=torch.uint16 if idx16 else torch.int32, device=dev)
    assert col_idx.element_size() == (2 if idx16 else 4)
    _check(fn(_ptr(bitmask), L, H, N, _ptr(row_ptr), _ptr(col_idx),
              col_idx.numel(), _ptr(workspace), C.byref(wsb), _stream(stream)))
    return row_ptr, col_idx


def chorus_visit_refresh(bitmask, nk_blk: int, group: int = 8, stream=None):
    L, H, nq, words = bitmask.shape
    assert bitmask.is_cuda and bitmask.is_contiguous() and bitmask.element_size() == 4
    _check(lib().chorus_visit_refresh(_ptr(bitmask), L, H, nq, nk_blk, group, _stream(stream)))
    return bitmask


def attn_shape(Q, K, V, O=None) -> AttnShape:
    B, N, H, d = Q.shape
    s = AttnShape(B=B, H=H, N=N, d=d)
    for name, t in (("q", Q), ("k", K), ("v", V), ("o", O)):
        if t is None:
            continue
        assert t.stride(3) == 1, "last dimension must be contiguous"
        setattr(s, f"{name}_stride_b", t.stride(0))
        setattr(s, f"{name}_stride_n", t.stride(1))
        setattr(s, f"{name}_stride_h", t.stride(2))
    return s


def chorus_block_sparse_attn_fwd(Q, K, V, row_ptr, col_idx, scale: float, dtype: int = CHORUS_BF16,
                                 O=None, fp8_scales=None, stream=None, lse=None, n_first=0, beta=1.0,
                                 geometry_64x128=False):
    """Q, K, V: cuda tensors indexed [B][N][H][d] (bf16, or uint8/float8_e4m3fn codes for FP8).
    row_ptr: this layer's H*nq+1 entries (a view into the full row_ptr is fine).  Returns O (bf16).
    n_first, beta: first-frame key enhancement (chorus_block_sparse_attn_fwd_first_frame).
    geometry_64x128: row_ptr / col_idx come from chorus_mask_to_index_64x128 (chorus_block_sparse_attn_fwd_64x128)."""
    assert Q.is_cuda and K.is_cuda and V.is_cuda
    B, N, H, d = Q.shape
    if Q.dtype == torch.float16:          # the paper's non-quantised path: fp16 in, fp16 out
        dtype = CHORUS_FP16
    if O is None:
        O = torch.empty((B, N, H, d), dtype=torch.float16 if dtype == CHORUS_FP16 else torch.bfloat16,
                        device=Q.device)
    shape = attn_shape(Q, K, V, O)
    sc = None
    if fp8_scales is not None:
        sc = Fp8Scales(*(x.data_ptr() for x in fp8_scales))
    if lse is not None:     # float32 [B][H][N], written by the kernel (natural-log row log-sum-exp)
        assert lse.dtype == torch.float32 and lse.is_contiguous() and lse.shape == (B, H, N)
    if col_idx.element_size() == 2:     # 16-bit index entries (chorus_mask_to_index_u16 / _64x128_u16)
        _check(lib().chorus_block_sparse_attn_fwd_idx16(
            _ptr(Q), _ptr(K), _ptr(V), _ptr(row_ptr), _ptr(col_idx), C.c_float(scale), dtype, _ptr(O),
            C.byref(shape), C.byref(sc) if sc is not None else None,
            _ptr(lse) if lse is not None else None, C.c_int(int(n_first)), C.c_float(float(beta)),
            C.c_int(int(bool(geometry_64x128))), _stream(stream)))
        return O
    if geometry_64x128:
        _check(lib().chorus_block_sparse_attn_fwd_64x128(
            _ptr(Q), _ptr(K), _ptr(V), _ptr(row_ptr), _ptr(col_idx), C.c_float(scale), dtype, _ptr(O),
            C.byref(shape), C.byref(sc) if sc is not None else None,
            _ptr(lse) if lse is not None else None, C.c_int(int(n_first)), C.c_float(float(beta)),
            _stream(stream)))
        return O
    if n_first != 0 or beta != 1.0:
        _check(lib().chorus_block_sparse_attn_fwd_first_frame(
            _ptr(Q), _ptr(K), _ptr(V), _ptr(row_ptr), _ptr(col_idx), C.c_float(scale), dtype, _ptr(O),
            C.byref(shape), C.byref(sc) if sc is not None else None,
            _ptr(lse) if lse is not None else None, C.c_int(int(n_first)), C.c_float(float(beta)),
            _stream(stream)))
        return O
    if lse is not None:
        _check(lib().chorus_block_sparse_attn_fwd_lse(_ptr(Q), _ptr(K), _ptr(V), _ptr(row_ptr), _ptr(col_idx),
                                                      C.c_float(scale), dtype, _ptr(O), C.byref(shape),
                                                      C.byref(sc) if sc is not None else None,
                                                      _ptr(lse), _stream(stream)))
        return O
    _check(lib().chorus_block_sparse_attn_fwd(_ptr(Q), _ptr(K), _ptr(V), _ptr(row_ptr), _ptr(col_idx),
                                              C.c_float(scale), dtype, _ptr(O), C.byref(shape),
                                              C.byref(sc) if sc is not None else None,
                                              _stream(stream)))
    return O


def chorus_quantize_fp8(Q, K, V, out=None, stream=None):
    """bf16 Q/K/V [B][N][H][d] -> (q8, k8, v8 uint8 packed, q_scale, k_scale, v_scale)."""
    B, N, H, d = Q.shape
    dev = Q.device
    nsb = (N + 127) // 128
    if out is None:
        out = tuple(torch.empty((B, N, H, d), dtype=torch.uint8, device=dev) for _ in range(3)) + (
            torch.empty((B, H, nsb), dtype=torch.float32, device=dev),
            torch.empty((B, H, nsb), dtype=torch.float32, device=dev),
            torch.empty((B, H, d), dtype=torch.float32, device=dev))
    shape = attn_shape(Q, K, V)
    _check(lib().chorus_quantize_fp8(_ptr(Q), _ptr(K), _ptr(V), C.byref(shape), *(_ptr(t) for t in out),
                                     _stream(stream)))
    return out


def retrieve_workspace_bytes(n: int, dim: int) -> int:
    b = C.c_size_t(0)
    _check(lib().chorus_retrieve_top1(None, n, dim, None, C.c_float(0), None, None, None, None,
                                      C.byref(b), None))
    return int(b.value)


def chorus_retrieve_top1(bank, query, tau: float, out=None, workspace=None, stream=None):
    """bank float32 [n][dim], query float32 [dim] (cuda).  Returns device tensors
    (best_idx int32[1], best_sim float32[1], hit int32[1]); nothing is synchronised."""
    n, dim = bank.shape
    dev = bank.device
    if out is None:
        out = (torch.empty(1, dtype=torch.int32, device=dev),
               torch.empty(1, dtype=torch.float32, device=dev),
               torch.empty(1, dtype=torch.int32, device=dev))
    if workspace is None:
        workspace = torch.empty(retrieve_workspace_bytes(n, dim), dtype=torch.uint8, device=dev)
    wsb = C.c_size_t(workspace.numel())
    _check(lib().chorus_retrieve_top1(_ptr(bank), n, dim, _ptr(query), C.c_float(tau), _ptr(out[0]),
                                      _ptr(out[1]), _ptr(out[2]), _ptr(workspace), C.byref(wsb),
                                      _stream(stream)))
    return out


def chorus_block_mass(Q, K, scale: float, mass=None, stream=None, lse=None, geometry_64x128=False):
    """bf16 Q, K [B][N][H][d] (cuda) -> float32 mass [B][H][ceil(N/128)][ceil(N/64)] of the dense
    attention; geometry_64x128: [B][H][ceil(N/64)][ceil(N/128)] (chorus_block_mass_64x128)."""
    B, N, H, d = Q.shape
    nq, nk = (N + BLOCK_Q - 1) // BLOCK_Q, (N + BLOCK_K - 1) // BLOCK_K
    if geometry_64x128:
        nq, nk = nk, nq
    if mass is None:
        mass = torch.empty((B, H, nq, nk), dtype=torch.float32, device=Q.device)
    assert mass.shape == (B, H, nq, nk) and mass.is_contiguous() and mass.dtype == torch.float32
    shape = attn_shape(Q, K, K)
    fn = lib().chorus_block_mass_64x128 if geometry_64x128 else lib().chorus_block_mass
    _check(fn(_ptr(Q), _ptr(K), C.c_float(scale), C.byref(shape), _ptr(lse), _ptr(mass), _stream(stream)))
    return mass


def chorus_mask_from_mass(mass, top_p: float, min_top_k: float, bitmask=None, kept=None, stream=None):
    """float32 mass [..., nk] (cuda) -> (bitmask int32-bits [..., ceil(nk/32)], kept int32 [...]):
    top-p with a top-k floor (PAPER.md:L81, L93 (2))."""
    assert mass.is_cuda and mass.is_contiguous() and mass.dtype == torch.float32
    nk = mass.shape[-1]
    rows = mass.numel() // nk
    if bitmask is None:
        bitmask = torch.empty(mass.shape[:-1] + ((nk + 31) // 32,), dtype=torch.int32, device=mass.device)
    if kept is None:
        kept = torch.empty(mass.shape[:-1], dtype=torch.int32, device=mass.device)
    _check(lib().chorus_mask_from_mass(_ptr(mass), rows, nk, C.c_double(top_p), C.c_double(min_top_k),
                                       _ptr(bitmask), _ptr(kept), _stream(stream)))
    return bitmask, kept


def chorus_mask_coverage(mass, bitmask, nk_blk: int, coverage=None, stream=None):
    """mass float32 [heads][nq][nk], bitmask [heads][nq][words] (cuda) -> float32 coverage [heads]."""
    heads, nq, nk = mass.shape
    assert nk == nk_blk and mass.is_contiguous() and bitmask.is_contiguous()
    if coverage is None:
        coverage = torch.empty(heads, dtype=torch.float32, device=mass.device)
    _check(lib().chorus_mask_coverage(_ptr(mass), _ptr(bitmask), heads, nq, nk, _ptr(coverage),
                                      _stream(stream)))
    return coverage


def chorus_head_costs(row_ptr, H: int, nq_blk: int, cost=None, stream=None):
    """Kept tiles per head from this layer's CSR row_ptr (cuda int32) -> int64 [H] (cuda)."""
    if cost is None:
        cost = torch.empty(H, dtype=torch.int64, device=row_ptr.device)
    _check(lib().chorus_head_costs(_ptr(row_ptr), H, nq_blk, _ptr(cost), _stream(stream)))
    return cost


def chorus_schedule_heads(cost, n_ranks: int):
    """Host call (appendix A): cost = int64 [H] (host tensor or sequence).  Returns
    (order int32 [n_ranks][cap], load int64 [n_ranks]); -1 marks unused slots."""
    cost = torch.as_tensor(cost, dtype=torch.int64).contiguous().cpu()
    H = cost.numel()
    cap = (H + n_ranks - 1) // n_ranks
    order = torch.empty((n_ranks, cap), dtype=torch.int32)
    load = torch.empty(n_ranks, dtype=torch.int64)
    _check(lib().chorus_schedule_heads(_ptr(cost), H, n_ranks, _ptr(order), _ptr(load)))
    return order, load


def _host_order(order, H):
    o = torch.as_tensor(order, dtype=torch.int32).reshape(-1).contiguous().cpu()
    assert o.numel() == H, (o.numel(), H)
    return o


def chorus_gather_heads(X, order, n_ranks: int, packed=None, stream=None):
    """X: cuda [n_tokens][H][d] (strided views are fine, last dim contiguous); order: H head indices (host).
    Returns packed [n_ranks][n_tokens][H/n_ranks][d]: chunk p holds the heads order[p*slots:(p+1)*slots]."""
    n, H, d = X.shape
    assert X.is_cuda and X.stride(2) == 1
    if packed is None:
        packed = torch.empty(X.numel(), dtype=X.dtype, device=X.device)
        if n_ranks > 0 and H % n_ranks == 0:          # otherwise the library reports the error
            packed = packed.view(n_ranks, n, H // n_ranks, d)
    assert packed.is_contiguous() and packed.dtype == X.dtype and packed.numel() == X.numel()
    o = _host_order(order, H)
    _check(lib().chorus_gather_heads(_ptr(X), n, H, d, X.element_size(), X.stride(0), X.stride(1), _ptr(o), n_ranks,
                                     _ptr(packed), _stream(stream)))
    return packed


def chorus_scatter_heads(packed, order, X, stream=None):
    """Inverse of chorus_gather_heads: packed [n_ranks][n_tokens][slots][d] -> X [n_tokens][H][d] (written)."""
    n_ranks, n, slots, d = packed.shape
    H = n_ranks * slots
    assert packed.is_cuda and packed.is_contiguous() and X.shape == (n, H, d) and X.stride(2) == 1
    o = _host_order(order, H)
    _check(lib().chorus_scatter_heads(_ptr(packed), n, H, d, X.element_size(), X.stride(0), X.stride(1), _ptr(o),
                                      n_ranks, _ptr(X), _stream(stream)))
    return X
