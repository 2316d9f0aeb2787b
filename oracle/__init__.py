"""CPU oracle for the Chorus II sparsity-reuse hot path — TEST INFRASTRUCTURE, NOT THE PRODUCT.

Thin ctypes binding over ``oracle/chorus_oracle.cpp`` (plain fp64 C++, written from the paper; see
the header of that file for citations and pin status).  Only ``tests/``, ``__graft_entry__.smoke()``
and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import this package.  It imports
nothing from ``paper_2606_25040_b200`` and the CUDA path imports nothing from here.

All arrays are numpy: bf16 tensors travel as ``uint16`` bit patterns, e4m3 tensors as ``uint8`` codes.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from .build import build as _build

BQ, BK = 128, 64
_lib = None


def lib():
    global _lib
    if _lib is None:
        # CHORUS_ORACLE_SANITIZE=1: the ASan + UBSan build (the process must preload libasan; see
        # tests/test_oracle_sanitizers.py)
        _lib = C.CDLL(_build(sanitize=os.environ.get("CHORUS_ORACLE_SANITIZE") == "1"))
        _lib.oracle_mask_to_index.restype = C.c_int64
        _lib.oracle_mask_to_index_64x128.restype = C.c_int64
        _lib.oracle_mask_to_index_u16.restype = C.c_int64
        _lib.oracle_mask_to_index_64x128_u16.restype = C.c_int64
        _lib.oracle_e4m3_to_double.restype = C.c_double
        _lib.oracle_e4m3_to_double.argtypes = [C.c_uint8]
        _lib.oracle_f16_to_double.restype = C.c_double
        _lib.oracle_f16_to_double.argtypes = [C.c_uint16]
        _lib.oracle_float_to_e4m3.restype = C.c_uint8
        _lib.oracle_float_to_e4m3.argtypes = [C.c_float]
        _lib.oracle_num_threads.restype = C.c_int
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _c(a, dtype):
    a = np.ascontiguousarray(a, dtype=dtype)
    return a


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def mask_to_index(bitmask: np.ndarray, nk: int, count_only: bool = False):
    """bitmask uint32 [L][H][nq][words] -> (row_ptr int32 [L*H*nq+1], col_idx int32 [nnz])."""
    bm = _c(bitmask, np.uint32)
    L, H, nq, words = bm.shape
    assert words == (nk + 31) // 32
    row_ptr = np.zeros(L * H * nq + 1, dtype=np.int32)
    nnz = lib().oracle_mask_to_index(_p(bm), L, H, nq, nk, _p(row_ptr), None)
    if count_only:
        return row_ptr, None
    col_idx = np.zeros(max(int(nnz), 1), dtype=np.int32)
    lib().oracle_mask_to_index(_p(bm), L, H, nq, nk, _p(row_ptr), _p(col_idx))
    return row_ptr, col_idx[:nnz]


def mask_to_index_64x128(bitmask: np.ndarray, N: int):
    """Paper geometry (64 query rows x 128 keys): bitmask uint32 [L][H][ceil(N/64)][words] ->
    (row_ptr int32 [L*H*ceil(N/128)+1], col_idx uint32: 64-key tile | bit 30 = rows 0-63 of the 128-row block do
    not keep it | bit 31 = rows 64-127 do not keep it)."""
    bm = _c(bitmask, np.uint32)
    L, H, nq64, words = bm.shape
    assert nq64 == (N + 63) // 64 and words == ((N + 127) // 128 + 31) // 32
    row_ptr = np.zeros(L * H * ((N + 127) // 128) + 1, dtype=np.int32)
    nnz = lib().oracle_mask_to_index_64x128(_p(bm), L, H, N, _p(row_ptr), None)
    col_idx = np.zeros(max(int(nnz), 1), dtype=np.uint32)
    lib().oracle_mask_to_index_64x128(_p(bm), L, H, N, _p(row_ptr), _p(col_idx))
    return row_ptr, col_idx[:nnz]


def mask_to_index_u16(bitmask: np.ndarray, nk: int):
    """mask_to_index with 16-bit entries (nk <= 65536): (row_ptr int32, col_idx uint16)."""
    bm = _c(bitmask, np.uint32)
    L, H, nq, words = bm.shape
    assert words == (nk + 31) // 32
    row_ptr = np.zeros(L * H * nq + 1, dtype=np.int32)
    nnz = lib().oracle_mask_to_index_u16(_p(bm), L, H, nq, nk, _p(row_ptr), None)
    if nnz < 0:
        raise ValueError("key-block index does not fit 16 bits")
    col_idx = np.zeros(max(int(nnz), 1), dtype=np.uint16)
    lib().oracle_mask_to_index_u16(_p(bm), L, H, nq, nk, _p(row_ptr), _p(col_idx))
    return row_ptr, col_idx[:nnz]


def mask_to_index_64x128_u16(bitmask: np.ndarray, N: int):
    """mask_to_index_64x128 with 16-bit entries: tile | bit 14 = upper half does not keep it | bit 15 = lower."""
    bm = _c(bitmask, np.uint32)
    L, H, nq64, words = bm.shape
    assert nq64 == (N + 63) // 64 and words == ((N + 127) // 128 + 31) // 32
    row_ptr = np.zeros(L * H * ((N + 127) // 128) + 1, dtype=np.int32)
    nnz = lib().oracle_mask_to_index_64x128_u16(_p(bm), L, H, N, _p(row_ptr), None)
    if nnz < 0:
        raise ValueError("tile index does not fit 14 bits")
    col_idx = np.zeros(max(int(nnz), 1), dtype=np.uint16)
    lib().oracle_mask_to_index_64x128_u16(_p(bm), L, H, N, _p(row_ptr), _p(col_idx))
    return row_ptr, col_idx[:nnz]


def _strides(a):
    # element strides of a [B][N][H][d] array whose last dim is contiguous
    es = a.dtype.itemsize
    assert a.strides[3] == es, "last dim must be contiguous"
    return [C.c_int64(a.strides[0] // es), C.c_int64(a.strides[1] // es),
            C.c_int64(a.strides[2] // es)]


def block_sparse_attn(Q, K, V, bitmask, scale, items=None, fp8_scales=None, n_threads=0,
                      return_weight_sum=False, return_lse=False, n_first=0, beta=1.0, block=(128, 64)):
    """fp64 block-sparse attention on the exact input bytes.

    block = (query rows, keys) per mask block: (128, 64) or the paper's (64, 128); items, the
    bitmask's shape and the output rows follow it.
    n_first, beta: first-frame key enhancement (eq. (1)): the keys of tokens
    0 .. n_first-1 are multiplied by beta (in fp64, on the exact input values) before the scores.

    Q, K, V: [B][N][H][d] numpy arrays, uint16 (bf16 bits), float16, or uint8 (e4m3 codes; then
    fp8_scales = (q_scale [B][H][ceil(N/128)], k_scale same, v_scale [B][H][d]) float32).
    bitmask: uint32 [H][nq][words] (one layer).  items: int array [n][3] of (b, h, qb); default all.
    Returns out float64 [n_items][128][d] (rows beyond N are 0)  (+ weight sums [n_items][128])
    (+ row log-sum-exp [n_items][128], natural log, -inf for empty rows, if return_lse).
    """
    assert Q.dtype == K.dtype == V.dtype and Q.dtype in (np.uint16, np.uint8, np.float16)
    dtype = {np.dtype(np.uint16): 0, np.dtype(np.uint8): 1, np.dtype(np.float16): 2}[Q.dtype]
    B, N, H, d = Q.shape
    BQ, BK = block
    assert (BQ, BK) in ((128, 64), (64, 128))
    nq, nk = (N + BQ - 1) // BQ, (N + BK - 1) // BK
    bm = _c(bitmask, np.uint32)
    assert bm.shape == (H, nq, (nk + 31) // 32), (bm.shape, (H, nq, (nk + 31) // 32))
    if items is None:
        items = np.array([(b, h, qb) for b in range(B) for h in range(H) for qb in range(nq)],
                         dtype=np.int32)
    items = np.asarray(items, dtype=np.int32).reshape(-1, 3)
    ib, ih, iq = (_c(items[:, k], np.int32) for k in range(3))
    n = items.shape[0]
    out = np.zeros((n, BQ, d), dtype=np.float64)
    ws = np.zeros((n, BQ), dtype=np.float64) if return_weight_sum else None
    lse = np.zeros((n, BQ), dtype=np.float64) if return_lse else None
    if dtype == 1:
        qs, ks, vs = (_c(x, np.float32) for x in fp8_scales)
        nsb = (N + 127) // 128
        assert qs.size == B * H * nsb and ks.size == B * H * nsb and vs.size == B * H * d
    else:
        qs = ks = vs = None
    lib().oracle_block_sparse_attn(
        _p(Q), _p(K), _p(V), C.c_int(dtype), B, H, N, d,
        *_strides(Q), *_strides(K), *_strides(V),
        _p(qs), _p(ks), _p(vs), _p(bm), C.c_double(scale),
        n, _p(ib), _p(ih), _p(iq), _p(out), _p(ws), _p(lse), C.c_int(n_threads),
        C.c_int(int(n_first)), C.c_double(float(beta)), C.c_int(BQ), C.c_int(BK))
    res = (out,) + ((ws,) if return_weight_sum else ()) + ((lse,) if return_lse else ())
    return res if len(res) > 1 else out


def scatter_items(out_items, items, N, H):
    """[n_items][128][d] -> dense [B=1][N][H][d] float64 for the covered (h, qb) items."""
    d = out_items.shape[2]
    O = np.zeros((1, N, H, d), dtype=np.float64)
    for t, (b, h, qb) in enumerate(np.asarray(items).reshape(-1, 3)):
        lo, hi = qb * BQ, min(N, (qb + 1) * BQ)
        O[b, lo:hi, h, :] = out_items[t, : hi - lo, :]
    return O


def quantize_fp8(Q, K, V):
    """bf16-bit arrays [B][N][H][d] -> (q8, k8, v8 uint8 packed, q_scale, k_scale, v_scale f32)."""
    B, N, H, d = Q.shape
    nsb = (N + 127) // 128
    q8, k8, v8 = (np.zeros((B, N, H, d), dtype=np.uint8) for _ in range(3))
    qs = np.zeros((B, H, nsb), dtype=np.float32)
    ks = np.zeros((B, H, nsb), dtype=np.float32)
    vs = np.zeros((B, H, d), dtype=np.float32)
    lib().oracle_quantize_fp8(_p(Q), _p(K), _p(V), B, H, N, d,
                              *_strides(Q), *_strides(K), *_strides(V),
                              _p(q8), _p(k8), _p(v8), _p(qs), _p(ks), _p(vs))
    return q8, k8, v8, qs, ks, vs


def e4m3_to_double(code: int) -> float:
    return float(lib().oracle_e4m3_to_double(int(code)))


def f16_to_double(bits: int) -> float:
    return float(lib().oracle_f16_to_double(int(bits)))


def float_to_e4m3(x: float) -> int:
    return int(lib().oracle_float_to_e4m3(float(x)))


def retrieve_top1(bank, query, tau):
    bank = _c(bank, np.float32)
    query = _c(query, np.float32)
    n, dim = bank.shape
    idx, hit, sim = C.c_int32(), C.c_int32(), C.c_double()
    lib().oracle_retrieve_top1(_p(bank), n, dim, _p(query), C.c_double(tau),
                               C.byref(idx), C.byref(sim), C.byref(hit))
    return idx.value, sim.value, bool(hit.value)


def visit_refresh(mask, nk, group=8):
    """mask uint32 [L][H][nq][words]; returns the refreshed copy (PAPER.md:L93 (1))."""
    m = np.array(mask, dtype=np.uint32, copy=True, order="C")
    L, H, nq, words = m.shape
    lib().oracle_visit_refresh(_p(m), L, H, nq, nk, group)
    return m


def block_mass(Q, K, scale, qblocks=None, n_threads=0, block=(128, 64)):
    """True (dense) attention mass per block pair: Q, K bf16-bit arrays
    [B][N][H][d] -> float64 [B][H][nq][nk]; every valid query row contributes exactly 1.
    qblocks: only these query blocks are computed (the rest of the output is 0).
    block: (query rows, keys) per block, (128, 64) or the paper's (64, 128)."""
    assert Q.dtype == K.dtype == np.uint16
    B, N, H, d = Q.shape
    assert tuple(block) in ((128, 64), (64, 128))
    nq, nk = (N + block[0] - 1) // block[0], (N + block[1] - 1) // block[1]
    out = np.zeros((B, H, nq, nk), dtype=np.float64)
    sel = _c(np.asarray([] if qblocks is None else qblocks), np.int32)
    lib().oracle_block_mass(_p(Q), _p(K), B, H, N, d, *_strides(Q), *_strides(K),
                            C.c_double(scale), _p(out), C.c_int(sel.size), _p(sel), C.c_int(n_threads),
                            C.c_int(block[0]), C.c_int(block[1]))
    return out


def mask_from_mass(mass, nk, top_p, min_top_k):
    """Top-p with a top-k floor (PAPER.md:L81, L93 (2)): mass float32 [..., nk] -> (bitmask uint32
    [..., words], kept int32 [...])."""
    m = _c(mass, np.float32)
    assert m.shape[-1] == nk
    rows = m.size // nk
    words = (nk + 31) // 32
    bm = np.zeros(m.shape[:-1] + (words,), dtype=np.uint32)
    kept = np.zeros(m.shape[:-1], dtype=np.int32)
    lib().oracle_mask_from_mass(_p(m), C.c_int64(rows), nk, C.c_double(top_p), C.c_double(min_top_k),
                                _p(bm), _p(kept))
    return bm, kept


def mask_coverage(mass, bitmask, nk):
    """Per-head coverage: mass float32 [heads][nq][nk], bitmask [heads][nq][words]."""
    m = _c(mass, np.float32)
    b = _c(bitmask, np.uint32)
    heads, nq = m.shape[0], m.shape[1]
    out = np.zeros(heads, dtype=np.float64)
    lib().oracle_mask_coverage(_p(m), _p(b), heads, nq, nk, _p(out))
    return out


def schedule_heads(cost, n_ranks):
    """Head-level scheduling (appendix A), followed step by step: heads with
    the heavier workload first, each "to the GPUs with the lightest current load"; a rank takes at
    most ceil(H / n_ranks) heads (equal head slots per rank under Ulysses, R24); ties:
    lower head, lower rank.  Returns (list of ascending head lists per rank, loads)."""
    cost = [int(c) for c in cost]
    H = len(cost)
    cap = -(-H // n_ranks)
    heads = sorted(range(H), key=lambda h: (-cost[h], h))
    mine = [[] for _ in range(n_ranks)]
    load = [0] * n_ranks
    for h in heads:
        best = None
        for r in range(n_ranks):
            if len(mine[r]) < cap and (best is None or load[r] < load[best]):
                best = r
        mine[best].append(h)
        load[best] += cost[h]
    return [sorted(m) for m in mine], load


def gather_heads(X, order, n_ranks):
    """PAPER.md:L95 / appendix A, the copy before the Ulysses all-to-all, written out: X [n][H][d] ->
    packed [n_ranks][n][H/n_ranks][d] with packed[p][i][s] = X[i][order[p * slots + s]]."""
    n, H, d = X.shape
    slots = H // n_ranks
    out = np.empty((n_ranks, n, slots, d), dtype=X.dtype)
    for p in range(n_ranks):
        for s in range(slots):
            out[p, :, s, :] = X[:, int(order[p * slots + s]), :]
    return out


def scatter_heads(packed, order):
    """The inverse copy: packed [n_ranks][n][slots][d] -> X [n][H][d]."""
    n_ranks, n, slots, d = packed.shape
    X = np.empty((n, n_ranks * slots, d), dtype=packed.dtype)
    for p in range(n_ranks):
        for s in range(slots):
            X[:, int(order[p * slots + s]), :] = packed[p, :, s, :]
    return X
