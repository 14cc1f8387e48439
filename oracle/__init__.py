"""ctypes front-end of the CPU oracle (oracle/saf3r_oracle.c).

TEST INFRASTRUCTURE, NOT PRODUCT CODE: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module.  It imports nothing from
paper_2607_03612_b200 and shares no code with the CUDA path.  Argument marshalling only; every
number is computed inside the C file, whose functions cite the PAPER.md passage they follow.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "saf3r_oracle.c")
_LIB = os.path.join(_HERE, "libsaf3r_oracle.so")

HEAD_DENSE, HEAD_UNIFORM_STRIDE, HEAD_STATIC, HEAD_QUERY_PROBE_TOPK, HEAD_BLOCK_TOPK = range(5)
STATIC_ANCHOR, STATIC_FRAME_LOCAL, STATIC_POSITION_BAND = range(3)
SCOPE_GLOBAL, SCOPE_PER_FRAME = range(2)
SCORE_DOT, SCORE_COSINE = range(2)


class OrcHeadCfg(C.Structure):
    _fields_ = [(n, C.c_int32) for n in (
        "type", "stride", "offset", "keep_blocks", "static_mode", "anchor_frame", "band_radius",
        "topk_scope", "topk_per_frame", "score_mode")]


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain C, -O2, OpenMP across independent rows only).  With SAF3R_ORACLE_SANITIZE=1 in the
    environment a second library is built with AddressSanitizer + UndefinedBehaviorSanitizer (-O1 -g, same source) and loaded
    instead; the process must then run with LD_PRELOAD=$(gcc -print-file-name=libasan.so) (profiles/r3_oracle_sanitizers.md)."""
    if os.environ.get("SAF3R_ORACLE_SANITIZE") == "1":
        out = os.path.join(_HERE, "libsaf3r_oracle_san.so")
        if force or not os.path.exists(out) or os.path.getmtime(out) < os.path.getmtime(_SRC):
            subprocess.check_call(["gcc", "-O1", "-g", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-fsanitize=address,undefined",
                                   "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer", "-o", out, _SRC, "-lm"])
        return out
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-o", _LIB, _SRC, "-lm"])
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        i64, i32, vp, dbl = C.c_int64, C.c_int32, C.c_void_p, C.c_double
        L.orc_pool.argtypes = [vp, i64, i32, i32, i32, vp]
        L.orc_mean_query.argtypes = [vp, i64, i32, vp]
        L.orc_score_row.argtypes = [vp, vp, i64, i32, dbl, vp]
        L.orc_topn.argtypes = [vp, i64, i64, i32, vp]
        L.orc_topn.restype = i64
        L.orc_select_head.argtypes = [vp, vp, i64, i64, i32, i32, C.POINTER(OrcHeadCfg), vp, vp, i64, vp]
        L.orc_select_head.restype = i64
        L.orc_attn_lists.argtypes = [vp, vp, vp, i64, i32, i32, vp, vp, vp, i64, vp, vp]
        L.orc_attn_dense.argtypes = [vp, vp, vp, i64, i32, i64, i64, vp, vp]
        L.orc_attn_tokens.argtypes = [vp, vp, vp, i64, i32, vp, i64, i64, i64, vp, vp]
        L.orc_token_probe.argtypes = [vp, vp, i64, i32, vp]
        L.orc_token_topk_per_frame.argtypes = [vp, i64, i64, i32, i64, i64, i64, vp]
        L.orc_token_cosine_row.argtypes = [vp, i64, i32, i64, vp]
        L.orc_attn_token_lists.argtypes = [vp, vp, vp, i64, i32, vp, i64, i64, i64, vp, vp]
        L.orc_attn_broadcast_frame0.argtypes = [vp, vp, vp, i64, i64, i32, vp, vp]
        L.orc_union_lists.argtypes = [vp, vp, vp, vp, i64, i64, vp, vp, i64]
        L.orc_union_lists.restype = i64
        L.orc_nmse.argtypes = [vp, vp, i64]
        L.orc_nmse.restype = dbl
        L.orc_num_threads.restype = i32
        _lib = L
    return _lib


def _p(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


def _u16(a) -> np.ndarray:
    a = np.ascontiguousarray(a)
    assert a.dtype == np.uint16, "bf16 tensors travel as uint16 bit patterns"
    return a


def make_cfg(**kw) -> OrcHeadCfg:
    c = OrcHeadCfg()
    for k, v in kw.items():
        setattr(c, k, int(v))
    return c


def num_threads() -> int:
    return int(lib().orc_num_threads())


def pool(x_bits: np.ndarray, B: int, cosine: bool = False) -> np.ndarray:
    x = _u16(x_bits)
    N, D = x.shape
    NB = (N + B - 1) // B
    out = np.empty((NB, D), np.float32)
    lib().orc_pool(_p(x), N, D, B, int(cosine), _p(out))
    return out


def mean_query(q_bits: np.ndarray) -> np.ndarray:
    q = _u16(q_bits)
    N, D = q.shape
    out = np.empty((D,), np.float32)
    lib().orc_mean_query(_p(q), N, D, _p(out))
    return out


def score_row(a: np.ndarray, kt: np.ndarray, c: float) -> np.ndarray:
    a = np.ascontiguousarray(a, np.float32)
    kt = np.ascontiguousarray(kt, np.float32)
    NB, D = kt.shape
    s = np.empty((NB,), np.float32)
    lib().orc_score_row(_p(a), _p(kt), NB, D, float(c), _p(s))
    return s


def topn(s: np.ndarray, n: int, use_sort: bool) -> np.ndarray:
    s = np.ascontiguousarray(s, np.float32)
    out = np.empty((s.shape[0],), np.int32)
    c = lib().orc_topn(_p(s), s.shape[0], n, int(use_sort), _p(out))
    return out[:c].copy()


@dataclass
class HeadLists:
    row_ptr: np.ndarray      # int64 [NB+1], relative to this head
    col_idx: np.ndarray      # int32, ascending per row
    scores: np.ndarray | None  # [NB][NB] (BLOCK_TOPK) or [1][NB] (QUERY_PROBE) when requested


def select_head(q_bits, k_bits, S: int, T: int, B: int, cfg: OrcHeadCfg, want_scores: bool = False) -> HeadLists:
    q, k = _u16(q_bits), _u16(k_bits)
    N, D = q.shape
    assert N == S * T
    NB = (N + B - 1) // B
    row_ptr = np.empty((NB + 1,), np.int64)
    scores = None
    if want_scores and cfg.type == HEAD_BLOCK_TOPK:
        scores = np.empty((NB, NB), np.float32)
    elif want_scores and cfg.type == HEAD_QUERY_PROBE_TOPK:
        scores = np.empty((1, NB), np.float32)
    cap = NB * NB
    col = np.empty((cap,), np.int32)
    cnt = lib().orc_select_head(_p(q), _p(k), S, T, D, B, C.byref(cfg), _p(row_ptr), _p(col), cap,
                                _p(scores) if scores is not None else None)
    assert cnt >= 0
    return HeadLists(row_ptr, col[:cnt].copy(), scores)


def attn_lists(q_bits, k_bits, v_bits, B: int, row_ptr, col_idx, qblocks=None, want_lse: bool = True):
    """Masked softmax attention of one head over CSR lists; returns (out [N][D] fp32, lse [N] fp32).
    Rows of q-blocks not in `qblocks` are left as NaN."""
    q, k, v = _u16(q_bits), _u16(k_bits), _u16(v_bits)
    N, D = q.shape
    NB = (N + B - 1) // B
    row_ptr = np.ascontiguousarray(row_ptr, np.int64)
    col_idx = np.ascontiguousarray(col_idx, np.int32)
    if col_idx.size == 0:
        col_idx = np.zeros((1,), np.int32)
    qb = np.arange(NB, dtype=np.int64) if qblocks is None else np.ascontiguousarray(qblocks, np.int64)
    out = np.full((N, D), np.nan, np.float32)
    lse = np.full((N,), np.nan, np.float32)
    lib().orc_attn_lists(_p(q), _p(k), _p(v), N, D, B, _p(row_ptr), _p(col_idx), _p(qb), qb.shape[0],
                         _p(out), _p(lse) if want_lse else None)
    return out, lse


def attn_dense(q_bits, k_bits, v_bits, i0: int = 0, i1: int | None = None):
    q, k, v = _u16(q_bits), _u16(k_bits), _u16(v_bits)
    N, D = q.shape
    i1 = N if i1 is None else i1
    out = np.full((N, D), np.nan, np.float32)
    lse = np.full((N,), np.nan, np.float32)
    lib().orc_attn_dense(_p(q), _p(k), _p(v), N, D, i0, i1, _p(out), _p(lse))
    return out, lse


def attn_tokens(q_bits, k_bits, v_bits, idx, i0: int = 0, i1: int | None = None):
    """Every query of rows [i0, i1) attends the same key-token set idx (ascending); returns (out [N][D], lse [N]), other rows NaN."""
    q, k, v = _u16(q_bits), _u16(k_bits), _u16(v_bits)
    N, D = q.shape
    i1 = N if i1 is None else i1
    idx = np.ascontiguousarray(idx, np.int64)
    out = np.full((N, D), np.nan, np.float32)
    lse = np.full((N,), np.nan, np.float32)
    pad = idx if idx.size else np.zeros((1,), np.int64)
    lib().orc_attn_tokens(_p(q), _p(k), _p(v), N, D, _p(pad), idx.size, i0, i1, _p(out), _p(lse))
    return out, lse


def token_probe(q_bits, k_bits) -> np.ndarray:
    """p[j] = qbar . k_j / sqrt(D) for every key token."""
    q, k = _u16(q_bits), _u16(k_bits)
    N, D = q.shape
    p = np.empty((N,), np.float32)
    lib().orc_token_probe(_p(q), _p(k), N, D, _p(p))
    return p


def token_probe_topk(q_bits, k_bits, K: int):
    """Query-Probe Top-K at token level: the K key tokens with the largest probe score (score desc, index asc), ascending.
    Returns (idx int64 [K], scores fp32 [N])."""
    p = token_probe(q_bits, k_bits)
    keep = topn(p, K, use_sort=True)
    return keep.astype(np.int64), p


def token_topk_per_frame(feat_bits, S: int, T: int, K: int, i0: int = 0, i1: int | None = None) -> np.ndarray:
    """Token-wise DINO Top-K: for the queries [i0, i1) the K most cosine-similar tokens of EVERY frame;
    returns int32 [(i1 - i0)][S][K] global token indices, ascending."""
    f = _u16(feat_bits)
    N, D = f.shape
    assert N == S * T and 1 <= K <= T
    i1 = N if i1 is None else i1
    out = np.empty((i1 - i0, S, K), np.int32)
    lib().orc_token_topk_per_frame(_p(f), S, T, D, K, i0, i1, _p(out))
    return out


def token_cosine_row(feat_bits, i: int) -> np.ndarray:
    f = _u16(feat_bits)
    N, D = f.shape
    out = np.empty((N,), np.float32)
    lib().orc_token_cosine_row(_p(f), N, D, i, _p(out))
    return out


def attn_token_lists(q_bits, k_bits, v_bits, idx: np.ndarray, i0: int = 0, i1: int | None = None):
    """Attention with per-query key lists: idx int32 [(i1 - i0)][L] (negative = padding).  Returns (out [N][D], lse [N]); rows
    outside [i0, i1) are NaN."""
    q, k, v = _u16(q_bits), _u16(k_bits), _u16(v_bits)
    N, D = q.shape
    i1 = N if i1 is None else i1
    idx = np.ascontiguousarray(idx, np.int32).reshape(i1 - i0, -1)
    out = np.full((N, D), np.nan, np.float32)
    lse = np.full((N,), np.nan, np.float32)
    lib().orc_attn_token_lists(_p(q), _p(k), _p(v), N, D, _p(idx), idx.shape[1], i0, i1, _p(out), _p(lse))
    return out, lse


def attn_broadcast_frame0(q_bits, k_bits, v_bits, S: int, T: int):
    """Static kernel broadcasting frame 0's local attention map to every frame pair (reading A18):
    returns (out [N][D] fp32, lse [N] fp32)."""
    q, k, v = _u16(q_bits), _u16(k_bits), _u16(v_bits)
    N, D = q.shape
    assert N == S * T
    out = np.empty((N, D), np.float32)
    lse = np.empty((N,), np.float32)
    lib().orc_attn_broadcast_frame0(_p(q), _p(k), _p(v), S, T, D, _p(out), _p(lse))
    return out, lse


def union_lists(row_ptr_a, col_a, row_ptr_b, col_b, NB: int):
    """Row-wise set union of two CSR block lists over the same rows; returns (row_ptr, col_idx), rows ascending."""
    ra, rb = np.ascontiguousarray(row_ptr_a, np.int64), np.ascontiguousarray(row_ptr_b, np.int64)
    ca, cb = np.ascontiguousarray(col_a, np.int32), np.ascontiguousarray(col_b, np.int32)
    assert ra.shape == rb.shape
    rows = ra.shape[0] - 1
    cap = int(ca.size + cb.size) + 1
    ro, co = np.empty((rows + 1,), np.int64), np.empty((cap,), np.int32)
    pa = ca if ca.size else np.zeros((1,), np.int32)
    pb = cb if cb.size else np.zeros((1,), np.int32)
    n = lib().orc_union_lists(_p(ra), _p(pa), _p(rb), _p(pb), rows, NB, _p(ro), _p(co), cap)
    assert n >= 0
    return ro, co[:n].copy()


def nmse(o_full: np.ndarray, o_sparse: np.ndarray) -> float:
    a = np.ascontiguousarray(o_full, np.float32)
    b = np.ascontiguousarray(o_sparse, np.float32)
    return float(lib().orc_nmse(_p(a), _p(b), a.size))
