"""paper_2607_03612_b200 -- thin Python binding of the SAF3R C-ABI library (include/saf3r.h).

Argument marshalling only: every step of the hot path (pool, score, select, block-sparse / dense attention) runs in the
hand-written sm_100a kernels of csrc/.  PyTorch is used for device memory and streams, nothing else.  There is no CPU
fallback: importing works anywhere, but creating a context without the built library or without an sm_100 GPU raises.

Function names mirror the C entry points: query_sizes, select, sparse_attn, dense_attn, layer_host.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libsaf3r.so")

MAX_HEADS = 64
OK, ERR_INVALID_ARG, ERR_UNSUPPORTED, ERR_CAPACITY, ERR_CUDA = range(5)
_STATUS = {0: "OK", 1: "INVALID_ARG", 2: "UNSUPPORTED", 3: "CAPACITY", 4: "CUDA"}

HEAD_DENSE, HEAD_UNIFORM_STRIDE, HEAD_STATIC, HEAD_QUERY_PROBE_TOPK, HEAD_BLOCK_TOPK, HEAD_CACHED = range(6)
STATIC_ANCHOR, STATIC_FRAME_LOCAL, STATIC_POSITION_BAND = range(3)
SCOPE_GLOBAL, SCOPE_PER_FRAME = range(2)
SCORE_DOT, SCORE_COSINE = range(2)

EXPORTS = ("saf3r_create", "saf3r_destroy", "saf3r_last_error", "saf3r_query_sizes", "saf3r_select", "saf3r_sparse_attn",
           "saf3r_dense_attn", "saf3r_layer_host_scratch_bytes", "saf3r_layer_host", "saf3r_launch_count",
           "saf3r_set_stage_timing", "saf3r_last_select_stage_ms", "saf3r_select_cached", "saf3r_token_stride_attn",
           "saf3r_token_query_sizes", "saf3r_token_probe_select", "saf3r_token_set_attn", "saf3r_check_lists", "saf3r_select_plan", "saf3r_union_lists",
           "saf3r_static_broadcast_workspace_bytes", "saf3r_static_broadcast_attn", "saf3r_token_topk_query_sizes",
           "saf3r_token_topk_select", "saf3r_token_lists_count", "saf3r_token_lists_fill", "saf3r_token_lists_attn", "saf3r_nmse_accumulate",
           "saf3r_token_probe_select_noalloc")


class Saf3rError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"saf3r: {_STATUS.get(status, status)}: {msg}")
        self.status = status


class HeadCfg(C.Structure):
    _fields_ = [(n, C.c_int32) for n in (
        "type", "stride", "offset", "keep_blocks", "static_mode", "anchor_frame", "band_radius",
        "topk_scope", "topk_per_frame", "score_mode")]


class ShapeC(C.Structure):
    _fields_ = [("num_frames", C.c_int32), ("tokens_per_frame", C.c_int32), ("num_heads", C.c_int32),
                ("head_dim", C.c_int32), ("block", C.c_int32), ("stride_head", C.c_int64), ("stride_token", C.c_int64)]


class ListsC(C.Structure):
    _fields_ = [("row_ptr", C.c_void_p), ("col_idx", C.c_void_p), ("capacity", C.c_int64)]


class TokenListsC(C.Structure):
    _fields_ = [("tile_ptr", C.c_void_p), ("key_idx", C.c_void_p), ("mask", C.c_void_p), ("capacity_tiles", C.c_int64)]


_lib = None


def load_library():
    """dlopen the in-tree libsaf3r.so; raises if it has not been built (python -m paper_2607_03612_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2607_03612_b200.build` "
                               "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, i64, i32 = C.c_void_p, C.c_int64, C.c_int
        L.saf3r_create.argtypes = [C.POINTER(vp), i32]
        L.saf3r_destroy.argtypes = [vp]
        L.saf3r_destroy.restype = None
        L.saf3r_last_error.argtypes = [vp]
        L.saf3r_last_error.restype = C.c_char_p
        L.saf3r_query_sizes.argtypes = [C.POINTER(ShapeC), C.POINTER(HeadCfg), C.POINTER(i64), C.POINTER(C.c_size_t)]
        L.saf3r_select.argtypes = [vp, vp, vp, C.POINTER(ShapeC), C.POINTER(HeadCfg), vp, C.c_size_t, C.POINTER(ListsC), vp]
        L.saf3r_select_cached.argtypes = [vp, vp, vp, C.POINTER(ShapeC), C.POINTER(HeadCfg), C.POINTER(ListsC), C.c_int32, vp,
                                          C.c_size_t, C.POINTER(ListsC), vp]
        L.saf3r_token_stride_attn.argtypes = [vp, vp, vp, vp, C.POINTER(ShapeC), C.c_int32, C.c_int32, vp, i32, vp, vp]
        L.saf3r_token_query_sizes.argtypes = [C.POINTER(ShapeC), C.c_int32, C.POINTER(C.c_size_t), C.POINTER(C.c_size_t)]
        L.saf3r_token_probe_select.argtypes = [vp, vp, vp, C.POINTER(ShapeC), C.c_int32, vp, C.c_size_t, vp, vp]
        L.saf3r_token_probe_select_noalloc.argtypes = [vp, vp, C.POINTER(ShapeC), C.c_int32, vp, vp, C.c_char_p, C.c_size_t]
        L.saf3r_token_set_attn.argtypes = [vp, vp, vp, vp, C.POINTER(ShapeC), vp, C.c_int32, vp, C.c_size_t, vp, i32, vp, vp]
        L.saf3r_check_lists.argtypes = [vp, C.POINTER(ShapeC), C.POINTER(ListsC), C.POINTER(i64), vp]
        L.saf3r_sparse_attn.argtypes = [vp, vp, vp, vp, C.POINTER(ShapeC), C.POINTER(ListsC), vp, i32, vp, vp]
        L.saf3r_dense_attn.argtypes = [vp, vp, vp, vp, C.POINTER(ShapeC), vp, i32, vp, vp]
        L.saf3r_layer_host_scratch_bytes.argtypes = [C.POINTER(ShapeC), C.POINTER(HeadCfg), C.POINTER(C.c_size_t)]
        L.saf3r_layer_host.argtypes = [vp, vp, vp, vp, C.POINTER(ShapeC), C.POINTER(HeadCfg), vp, C.c_size_t, vp, vp]
        L.saf3r_select_plan.argtypes = [vp, C.POINTER(ShapeC), C.POINTER(HeadCfg), C.POINTER(C.c_int32), C.POINTER(C.c_size_t)]
        L.saf3r_union_lists.argtypes = [vp, C.POINTER(ShapeC), C.POINTER(ListsC), C.POINTER(ListsC), C.POINTER(ListsC), vp]
        L.saf3r_static_broadcast_workspace_bytes.argtypes = [C.POINTER(ShapeC), C.POINTER(C.c_size_t)]
        L.saf3r_static_broadcast_attn.argtypes = [vp, vp, vp, vp, C.POINTER(ShapeC), vp, C.c_size_t, vp, i32, vp, vp]
        L.saf3r_token_topk_query_sizes.argtypes = [C.POINTER(ShapeC), C.c_int32, C.POINTER(C.c_size_t), C.POINTER(i64), C.POINTER(i64)]
        L.saf3r_token_topk_select.argtypes = [vp, vp, C.POINTER(ShapeC), C.c_int32, vp, C.c_size_t, vp, vp]
        L.saf3r_token_lists_count.argtypes = [vp, C.POINTER(ShapeC), C.c_int32, vp, vp, vp]
        L.saf3r_token_lists_fill.argtypes = [vp, C.POINTER(ShapeC), C.c_int32, vp, C.POINTER(TokenListsC), vp]
        L.saf3r_token_lists_attn.argtypes = [vp, vp, vp, vp, C.POINTER(ShapeC), C.POINTER(TokenListsC), vp, i32, vp, vp]
        L.saf3r_nmse_accumulate.argtypes = [vp, vp, vp, C.POINTER(ShapeC), i32, vp, vp]
        L.saf3r_launch_count.argtypes = [vp]
        L.saf3r_launch_count.restype = i64
        L.saf3r_set_stage_timing.argtypes = [vp, i32]
        L.saf3r_last_select_stage_ms.argtypes = [vp, C.POINTER(C.c_float), C.POINTER(C.c_float)]
        _lib = L
    return _lib


def make_cfgs(cfgs) -> "C.Array[HeadCfg]":
    """cfgs: list of dicts (the ten int32 fields) or HeadCfg."""
    arr = (HeadCfg * len(cfgs))()
    for i, c in enumerate(cfgs):
        if isinstance(c, HeadCfg):
            arr[i] = c
        else:
            for k, v in c.items():
                setattr(arr[i], k, int(v))
    return arr


def make_shape(S: int, T: int, H: int, D: int, B: int, stride_head: int | None = None, stride_token: int | None = None) -> ShapeC:
    st = D if stride_token is None else stride_token
    sh = S * T * st if stride_head is None else stride_head
    return ShapeC(S, T, H, D, B, sh, st)


@dataclass
class TokenLists:
    tile_ptr: "torch.Tensor"  # int64 [NB+1], device
    key_idx: "torch.Tensor"   # int32 [tiles*block], device
    mask: "torch.Tensor"      # int32 [tiles][block][block/32], device (bit patterns)
    tiles: int

    def c(self) -> TokenListsC:
        return TokenListsC(self.tile_ptr.data_ptr(), self.key_idx.data_ptr(), self.mask.data_ptr(), self.tiles)


@dataclass
class Lists:
    row_ptr: "torch.Tensor"   # int64 [H*NB+1], device
    col_idx: "torch.Tensor"   # int32 [capacity], device

    def c(self) -> ListsC:
        return ListsC(self.row_ptr.data_ptr(), self.col_idx.data_ptr(), self.col_idx.numel())


def _stream_ptr(stream=None):
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def _on_stream(stream, *tensors):
    """Tensors this binding allocated itself (on torch's CURRENT stream) and that kernels enqueued on `stream` touch.  Two hazards
    of the caching allocator when `stream` is not the current stream: (1) the block may have been recycled from a tensor that
    kernels already queued on the current stream still use - so `stream` first waits for the current stream's work queued so far;
    (2) the block may be handed to another allocation while kernels on `stream` still run - so the tensors are recorded on it."""
    if stream is not None:
        import torch
        cur = torch.cuda.current_stream()
        if stream != cur:
            stream.wait_stream(cur)
        for t in tensors:
            if t is not None:
                t.record_stream(stream)


class Context:
    """Owns one saf3r_ctx on a CUDA device."""

    def __init__(self, device: int = 0):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("saf3r needs a CUDA device (sm_100a); there is no CPU fallback")
        self.lib = load_library()
        self.device = device
        h = C.c_void_p()
        st = self.lib.saf3r_create(C.byref(h), device)
        if st != OK:
            raise Saf3rError(st, "saf3r_create failed (needs an sm_100 device)")
        self.h = h

    def close(self):
        if getattr(self, "h", None):
            self.lib.saf3r_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, st: int):
        if st != OK:
            raise Saf3rError(st, self.lib.saf3r_last_error(self.h).decode())

    def launch_count(self) -> int:
        return int(self.lib.saf3r_launch_count(self.h))

    # ---- saf3r_set_stage_timing / saf3r_last_select_stage_ms
    def set_stage_timing(self, enable: bool):
        self._check(self.lib.saf3r_set_stage_timing(self.h, int(enable)))

    def last_select_stage_ms(self) -> tuple[float, float]:
        a, b = C.c_float(), C.c_float()
        self._check(self.lib.saf3r_last_select_stage_ms(self.h, C.byref(a), C.byref(b)))
        return float(a.value), float(b.value)

    # ---- saf3r_query_sizes / saf3r_select_plan
    def query_sizes(self, shape: ShapeC, cfgs) -> tuple[int, int]:
        return query_sizes(shape, cfgs)

    def select_plan(self, shape: ShapeC, cfgs) -> tuple[int, int]:
        """(rows per score strip, dynamic shared-memory bytes) of the score + select launch for (shape, cfgs)."""
        arr = make_cfgs(cfgs)
        r, b = C.c_int32(), C.c_size_t()
        self._check(self.lib.saf3r_select_plan(self.h, C.byref(shape), arr, C.byref(r), C.byref(b)))
        return int(r.value), int(b.value)

    # ---- saf3r_select / saf3r_select_cached
    def select(self, q, k, shape: ShapeC, cfgs, workspace=None, lists: Lists | None = None, stream=None,
               cache: Lists | None = None, cache_heads: int = 0) -> Lists:
        """cache: lists of `cache_heads` heads built once per sequence (an ordinary select on features); heads of type
        HEAD_CACHED copy their rows from cache head cfg['offset'] (saf3r_select_cached)."""
        import torch
        arr = make_cfgs(cfgs)
        entries, ws_bytes = query_sizes(shape, arr)
        dev = q.device
        if workspace is None:
            workspace = torch.empty(ws_bytes, dtype=torch.uint8, device=dev)
            _on_stream(stream, workspace)
        if lists is None:
            N = shape.num_frames * shape.tokens_per_frame
            NB = (N + shape.block - 1) // shape.block
            lists = Lists(torch.empty(shape.num_heads * NB + 1, dtype=torch.int64, device=dev),
                          torch.empty(max(entries, 1), dtype=torch.int32, device=dev))
            _on_stream(stream, lists.row_ptr, lists.col_idx)
        lc = lists.c()
        if cache is not None:
            cc = cache.c()
            self._check(self.lib.saf3r_select_cached(self.h, q.data_ptr(), k.data_ptr(), C.byref(shape), arr, C.byref(cc),
                                                     int(cache_heads), workspace.data_ptr(),
                                                     workspace.numel() * workspace.element_size(), C.byref(lc), _stream_ptr(stream)))
        else:
            self._check(self.lib.saf3r_select(self.h, q.data_ptr(), k.data_ptr(), C.byref(shape), arr, workspace.data_ptr(),
                                              workspace.numel() * workspace.element_size(), C.byref(lc), _stream_ptr(stream)))
        return lists

    # ---- saf3r_check_lists
    def check_lists(self, shape: ShapeC, lists: Lists, stream=None) -> int:
        """Number of malformed rows of caller-made lists (synchronises the stream)."""
        lc, bad = lists.c(), C.c_int64()
        self._check(self.lib.saf3r_check_lists(self.h, C.byref(shape), C.byref(lc), C.byref(bad), _stream_ptr(stream)))
        return int(bad.value)

    # ---- saf3r_union_lists
    def union_lists(self, shape: ShapeC, a: Lists, b: Lists, out: Lists | None = None, stream=None) -> Lists:
        """Row-wise union of two sets of block lists (ascending, unique); out defaults to a buffer of entries(a) + entries(b)."""
        import torch
        if out is None:
            out = Lists(torch.empty_like(a.row_ptr), torch.empty(a.col_idx.numel() + b.col_idx.numel(), dtype=torch.int32,
                                                                 device=a.col_idx.device))
            _on_stream(stream, out.row_ptr, out.col_idx)
        ca, cb, co = a.c(), b.c(), out.c()
        self._check(self.lib.saf3r_union_lists(self.h, C.byref(shape), C.byref(ca), C.byref(cb), C.byref(co), _stream_ptr(stream)))
        return out

    # ---- saf3r_sparse_attn / saf3r_dense_attn
    def sparse_attn(self, q, k, v, shape: ShapeC, lists: Lists, out=None, out_fp32: bool = False, want_lse: bool = False, stream=None):
        return self._attn(q, k, v, shape, lists, out, out_fp32, want_lse, stream)

    def dense_attn(self, q, k, v, shape: ShapeC, out=None, out_fp32: bool = False, want_lse: bool = False, stream=None):
        return self._attn(q, k, v, shape, None, out, out_fp32, want_lse, stream)

    def _attn(self, q, k, v, shape, lists, out, out_fp32, want_lse, stream):
        import torch
        out, lse = self._out_lse(q, shape, out, out_fp32, want_lse, stream)
        lp = lse.data_ptr() if lse is not None else None
        if lists is not None:
            lc = lists.c()
            st = self.lib.saf3r_sparse_attn(self.h, q.data_ptr(), k.data_ptr(), v.data_ptr(), C.byref(shape), C.byref(lc),
                                            out.data_ptr(), int(out_fp32), lp, _stream_ptr(stream))
        else:
            st = self.lib.saf3r_dense_attn(self.h, q.data_ptr(), k.data_ptr(), v.data_ptr(), C.byref(shape),
                                           out.data_ptr(), int(out_fp32), lp, _stream_ptr(stream))
        self._check(st)
        return (out, lse) if want_lse else out

    # ---- token-granular variants: saf3r_token_stride_attn / saf3r_token_probe_select / saf3r_token_set_attn
    def _out_lse(self, q, shape, out, out_fp32, want_lse, stream=None):
        import torch
        if out is None:
            out = torch.empty(q.shape, dtype=torch.float32 if out_fp32 else torch.bfloat16, device=q.device)
            _on_stream(stream, out)
        N = shape.num_frames * shape.tokens_per_frame
        lse = torch.empty((shape.num_heads, N), dtype=torch.float32, device=q.device) if want_lse else None
        _on_stream(stream, lse)
        return out, lse

    def token_stride_attn(self, q, k, v, shape: ShapeC, stride: int, offset: int = 0, out=None, out_fp32=False, want_lse=False,
                          stream=None):
        out, lse = self._out_lse(q, shape, out, out_fp32, want_lse, stream)
        self._check(self.lib.saf3r_token_stride_attn(self.h, q.data_ptr(), k.data_ptr(), v.data_ptr(), C.byref(shape), int(stride),
                                                     int(offset), out.data_ptr(), int(out_fp32),
                                                     lse.data_ptr() if lse is not None else None, _stream_ptr(stream)))
        return (out, lse) if want_lse else out

    def token_probe_select(self, q, k, shape: ShapeC, K: int, workspace=None, idx=None, stream=None):
        """Returns idx int32 [H][K] (device): the K key tokens with the largest probe score per head, ascending."""
        import torch
        sel_ws, _ = token_query_sizes(shape, K)
        if workspace is None:
            workspace = torch.empty(sel_ws, dtype=torch.uint8, device=q.device)
            _on_stream(stream, workspace)
        if idx is None:
            idx = torch.empty((shape.num_heads, K), dtype=torch.int32, device=q.device)
            _on_stream(stream, idx)
        self._check(self.lib.saf3r_token_probe_select(self.h, q.data_ptr(), k.data_ptr(), C.byref(shape), int(K), workspace.data_ptr(),
                                                      workspace.numel(), idx.data_ptr(), _stream_ptr(stream)))
        return idx

    def token_set_attn(self, q, k, v, shape: ShapeC, idx, workspace=None, out=None, out_fp32=False, want_lse=False, stream=None):
        import torch
        K = int(idx.shape[1])
        _, att_ws = token_query_sizes(shape, K)
        if workspace is None:
            workspace = torch.empty(att_ws, dtype=torch.uint8, device=q.device)
            _on_stream(stream, workspace)
        out, lse = self._out_lse(q, shape, out, out_fp32, want_lse, stream)
        self._check(self.lib.saf3r_token_set_attn(self.h, q.data_ptr(), k.data_ptr(), v.data_ptr(), C.byref(shape), idx.data_ptr(), K,
                                                  workspace.data_ptr(), workspace.numel(), out.data_ptr(), int(out_fp32),
                                                  lse.data_ptr() if lse is not None else None, _stream_ptr(stream)))
        return (out, lse) if want_lse else out

    # ---- token-wise per-frame Top-K: saf3r_token_topk_select / saf3r_token_lists_count / _fill / _attn
    def token_topk_select(self, feat, shape: ShapeC, K: int, workspace=None, idx=None, stream=None):
        """feat: [N][64] bf16 device tensor (per-sequence features).  Returns idx int32 [N][S][K]: per query and frame the K most
        cosine-similar tokens of that frame, ascending."""
        import torch
        ws_bytes, _, _ = token_topk_query_sizes(shape, K)
        N = shape.num_frames * shape.tokens_per_frame
        if workspace is None:
            workspace = torch.empty(ws_bytes, dtype=torch.uint8, device=feat.device)
            _on_stream(stream, workspace)
        if idx is None:
            idx = torch.empty((N, shape.num_frames, K), dtype=torch.int32, device=feat.device)
            _on_stream(stream, idx)
        fshape = ShapeC(shape.num_frames, shape.tokens_per_frame, 1, shape.head_dim, shape.block, N * feat.stride(0), feat.stride(0))
        self._check(self.lib.saf3r_token_topk_select(self.h, feat.data_ptr(), C.byref(fshape), int(K), workspace.data_ptr(),
                                                     workspace.numel(), idx.data_ptr(), _stream_ptr(stream)))
        return idx

    def token_lists_build(self, shape: ShapeC, idx, stream=None) -> TokenLists:
        """Per q-tile union of the queries' keys + per-(query, key) masks (once per sequence).  Counts first, reads the total back
        (one synchronisation), allocates exactly, then fills."""
        import torch
        K = int(idx.shape[2])
        N = shape.num_frames * shape.tokens_per_frame
        NB = (N + shape.block - 1) // shape.block
        tile_ptr = torch.empty(NB + 1, dtype=torch.int64, device=idx.device)
        _on_stream(stream, tile_ptr)
        self._check(self.lib.saf3r_token_lists_count(self.h, C.byref(shape), K, idx.data_ptr(), tile_ptr.data_ptr(), _stream_ptr(stream)))
        (torch.cuda.current_stream() if stream is None else stream).synchronize()
        tiles = int(tile_ptr[-1].item())
        B = shape.block
        lists = TokenLists(tile_ptr, torch.empty(max(tiles, 1) * B, dtype=torch.int32, device=idx.device),
                           torch.empty((max(tiles, 1), B, B // 32), dtype=torch.int32, device=idx.device), tiles)
        _on_stream(stream, lists.key_idx, lists.mask)
        lc = lists.c()
        self._check(self.lib.saf3r_token_lists_fill(self.h, C.byref(shape), K, idx.data_ptr(), C.byref(lc), _stream_ptr(stream)))
        return lists

    def token_lists_attn(self, q, k, v, shape: ShapeC, lists: TokenLists, out=None, out_fp32=False, want_lse=False, stream=None):
        out, lse = self._out_lse(q, shape, out, out_fp32, want_lse, stream)
        lc = lists.c()
        self._check(self.lib.saf3r_token_lists_attn(self.h, q.data_ptr(), k.data_ptr(), v.data_ptr(), C.byref(shape), C.byref(lc),
                                                    out.data_ptr(), int(out_fp32), lse.data_ptr() if lse is not None else None,
                                                    _stream_ptr(stream)))
        return (out, lse) if want_lse else out

    # ---- saf3r_nmse_accumulate
    def nmse(self, o_full, o_sparse, shape: ShapeC, stream=None) -> list[float]:
        """Eq. 1 per head for one sample: ||O_full - O_sparse||^2 / ||O_full||^2, both sums in the library."""
        import torch
        acc = torch.zeros(2 * shape.num_heads, dtype=torch.float64, device=o_full.device)
        _on_stream(stream, acc)
        assert o_full.dtype == o_sparse.dtype
        self._check(self.lib.saf3r_nmse_accumulate(self.h, o_full.data_ptr(), o_sparse.data_ptr(), C.byref(shape),
                                                   int(o_full.dtype == torch.float32), acc.data_ptr(), _stream_ptr(stream)))
        (stream or torch.cuda.current_stream()).synchronize()   # the copy below runs on the current stream, the kernel on `stream`
        a = acc.cpu().tolist()
        H = shape.num_heads
        return [a[h] / a[H + h] if a[H + h] > 0 else float("nan") for h in range(H)]   # ||O_full|| = 0: Eq. 1 is undefined

    # ---- saf3r_static_broadcast_attn
    def static_broadcast_attn(self, q, k, v, shape: ShapeC, workspace=None, out=None, out_fp32=False, want_lse=False, stream=None):
        """Static kernel that broadcasts frame 0's local attention map to every frame pair."""
        import torch
        b = C.c_size_t()
        st = self.lib.saf3r_static_broadcast_workspace_bytes(C.byref(shape), C.byref(b))
        if st != OK:
            raise Saf3rError(st, "saf3r_static_broadcast_workspace_bytes rejected the shape")
        if workspace is None:
            workspace = torch.empty(int(b.value), dtype=torch.uint8, device=q.device)
            _on_stream(stream, workspace)
        out, lse = self._out_lse(q, shape, out, out_fp32, want_lse, stream)
        self._check(self.lib.saf3r_static_broadcast_attn(self.h, q.data_ptr(), k.data_ptr(), v.data_ptr(), C.byref(shape),
                                                         workspace.data_ptr(), workspace.numel(), out.data_ptr(), int(out_fp32),
                                                         lse.data_ptr() if lse is not None else None, _stream_ptr(stream)))
        return (out, lse) if want_lse else out

    # ---- saf3r_layer_host
    def layer_host_scratch_bytes(self, shape: ShapeC, cfgs) -> int:
        arr = make_cfgs(cfgs)
        b = C.c_size_t()
        self._check(self.lib.saf3r_layer_host_scratch_bytes(C.byref(shape), arr, C.byref(b)))
        return int(b.value)

    def layer_host(self, q_host, k_host, v_host, shape: ShapeC, cfgs, scratch, out_host, stream=None):
        """q_host/k_host/v_host/out_host: (pinned) CPU tensors, contiguous [H][N][D] bf16.  Enqueues H2D + select +
        sparse_attn + D2H on the stream; synchronise before reading out_host."""
        arr = make_cfgs(cfgs)
        self._check(self.lib.saf3r_layer_host(self.h, q_host.data_ptr(), k_host.data_ptr(), v_host.data_ptr(), C.byref(shape),
                                              arr, scratch.data_ptr(), scratch.numel() * scratch.element_size(),
                                              out_host.data_ptr(), _stream_ptr(stream)))
        return out_host


NOALLOC_MAX_KEYS = 1 << 20  # SAF3R_NOALLOC_MAX_KEYS: num_heads * N the built-in scratch of the call below is sized for


def token_probe_select_noalloc(q, k, shape: ShapeC, K: int, idx, stream=None):
    """saf3r_token_probe_select_noalloc: token-level Query-Probe Top-K for hosts that cannot allocate device memory when they
    call (a plug-in whose engine owns the whole GPU heap, a process under a memory quota, a loop that may not stall on
    cudaMalloc).  No Context and no workspace: the scratch is a fixed ~4.6 MiB array inside libsaf3r.so, so num_heads * N must
    stay <= NOALLOC_MAX_KEYS (Saf3rError with status ERR_CAPACITY otherwise).  `idx` is the caller's int32 [H][K] device tensor and
    receives the same indices Context.token_probe_select returns; q / k / idx must be on the current CUDA device.  All calls on a
    device share the one array: keep them in one stream order.  The first call per device does a one-off address look-up; make it
    at start-up.  This wrapper allocates nothing either."""
    L = load_library()
    err = C.create_string_buffer(512)
    st = L.saf3r_token_probe_select_noalloc(q.data_ptr(), k.data_ptr(), C.byref(shape), int(K), idx.data_ptr(), _stream_ptr(stream),
                                            err, len(err))
    if st != OK:
        raise Saf3rError(st, err.value.decode())
    return idx


def token_topk_query_sizes(shape: ShapeC, K: int) -> tuple[int, int, int]:
    """Host-only: (select workspace bytes, idx entries = N*S*K, worst-case tiles) of the token-wise per-frame Top-K calls."""
    L = load_library()
    a, b, c = C.c_size_t(), C.c_int64(), C.c_int64()
    st = L.saf3r_token_topk_query_sizes(C.byref(shape), int(K), C.byref(a), C.byref(b), C.byref(c))
    if st != OK:
        raise Saf3rError(st, "saf3r_token_topk_query_sizes rejected (shape, K)")
    return int(a.value), int(b.value), int(c.value)


def token_query_sizes(shape: ShapeC, K: int) -> tuple[int, int]:
    """Host-only: (select workspace bytes, attention workspace bytes) of the token-granular calls."""
    L = load_library()
    a, b = C.c_size_t(), C.c_size_t()
    st = L.saf3r_token_query_sizes(C.byref(shape), int(K), C.byref(a), C.byref(b))
    if st != OK:
        raise Saf3rError(st, "saf3r_token_query_sizes rejected (shape, K)")
    return int(a.value), int(b.value)


def query_sizes(shape: ShapeC, cfgs) -> tuple[int, int]:
    """Host-only: (list entries, workspace bytes) saf3r_select needs.  Works without a GPU."""
    L = load_library()
    arr = cfgs if isinstance(cfgs, C.Array) else make_cfgs(cfgs)
    n, w = C.c_int64(), C.c_size_t()
    st = L.saf3r_query_sizes(C.byref(shape), arr, C.byref(n), C.byref(w))
    if st != OK:
        raise Saf3rError(st, "saf3r_query_sizes rejected (shape, cfg)")
    return int(n.value), int(w.value)
