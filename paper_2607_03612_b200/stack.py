"""The global-attention stack with an index cache.

The paper computes its similarity Top-K indices ONCE per input from encoder features and reuses them in every layer's
correspondence heads ("the indices are cached and reused by all subsequent DINO Top-K kernels").  Here:
  build_cache(features)  one ordinary saf3r_select on (features, features) with BLOCK_TOPK / COSINE rules -> cache lists
  run()                  per layer: saf3r_select_cached (CACHED heads copy their rows from the cache, so the layer pools and
                         scores only for its QUERY_PROBE heads) + saf3r_sparse_attn
  capture() / replay()   the whole stack (select + attention of every layer) as ONE CUDA graph: the C entry points only
                         enqueue kernels on the given stream (no allocation, no synchronisation), so they can be captured
Argument marshalling and buffer ownership only; every step runs in the library's kernels.
"""
from __future__ import annotations

from . import HEAD_BLOCK_TOPK, HEAD_CACHED, Context, Lists, ShapeC, query_sizes


def cached_cfgs(cfgs: list[dict], cache_cfgs: list[dict], slot_of_head: dict[int, int]) -> list[dict]:
    """Rewrite the BLOCK_TOPK heads named in slot_of_head {head -> cache slot} as CACHED heads that repeat the rule of the
    cache slot they read (the rule fixes the list lengths)."""
    out = []
    for h, c in enumerate(cfgs):
        if h in slot_of_head:
            src = cache_cfgs[slot_of_head[h]]
            assert src["type"] == HEAD_BLOCK_TOPK
            d = dict(src)
            d.update(type=HEAD_CACHED, offset=slot_of_head[h])
            out.append(d)
        else:
            out.append(dict(c))
    return out


class GlobalStack:
    def __init__(self, ctx: Context, shape: ShapeC, layer_cfgs: list[list[dict]], cache_cfgs: list[dict] | None = None,
                 device="cuda:0"):
        import torch
        self.ctx, self.shape, self.layer_cfgs, self.cache_cfgs = ctx, shape, layer_cfgs, cache_cfgs
        self.dev = torch.device(device)
        N = shape.num_frames * shape.tokens_per_frame
        self.NB = (N + shape.block - 1) // shape.block
        self.lists, ws_max = [], 0
        for cfgs in layer_cfgs:
            entries, ws = query_sizes(shape, cfgs)
            ws_max = max(ws_max, ws)
            self.lists.append(Lists(torch.empty(shape.num_heads * self.NB + 1, dtype=torch.int64, device=self.dev),
                                    torch.empty(max(entries, 1), dtype=torch.int32, device=self.dev)))
        self.cache = None
        self.cache_shape = None
        if cache_cfgs:
            self.cache_shape = ShapeC(shape.num_frames, shape.tokens_per_frame, len(cache_cfgs), shape.head_dim, shape.block,
                                      N * shape.head_dim, shape.head_dim)
            entries, ws = query_sizes(self.cache_shape, cache_cfgs)
            ws_max = max(ws_max, ws)
            self.cache = Lists(torch.empty(len(cache_cfgs) * self.NB + 1, dtype=torch.int64, device=self.dev),
                               torch.empty(max(entries, 1), dtype=torch.int32, device=self.dev))
        self.ws = torch.empty(ws_max, dtype=torch.uint8, device=self.dev)   # one workspace: the stack is stream-ordered
        self.qkv, self.out, self.graph = None, None, None

    def bind(self, qkv, out=None):
        """qkv: per layer (q, k, v) device tensors [H][N][D] bf16 (static addresses if the stack is captured)."""
        import torch
        assert len(qkv) == len(self.layer_cfgs)
        self.qkv = qkv
        self.out = out if out is not None else [torch.empty_like(q) for q, _, _ in qkv]
        self.graph = None

    def build_cache(self, features, stream=None):
        """features: [C][N][D] bf16 device tensor, C = len(cache_cfgs) (one slot per rule; slots may share storage)."""
        self.ctx.select(features, features, self.cache_shape, self.cache_cfgs, workspace=self.ws, lists=self.cache, stream=stream)

    def run(self, stream=None):
        n_cache = len(self.cache_cfgs) if self.cache_cfgs else 0
        for (q, k, v), cfgs, lists, out in zip(self.qkv, self.layer_cfgs, self.lists, self.out):
            self.ctx.select(q, k, self.shape, cfgs, workspace=self.ws, lists=lists, stream=stream,
                            cache=self.cache, cache_heads=n_cache)
            self.ctx.sparse_attn(q, k, v, self.shape, lists, out=out, stream=stream)
        return self.out

    def capture(self):
        """Capture run() as one CUDA graph (the cache must have been built; its buffers are read, not re-captured)."""
        import torch
        s = torch.cuda.Stream(device=self.dev)
        s.wait_stream(torch.cuda.current_stream(self.dev))
        with torch.cuda.stream(s):
            self.run(stream=s)                                   # warm-up outside capture (tensor-map cache, lazy init)
        torch.cuda.current_stream(self.dev).wait_stream(s)
        torch.cuda.synchronize(self.dev)
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):
            self.run(stream=s)
        self.graph = g
        return g

    def replay(self):
        self.graph.replay()
        return self.out
