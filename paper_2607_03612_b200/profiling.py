"""Offline head profiling (Sec. 4.2): a driver over the library, not a kernel.

For every head: start from the baseline c_base (uniform sampling at sparsity sigma), evaluate a candidate
set C_h of alternative kernels / settings with equal or higher sparsity, score each by the NMSE of Eq. 1

    E(c) = E_calib[ ||O_full - O_sparse(c)||^2 / ||O_full||^2 ]

and keep   c* = argmin_{c in C_h + {c_base}} E(c)  s.t.  Omega(c) <= Omega(c_base)   (Eq. 2),

with Omega = executed FLOP of the block-sparse attention (4*B^2*D per listed block pair, a closed form of (shape, c)).
O_full comes from saf3r_dense_attn, O_sparse from saf3r_select + saf3r_sparse_attn; heads are independent, so one call
evaluates a candidate on every head at once.  The two sums of Eq. 1 run in the library too (saf3r_nmse_accumulate).
The paper's calibration data (10 ETH3D sequences) is not available; callers pass their own layers.
"""
from __future__ import annotations

from dataclasses import dataclass, field

from . import (HEAD_BLOCK_TOPK, HEAD_QUERY_PROBE_TOPK, HEAD_STATIC, HEAD_UNIFORM_STRIDE, SCOPE_GLOBAL, SCOPE_PER_FRAME,
               STATIC_ANCHOR, STATIC_FRAME_LOCAL, Context, ShapeC, query_sizes)

_FIELDS = ("type", "stride", "offset", "keep_blocks", "static_mode", "anchor_frame", "band_radius", "topk_scope",
           "topk_per_frame", "score_mode")


def _cfg(**kw) -> dict:
    d = {k: 0 for k in _FIELDS}
    d.update(kw)
    return d


def num_blocks(shape: ShapeC) -> int:
    return (shape.num_frames * shape.tokens_per_frame + shape.block - 1) // shape.block


def cost_flop(shape: ShapeC, cfg: dict) -> int:
    """Omega(c): executed FLOP of one head under configuration c (closed form; no data, no GPU)."""
    one = ShapeC(shape.num_frames, shape.tokens_per_frame, 1, shape.head_dim, shape.block, shape.stride_head, shape.stride_token)
    entries, _ = query_sizes(one, [cfg])
    return int(entries) * 4 * shape.block * shape.block * shape.head_dim


def baseline_cfg(shape: ShapeC, sigma: float) -> dict:
    """c_base: uniform sampling kernel at sparsity sigma (sigma = 0.85 in the paper, L161)."""
    return _cfg(type=HEAD_UNIFORM_STRIDE, stride=0, keep_blocks=max(1, round((1.0 - sigma) * num_blocks(shape))))


def candidate_set(shape: ShapeC, sigma: float) -> list[dict]:
    """C_h: the other kernels under several settings, all with sparsity >= the baseline's (checked by the
    caller through Omega).  Static (frame-local, anchor frame 0), query-probe top-n and block top-k (global n, per-frame k_f)
    on a geometric ladder of budgets below the baseline's."""
    NB = num_blocks(shape)
    n_base = max(1, round((1.0 - sigma) * NB))
    ladder = sorted({max(1, n_base >> s) for s in range(0, 4)}, reverse=True)
    out = [_cfg(type=HEAD_STATIC, static_mode=STATIC_FRAME_LOCAL), _cfg(type=HEAD_STATIC, static_mode=STATIC_ANCHOR, anchor_frame=0)]
    for n in ladder:
        out.append(_cfg(type=HEAD_QUERY_PROBE_TOPK, keep_blocks=n))
        out.append(_cfg(type=HEAD_BLOCK_TOPK, topk_scope=SCOPE_GLOBAL, keep_blocks=n))
    for kf in (1, 2, 3):
        out.append(_cfg(type=HEAD_BLOCK_TOPK, topk_scope=SCOPE_PER_FRAME, topk_per_frame=kf))
    return out


def nmse_per_head(ctx: Context, o_full, o_sparse, shape: ShapeC):
    """Eq. 1 for one calibration sample: ||O_full - O_sparse||_F^2 / ||O_full||_F^2 per head ([H][N][D] tensors); both sums run in
    the library (saf3r_nmse_accumulate, double accumulators)."""
    return ctx.nmse(o_full, o_sparse, shape)


@dataclass
class HeadProfile:
    cfg: dict                      # c*
    nmse: float                    # E(c*)
    nmse_base: float               # E(c_base)
    cost: int                      # Omega(c*)
    cost_base: int                 # Omega(c_base)
    table: list = field(default_factory=list)   # (cfg, E(c), Omega(c), admissible) for every evaluated configuration


def profile_heads(ctx: Context, layers, shape: ShapeC, sigma: float = 0.85, candidates: list[dict] | None = None) -> list[HeadProfile]:
    """layers: calibration samples, each (q, k, v) device tensors [H][N][D] bf16 of the SAME layer of the model (Eq. 1's
    expectation runs over them).  Returns one HeadProfile per head."""
    import torch
    H = shape.num_heads
    base = baseline_cfg(shape, sigma)
    cands = [base] + (candidates if candidates is not None else candidate_set(shape, sigma))
    cost = [cost_flop(shape, c) for c in cands]
    admissible = [w <= cost[0] for w in cost]                 # Omega(c) <= Omega(c_base)
    err = [[0.0] * H for _ in cands]
    for (q, k, v) in layers:
        o_full = ctx.dense_attn(q, k, v, shape, out_fp32=True)
        for ci, c in enumerate(cands):
            if not admissible[ci]:
                continue
            lists = ctx.select(q, k, shape, [c] * H)
            o = ctx.sparse_attn(q, k, v, shape, lists, out_fp32=True)
            e = nmse_per_head(ctx, o_full, o, shape)
            for h in range(H):
                err[ci][h] += e[h] / len(layers)
        torch.cuda.synchronize()
    out = []
    for h in range(H):
        best = 0                                               # progressive substitution from c_base
        for ci in range(1, len(cands)):
            if admissible[ci] and err[ci][h] < err[best][h]:
                best = ci
        out.append(HeadProfile(dict(cands[best]), err[best][h], err[0][h], cost[best], cost[0],
                               [(dict(c), err[ci][h] if admissible[ci] else None, cost[ci], admissible[ci])
                                for ci, c in enumerate(cands)]))
    return out
