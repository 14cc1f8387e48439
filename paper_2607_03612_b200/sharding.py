"""Host-side sharding helpers for N > 1 processes (one per GPU).

The hot path has no exchange step inside it: pooling, scoring, selection and attention of head h touch only Q_h, K_h, V_h
("for each head h", L124), and layers are independent problems.  So N ranks split LAYERS (what bench.py does:
weak scaling, no data-path collective) or HEADS of one layer (no collective either; an all-gather of O only if the caller's
next op wants every head on every GPU).  This module holds the partitioning arithmetic and the max-over-ranks reduction
bench.py uses for timing; it launches nothing on the GPU.
"""
from __future__ import annotations

from . import ShapeC, make_cfgs, query_sizes


def head_costs(shape: ShapeC, cfgs) -> list[int]:
    """Executed FLOP of saf3r_sparse_attn per head: 4*B^2*D per listed (q-block, k-block) pair (reading A15).
    List lengths are a closed form of (shape, cfg), so this needs no data and no GPU (saf3r_query_sizes, one head at a time)."""
    arr = make_cfgs(cfgs)
    one = ShapeC(shape.num_frames, shape.tokens_per_frame, 1, shape.head_dim, shape.block, shape.stride_head, shape.stride_token)
    out = []
    for h in range(len(arr)):
        entries, _ = query_sizes(one, make_cfgs([arr[h]]))
        out.append(int(entries) * 4 * shape.block * shape.block * shape.head_dim)
    return out


def assign_heads(costs: list[int], world: int) -> list[list[int]]:
    """Longest-processing-time-first assignment of heads to ranks by cost; deterministic (ties: lower head index, lower
    rank).  Every head appears exactly once; ranks may be empty when world > len(costs)."""
    if world < 1:
        raise ValueError("world must be >= 1")
    order = sorted(range(len(costs)), key=lambda h: (-costs[h], h))
    load = [0] * world
    parts: list[list[int]] = [[] for _ in range(world)]
    for h in order:
        r = min(range(world), key=lambda i: (load[i], i))
        parts[r].append(h)
        load[r] += costs[h]
    return [sorted(p) for p in parts]


def layers_for_rank(n_layers: int, rank: int, world: int) -> list[int]:
    """Round-robin split of independent layers."""
    return list(range(rank, n_layers, world))


def max_over_ranks(value: float, device=None) -> float:
    """MAX all-reduce of a scalar over the default process group (gloo: CPU tensor, nccl: pass the CUDA device).
    Returns `value` unchanged when torch.distributed is not initialised."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
