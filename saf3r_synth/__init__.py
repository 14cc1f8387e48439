"""Seeded synthetic inputs for the SAF3R hot path (shared by the oracle-side tests and the CUDA-side tests/bench).

This module holds NONE of the method's arithmetic (no pooling, scoring, selection or attention): it only
draws Q/K/V tensors shaped like VGGT-style global attention and the per-head configuration values, following
the recipe in DESIGN.md "Input recipe".  It imports neither the oracle nor the CUDA package.

Stand-in statement: the paper measures on real scenes pushed through trained VGGT / pi^3 / DA3 weights
(PAPER.md:L132-136, L213); none of those exist here.  These inputs take the paper's shapes (tokens per frame,
frames, heads, layers), its sparsity levels and the four head types of PAPER.md:L80.

bf16 tensors travel as numpy uint16 bit patterns, layout [H][N][D].  Head configurations travel as plain dicts
with the ten int32 fields (type, stride, offset, keep_blocks, static_mode, anchor_frame, band_radius, topk_scope,
topk_per_frame, score_mode); each side marshals them into its own struct.
"""
from __future__ import annotations

import math
from concurrent.futures import ThreadPoolExecutor
from dataclasses import dataclass, field

import numpy as np

# enum values (restated here as data, see include/saf3r.h for the CUDA side and oracle/saf3r_oracle.c for the oracle)
HEAD_DENSE, HEAD_UNIFORM_STRIDE, HEAD_STATIC, HEAD_QUERY_PROBE_TOPK, HEAD_BLOCK_TOPK, HEAD_CACHED = range(6)
STATIC_ANCHOR, STATIC_FRAME_LOCAL, STATIC_POSITION_BAND = range(3)
SCOPE_GLOBAL, SCOPE_PER_FRAME = range(2)
SCORE_DOT, SCORE_COSINE = range(2)

CFG_FIELDS = ("type", "stride", "offset", "keep_blocks", "static_mode", "anchor_frame", "band_radius",
              "topk_scope", "topk_per_frame", "score_mode")

GEN_UNIFORM, GEN_FRAME_LOCAL, GEN_SAME_POSITION, GEN_SINK, GEN_ANCHOR = "uniform", "frame_local", "same_position", "sink", "anchor"
NUM_SPECIAL = 5          # camera/register tokens per frame (BASELINE.json: 16x16+5, 37x37+5)
NOISE_STD = 0.1          # BASELINE.json config 1: "+ N(0,0.1) noise"
SCAN_STD = 1.0           # scanning heads: diffuse but non-constant logits (std 1 after the 1/sqrt(D) scale)
MATCH_LOGIT = 12.0       # g^2/sqrt(D): matched logit exceeds unmatched ones by ~12 ("scaled so softmax is peaked")


def cfg(**kw) -> dict:
    d = {k: 0 for k in CFG_FIELDS}
    d["stride"] = 1
    for k, v in kw.items():
        assert k in d, k
        d[k] = int(v)
    return d


def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """Round-to-nearest-even fp32 -> bf16, returned as uint16 bit patterns (finite inputs)."""
    u = np.ascontiguousarray(x, np.float32).view(np.uint32)
    r = ((u >> 16) & 1) + np.uint32(0x7FFF)
    return ((u + r) >> 16).astype(np.uint16)


def bf16_bits_to_f32(b: np.ndarray) -> np.ndarray:
    return (np.ascontiguousarray(b, np.uint16).astype(np.uint32) << 16).view(np.float32)


@dataclass
class Shape:
    S: int   # frames
    G: int   # patch grid side; T = G*G + NUM_SPECIAL tokens per frame (special tokens first, reading A17)
    H: int
    D: int
    B: int

    @property
    def T(self) -> int:
        return self.G * self.G + NUM_SPECIAL

    @property
    def N(self) -> int:
        return self.S * self.T

    @property
    def NB(self) -> int:
        return (self.N + self.B - 1) // self.B


@dataclass
class Layer:
    shape: Shape
    q: np.ndarray            # uint16 [H][N][D]
    k: np.ndarray
    v: np.ndarray
    cfgs: list               # H dicts
    gens: list               # H generator names
    planted: list = field(default_factory=list)


def _rng(seed: int, layer: int, head: int, tensor: int) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(key=[(seed << 32) ^ (layer << 16) ^ head, tensor]))


def _unit(r: np.random.Generator, n: int, D: int) -> np.ndarray:
    x = r.standard_normal((n, D), dtype=np.float32)
    return x / np.linalg.norm(x, axis=1, keepdims=True)


def _position_codes(r: np.random.Generator, G: int, D: int) -> np.ndarray:
    """[T][D]: random unit codes for the special tokens, random-Fourier codes for patches
    phi(x,y) = sqrt(2/D) cos(W (x,y)/l + b) with l = 1.5 patches, so phi(p).phi(p') ~ exp(-|dp|^2 / 2 l^2)."""
    W = r.standard_normal((D, 2), dtype=np.float32)
    b = r.uniform(0.0, 2.0 * math.pi, (D,)).astype(np.float32)
    ys, xs = np.meshgrid(np.arange(G, dtype=np.float32), np.arange(G, dtype=np.float32), indexing="ij")
    xy = np.stack([xs.ravel(), ys.ravel()], axis=1)                       # row-major patches
    phi = math.sqrt(2.0 / D) * np.cos(xy @ W.T / 1.5 + b)
    return np.concatenate([_unit(r, NUM_SPECIAL, D), phi.astype(np.float32)], axis=0)


def make_head(gen: str, sh: Shape, seed: int, layer: int, head: int):
    """One head's (q, k, v) as uint16 [N][D] bf16 bit patterns."""
    S, T, N, D = sh.S, sh.T, sh.N, sh.D
    g = math.sqrt(MATCH_LOGIT * math.sqrt(D))
    rq, rk, rv, rc = (_rng(seed, layer, head, t) for t in range(4))
    std = SCAN_STD if gen == GEN_UNIFORM else NOISE_STD
    q = rq.standard_normal((N, D), dtype=np.float32) * np.float32(std)
    k = rk.standard_normal((N, D), dtype=np.float32) * np.float32(std)
    v = rv.standard_normal((N, D), dtype=np.float32)
    pos = np.arange(N) % T
    frm = np.arange(N) // T
    if gen == GEN_FRAME_LOCAL:
        e = _unit(rc, S, D) * np.float32(g)
        q += e[frm]
        k += e[frm]
    elif gen == GEN_SAME_POSITION:
        code = _position_codes(rc, sh.G, D) * np.float32(g)
        q += code[pos]
        k += code[pos]
    elif gen == GEN_SINK:
        u = _unit(rc, 1, D)[0] * np.float32(g)
        q += u
        k[pos < NUM_SPECIAL] += u
    elif gen == GEN_ANCHOR:
        u = _unit(rc, 1, D)[0] * np.float32(g)
        q += u
        k[frm == 0] += u
    elif gen != GEN_UNIFORM:
        raise ValueError(gen)
    return f32_to_bf16_bits(q), f32_to_bf16_bits(k), f32_to_bf16_bits(v)


def make_layer(sh: Shape, gens: list, cfgs: list, seed: int, layer: int = 0, threads: int = 8) -> Layer:
    assert len(gens) == sh.H == len(cfgs)
    q = np.empty((sh.H, sh.N, sh.D), np.uint16)
    k = np.empty_like(q)
    v = np.empty_like(q)

    def one(h):
        q[h], k[h], v[h] = make_head(gens[h], sh, seed, layer, h)

    with ThreadPoolExecutor(max_workers=threads) as ex:
        list(ex.map(one, range(sh.H)))
    return Layer(sh, q, k, v, list(cfgs), list(gens))


# ------------------------------------------------------------------------------------------------------------
# BASELINE.json configs restated as concrete recipes
# ------------------------------------------------------------------------------------------------------------
def shape_c1() -> Shape:
    return Shape(S=4, G=16, H=4, D=64, B=64)          # T=261, N=1044, NB=17, tail 20


def shape_c2() -> Shape:
    return Shape(S=32, G=37, H=16, D=64, B=128)       # T=1374, N=43968, NB=344, tail 64


def shape_c3() -> Shape:
    return Shape(S=100, G=37, H=16, D=64, B=128)      # N=137400, NB=1074, tail 56


def shape_c4() -> Shape:
    return Shape(S=200, G=37, H=16, D=64, B=128)      # N=274800, NB=2147, tail 112


def shape_c5() -> Shape:
    return Shape(S=500, G=37, H=16, D=64, B=128)      # N=687000, NB=5368, tail 24


def config_c1(seed: int = 1) -> Layer:
    sh = shape_c1()
    gens = [GEN_UNIFORM, GEN_FRAME_LOCAL, GEN_SAME_POSITION, GEN_SINK]
    cfgs = [cfg(type=HEAD_UNIFORM_STRIDE, stride=2),
            cfg(type=HEAD_STATIC, static_mode=STATIC_FRAME_LOCAL),
            cfg(type=HEAD_BLOCK_TOPK, topk_scope=SCOPE_PER_FRAME, topk_per_frame=1),
            cfg(type=HEAD_QUERY_PROBE_TOPK, keep_blocks=4)]
    return make_layer(sh, gens, cfgs, seed)


def mixed_heads(sh: Shape):
    """C2's mix: 4 heads per generator, per-head sparsity 80-95 %."""
    NB, S = sh.NB, sh.S
    gens, cfgs = [], []
    for s in (5, 8, 12, 20):
        gens.append(GEN_UNIFORM); cfgs.append(cfg(type=HEAD_UNIFORM_STRIDE, stride=s))
    for _ in range(4):
        gens.append(GEN_FRAME_LOCAL); cfgs.append(cfg(type=HEAD_STATIC, static_mode=STATIC_FRAME_LOCAL))
    for rho in (0.20, 0.15, 0.10, 0.05):
        gens.append(GEN_SAME_POSITION)
        cfgs.append(cfg(type=HEAD_BLOCK_TOPK, topk_scope=SCOPE_GLOBAL, keep_blocks=max(1, round(rho * NB))))
    for n in (S, S, 2 * S, 2 * S):
        gens.append(GEN_SINK); cfgs.append(cfg(type=HEAD_QUERY_PROBE_TOPK, keep_blocks=min(NB, n)))
    return gens, cfgs


def config_c2(seed: int = 2) -> Layer:
    sh = shape_c2()
    gens, cfgs = mixed_heads(sh)
    return make_layer(sh, gens, cfgs, seed)


def stack_layer_heads(sh: Shape, layer: int, seed: int = 3):
    """C3: per layer a seeded mix of head types (4 each +- 2) and a per-layer sparsity sigma ~ U(0.70, 0.97)
    mapped to n = max(1, round((1 - sigma) NB)); frame-local heads keep their closed-form set."""
    r = np.random.Generator(np.random.Philox(key=[seed * 1000 + layer, 77]))
    sigma = float(r.uniform(0.70, 0.97))
    n = max(1, round((1.0 - sigma) * sh.NB))
    counts = np.array([4, 4, 4, 4]) + r.integers(-2, 3, size=4)
    while counts.sum() != sh.H:                      # re-balance to exactly H heads
        i = int(r.integers(0, 4))
        counts[i] += 1 if counts.sum() < sh.H else (-1 if counts[i] > 1 else 0)
    kinds = [GEN_UNIFORM] * counts[0] + [GEN_FRAME_LOCAL] * counts[1] + [GEN_SAME_POSITION] * counts[2] + [GEN_SINK] * counts[3]
    kinds = [kinds[i] for i in r.permutation(len(kinds))]
    cfgs = []
    for kd in kinds:
        if kd == GEN_UNIFORM:
            cfgs.append(cfg(type=HEAD_UNIFORM_STRIDE, stride=0, keep_blocks=n))
        elif kd == GEN_FRAME_LOCAL:
            cfgs.append(cfg(type=HEAD_STATIC, static_mode=STATIC_FRAME_LOCAL))
        elif kd == GEN_SAME_POSITION:
            cfgs.append(cfg(type=HEAD_BLOCK_TOPK, topk_scope=SCOPE_GLOBAL, keep_blocks=n))
        else:
            cfgs.append(cfg(type=HEAD_QUERY_PROBE_TOPK, keep_blocks=n))
    return kinds, cfgs, sigma


def config_c3_layer(layer: int, seed: int = 3, sh: Shape | None = None) -> Layer:
    sh = sh or shape_c3()
    gens, cfgs, _ = stack_layer_heads(sh, layer, seed)
    return make_layer(sh, gens, cfgs, seed * 1000 + layer, layer)


def sweep_heads(sh: Shape, gen: str, ratio: float):
    """C4: all heads one generator type, kept-block ratio `ratio`."""
    n = max(1, round(ratio * sh.NB))
    if gen == GEN_UNIFORM:
        c = cfg(type=HEAD_UNIFORM_STRIDE, stride=0, keep_blocks=n)
    elif gen == GEN_SAME_POSITION:
        c = cfg(type=HEAD_BLOCK_TOPK, topk_scope=SCOPE_GLOBAL, keep_blocks=n)
    elif gen == GEN_SINK:
        c = cfg(type=HEAD_QUERY_PROBE_TOPK, keep_blocks=n)
    else:
        raise ValueError(gen)
    return [gen] * sh.H, [dict(c) for _ in range(sh.H)]


def make_features(sh: Shape, seed: int) -> np.ndarray:
    """[N][D] bf16 bits: per-sequence patch features standing in for the encoder's last-block output (PAPER.md:L126 uses DINO
    features; none exist here): the same-position code of every token + N(0, 0.1) noise, shared by all layers."""
    return make_head(GEN_SAME_POSITION, sh, seed, layer=9999, head=0)[0]
