"""Pins P1-P13: the CPU oracle checked against what the paper and the mathematics fix --
closed forms, brute force in numpy float64 on tiny inputs, invariants, library routines.  CPU only."""
import os

import numpy as np
import pytest

import oracle as orc
import saf3r_synth as sy

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def rand_bits(rng, shape, scale=1.0):
    return sy.f32_to_bf16_bits(rng.standard_normal(shape).astype(np.float32) * np.float32(scale))


def ocfg(d):
    return orc.make_cfg(**d)


def lists_to_mask(row_ptr, col_idx, N, B):
    NB = (N + B - 1) // B
    m = np.zeros((N, N), bool)
    for I in range(NB):
        for J in col_idx[row_ptr[I]:row_ptr[I + 1]]:
            m[I * B:(I + 1) * B, J * B:(J + 1) * B] = True
    return m


def brute_masked_attention(q, k, v, mask):
    """softmax(QK^T/sqrt(D) restricted to mask) V in float64 with a dense matrix (plain definition)."""
    qf, kf, vf = (sy.bf16_bits_to_f32(x).astype(np.float64) for x in (q, k, v))
    z = qf @ kf.T / np.sqrt(qf.shape[1])
    z = np.where(mask, z, -np.inf)
    m = z.max(axis=1, keepdims=True)
    m = np.where(np.isfinite(m), m, 0.0)
    w = np.exp(z - m)
    l = w.sum(axis=1, keepdims=True)
    out = np.where(l > 0, (w @ vf) / np.where(l > 0, l, 1.0), 0.0)
    with np.errstate(divide="ignore"):
        lse = (m + np.log(l))[:, 0]
    return out, lse


ALL_CFGS_TINY = [
    sy.cfg(type=sy.HEAD_DENSE),
    sy.cfg(type=sy.HEAD_UNIFORM_STRIDE, stride=3, offset=1),
    sy.cfg(type=sy.HEAD_UNIFORM_STRIDE, stride=0, keep_blocks=5),
    sy.cfg(type=sy.HEAD_STATIC, static_mode=sy.STATIC_ANCHOR, anchor_frame=1),
    sy.cfg(type=sy.HEAD_STATIC, static_mode=sy.STATIC_FRAME_LOCAL),
    sy.cfg(type=sy.HEAD_STATIC, static_mode=sy.STATIC_POSITION_BAND, band_radius=2),
    sy.cfg(type=sy.HEAD_QUERY_PROBE_TOPK, keep_blocks=4),
    sy.cfg(type=sy.HEAD_BLOCK_TOPK, topk_scope=sy.SCOPE_GLOBAL, keep_blocks=3),
    sy.cfg(type=sy.HEAD_BLOCK_TOPK, topk_scope=sy.SCOPE_GLOBAL, keep_blocks=3, score_mode=sy.SCORE_COSINE),
    sy.cfg(type=sy.HEAD_BLOCK_TOPK, topk_scope=sy.SCOPE_PER_FRAME, topk_per_frame=1),
    sy.cfg(type=sy.HEAD_BLOCK_TOPK, topk_scope=sy.SCOPE_PER_FRAME, topk_per_frame=2, score_mode=sy.SCORE_COSINE),
]


# ---------------------------------------------------------------- P1
@pytest.mark.parametrize("N,B,D", [(90, 8, 8), (1044, 64, 64)])
def test_p1_keep_all_lists_reproduce_dense(N, B, D):
    rng = np.random.default_rng(1)
    q, k, v = (rand_bits(rng, (N, D)) for _ in range(3))
    NB = (N + B - 1) // B
    row_ptr = np.arange(NB + 1, dtype=np.int64) * NB
    col = np.tile(np.arange(NB, dtype=np.int32), NB)
    rows = slice(0, N) if N < 200 else slice(0, 128)
    qb = None if N < 200 else np.array([0, 1], np.int64)
    o1, l1 = orc.attn_lists(q, k, v, B, row_ptr, col, qb)
    o2, l2 = orc.attn_dense(q, k, v, rows.start, rows.stop)
    assert np.abs(o1[rows] - o2[rows]).max() <= 1e-6
    assert np.abs(l1[rows] - l2[rows]).max() <= 1e-5


# ---------------------------------------------------------------- P2
@pytest.mark.parametrize("ci", range(len(ALL_CFGS_TINY)))
@pytest.mark.parametrize("S,T,B,D", [(4, 23, 8, 8), (3, 32, 4, 8)])
def test_p2_bruteforce_tiny(ci, S, T, B, D):
    rng = np.random.default_rng(100 + ci)
    N = S * T
    q, k, v = rand_bits(rng, (N, D), 1.5), rand_bits(rng, (N, D), 1.5), rand_bits(rng, (N, D))
    hl = orc.select_head(q, k, S, T, B, ocfg(ALL_CFGS_TINY[ci]))
    NB = (N + B - 1) // B
    for I in range(NB):
        row = hl.col_idx[hl.row_ptr[I]:hl.row_ptr[I + 1]]
        assert len(row) >= 1 and np.all(np.diff(row) > 0) and row[0] >= 0 and row[-1] < NB
    out, lse = orc.attn_lists(q, k, v, B, hl.row_ptr, hl.col_idx)
    ref, ref_lse = brute_masked_attention(q, k, v, lists_to_mask(hl.row_ptr, hl.col_idx, N, B))
    assert np.abs(out - ref).max() <= 2e-6
    assert np.abs(lse - ref_lse).max() <= 2e-6


def test_p2_empty_list_convention():
    rng = np.random.default_rng(5)
    N, B, D = 40, 8, 8
    q, k, v = (rand_bits(rng, (N, D)) for _ in range(3))
    row_ptr = np.array([0, 0, 2, 2, 3, 3], np.int64)
    col = np.array([1, 4, 0], np.int32)
    out, lse = orc.attn_lists(q, k, v, B, row_ptr, col)
    for I in (0, 2, 4):
        assert np.all(out[I * B:(I + 1) * B] == 0) and np.all(np.isneginf(lse[I * B:(I + 1) * B]))
    ref, _ = brute_masked_attention(q, k, v, lists_to_mask(row_ptr, col, N, B))
    assert np.abs(out - ref).max() <= 2e-6


# ---------------------------------------------------------------- P3
def test_p3_rows_sum_to_one_and_lse_bound():
    rng = np.random.default_rng(3)
    S, T, B, D = 4, 23, 8, 8
    N = S * T
    q, k = rand_bits(rng, (N, D), 2.0), rand_bits(rng, (N, D), 2.0)
    ones = sy.f32_to_bf16_bits(np.ones((N, D), np.float32))
    _, lse_dense = orc.attn_dense(q, k, ones)
    for c in ALL_CFGS_TINY:
        hl = orc.select_head(q, k, S, T, B, ocfg(c))
        out, lse = orc.attn_lists(q, k, ones, B, hl.row_ptr, hl.col_idx)
        assert np.abs(out - 1.0).max() <= 1e-6          # sum_j softmax_ij * 1 = 1
        assert np.all(lse <= lse_dense + 1e-6)          # a subset of the keys cannot have a larger log-sum-exp


# ---------------------------------------------------------------- P4
def test_p4_uniform_stride_closed_form():
    rng = np.random.default_rng(4)
    S, T, B, D = 5, 29, 4, 8
    N = S * T
    NB = (N + B - 1) // B
    q, k = rand_bits(rng, (N, D)), rand_bits(rng, (N, D))
    for s, o in [(1, 0), (2, 0), (3, 2), (7, 6), (NB, 0), (NB + 5, 3)]:
        hl = orc.select_head(q, k, S, T, B, ocfg(sy.cfg(type=sy.HEAD_UNIFORM_STRIDE, stride=s, offset=o)))
        expect = np.arange(o, NB, s, dtype=np.int32)
        assert len(expect) == -(-(NB - o) // s)                     # ceil((NB - o)/s), "fixed stride"
        for I in range(NB):
            assert np.array_equal(hl.col_idx[hl.row_ptr[I]:hl.row_ptr[I + 1]], expect)
    for n in (1, 2, 5, NB // 2, NB):
        hl = orc.select_head(q, k, S, T, B, ocfg(sy.cfg(type=sy.HEAD_UNIFORM_STRIDE, stride=0, keep_blocks=n)))
        row = hl.col_idx[hl.row_ptr[0]:hl.row_ptr[1]]
        assert len(row) == n and row[0] == 0 and np.all(np.diff(row) > 0)
        assert np.array_equal(hl.col_idx, np.tile(row, NB))
    # keep_blocks form when n does not divide NB: block i of the n kept ones is floor(i * NB / n) (reading A1; a ceiling or a
    # rounding would pass every check above).  NB = 37 is prime, so no n in 2..36 divides it.
    S3, T3 = 4, 37          # N = 148, B = 4 -> NB = 37
    q3, k3 = rand_bits(rng, (148, D)), rand_bits(rng, (148, D))
    for n in (2, 5, 7, 19, 36):
        hl = orc.select_head(q3, k3, S3, T3, 4, ocfg(sy.cfg(type=sy.HEAD_UNIFORM_STRIDE, stride=0, keep_blocks=n)))
        expect = np.floor(np.arange(n) * 37 / n).astype(np.int32)
        assert len(set(expect.tolist())) == n
        for I in range(37):
            assert np.array_equal(hl.col_idx[hl.row_ptr[I]:hl.row_ptr[I + 1]], expect), f"keep_blocks={n} row {I}"
    # keep_blocks form equals the stride set when s | NB
    S2, T2 = 4, 24          # N = 96, B = 4 -> NB = 24
    q2, k2 = rand_bits(rng, (96, D)), rand_bits(rng, (96, D))
    for s in (2, 3, 4, 6, 8):
        a = orc.select_head(q2, k2, S2, T2, 4, ocfg(sy.cfg(type=sy.HEAD_UNIFORM_STRIDE, stride=s)))
        b = orc.select_head(q2, k2, S2, T2, 4, ocfg(sy.cfg(type=sy.HEAD_UNIFORM_STRIDE, stride=0, keep_blocks=24 // s)))
        assert np.array_equal(a.col_idx, b.col_idx)


# ---------------------------------------------------------------- P5
def test_p5_probe_equals_column_mean_of_full_scores():
    """ranking keys by the column-wise average of S = QK^T/sqrt(D) equals ranking by qbar K^T/sqrt(D);
    block-lifted: the probe of block J is the mean of S over all queries and the keys of J."""
    rng = np.random.default_rng(6)
    S, T, B, D = 4, 23, 8, 8
    N = S * T
    NB = (N + B - 1) // B
    q, k = rand_bits(rng, (N, D), 1.3), rand_bits(rng, (N, D), 1.3)
    qf, kf = sy.bf16_bits_to_f32(q).astype(np.float64), sy.bf16_bits_to_f32(k).astype(np.float64)
    Sfull = qf @ kf.T / np.sqrt(D)
    colmean = Sfull.mean(axis=0)
    blockmean = np.array([colmean[J * B:(J + 1) * B].mean() for J in range(NB)])
    n = 4
    hl = orc.select_head(q, k, S, T, B, ocfg(sy.cfg(type=sy.HEAD_QUERY_PROBE_TOPK, keep_blocks=n)), want_scores=True)
    assert np.abs(hl.scores[0] - blockmean).max() <= 1e-6
    expect = np.sort(np.argsort(-blockmean, kind="stable")[:n])
    for I in range(NB):
        assert np.array_equal(hl.col_idx[hl.row_ptr[I]:hl.row_ptr[I + 1]], expect)
    # token level (B = 1): exactly the paper's statement
    hl1 = orc.select_head(q, k, S, T, 1, ocfg(sy.cfg(type=sy.HEAD_QUERY_PROBE_TOPK, keep_blocks=7)), want_scores=True)
    assert np.abs(hl1.scores[0] - colmean).max() <= 1e-6
    assert np.array_equal(hl1.col_idx[:7], np.sort(np.argsort(-colmean, kind="stable")[:7]))


# ---------------------------------------------------------------- P6
def test_p6_per_frame_topk_counts_match_paper_fractions():
    gold = {}
    for line in open(os.path.join(GOLD, "paper_key_fractions.txt")):
        if line.strip() and not line.startswith("#"):
            name, val = line.split()
            gold[name] = float(val)
    # token granularity (B = 1) is the paper's own setting: K keys from each frame's T tokens -> K/T of all keys.
    rng = np.random.default_rng(7)
    S, T, D = 3, 40, 8
    N = S * T
    q, k = rand_bits(rng, (N, D)), rand_bits(rng, (N, D))
    for K in (2, 4):
        hl = orc.select_head(q, k, S, T, 1, ocfg(sy.cfg(type=sy.HEAD_BLOCK_TOPK, topk_scope=sy.SCOPE_PER_FRAME, topk_per_frame=K)))
        assert np.all(np.diff(hl.row_ptr) == S * K)
        frac = (S * K) / N
        assert abs(frac - K / T) < 1e-12
    # the paper's printed numbers: K/T at T = 1024 tokens per frame gives 0.2 % / 0.4 %, and (1/32)/(2/T) = 16
    T_paper = 1024
    assert round(100 * 2 / T_paper, 1) == gold["topk_k2_fraction_percent"]
    assert round(100 * 4 / T_paper, 1) == gold["topk_k4_fraction_percent"]
    assert (1 / 32) / (2 / T_paper) == gold["stride32_vs_k2_sparsity_ratio"]
    # block granularity: S * k_f blocks per q-block when k_f <= min_g |C_g|
    S, T, B = 4, 23, 4
    N = S * T
    q, k = rand_bits(rng, (N, D)), rand_bits(rng, (N, D))
    for kf in (1, 2, 3):
        hl = orc.select_head(q, k, S, T, B, ocfg(sy.cfg(type=sy.HEAD_BLOCK_TOPK, topk_scope=sy.SCOPE_PER_FRAME, topk_per_frame=kf)), want_scores=True)
        assert np.all(np.diff(hl.row_ptr) == S * kf)
        NB = (N + B - 1) // B
        frame_of_block = (np.arange(NB) * B) // T
        for I in range(NB):
            row = hl.col_idx[hl.row_ptr[I]:hl.row_ptr[I + 1]]
            for g in range(S):
                kept = [J for J in row if frame_of_block[J] == g]
                rest = [J for J in range(NB) if frame_of_block[J] == g and J not in kept]
                assert len(kept) == kf
                assert min(hl.scores[I][kept]) >= max(hl.scores[I][rest])     # property: kept dominate the rest of the frame


# ---------------------------------------------------------------- P7
@pytest.mark.parametrize("cosine", [False, True])
def test_p7_pooled_score_is_mean_of_token_pair_scores(cosine):
    """PAPER.md:L126 "block-level similarities averaged over multiple tokens": s[I][J] = mean over token pairs."""
    rng = np.random.default_rng(8)
    S, T, B, D = 3, 23, 8, 8          # N = 69, tail block of 5 tokens
    N = S * T
    NB = (N + B - 1) // B
    q, k = rand_bits(rng, (N, D), 1.2), rand_bits(rng, (N, D), 1.2)
    qf, kf = sy.bf16_bits_to_f32(q).astype(np.float64), sy.bf16_bits_to_f32(k).astype(np.float64)
    if cosine:
        tok = (qf / np.linalg.norm(qf, axis=1, keepdims=True)) @ (kf / np.linalg.norm(kf, axis=1, keepdims=True)).T
    else:
        tok = qf @ kf.T / np.sqrt(D)
    expect = np.array([[tok[I * B:(I + 1) * B, J * B:(J + 1) * B].mean() for J in range(NB)] for I in range(NB)])
    c = sy.cfg(type=sy.HEAD_BLOCK_TOPK, keep_blocks=2, score_mode=sy.SCORE_COSINE if cosine else sy.SCORE_DOT)
    hl = orc.select_head(q, k, S, T, B, ocfg(c), want_scores=True)
    assert np.abs(hl.scores - expect).max() <= 1e-6
    # and the pieces: pooled vectors and a single score row
    qt, kt = orc.pool(q, B, cosine), orc.pool(k, B, cosine)
    row = orc.score_row(qt[2], kt, 1.0 if cosine else 1.0 / np.sqrt(D))
    assert np.abs(row - expect[2]).max() <= 1e-6
    assert np.abs(orc.mean_query(q) - qf.mean(axis=0)).max() <= 1e-6


# ---------------------------------------------------------------- P8
def test_p8_static_closed_forms():
    rng = np.random.default_rng(9)
    D = 8
    for S, T, B in [(4, 23, 8), (5, 261, 64), (3, 1374, 128)]:
        N = S * T
        NB = (N + B - 1) // B
        q = k = rand_bits(rng, (N, D))
        for a in range(S):
            hl = orc.select_head(q, k, S, T, B, ocfg(sy.cfg(type=sy.HEAD_STATIC, static_mode=sy.STATIC_ANCHOR, anchor_frame=a)))
            lo, hi = (a * T) // B, ((a + 1) * T - 1) // B
            assert np.all(np.diff(hl.row_ptr) == hi - lo + 1)
            assert np.array_equal(hl.col_idx[:hi - lo + 1], np.arange(lo, hi + 1))
            # every token of the anchor frame is covered and no block lies fully outside the frame
            assert lo * B <= a * T and (hi + 1) * B >= min(N, (a + 1) * T)
        # frame-local: a q-block's list covers exactly the frames of its tokens
        hl = orc.select_head(q, k, S, T, B, ocfg(sy.cfg(type=sy.HEAD_STATIC, static_mode=sy.STATIC_FRAME_LOCAL)))
        tok_frame = np.arange(N) // T
        for I in range(NB):
            row = hl.col_idx[hl.row_ptr[I]:hl.row_ptr[I + 1]]
            frames = set(tok_frame[I * B:(I + 1) * B])
            need = {j // B for j in range(N) if tok_frame[j] in frames}
            assert set(row) == need
        # position band with r >= T is dense
        hl = orc.select_head(q, k, S, T, B, ocfg(sy.cfg(type=sy.HEAD_STATIC, static_mode=sy.STATIC_POSITION_BAND, band_radius=T)))
        assert np.all(np.diff(hl.row_ptr) == NB)
    # S = 1: frame-local == dense
    q = k = rand_bits(rng, (50, D))
    hl = orc.select_head(q, k, 1, 50, 8, ocfg(sy.cfg(type=sy.HEAD_STATIC, static_mode=sy.STATIC_FRAME_LOCAL)))
    assert np.all(np.diff(hl.row_ptr) == 7)
    # position band r = 0 at token granularity (B = 1): query (f, p) attends key (g, p) for every frame g
    S, T = 4, 11
    q = k = rand_bits(rng, (S * T, D))
    hl = orc.select_head(q, k, S, T, 1, ocfg(sy.cfg(type=sy.HEAD_STATIC, static_mode=sy.STATIC_POSITION_BAND, band_radius=0)))
    for i in range(S * T):
        assert np.array_equal(hl.col_idx[hl.row_ptr[i]:hl.row_ptr[i + 1]], np.arange(S) * T + i % T)
    hl = orc.select_head(q, k, S, T, 1, ocfg(sy.cfg(type=sy.HEAD_STATIC, static_mode=sy.STATIC_POSITION_BAND, band_radius=2)))
    for i in range(S * T):
        p = i % T
        exp = sorted(g * T + pp for g in range(S) for pp in range(max(0, p - 2), min(T - 1, p + 2) + 1))
        assert list(hl.col_idx[hl.row_ptr[i]:hl.row_ptr[i + 1]]) == exp


@pytest.mark.parametrize("S,T,B", [(4, 23, 8), (5, 261, 64), (3, 1374, 128), (6, 10, 16), (4, 24, 8), (5, 12, 8)])
def test_p8_position_band_and_anchor_per_token_at_block_granularity(S, T, B):
    """P8 at B > 1, derived per TOKEN ("fixed across all image blocks", L96; readings A5/A6/A12): q-blocks straddle
    frames here, so a row can hold two position intervals, each clipped to [0, T-1] in its own frame.  The expected block set of
    q-block I is built token by token -- every token t of I reaches the positions p(t)-r .. p(t)+r (clipped) of EVERY frame g --
    and only then lifted to blocks; nothing of the oracle's interval arithmetic is restated.  (B=16 > T=10: whole frames inside
    one q-block; T=24, B=8: frame
    boundaries coincide with block boundaries, where clipping at T instead of T-1 would leak into the next frame's first block.)"""
    rng = np.random.default_rng(19)
    N, D = S * T, 8
    NB = (N + B - 1) // B
    q = k = rand_bits(rng, (N, D))
    for r in (0, 3, T // 2):
        hl = orc.select_head(q, k, S, T, B, ocfg(sy.cfg(type=sy.HEAD_STATIC, static_mode=sy.STATIC_POSITION_BAND, band_radius=r)))
        for I in range(NB):
            expect = set()
            for t in range(I * B, min(N, (I + 1) * B)):
                p = t % T
                for pp in range(max(0, p - r), min(T - 1, p + r) + 1):
                    expect.update((g * T + pp) // B for g in range(S))
            row = hl.col_idx[hl.row_ptr[I]:hl.row_ptr[I + 1]]
            assert np.all(np.diff(row) > 0)
            assert set(row.tolist()) == expect, f"POSITION_BAND S={S} T={T} B={B} r={r} row {I}"
    for a in range(S):                                            # ANCHOR: the blocks that hold a token of frame a, from the token list
        hl = orc.select_head(q, k, S, T, B, ocfg(sy.cfg(type=sy.HEAD_STATIC, static_mode=sy.STATIC_ANCHOR, anchor_frame=a)))
        expect = sorted({t // B for t in range(N) if t // T == a})
        for I in range(NB):
            assert hl.col_idx[hl.row_ptr[I]:hl.row_ptr[I + 1]].tolist() == expect, f"ANCHOR a={a} row {I}"


# ---------------------------------------------------------------- P9
def test_p9_softmax_special_cases():
    rng = np.random.default_rng(10)
    N, B, D = 44, 8, 8
    NB = 6
    k, v = rand_bits(rng, (N, D)), rand_bits(rng, (N, D))
    row_ptr = np.arange(NB + 1, dtype=np.int64) * 2
    col = np.array([0, 5, 1, 2, 0, 3, 2, 4, 1, 5, 3, 4], np.int32)
    vf = sy.bf16_bits_to_f32(v).astype(np.float64)
    # Q = 0  =>  o_i = mean of v over A(i)
    zero = np.zeros((N, D), np.uint16)
    out, lse = orc.attn_lists(zero, k, v, B, row_ptr, col)
    for I in range(NB):
        keys = np.concatenate([np.arange(J * B, min(N, (J + 1) * B)) for J in col[2 * I:2 * I + 2]])
        assert np.abs(out[I * B:(I + 1) * B] - vf[keys].mean(axis=0)).max() <= 1e-6
        assert np.abs(lse[I * B:(I + 1) * B] - np.log(len(keys))).max() <= 1e-6
    # V constant => o = that constant
    q = rand_bits(rng, (N, D), 3.0)
    cst = sy.f32_to_bf16_bits(np.full((N, D), 0.375, np.float32))
    out, _ = orc.attn_lists(q, k, cst, B, row_ptr, col)
    assert np.abs(out - 0.375).max() <= 1e-6
    # one dominant key => o_i -> v_j
    kd = sy.bf16_bits_to_f32(k).copy() * 0.01
    qd = np.zeros((N, D), np.float32)
    qd[:, 0] = 40.0
    kd[13, 0] = 40.0                                         # key 13 (block 1) gets logit 40*40/sqrt(8)
    out, _ = orc.attn_lists(sy.f32_to_bf16_bits(qd), sy.f32_to_bf16_bits(kd), v, B,
                            np.arange(NB + 1, dtype=np.int64), np.ones(NB, np.int32))
    assert np.abs(out - vf[13]).max() <= 1e-6
    # permuting tokens inside a k-block (K and V together) leaves O unchanged
    perm = np.arange(N)
    perm[8:16] = 8 + rng.permutation(8)
    o1, _ = orc.attn_lists(q, k, v, B, row_ptr, col)
    o2, _ = orc.attn_lists(q, k[perm], v[perm], B, row_ptr, col)
    assert np.abs(o1 - o2).max() <= 1e-6


# ---------------------------------------------------------------- P10
def test_p10_topn_total_order():
    rng = np.random.default_rng(11)
    for NB in (1, 5, 33, 200):
        s = rng.standard_normal(NB).astype(np.float32)
        s[rng.integers(0, NB, NB // 3)] = 0.5                # planted ties
        if NB > 4:
            s[[1, 3]] = s.max() + 1                          # tie at the top
        for n in {1, 2, NB // 2 + 1, NB}:
            expect = np.sort(np.argsort(-s.astype(np.float64), kind="stable")[:n])    # library: stable sort = (score desc, index asc)
            assert np.array_equal(orc.topn(s, n, False), expect)
            assert np.array_equal(orc.topn(s, n, True), expect)
    s = np.array([1, 7, 7, 7, 3], np.float32)
    assert list(orc.topn(s, 2, True)) == [1, 2] and list(orc.topn(s, 2, False)) == [1, 2]


# ---------------------------------------------------------------- P11
def test_p11_planted_structure_is_recovered_on_c1():
    L = sy.config_c1()
    sh = L.shape
    S, T, B, NB = sh.S, sh.T, sh.B, sh.NB
    # head 2: same-position, per-frame top-1 -> in every OTHER frame the kept block overlaps the q-block's own positions
    hl = orc.select_head(L.q[2], L.k[2], S, T, B, ocfg(L.cfgs[2]))
    hits = tot = 0
    for I in range(NB):
        t0, t1 = I * B, min(sh.N, (I + 1) * B)
        if t0 // T != (t1 - 1) // T:
            continue
        p0, p1 = t0 % T, (t1 - 1) % T
        for J in hl.col_idx[hl.row_ptr[I]:hl.row_ptr[I + 1]]:
            j0, j1 = J * B, min(sh.N, (J + 1) * B) - 1
            # positions covered by block J (may wrap a frame boundary)
            pos = {j % T for j in range(j0, j1 + 1)}
            tot += 1
            hits += bool(pos & set(range(max(0, p0 - 20), min(T, p1 + 21))))
    assert hits / tot >= 0.9
    # head 3: sink -> probe top-S picks the S blocks that hold the special tokens (positions 0..4 of each frame)
    hl = orc.select_head(L.q[3], L.k[3], S, T, B, ocfg(L.cfgs[3]))
    assert sorted(hl.col_idx[:S]) == sorted({(f * T) // B for f in range(S)})


# ---------------------------------------------------------------- P12
def test_p12_masked_attention_matches_torch_sdpa_on_c1():
    import torch
    L = sy.config_c1()
    sh = L.shape
    for h in range(sh.H):
        hl = orc.select_head(L.q[h], L.k[h], sh.S, sh.T, sh.B, ocfg(L.cfgs[h]))
        out, _ = orc.attn_lists(L.q[h], L.k[h], L.v[h], sh.B, hl.row_ptr, hl.col_idx)
        mask = torch.from_numpy(lists_to_mask(hl.row_ptr, hl.col_idx, sh.N, sh.B))
        qf, kf, vf = (torch.from_numpy(sy.bf16_bits_to_f32(x)) for x in (L.q[h], L.k[h], L.v[h]))
        ref = torch.nn.functional.scaled_dot_product_attention(qf[None], kf[None], vf[None], attn_mask=mask[None])[0].numpy()
        assert np.abs(out - ref).max() <= 1e-5


# ---------------------------------------------------------------- P13
def test_p13_nmse():
    rng = np.random.default_rng(13)
    a = rng.standard_normal((50, 8)).astype(np.float32)
    assert orc.nmse(a, a) == 0.0
    b = a + np.float32(0.1) * rng.standard_normal((50, 8)).astype(np.float32)
    exp = ((a.astype(np.float64) - b) ** 2).sum() / (a.astype(np.float64) ** 2).sum()
    assert abs(orc.nmse(a, b) - exp) <= 1e-12
    assert abs(orc.nmse(a, np.zeros_like(a)) - 1.0) <= 1e-12       # dropping the head entirely ("Skip")


# ------------------------------------------------------------------------------------------------ P14-P16: token-granular variants
def _rand_bits(rng, shape, scale=1.0):
    return sy.f32_to_bf16_bits((rng.standard_normal(shape) * scale).astype(np.float32))


def test_p14_attn_tokens_bruteforce_and_reductions():
    """O4-token against what fixes it: numpy float64 brute force with an explicit key mask; idx = all tokens == the
    separately coded dense function; idx = the tokens of a block list == the block-list function; empty set convention;
    and the library routine torch SDPA with a boolean mask."""
    rng = np.random.default_rng(14)
    N, D = 75, 16
    q, k, v = _rand_bits(rng, (N, D), 1.5), _rand_bits(rng, (N, D), 1.5), _rand_bits(rng, (N, D))
    qf, kf, vf = (sy.bf16_bits_to_f32(x).astype(np.float64) for x in (q, k, v))
    idx = np.array(sorted(rng.choice(N, 17, replace=False)), np.int64)
    out, lse = orc.attn_tokens(q, k, v, idx)
    z = qf @ kf[idx].T / np.sqrt(D)
    w = np.exp(z - z.max(1, keepdims=True))
    ref = (w / w.sum(1, keepdims=True)) @ vf[idx]
    assert np.abs(out - ref).max() <= 1e-6
    assert np.abs(lse - (z.max(1) + np.log(w.sum(1)))).max() <= 1e-5
    # all tokens == dense
    o_all, l_all = orc.attn_tokens(q, k, v, np.arange(N))
    o_d, l_d = orc.attn_dense(q, k, v)
    assert np.abs(o_all - o_d).max() <= 1e-6 and np.abs(l_all - l_d).max() <= 1e-6
    # tokens of a block list == block-list attention (B = 8, blocks {1, 4, 9 (tail)})
    B, blocks = 8, [1, 4, 9]
    tok = np.concatenate([np.arange(b * B, min((b + 1) * B, N)) for b in blocks])
    NB = (N + B - 1) // B
    rp = np.arange(NB + 1, dtype=np.int64) * len(blocks)
    col = np.tile(np.array(blocks, np.int32), NB)
    o_b, _ = orc.attn_lists(q, k, v, B, rp, col)
    o_t, _ = orc.attn_tokens(q, k, v, tok)
    assert np.abs(o_b - o_t).max() <= 1e-6
    # empty set, and a sub-range of rows
    o_e, l_e = orc.attn_tokens(q, k, v, np.zeros(0, np.int64))
    assert np.all(o_e == 0) and np.all(np.isneginf(l_e))
    o_r, _ = orc.attn_tokens(q, k, v, idx, 10, 20)
    assert np.isnan(o_r[:10]).all() and np.isnan(o_r[20:]).all() and np.abs(o_r[10:20] - ref[10:20]).max() <= 1e-6
    # library routine
    import torch
    mask = torch.zeros(N, N, dtype=torch.bool)
    mask[:, torch.from_numpy(idx)] = True
    sd = torch.nn.functional.scaled_dot_product_attention(torch.from_numpy(qf)[None], torch.from_numpy(kf)[None],
                                                          torch.from_numpy(vf)[None], attn_mask=mask)[0].numpy()
    assert np.abs(out - sd).max() <= 1e-6


def test_p15_token_stride_closed_form():
    """Uniform sampling at token level: keys {o + i*s}; count ceil((N-o)/s) = the 1/s of PAPER.md:L241 (s = 32
    -> 3.1 %, s = 64 -> 1.6 %); s = 1 is dense; attending a strided set == dense attention over the sub-sampled K/V arrays."""
    rng = np.random.default_rng(15)
    N, D = 203, 8
    q, k, v = _rand_bits(rng, (N, D)), _rand_bits(rng, (N, D)), _rand_bits(rng, (N, D))
    for s, o in ((1, 0), (3, 0), (3, 2), (32, 5), (64, 0)):
        idx = np.arange(o, N, s)
        assert len(idx) == -(-(N - o) // s)
        out, _ = orc.attn_tokens(q, k, v, idx)
        if s == 1:
            assert np.abs(out - orc.attn_dense(q, k, v)[0]).max() <= 1e-6
        # same numbers from the dense function on the sub-sampled keys (queries padded / truncated to the same count)
        ks, vs = np.ascontiguousarray(k[o::s]), np.ascontiguousarray(v[o::s])
        m = len(ks)
        qs = np.ascontiguousarray(np.concatenate([q, q])[:m]) if m <= 2 * N else None
        d, _ = orc.attn_dense(qs, ks, vs)
        take = min(m, N)
        assert np.abs(out[:take] - d[:take]).max() <= 1e-6
    # the paper's printed ratio (tests/golden/paper_key_fractions.txt): stride 32 keeps 16x the keys of K = 2 per
    # frame at T = 1024 tokens per frame, with the token-level count of this function
    vals = dict(l.split() for l in open(os.path.join(GOLD, "paper_key_fractions.txt")) if l.strip() and not l.startswith("#"))
    T = 1024
    assert len(np.arange(0, 8 * T, 32)) / (8 * 2) == float(vals["stride32_vs_k2_sparsity_ratio"])


def test_p16_token_probe_is_column_mean_of_scores_and_topk_order():
    """the probe equals the column-wise average of S = QK^T/sqrt(D) (numpy float64) and induces the same
    ranking; the top-K set follows the total order (score desc, index asc) - checked against numpy's stable argsort with
    planted exact ties (duplicated key rows)."""
    rng = np.random.default_rng(16)
    N, D, K = 120, 16, 9
    q, k = _rand_bits(rng, (N, D)), _rand_bits(rng, (N, D))
    k[40] = k[7]
    k[41] = k[7]
    k[99] = k[7]
    qf, kf = sy.bf16_bits_to_f32(q).astype(np.float64), sy.bf16_bits_to_f32(k).astype(np.float64)
    col_mean = (qf @ kf.T / np.sqrt(D)).mean(0)
    idx, p = orc.token_probe_topk(q, k, K)
    assert np.abs(p - col_mean).max() <= 1e-6
    assert p[40] == p[7] == p[41] == p[99]
    order = np.argsort(-p.astype(np.float64), kind="stable")     # score desc, index asc
    assert np.array_equal(idx, np.sort(order[:K]))
    # a cut that falls inside the tie group takes the lower indices
    rank7 = int(np.nonzero(order == 7)[0][0])
    idx2, _ = orc.token_probe_topk(q, k, rank7 + 2)
    assert 7 in idx2 and 40 in idx2 and 41 not in idx2 and 99 not in idx2


# ---------------------------------------------------------------- P17 (NEXT-4: Top-K U stride)
def test_p17_union_lists_is_the_set_union():
    """orc_union_lists against numpy's union1d (a library routine) row by row on random ascending lists, with empty rows; the
    algebra of a union (idempotent, commutative, identity = empty lists, |A U B| = |A| + |B| - |A n B|); and the case the paper
    names ("combining Top-K with uniform striding"): block top-k lists U stride lists of the same head contain both,
    and the attention over the union equals the brute-force masked attention with mask_topk OR mask_stride."""
    rng = np.random.default_rng(17)
    NB, rows = 37, 23

    def rand_lists():
        rp, cols = [0], []
        for _ in range(rows):
            n = int(rng.integers(0, NB + 1)) if rng.random() > 0.2 else 0
            cols.append(np.sort(rng.choice(NB, n, replace=False)).astype(np.int32))
            rp.append(rp[-1] + n)
        return np.array(rp, np.int64), (np.concatenate(cols) if cols else np.zeros(0, np.int32))

    (ra, ca), (rb, cb) = rand_lists(), rand_lists()
    ro, co = orc.union_lists(ra, ca, rb, cb, NB)
    inter = 0
    for I in range(rows):
        a, b = ca[ra[I]:ra[I + 1]], cb[rb[I]:rb[I + 1]]
        assert np.array_equal(co[ro[I]:ro[I + 1]], np.union1d(a, b))
        inter += len(np.intersect1d(a, b))
    assert len(co) == len(ca) + len(cb) - inter
    r2, c2 = orc.union_lists(rb, cb, ra, ca, NB)
    assert np.array_equal(r2, ro) and np.array_equal(c2, co)                       # commutative
    r3, c3 = orc.union_lists(ra, ca, ra, ca, NB)
    assert np.array_equal(r3, ra) and np.array_equal(c3, ca)                       # idempotent
    r4, c4 = orc.union_lists(ra, ca, np.zeros(rows + 1, np.int64), np.zeros(0, np.int32), NB)
    assert np.array_equal(r4, ra) and np.array_equal(c4, ca)                       # empty lists are the identity
    # Top-K U stride on a tiny head, attention against the explicit OR of the two masks
    S, T, B, D = 4, 23, 8, 8
    N = S * T
    q, k, v = rand_bits(rng, (N, D), 1.5), rand_bits(rng, (N, D), 1.5), rand_bits(rng, (N, D))
    top = orc.select_head(q, k, S, T, B, ocfg(sy.cfg(type=sy.HEAD_BLOCK_TOPK, topk_scope=sy.SCOPE_GLOBAL, keep_blocks=2)))
    strd = orc.select_head(q, k, S, T, B, ocfg(sy.cfg(type=sy.HEAD_UNIFORM_STRIDE, stride=4, offset=1)))
    ru, cu = orc.union_lists(top.row_ptr, top.col_idx, strd.row_ptr, strd.col_idx, (N + B - 1) // B)
    out, lse = orc.attn_lists(q, k, v, B, ru, cu)
    mask = lists_to_mask(top.row_ptr, top.col_idx, N, B) | lists_to_mask(strd.row_ptr, strd.col_idx, N, B)
    ref, ref_lse = brute_masked_attention(q, k, v, mask)
    assert np.abs(out - ref).max() <= 2e-6 and np.abs(lse - ref_lse).max() <= 2e-6


# ---------------------------------------------------------------- P18 (NEXT-4: static broadcast of frame 0's local map)
def test_p18_broadcast_of_frame0_local_map():
    """orc_attn_broadcast_frame0 (reading A18) against: (a) the explicit N x N matrix whose every T x T image block
    is frame 0's unnormalised map, row-normalised, times V (numpy float64 brute force); (b) S = 1: the separately written dense
    function on frame 0; (c) V identical in every frame: frame 0's dense local attention, for every frame; (d) rows sum to one
    (V = 1 gives 1) and the output does not depend on the queries or keys of frames >= 1."""
    rng = np.random.default_rng(18)
    S, T, D = 4, 23, 8
    N = S * T
    q, k, v = rand_bits(rng, (N, D), 1.5), rand_bits(rng, (N, D), 1.5), rand_bits(rng, (N, D))
    out, lse = orc.attn_broadcast_frame0(q, k, v, S, T)
    qf, kf, vf = (sy.bf16_bits_to_f32(x).astype(np.float64) for x in (q, k, v))
    z0 = qf[:T] @ kf[:T].T / np.sqrt(D)
    A = np.tile(np.exp(z0 - z0.max(axis=1, keepdims=True)), (S, S))                # every image block = frame 0's block
    A /= A.sum(axis=1, keepdims=True)
    assert np.abs(out - A @ vf).max() <= 2e-6
    ref_lse = np.tile(np.log(np.exp(z0).sum(axis=1) * S), S)
    assert np.abs(lse - ref_lse).max() <= 2e-6
    o1, l1 = orc.attn_broadcast_frame0(q[:T], k[:T], v[:T], 1, T)                    # (b)
    o2, l2 = orc.attn_dense(q[:T], k[:T], v[:T])
    assert np.abs(o1 - o2).max() <= 1e-6 and np.abs(l1 - l2).max() <= 1e-5
    vrep = np.tile(v[:T], (S, 1))                                                    # (c)
    o3, _ = orc.attn_broadcast_frame0(q, k, vrep, S, T)
    assert np.abs(o3 - np.tile(o2, (S, 1))).max() <= 1e-6
    ones = sy.f32_to_bf16_bits(np.ones((N, D), np.float32))                          # (d)
    o4, _ = orc.attn_broadcast_frame0(q, k, ones, S, T)
    assert np.abs(o4 - 1.0).max() <= 1e-6
    q2, k2 = q.copy(), k.copy()
    q2[T:], k2[T:] = rand_bits(rng, (N - T, D)), rand_bits(rng, (N - T, D))
    o5, _ = orc.attn_broadcast_frame0(q2, k2, v, S, T)
    assert np.array_equal(o5, out)


# ---------------------------------------------------------------- P19 (NEXT-2 iii: token-wise per-frame Top-K)
def test_p19_token_topk_per_frame_and_per_query_attention():
    """orc_token_topk_per_frame / orc_token_cosine_row / orc_attn_token_lists against numpy:
    (a) the cosine row equals the normalised float64 Gram matrix; (b) per query and per frame the kept set equals numpy's stable
    argsort of (-cos) cut at K, with planted EXACT ties (duplicated feature rows) going to the lower index; (c) the kept fraction is
    K/T, the paper's printed 0.2 % / 0.4 % for K = 2 / 4 (tests/golden/paper_key_fractions.txt);
    (d) K = T keeps every token and the per-query attention equals the separately written dense function; (e) the per-query
    attention equals the brute-force masked softmax with the explicit N x N boolean mask; (f) identical lists for all queries
    reduce to orc_attn_tokens; padding entries (-1) are ignored and an all-padding list gives 0 / -inf."""
    rng = np.random.default_rng(19)
    S, T, D, K = 4, 23, 8, 3
    N = S * T
    feat = rand_bits(rng, (N, D))
    feat[T + 5] = feat[T + 2]                                   # exact ties inside frame 1 ...
    feat[2 * T + 7] = feat[2 * T + 1]
    feat[2 * T + 9] = feat[2 * T + 1]                           # ... and a triple inside frame 2
    ff = sy.bf16_bits_to_f32(feat).astype(np.float64)
    fn = ff / np.linalg.norm(ff, axis=1, keepdims=True)
    G = fn @ fn.T
    for i in (0, T + 2, N - 1):
        assert np.abs(orc.token_cosine_row(feat, i) - G[i]).max() <= 1e-6                      # (a)
    idx = orc.token_topk_per_frame(feat, S, T, K)
    assert idx.shape == (N, S, K)
    for i in range(N):
        c32 = orc.token_cosine_row(feat, i)                    # ranking happens on the stored fp32 values
        for g in range(S):
            order = np.argsort(-c32[g * T:(g + 1) * T], kind="stable")[:K]
            assert np.array_equal(idx[i, g], np.sort(order) + g * T), (i, g)                   # (b)
            assert np.all(np.diff(idx[i, g]) > 0)
        assert i in idx[i, i // T]                              # reading A19: the query itself is its own best match
    # planted ties: for a query outside frame 2 with K = 1.. the lower index of an exact tie wins
    one = orc.token_topk_per_frame(feat, S, T, 1)
    i = 2 * T + 7                                               # its own frame holds two exact copies (indices 2T+1, 2T+7, 2T+9 all cos = 1)
    assert one[i, 2, 0] == 2 * T + 1
    lines = [l.split() for l in open(os.path.join(GOLD, "paper_key_fractions.txt")) if l.strip() and not l.startswith("#")]
    gold = {l[0]: l[1:] for l in lines}                         # (c)
    Tp = int(round(32 * 2 * float(gold["stride32_vs_k2_sparsity_ratio"][0])))   # (1/32) / (2/T) = 16  =>  T = 1024
    for key, kk in (("topk_k2_fraction_percent", 2), ("topk_k4_fraction_percent", 4)):
        full_count = orc.token_topk_per_frame(rand_bits(rng, (2 * Tp, D)), 2, Tp, kk, 0, 1).size    # keys of one query: S * K
        assert abs(100.0 * full_count / (2 * Tp) - float(gold[key][0])) < 0.05
    assert idx.shape[1] * idx.shape[2] / N == K / T
    q, k, v = rand_bits(rng, (N, D), 1.5), rand_bits(rng, (N, D), 1.5), rand_bits(rng, (N, D))
    full = orc.token_topk_per_frame(feat, S, T, T)              # (d)
    assert np.array_equal(full.reshape(N, N), np.tile(np.arange(N, dtype=np.int32), (N, 1)))
    o1, l1 = orc.attn_token_lists(q, k, v, full.reshape(N, -1))
    o2, l2 = orc.attn_dense(q, k, v)
    assert np.abs(o1 - o2).max() <= 1e-6 and np.abs(l1 - l2).max() <= 1e-5
    mask = np.zeros((N, N), bool)                               # (e)
    for i in range(N):
        mask[i, idx[i].ravel()] = True
    o3, l3 = orc.attn_token_lists(q, k, v, idx.reshape(N, -1))
    ref, ref_lse = brute_masked_attention(q, k, v, mask)
    assert np.abs(o3 - ref).max() <= 2e-6 and np.abs(l3 - ref_lse).max() <= 2e-6
    same = np.sort(rng.choice(N, 11, replace=False)).astype(np.int32)                          # (f)
    lists = np.tile(np.concatenate([same, [-1, -1]]).astype(np.int32), (N, 1))
    o4, l4 = orc.attn_token_lists(q, k, v, lists)
    o5, l5 = orc.attn_tokens(q, k, v, same.astype(np.int64))
    assert np.abs(o4 - o5).max() <= 1e-6 and np.abs(l4 - l5).max() <= 1e-5
    o6, l6 = orc.attn_token_lists(q, k, v, np.full((N, 4), -1, np.int32))
    assert np.all(o6 == 0) and np.all(np.isneginf(l6))


# ---------------------------------------------------------------- P20
@pytest.mark.parametrize("mode", ["dot", "cosine", "probe"])
def test_p20_global_topn_kept_set_is_the_argsort_of_the_mean_token_pair_scores(mode):
    """PAPER.md:L126 (block-wise similarity Top-K), L98/L124 (query probe): the kept set of row I of a BLOCK_TOPK / GLOBAL head is
    the n largest of that row's block scores, ties to the lower index, written ascending - checked against numpy on the
    mean-of-token-pair matrix built here from the tokens (what P7 pins the scores to), never on the oracle's own scores.  A cut one
    short or one long (n - 1, n + 1), a ranking of a neighbouring row, or a descending / unsorted list fails this.  The oracle
    ranks the fp32 it stores, so the expected scores are rounded to fp32 before ranking."""
    cosine, probe = mode == "cosine", mode == "probe"
    rng = np.random.default_rng(200 + int(cosine))
    S, T, B, D = 3, 23, 8, 8          # N = 69, NB = 9, tail block of 5 tokens
    N = S * T
    NB = (N + B - 1) // B
    q, k = rand_bits(rng, (N, D), 1.2), rand_bits(rng, (N, D), 1.2)
    qf, kf = sy.bf16_bits_to_f32(q).astype(np.float64), sy.bf16_bits_to_f32(k).astype(np.float64)
    if cosine:
        tok = (qf / np.linalg.norm(qf, axis=1, keepdims=True)) @ (kf / np.linalg.norm(kf, axis=1, keepdims=True)).T
    else:
        tok = qf @ kf.T / np.sqrt(D)
    if probe:    # one row for every I: the mean over ALL queries and the keys of block J
        E = np.array([[tok[:, J * B:(J + 1) * B].mean() for J in range(NB)]] * NB)
    else:
        E = np.array([[tok[I * B:(I + 1) * B, J * B:(J + 1) * B].mean() for J in range(NB)] for I in range(NB)])
    E32 = E.astype(np.float32)
    gaps = np.diff(np.sort(E32, axis=1), axis=1).min()
    assert gaps > 1e-5, "the seeded scores must be tie-free for this pin to be unambiguous"
    assert len({tuple(np.argsort(-E32[I], kind="stable")[:2]) for I in range(NB)}) > 1 or probe   # rows really differ
    for n in (1, 2, NB // 2, NB - 1, NB):
        if probe:
            c = sy.cfg(type=sy.HEAD_QUERY_PROBE_TOPK, keep_blocks=n)
        else:
            c = sy.cfg(type=sy.HEAD_BLOCK_TOPK, topk_scope=sy.SCOPE_GLOBAL, keep_blocks=n,
                       score_mode=sy.SCORE_COSINE if cosine else sy.SCORE_DOT)
        hl = orc.select_head(q, k, S, T, B, ocfg(c))
        assert np.array_equal(hl.row_ptr, np.arange(NB + 1, dtype=np.int64) * n)
        for I in range(NB):
            expect = np.sort(np.argsort(-E32[I], kind="stable")[:n]).astype(np.int32)
            assert np.array_equal(hl.col_idx[hl.row_ptr[I]:hl.row_ptr[I + 1]], expect), f"n={n} row {I}"


def test_p20_global_topn_breaks_exact_ties_towards_the_lower_index():
    """The total order of include/saf3r.h (score descending, then index ascending) at the level of select_head: two k-blocks made
    of identical tokens have bit-identical scores in every row; when the cut falls between them the lower index is kept."""
    rng = np.random.default_rng(210)
    S, T, B, D = 4, 16, 8, 8          # N = 64, NB = 8, no tail
    N, NB = S * T, 8
    q, k = rand_bits(rng, (N, D), 1.2), rand_bits(rng, (N, D), 1.2)
    k[5 * B:6 * B] = k[2 * B:3 * B]   # block 5 == block 2
    kf = sy.bf16_bits_to_f32(k).astype(np.float64)
    qf = sy.bf16_bits_to_f32(q).astype(np.float64)
    E = np.array([[(qf[I * B:(I + 1) * B] @ kf[J * B:(J + 1) * B].T).mean() for J in range(NB)] for I in range(NB)]) / np.sqrt(D)
    for n in range(1, NB + 1):
        hl = orc.select_head(q, k, S, T, B, ocfg(sy.cfg(type=sy.HEAD_BLOCK_TOPK, topk_scope=sy.SCOPE_GLOBAL, keep_blocks=n)))
        for I in range(NB):
            row = hl.col_idx[hl.row_ptr[I]:hl.row_ptr[I + 1]].tolist()
            rank = np.argsort(-E[I].astype(np.float32), kind="stable")
            others = [J for J in rank if J not in (2, 5)]
            pos2 = int(np.sum(E[I][others] > E[I][2]))              # blocks strictly ahead of the tied pair
            if n == pos2 + 1:
                assert 2 in row and 5 not in row, f"n={n} row {I}: the cut splits the tie, block 2 must win"
            elif n >= pos2 + 2:
                assert 2 in row and 5 in row
            else:
                assert 2 not in row and 5 not in row
