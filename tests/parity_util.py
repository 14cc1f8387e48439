"""Helpers shared by the GPU parity tests: upload synthetic layers, compare block lists under the near-tie rule
(reading A11), compare attention outputs under the north_star tolerances."""
from __future__ import annotations

import numpy as np

import oracle as orc
import saf3r_synth as sy

MAX_ABS_TOL = 1e-2     # north_star: attention outputs within max-abs 1e-2 ...
MEAN_ABS_TOL = 1e-3    # ... and mean-abs 1e-3 of the oracle
TIE_REL = 1e-4         # north_star: near-ties within 1e-4 relative of the selection cut


def to_dev(bits: np.ndarray, dev="cuda:0"):
    import torch
    return torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).to(dev).view(torch.bfloat16)


def upload(L: sy.Layer, dev="cuda:0"):
    return to_dev(L.q, dev), to_dev(L.k, dev), to_dev(L.v, dev)


def c_shape(sf, sh: sy.Shape):
    return sf.make_shape(sh.S, sh.T, sh.H, sh.D, sh.B)


def oracle_lists(L: sy.Layer, want_scores=True):
    sh = L.shape
    return [orc.select_head(L.q[h], L.k[h], sh.S, sh.T, sh.B, orc.make_cfg(**L.cfgs[h]), want_scores=want_scores)
            for h in range(sh.H)]


def concat_lists(hls):
    """Per-head oracle lists -> one CSR over H*NB rows."""
    row_ptr = [np.zeros(1, np.int64)]
    cols = []
    base = 0
    for hl in hls:
        row_ptr.append(hl.row_ptr[1:] + base)
        cols.append(hl.col_idx)
        base += hl.row_ptr[-1]
    return np.concatenate(row_ptr), np.concatenate(cols) if cols else np.zeros(0, np.int32)


LIST_REPORT: dict = {}  # tag -> near-tie statistics of compare_lists (written next to REPORT)


def compare_lists(L: sy.Layer, gpu_row_ptr: np.ndarray, gpu_col: np.ndarray, hls, tag: str | None = None) -> dict:
    """Bit-exact comparison except at near-ties of the selection cut.  Returns counts; raises on a real mismatch."""
    sh = L.shape
    NB, S, T, B = sh.NB, sh.S, sh.T, sh.B
    stats = {"rows": 0, "entries": 0, "tie_floored": 0, "tie_strict": 0}
    frame_of_block = (np.arange(NB, dtype=np.int64) * B) // T
    for h, hl in enumerate(hls):
        rp = gpu_row_ptr[h * NB:(h + 1) * NB + 1]
        assert np.array_equal(rp - rp[0], hl.row_ptr), f"head {h}: row_ptr differs"
        g = gpu_col[rp[0]:rp[-1]]
        stats["rows"] += NB
        stats["entries"] += len(g)
        if np.array_equal(g, hl.col_idx):
            continue
        c = L.cfgs[h]
        assert c["type"] in (sy.HEAD_QUERY_PROBE_TOPK, sy.HEAD_BLOCK_TOPK), f"head {h}: closed-form list differs"
        for I in range(NB):
            a = g[hl.row_ptr[I]:hl.row_ptr[I + 1]]
            b = hl.col_idx[hl.row_ptr[I]:hl.row_ptr[I + 1]]
            if np.array_equal(a, b):
                continue
            assert np.all(np.diff(a) > 0), f"head {h} row {I}: GPU list not ascending/unique"
            srow = hl.scores[0] if c["type"] == sy.HEAD_QUERY_PROBE_TOPK else hl.scores[I]
            smax = float(np.abs(srow).max())
            for J in np.setxor1d(a, b):
                if c["type"] == sy.HEAD_BLOCK_TOPK and c["topk_scope"] == sy.SCOPE_PER_FRAME:
                    cand = np.nonzero(frame_of_block == frame_of_block[J])[0]
                    n = min(c["topk_per_frame"], len(cand))
                else:
                    cand = np.arange(NB)
                    n = min(c["keep_blocks"], NB)
                tau = float(np.sort(srow[cand])[::-1][n - 1])
                d = abs(float(srow[J]) - tau)
                assert d <= TIE_REL * max(abs(tau), smax), \
                    f"head {h} row {I}: block {J} differs and is not a near-tie (|s-tau|={d:.3e}, tau={tau:.3e})"
                stats["tie_floored"] += 1
                stats["tie_strict"] += int(d <= TIE_REL * abs(tau))
    if tag:
        LIST_REPORT[tag] = dict(stats)
    return stats


REPORT: dict = {}      # tag -> [worst max-abs, worst mean-abs, checks]; written to gpurun_out/ at session end (conftest.py)


def check_attention(out: np.ndarray, ref: np.ndarray, what: str = "", tag: str | None = None) -> tuple[float, float]:
    """Asserts the north_star tolerances, prints (max-abs, mean-abs) (visible under -s) and keeps the worst per tag (default:
    the first word of `what`, e.g. "C3") for the parity report."""
    mask = ~np.isnan(ref)
    assert mask.any()
    assert not np.isnan(out[mask]).any(), f"{what}: NaN in GPU output"
    d = np.abs(out[mask].astype(np.float64) - ref[mask])
    mx, mean = float(d.max()), float(d.mean())
    print(f"parity {what}: max-abs {mx:.3e} (budget {MAX_ABS_TOL:g}), mean-abs {mean:.3e} (budget {MEAN_ABS_TOL:g})")
    r = REPORT.setdefault(tag or (what.split()[0] if what else "?"), [0.0, 0.0, 0])
    r[0], r[1], r[2] = max(r[0], mx), max(r[1], mean), r[2] + 1
    assert mx <= MAX_ABS_TOL, f"{what}: max-abs {mx:.3e} > {MAX_ABS_TOL}"
    assert mean <= MEAN_ABS_TOL, f"{what}: mean-abs {mean:.3e} > {MEAN_ABS_TOL}"
    return mx, mean
