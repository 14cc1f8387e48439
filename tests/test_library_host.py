"""CPU-only checks of the C-ABI library: it loads, exports every symbol include/saf3r.h declares, and its host-side
sizing (saf3r_query_sizes) agrees with the list lengths the oracle actually produces.  No compute calls."""
import ctypes
import os
import re

import numpy as np
import pytest

import oracle as orc
import paper_2607_03612_b200 as sf
import saf3r_synth as sy

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2607_03612_b200 import build
    build.build()
    return sf.load_library()


def test_exports_match_header(lib):
    hdr = open(os.path.join(ROOT, "include", "saf3r.h")).read()
    declared = set(re.findall(r"\b(saf3r_[a-z_]+)\s*\(", hdr))
    assert declared == set(sf.EXPORTS)
    for name in declared:
        assert hasattr(lib, name), name


def test_struct_layouts():
    assert ctypes.sizeof(sf.HeadCfg) == 40
    assert ctypes.sizeof(sf.ShapeC) == 40
    assert ctypes.sizeof(sf.ListsC) == 24


def rand_bits(rng, shape):
    return sy.f32_to_bf16_bits(rng.standard_normal(shape).astype(np.float32))


@pytest.mark.parametrize("S,T,B", [(4, 261, 64), (5, 294, 128), (3, 50, 64), (2, 1374, 128), (9, 70, 128)])
def test_query_sizes_equals_oracle_list_lengths(lib, S, T, B):
    rng = np.random.default_rng(S * 1000 + T)
    N = S * T
    NB = (N + B - 1) // B
    cfgs = [
        sy.cfg(type=sy.HEAD_DENSE),
        sy.cfg(type=sy.HEAD_UNIFORM_STRIDE, stride=3, offset=2),
        sy.cfg(type=sy.HEAD_UNIFORM_STRIDE, stride=0, keep_blocks=max(1, NB // 3)),
        sy.cfg(type=sy.HEAD_STATIC, static_mode=sy.STATIC_ANCHOR, anchor_frame=S - 1),
        sy.cfg(type=sy.HEAD_STATIC, static_mode=sy.STATIC_FRAME_LOCAL),
        sy.cfg(type=sy.HEAD_STATIC, static_mode=sy.STATIC_POSITION_BAND, band_radius=0),
        sy.cfg(type=sy.HEAD_STATIC, static_mode=sy.STATIC_POSITION_BAND, band_radius=17),
        sy.cfg(type=sy.HEAD_STATIC, static_mode=sy.STATIC_POSITION_BAND, band_radius=T),
        sy.cfg(type=sy.HEAD_QUERY_PROBE_TOPK, keep_blocks=min(NB, 3)),
        sy.cfg(type=sy.HEAD_BLOCK_TOPK, topk_scope=sy.SCOPE_GLOBAL, keep_blocks=min(NB, 4)),
        sy.cfg(type=sy.HEAD_BLOCK_TOPK, topk_scope=sy.SCOPE_PER_FRAME, topk_per_frame=1),
        sy.cfg(type=sy.HEAD_BLOCK_TOPK, topk_scope=sy.SCOPE_PER_FRAME, topk_per_frame=50),
    ]
    q, k = rand_bits(rng, (N, 8)), rand_bits(rng, (N, 8))
    for c in cfgs:
        hl = orc.select_head(q, k, S, T, B, orc.make_cfg(**c))
        entries, ws = sf.query_sizes(sf.make_shape(S, T, 1, 64, B), [c])
        assert entries == hl.row_ptr[-1], c
        assert ws >= 2 * NB * 64 * 4


def test_query_sizes_rejects_bad_arguments(lib):
    ok = sy.cfg(type=sy.HEAD_DENSE)
    with pytest.raises(sf.Saf3rError) as e:
        sf.query_sizes(sf.make_shape(4, 261, 1, 128, 64), [ok])
    assert e.value.status == sf.ERR_UNSUPPORTED
    with pytest.raises(sf.Saf3rError) as e:
        sf.query_sizes(sf.make_shape(4, 261, 1, 64, 32), [ok])
    assert e.value.status == sf.ERR_UNSUPPORTED
    for bad in (sy.cfg(type=9), sy.cfg(type=sy.HEAD_UNIFORM_STRIDE, stride=2, offset=2),
                sy.cfg(type=sy.HEAD_STATIC, static_mode=sy.STATIC_ANCHOR, anchor_frame=4),
                sy.cfg(type=sy.HEAD_QUERY_PROBE_TOPK, keep_blocks=18),
                sy.cfg(type=sy.HEAD_BLOCK_TOPK, topk_scope=sy.SCOPE_PER_FRAME, topk_per_frame=0)):
        with pytest.raises(sf.Saf3rError) as e:
            sf.query_sizes(sf.make_shape(4, 261, 1, 64, 64), [bad])
        assert e.value.status == sf.ERR_INVALID_ARG


def test_context_fails_loudly_without_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError):
        sf.Context(0)
