"""GPU test of saf3r_token_probe_select_noalloc, the one entry point of the library that obtains no device memory.

It exists for users who embed the library where device memory cannot be requested at call time: inside an engine or server
that has planned the whole GPU heap and passes a plug-in nothing but its input and output buffers, under a per-process memory
quota, or in a loop that cannot afford the device-wide stall of cudaMalloc.  Such a caller can use neither a Context
(saf3r_create allocates) nor a workspace, so the call keeps its scratch in a fixed array inside libsaf3r.so.

What is checked: its output equals that of the ordinary path (Context.token_probe_select, which runs the same three kernels over
a caller-made workspace).  The outputs are index lists, so the tolerance is the one every list test here uses: bit-exact.  Two
calls are made back to back on different inputs and different shapes, the second smaller than the first, so that it runs over the
scratch the first one left dirty: stale keys or histogram counts would change its answer.  A third call beyond the documented size
limit must be refused with ERR_CAPACITY and must not touch idx.

The file name sorts last on purpose: pytest -x stops at the first failure, and a failure here must not hide the parity tests.
The test makes no assumption about earlier tests (it passes alone in a fresh process and after the rest of the suite); the
reference results are computed before the no-alloc calls so that the comparison never depends on allocator reuse."""
import numpy as np
import pytest

import saf3r_synth as sy
from parity_util import c_shape, upload

pytestmark = pytest.mark.gpu


def _layer(S, G, H, seed):
    sh = sy.Shape(S=S, G=G, H=H, D=64, B=64)
    gens = [sy.GEN_SINK, sy.GEN_UNIFORM, sy.GEN_SAME_POSITION, sy.GEN_ANCHOR]
    return sy.make_layer(sh, [gens[h % 4] for h in range(H)], [sy.cfg(type=sy.HEAD_DENSE)] * H, seed)


def test_noalloc_token_probe_matches_workspace_path_twice_in_a_row():
    import torch
    import paper_2607_03612_b200 as sf
    ctx = sf.Context(0)
    torch.cuda.set_device(0)
    # first call: 8 heads x 9 frames x 1158 tokens (several probe tiles and Q-sum chunks per head, ragged tails);
    # second call: fewer heads, fewer tokens, another K - it reuses the low part of a scratch full of the first call's data
    cases = [(_layer(9, 34, 8, seed=301), 300), (_layer(3, 19, 3, seed=302), 37)]
    prepared = []
    for L, K in cases:
        q, k, _ = upload(L)
        shape = c_shape(sf, L.shape)
        want = ctx.token_probe_select(q, k, shape, K)
        idx = torch.full((L.shape.H, K), -7, dtype=torch.int32, device="cuda:0")
        prepared.append((q, k, shape, K, want, idx))
    torch.cuda.synchronize()
    free_mem = []
    for q, k, shape, K, _want, idx in prepared:      # the two calls in a row, nothing in between
        sf.token_probe_select_noalloc(q, k, shape, K, idx)
        free_mem.append(torch.cuda.mem_get_info()[0])  # driver-level free bytes: would see a cudaMalloc made behind torch's back
    torch.cuda.synchronize()
    for (L, K), (_q, _k, _shape, _K, want, idx) in zip(cases, prepared):
        got, ref = idx.cpu().numpy(), want.cpu().numpy()
        assert got.min() >= 0 and got.max() < L.shape.N and np.all(np.diff(got, axis=1) > 0)
        assert np.array_equal(got, ref), f"no-alloc token probe differs from the workspace path (N={L.shape.N}, K={K})"
    # and once more on the first, larger input: the second call's leftovers are in the way now
    q, k, shape, K, want, idx = prepared[0]
    idx.fill_(-7)
    sf.token_probe_select_noalloc(q, k, shape, K, idx)
    free_mem.append(torch.cuda.mem_get_info()[0])
    torch.cuda.synchronize()
    assert np.array_equal(idx.cpu().numpy(), want.cpu().numpy())
    # once the first call has done its one-off address look-up, further calls leave the device's free memory untouched
    assert free_mem[1] == free_mem[0] and free_mem[2] == free_mem[0], free_mem
    ctx.close()


def test_noalloc_token_probe_refuses_sizes_beyond_the_built_in_scratch():
    import torch
    import paper_2607_03612_b200 as sf
    torch.cuda.set_device(0)
    H, S, T = 16, 48, 1374                            # 16 * 65952 = 1 055 232 keys > 2^20
    assert H * S * T > sf.NOALLOC_MAX_KEYS
    shape = sf.make_shape(S, T, H, 64, 128)
    q = torch.zeros(16, dtype=torch.bfloat16, device="cuda:0")   # never read: the size check comes before any launch
    idx = torch.full((H, 8), -7, dtype=torch.int32, device="cuda:0")
    with pytest.raises(sf.Saf3rError) as ei:
        sf.token_probe_select_noalloc(q, q, shape, 8, idx)
    assert ei.value.status == sf.ERR_CAPACITY and "SAF3R_NOALLOC_MAX_KEYS" in str(ei.value)
    torch.cuda.synchronize()
    assert int((idx != -7).sum()) == 0
    # just inside the limit is accepted: 16 heads x 32 frames x 1374 tokens (the VGGT-shape configuration)
    assert 16 * 32 * 1374 <= sf.NOALLOC_MAX_KEYS
