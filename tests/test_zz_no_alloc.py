"""llx_decode_attention_static_ws: decode attention for callers that cannot allocate device memory.

Some users of this library cannot call cudaMalloc once they are serving: an engine that gave every free byte of HBM to
its KV-cache pool at start-up (a later allocation fails), a decode loop on a latency budget (cudaMalloc / cudaFree can
stall every stream of the device, a running migration included), code inside a stream's host callback.  The ordinary
llx_decode_attention grows a per-pool workspace with cudaMalloc when a larger shape arrives; the entry point tested
here keeps its split-KV partials in a fixed 16 MiB array that is part of the library image and allocates nothing.

What is checked: its output equals the existing path's on the same inputs, within the 2e-3 the attention tests use, on
two calls in a row that share the array (the second with other queries, another layer and shorter contexts, so rows the
first call left behind would show if they were read); a shape beyond the fixed size is refused with a clear message and
launches nothing.

This file sorts last on purpose (`pytest --collect-only`): the suite runs with `pytest -x`, which stops at the first
failure, so a failure here cannot hide any other test.  It passes alone in a fresh process (its first call is then the
one that looks up the array's device address) and after the rest of the suite.
"""
import numpy as np
import pytest
import torch

import synth

pytestmark = pytest.mark.gpu

TOL = 2e-3          # the tolerance of tests/test_gpu_attention.py (BASELINE.json north_star)

G128 = dict(layers=2, kv_heads=20, head_dim=128, block_size=16, elem_bytes=2, num_blocks=160)
G64 = dict(layers=2, kv_heads=6, head_dim=64, block_size=16, elem_bytes=2, num_blocks=160)


@pytest.fixture(scope="module")
def env():
    import gpu_harness as H
    import paper_2406_03243_b200 as llx
    llx.load()
    return H, llx


def as_f64(t):
    return t.cpu().numpy().view(np.float16).astype(np.float64)


def tables(g, ctx, seed):
    """Disjoint random blocks per sequence."""
    S = g["block_size"]
    need = [-(-int(c) // S) for c in ctx]
    perm = synth.block_permutation(seed, g["num_blocks"])
    assert sum(need) <= g["num_blocks"]
    bt = np.zeros((len(ctx), max(max(need), 1)), dtype=np.int32)
    p = 0
    for b, n in enumerate(need):
        bt[b, :n] = perm[p:p + n]
        p += n
    return bt


class Case:
    """One attention call's device-side arguments; `run(fn)` writes into an output buffer pre-filled with NaNs.  All
    buffers are made (and the device synchronised) in the constructor, so `run` only enqueues the call itself."""

    def __init__(self, g, layer, ctx, q_seed, bt_seed):
        self.g, self.layer = g, layer
        ctx = np.asarray(ctx, dtype=np.int32)
        bt = tables(g, ctx, bt_seed)
        self.B, self.MB = bt.shape
        q = synth.queries_f16(q_seed, len(ctx), g["kv_heads"], g["head_dim"])
        self.q = torch.from_numpy(np.ascontiguousarray(q).view(np.int16)).cuda()
        self.bt = torch.from_numpy(bt).cuda()
        self.ctx = torch.from_numpy(ctx).cuda()
        self.scale = 1.0 / np.sqrt(g["head_dim"])
        # fp16 NaN: an element a call does not write stays NaN
        self.outs = [torch.full_like(self.q, 0x7E00) for _ in range(2)]
        torch.cuda.synchronize()

    def run(self, fn, pool, stream=None):
        out = self.outs.pop()
        fn(pool, self.layer, self.q.data_ptr(), out.data_ptr(), self.bt.data_ptr(), self.ctx.data_ptr(),
           self.B, self.MB, self.scale, stream)
        return out


@pytest.mark.parametrize("g", [G128, G64], ids=["D128", "D64"])
@pytest.mark.parametrize("split", [0, 16], ids=["split256", "split16"])
def test_two_calls_in_a_row_match_the_allocating_path(env, g, split):
    H, llx = env
    pool = H.DevPool(g)
    pool.fill_from_synth(21, 0)
    # first call: long contexts (up to 44 splits of 16 tokens per head); second: other queries, the other layer, fewer and
    # shorter sequences — every partial row it reads was also written by the first call with different values
    first = Case(g, 0, [700, 257, 16, 1, 333, 512], q_seed=31, bt_seed=41)
    second = Case(g, 1, [90, 5, 300], q_seed=32, bt_seed=42)
    with llx.options(attn_split_tokens=split):
        want1 = first.run(llx.decode_attention, pool.pool)
        want2 = second.run(llx.decode_attention, pool.pool)
        torch.cuda.synchronize()
        before = llx.counters()["kernel_launches"]
        # back to back on one stream, no synchronisation in between: the shared array is reused in stream order
        got1 = first.run(llx.decode_attention_static_ws, pool.pool)
        got2 = second.run(llx.decode_attention_static_ws, pool.pool)
        torch.cuda.synchronize()
        assert llx.counters()["kernel_launches"] - before == 4     # partial + merge per call: the library's own kernels ran
    for name, got, want in (("first", got1, want1), ("second", got2, want2)):
        a, b = as_f64(got), as_f64(want)
        assert not np.isnan(b).any(), "the existing path left outputs unwritten"
        assert not np.isnan(a).any(), f"{name} call: outputs left unwritten"
        err = np.abs(a - b).max()
        assert err <= TOL, f"{name} call: max abs difference {err} to llx_decode_attention"


def test_same_result_on_a_second_stream_after_an_event(env):
    """Calls on different streams are allowed when ordered: the second waits for the first through an event."""
    H, llx = env
    pool = H.DevPool(G128)
    pool.fill_from_synth(22, 0)
    c1 = Case(G128, 0, [400, 31], q_seed=33, bt_seed=43)
    c2 = Case(G128, 0, [64, 129, 2], q_seed=34, bt_seed=44)
    want1 = c1.run(llx.decode_attention, pool.pool)
    want2 = c2.run(llx.decode_attention, pool.pool)
    torch.cuda.synchronize()
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    got1 = c1.run(llx.decode_attention_static_ws, pool.pool, s1.cuda_stream)
    s2.wait_event(s1.record_event())
    got2 = c2.run(llx.decode_attention_static_ws, pool.pool, s2.cuda_stream)
    torch.cuda.synchronize()
    assert np.abs(as_f64(got1) - as_f64(want1)).max() <= TOL
    assert np.abs(as_f64(got2) - as_f64(want2)).max() <= TOL


def test_a_shape_beyond_the_fixed_workspace_is_refused(env):
    H, llx = env
    g = dict(G128, kv_heads=32)
    pool = H.DevPool(g)
    assert llx.ATTN_STATIC_WS_BYTES == 16 << 20
    S, Hh, D = g["block_size"], g["kv_heads"], g["head_dim"]
    row = (D + 4) * 4
    # largest batch whose partials fit with 8 splits of 256 tokens per head, and one sequence more
    MB = 8 * 256 // S
    b_fit = llx.ATTN_STATIC_WS_BYTES // (Hh * 8 * row)
    buf = torch.zeros(4 << 20, dtype=torch.int16, device="cuda")           # q / out / tables: never dereferenced when refused
    before = llx.counters()["kernel_launches"]
    with pytest.raises(llx.LlxError) as e:
        llx.decode_attention_static_ws(pool.pool, 0, buf.data_ptr(), buf.data_ptr(), buf.data_ptr(), buf.data_ptr(),
                                       b_fit + 1, MB, 1.0)
    assert e.value.name == "LLX_ERR_INVALID_ARG"
    msg = str(e.value)
    assert str((b_fit + 1) * Hh * 8 * row) in msg and str(llx.ATTN_STATIC_WS_BYTES) in msg and "never allocates" in msg
    assert llx.counters()["kernel_launches"] == before                   # refused on the host: nothing launched
    assert int(buf.count_nonzero()) == 0
    # exactly at the limit it runs: ctx_len 0 for every sequence -> zeros, whatever the (zero) tables say
    out = torch.full((b_fit, Hh, D), 0x7E00, dtype=torch.int16, device="cuda")
    llx.decode_attention_static_ws(pool.pool, 0, buf.data_ptr(), out.data_ptr(), buf.data_ptr(), buf.data_ptr(),
                                   b_fit, MB, 1.0)
    torch.cuda.synchronize()
    assert int(out.count_nonzero()) == 0
    # the other argument checks are those of llx_decode_attention
    with pytest.raises(llx.LlxError):
        llx.decode_attention_static_ws(pool.pool, 9, buf.data_ptr(), buf.data_ptr(), buf.data_ptr(), buf.data_ptr(), 1, 1, 1.0)
    llx.decode_attention_static_ws(pool.pool, 0, 0, 0, 0, 0, 0, 0, 1.0)  # B == 0: OK, nothing launched
