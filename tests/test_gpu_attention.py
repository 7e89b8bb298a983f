"""GPU decode attention (S7 stand-in) against the fp64 oracle: max abs error <= 2e-3 (north_star),
plus the special cases of SURVEY.md §8(c) P11 and the resume equivalence P10.  Through the C-ABI."""
import numpy as np
import pytest
import torch

import synth
from oracle import kv_migration as om
from oracle.decode_attention import decode_attention_fp64

pytestmark = pytest.mark.gpu

TOL = 2e-3          # BASELINE.json north_star: "decode attention must agree within max abs error 2e-3"
SENT = synth.SENTINEL_U16

# D=128 with 20 heads (a ragged head group: 16 + 4) and D=64 (Tiny's head_dim) with 6 heads (ragged warp)
G128 = dict(layers=2, kv_heads=20, head_dim=128, block_size=16, elem_bytes=2, num_blocks=128)
G64 = dict(layers=2, kv_heads=6, head_dim=64, block_size=16, elem_bytes=2, num_blocks=128)
G64S = dict(layers=1, kv_heads=4, head_dim=64, block_size=5, elem_bytes=2, num_blocks=200)    # odd block size


@pytest.fixture(scope="module")
def env():
    import gpu_harness as H
    import paper_2406_03243_b200 as llx
    llx.load()
    return H, llx


def gpu_attention(llx, pool, layer, q_bits, bt, ctx, g, scale=None):
    B, MB = bt.shape
    q = torch.from_numpy(np.ascontiguousarray(q_bits).view(np.int16)).cuda()
    out = torch.zeros_like(q)
    d_bt = torch.from_numpy(np.ascontiguousarray(bt, dtype=np.int32)).cuda()
    d_ctx = torch.from_numpy(np.ascontiguousarray(ctx, dtype=np.int32)).cuda()
    if scale is None:
        scale = 1.0 / np.sqrt(g["head_dim"])
    llx.decode_attention(pool, layer, q.data_ptr(), out.data_ptr(), d_bt.data_ptr(), d_ctx.data_ptr(), B, MB, scale)
    torch.cuda.synchronize()
    return out.cpu().numpy().view(np.uint16)


def as_f64(bits):
    return np.ascontiguousarray(bits).view(np.float16).astype(np.float64)


def disjoint_tables(g, ctx, seed):
    """Every sequence gets its own random blocks (A12: no artificial sharing)."""
    S = g["block_size"]
    need = [-(-int(c) // S) for c in ctx]
    MB = max(max(need), 1)
    perm = synth.block_permutation(seed, g["num_blocks"])
    assert sum(need) <= g["num_blocks"]
    bt = np.zeros((len(ctx), MB), dtype=np.int32)
    p = 0
    for b, n in enumerate(need):
        bt[b, :n] = perm[p:p + n]
        p += n
    return bt


@pytest.mark.parametrize("g,ctx", [
    (G128, [1, 15, 16, 17, 255, 256, 257, 700]),
    (G64, [3, 64, 129, 511, 640]),
    (G64S, [1, 4, 5, 6, 333, 600]),
])
@pytest.mark.parametrize("split", [0, 8, 64])
def test_matches_fp64_oracle(env, g, ctx, split):
    H, llx = env
    pool = H.DevPool(g)
    pool.fill_from_synth(0, 0)
    h_pool = H.host_pool_from_synth(g, 0, 0)
    ctx = np.array(ctx, dtype=np.int32)
    bt = disjoint_tables(g, ctx, seed=6)
    q = synth.queries_f16(5, len(ctx), g["kv_heads"], g["head_dim"])
    with llx.options(attn_split_tokens=split):
        for layer in range(g["layers"]):
            got = as_f64(gpu_attention(llx, pool.pool, layer, q, bt, ctx, g))
            want = decode_attention_fp64(h_pool, layer, q, bt, ctx, g["block_size"], g["kv_heads"], g["head_dim"])
            err = np.abs(got - want).max()
            assert err <= TOL, f"layer {layer}: max abs err {err}"


def test_sharp_softmax_and_custom_scale(env):
    """Large scale -> near one-hot softmax: exercises the running-max rescale across groups and splits."""
    H, llx = env
    g = G128
    pool = H.DevPool(g)
    pool.fill_from_synth(1, 0)
    h_pool = H.host_pool_from_synth(g, 1, 0)
    ctx = np.array([300, 41], dtype=np.int32)
    bt = disjoint_tables(g, ctx, seed=7)
    q = synth.queries_f16(8, 2, g["kv_heads"], g["head_dim"])
    for scale in (1.0, 4.0):
        with llx.options(attn_split_tokens=32):
            got = as_f64(gpu_attention(llx, pool.pool, 1, q, bt, ctx, g, scale=scale))
        want = decode_attention_fp64(h_pool, 1, q, bt, ctx, g["block_size"], g["kv_heads"], g["head_dim"], scale=scale)
        assert np.abs(got - want).max() <= TOL


def test_special_cases(env):                                           # P11
    H, llx = env
    g = G64
    pool = H.DevPool(g)
    pool.fill_from_synth(2, 0)
    h_pool = H.host_pool_from_synth(g, 2, 0)
    S, Hh, D = g["block_size"], g["kv_heads"], g["head_dim"]
    ctx = np.array([1, 100], dtype=np.int32)
    bt = disjoint_tables(g, ctx, seed=9)
    # ctx_len = 1  =>  o = v_0 exactly (fp16 in, fp16 out)
    q = synth.queries_f16(5, 2, Hh, D)
    got = gpu_attention(llx, pool.pool, 0, q, bt, ctx, g)
    v0 = h_pool[0, 1, bt[0, 0]].reshape(S, Hh, D)[0]
    assert np.array_equal(got[0], v0)
    # q = 0  =>  o = mean_t v_t
    got = as_f64(gpu_attention(llx, pool.pool, 0, np.zeros_like(q), bt, ctx, g))
    rows = np.concatenate([h_pool[0, 1, b].reshape(S, Hh, D) for b in bt[1]])[:100]
    assert np.abs(got[1] - as_f64(rows).mean(axis=0)).max() <= TOL
    # ctx_len = 0  =>  zeros
    got = gpu_attention(llx, pool.pool, 0, q, bt, np.array([0, 0], dtype=np.int32), g)
    assert np.all(got == 0)


def test_resume_on_destination_is_bit_identical(env):                  # P10 ("resumes on the destination")
    H, llx = env
    g = G128
    src = H.DevPool(g)
    src.fill_from_synth(3, 0)
    dst = H.DevPool(g, num_blocks=130, fill=SENT)
    ctx = np.array([500, 77, 16], dtype=np.int32)
    bt_src = disjoint_tables(g, ctx, seed=10)
    need = [-(-int(c) // 16) for c in ctx]
    perm_d = synth.block_permutation(11, 130)
    bt_dst = np.zeros_like(bt_src)
    p = 0
    for b, n in enumerate(need):
        bt_dst[b, :n] = perm_d[p:p + n]
        llx.migrate_stage(src.pool, bt_src[b, :n], dst.pool, bt_dst[b, :n])
        p += n
    q = synth.queries_f16(12, 3, g["kv_heads"], g["head_dim"])
    for layer in range(g["layers"]):
        a = gpu_attention(llx, src.pool, layer, q, bt_src, ctx, g)
        b = gpu_attention(llx, dst.pool, layer, q, bt_dst, ctx, g)
        assert np.array_equal(a, b)
    h_src = H.host_pool_from_synth(g, 3, 0)
    want = decode_attention_fp64(h_src, 0, q, bt_src, ctx, 16, g["kv_heads"], g["head_dim"])
    assert np.abs(as_f64(gpu_attention(llx, dst.pool, 0, q, bt_dst, ctx, g)) - want).max() <= TOL


def test_attention_argument_errors(env):
    H, llx = env
    g = dict(G64, head_dim=32)
    pool = H.DevPool(g)
    buf = torch.zeros(1024, dtype=torch.int32, device="cuda")
    with pytest.raises(llx.LlxError) as e:
        llx.decode_attention(pool.pool, 0, buf.data_ptr(), buf.data_ptr(), buf.data_ptr(), buf.data_ptr(), 1, 1, 1.0)
    assert e.value.name == "LLX_ERR_INVALID_ARG"
    pool64 = H.DevPool(G64)
    with pytest.raises(llx.LlxError):
        llx.decode_attention(pool64.pool, 5, buf.data_ptr(), buf.data_ptr(), buf.data_ptr(), buf.data_ptr(), 1, 1, 1.0)
    llx.decode_attention(pool64.pool, 0, 0, 0, 0, 0, 0, 0, 1.0)        # B == 0: OK, nothing launched


def test_configs4_decode_batch_shape_within_tolerance(env):
    """BASELINE.json configs[4]'s own decode batch — the shape the interference numbers are quoted on: B = 32, context
    lengths uniform in [128, 4096] (synth seed 4), H = 32, D = 128, disjoint block tables in an 8448-block pool (reading
    A12), default KV split, 2 layers.  max |o - o_fp64| <= 2e-3 on every output element.  Prints the oracle's wall time
    ("the fp64 attention oracle is timed once")."""
    import time
    H, llx = env
    g = dict(synth.CONFIGS["llama7b"], layers=2, num_blocks=32 * 256 + 128 + 128)
    B, S, Hh, D = 32, g["block_size"], g["kv_heads"], g["head_dim"]
    ctx = synth.context_lengths(4, B, 128, 4096)
    bt = disjoint_tables(g, ctx, seed=6)
    assert bt.shape[1] <= 256 and int(ctx.sum()) > 32 * 1500
    pool = H.DevPool(g)
    # seeded fp16 U[-1,1) generated on the device (input generation only) and read back for the oracle: a host-side
    # fill of the 8448-block pool would spend minutes in the generator for blocks no sequence uses
    gen = torch.Generator(device="cuda")
    gen.manual_seed(4)
    flat = pool.raw.view(torch.float16)
    step = 1 << 27
    for a in range(0, flat.numel(), step):
        b = min(flat.numel(), a + step)
        flat[a:b] = (torch.rand(b - a, generator=gen, device="cuda", dtype=torch.float32) * 2 - 1).half()
    h_pool = pool.host()
    q = synth.queries_f16(5, B, Hh, D)
    worst, t_oracle = 0.0, 0.0
    for layer in range(g["layers"]):
        got = as_f64(gpu_attention(llx, pool.pool, layer, q, bt, ctx, g))
        t0 = time.perf_counter()
        want = decode_attention_fp64(h_pool, layer, q, bt, ctx, S, Hh, D)
        t_oracle += time.perf_counter() - t0
        err = np.abs(got - want).max()
        worst = max(worst, err)
        assert err <= TOL, f"layer {layer}: max abs err {err}"
    print(f"configs[4] decode batch: max abs err {worst:.3e} (bound {TOL}); fp64 oracle {t_oracle / g['layers']:.1f} s per layer "
          f"for {int(ctx.sum())} context tokens")


def test_ctx_len_beyond_the_table_row_is_clamped(env):
    """llx.h precondition: ctx_len <= max_blocks*block_size; a longer one is clamped in the kernels — the result is the
    attention over the row's max_blocks*block_size tokens, not a read past the table row."""
    H, llx = env
    g = G64
    pool = H.DevPool(g)
    pool.fill_from_synth(6, 0)
    h_pool = H.host_pool_from_synth(g, 6, 0)
    ctx_ok = np.array([48, 32], dtype=np.int32)
    bt = disjoint_tables(g, ctx_ok, seed=12)                             # 3 blocks per row
    q = synth.queries_f16(7, 2, g["kv_heads"], g["head_dim"])
    got = as_f64(gpu_attention(llx, pool.pool, 0, q, bt, np.array([10_000, 32], dtype=np.int32), g))
    want = decode_attention_fp64(h_pool, 0, q, bt, np.array([48, 32]), g["block_size"], g["kv_heads"], g["head_dim"])
    assert np.abs(got - want).max() <= TOL
