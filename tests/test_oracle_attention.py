"""Pins for oracle/decode_attention.py.  CPU only."""
import numpy as np
import torch

import brute
import synth
from oracle import kv_migration as om
from oracle.decode_attention import decode_attention_fp64

G = dict(layers=2, kv_heads=3, head_dim=8, block_size=4, num_blocks=16)


def make_pool(seed=0):
    te = G["block_size"] * G["kv_heads"] * G["head_dim"]
    p = om.new_pool(G["layers"], G["num_blocks"], te)
    for l in range(G["layers"]):
        for kv in range(2):
            p[l, kv] = synth.slice_values_f16(seed, 0, l, kv, G["num_blocks"], te)
    return p


def f64(bits):
    return np.ascontiguousarray(bits).view(np.float16).astype(np.float64)


def tables(batch, max_blocks, seed=1):
    perm = synth.block_permutation(seed, G["num_blocks"])
    return perm[: batch * max_blocks].reshape(batch, max_blocks)


def run(pool, layer, q, bt, ctx):
    return decode_attention_fp64(pool, layer, q, bt, ctx, G["block_size"], G["kv_heads"], G["head_dim"])


def test_against_torch_sdpa_float64_and_bruteforce():
    pool = make_pool()
    B, MB = 3, 5
    bt = tables(B, MB)
    ctx = np.array([1, 7, 20], dtype=np.int32)
    q = synth.queries_f16(5, B, G["kv_heads"], G["head_dim"])
    S, H, D = G["block_size"], G["kv_heads"], G["head_dim"]
    for layer in range(G["layers"]):
        o = run(pool, layer, q, bt, ctx)
        for b in range(B):
            n = int(ctx[b])
            # independent gather: whole blocks via torch.index_select, then trim to ctx
            K = torch.from_numpy(f64(pool[layer, 0]).reshape(-1, S, H, D))
            V = torch.from_numpy(f64(pool[layer, 1]).reshape(-1, S, H, D))
            idx = torch.from_numpy(bt[b].astype(np.int64))
            k = K.index_select(0, idx).reshape(-1, H, D)[:n].permute(1, 0, 2)      # [H,n,D]
            v = V.index_select(0, idx).reshape(-1, H, D)[:n].permute(1, 0, 2)
            qq = torch.from_numpy(f64(q[b])).reshape(H, 1, D)
            ref = torch.nn.functional.scaled_dot_product_attention(qq, k, v)       # default scale 1/sqrt(D)
            assert np.abs(ref.reshape(H, D).numpy() - o[b]).max() <= 1e-12
            # pure-Python textbook softmax, head by head
            for h in range(H):
                o_b = brute.attention(k[h].tolist(), v[h].tolist(), qq[h, 0].tolist(), 1.0 / np.sqrt(D))
                assert np.abs(np.array(o_b) - o[b, h]).max() <= 1e-12


def test_ctx_len_one_returns_v0_exactly():
    pool = make_pool()
    bt = tables(2, 2)
    q = synth.queries_f16(5, 2, G["kv_heads"], G["head_dim"])
    o = run(pool, 1, q, bt, np.array([1, 1]))
    S, H, D = G["block_size"], G["kv_heads"], G["head_dim"]
    for b in range(2):
        v0 = f64(pool[1, 1, bt[b, 0]]).reshape(S, H, D)[0]
        assert np.array_equal(o[b], v0)


def test_zero_query_and_equal_keys_give_mean_of_values():
    pool = make_pool()
    S, H, D = G["block_size"], G["kv_heads"], G["head_dim"]
    bt = tables(1, 3)
    n = 10
    q0 = np.zeros((1, H, D), dtype=np.uint16)
    o = run(pool, 0, q0, bt, np.array([n]))
    v = np.concatenate([f64(pool[0, 1, b]).reshape(S, H, D) for b in bt[0]])[:n]
    assert np.abs(o[0] - v.mean(axis=0)).max() <= 1e-15
    # all keys equal (copy key of token 0 over every slot of every listed block) with a nonzero query
    pool2 = pool.copy()
    k0 = pool2[0, 0, bt[0, 0]].reshape(S, H * D)[0].copy()
    for b in bt[0]:
        pool2[0, 0, b] = np.tile(k0, S)
    q = synth.queries_f16(5, 1, H, D)
    o2 = run(pool2, 0, q, bt, np.array([n]))
    assert np.abs(o2[0] - v.mean(axis=0)).max() <= 1e-14


def test_softmax_weights_follow_scores_and_scale():
    """One head, D=8: keys e_0*a_t make the scores q_0*a_t/sqrt(D); check against the closed form."""
    S, H, D = G["block_size"], G["kv_heads"], G["head_dim"]
    pool = np.zeros((1, 2, 4, S * H * D), dtype=np.uint16)
    a = np.array([0.0, 1.0, 2.0, 3.0, -1.0], dtype=np.float16)
    bt = np.array([[2, 0]])
    vals = np.arange(1, 6, dtype=np.float16)
    for t in range(5):
        blk, slot = bt[0, t // S], t % S
        kview = pool[0, 0, blk].view(np.float16).reshape(S, H, D)
        vview = pool[0, 1, blk].view(np.float16).reshape(S, H, D)
        kview[slot, 1, 0] = a[t]
        vview[slot, 1, :] = vals[t]
    q = np.zeros((1, H, D), dtype=np.float16)
    q[0, 1, 0] = 2.0
    o = run(pool, 0, q.view(np.uint16), bt, np.array([5]))
    s = 2.0 * a.astype(np.float64) / np.sqrt(8.0)
    w = np.exp(s) / np.exp(s).sum()
    assert np.abs(o[0, 1] - (w * vals.astype(np.float64)).sum()).max() <= 1e-14
    # heads with zero keys: uniform mean of zeros values -> 0
    assert np.all(o[0, 0] == 0) and np.all(o[0, 2] == 0)


def test_resume_equivalence_on_the_oracle():
    """P10 on the CPU side: attention over (dst pool, dst table) after migration == over (src pool, src table)."""
    pool = make_pool()
    dst = om.new_pool(G["layers"], G["num_blocks"], pool.shape[3], synth.SENTINEL_U16)
    s_tab = synth.block_permutation(1, G["num_blocks"])[:5]
    d_tab = synth.block_permutation(2, G["num_blocks"])[:5]
    om.migrate_stage(pool, s_tab, dst, d_tab)
    q = synth.queries_f16(5, 1, G["kv_heads"], G["head_dim"])
    a = run(pool, 1, q, s_tab[None, :], np.array([18]))
    b = run(dst, 1, q, d_tab[None, :], np.array([18]))
    assert np.array_equal(a, b)
