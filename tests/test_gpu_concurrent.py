"""BASELINE.json configs[4]'s defining scenario as a parity test: a 2048-token request migrates in three
stages on a LOW-priority stream while a batch-32 decode-attention step keeps running over the same source pool on the
decode stream, with the request's appends on the decode stream too (PAPER.md:134 Fig. 6, :235 own stream, :289 the
co-running batch).  Concurrency is where the co-residency machinery lives (the paced register-staged kernel, sliced
budgeted launches, the kernel switch while a paced stage is in flight), so each of three launch policies is checked:
unthrottled, a 25 GB/s budget on the non-final stages, and the copy-engine route.

Asserted for every policy: the destination equals oracle.staged_migration word for word on the sampled layers and keeps
the sentinel elsewhere; every attention output produced WHILE the migration ran is bit-identical to the same launch run
alone and within 2e-3 of the fp64 oracle; attention over the migrated request on the destination is bit-identical to
attention over it on the source (resume equivalence).

LLaMA-7B tiles and heads, 4 layers (the attention step is per layer; the copy treats layers alike), decode batch of
configs[4]: 32 sequences, context lengths uniform in [128, 4096] (synth seed 4), disjoint block tables (reading A12)."""
import numpy as np
import pytest
import torch

import synth
from oracle import kv_migration as om
from oracle.decode_attention import decode_attention_fp64

pytestmark = pytest.mark.gpu

TOL = 2e-3
SENT = synth.SENTINEL_U16
SENT_I16 = int(np.array(SENT, np.uint16).view(np.int16))
SCHEDULE, APPENDS, START = (112, 14, 2), (8, 8), 2032
L = 4
SAMPLE = [0, 3]                     # layers mirrored on the host; attention runs on these


@pytest.fixture(scope="module")
def env():
    import gpu_harness as H
    import paper_2406_03243_b200 as llx
    llx.load()
    return H, llx


@pytest.fixture(scope="module")
def scene(env):
    H, llx = env
    g = dict(synth.CONFIGS["llama7b"], layers=L)
    S, Hh, D = g["block_size"], g["kv_heads"], g["head_dim"]
    B = 32
    ctx = synth.context_lengths(4, B, 128, 4096)
    need = [-(-int(c) // S) for c in ctx]
    nb_src = sum(need) + 128 + 64
    g["num_blocks"] = nb_src
    src = H.DevPool(g)
    gen = torch.Generator(device="cuda")
    gen.manual_seed(44)
    flat = src.raw.view(torch.float16)                    # seeded fp16 U[-1,1) made on the device: input generation only
    step = 1 << 27
    for a in range(0, flat.numel(), step):
        b = min(flat.numel(), a + step)
        flat[a:b] = (torch.rand(b - a, generator=gen, device="cuda", dtype=torch.float32) * 2 - 1).half()
    dst = H.DevPool(g, num_blocks=300, fill=SENT)
    perm = synth.block_permutation(6, nb_src)
    MB = max(need)
    bt = np.zeros((B, MB), dtype=np.int32)
    pos = 0
    for b, n in enumerate(need):
        bt[b, :n] = perm[pos:pos + n]
        pos += n
    s_tab = perm[pos:pos + 128].astype(np.int32)          # the migrating request: blocks no sequence of the batch uses
    d_tab = synth.block_permutation(2, 300)[:128].astype(np.int32)
    te, te_tok = src.te, Hh * D
    vals = np.empty((sum(APPENDS), L, 2, te_tok), dtype=np.uint16)
    for j in range(sum(APPENDS)):
        for l in range(L):
            for kv in range(2):
                vals[j, l, kv] = synth.append_values_f16(3, START + j, l, kv, te_tok)
    # ---- the oracle, once: sampled layers of the source as generated, the staged migration, the batch's attention
    h_src = np.stack([src.host_layer(l)[0] for l in SAMPLE])                   # [len(SAMPLE), 2, nb, te]
    q = synth.queries_f16(5, B, Hh, D)
    want_attn = {l: decode_attention_fp64(h_src[i:i + 1], 0, q, bt, ctx, S, Hh, D) for i, l in enumerate(SAMPLE)}
    h_dst = om.new_pool(len(SAMPLE), 300, te, fill=SENT)
    h_work = h_src.copy()
    om.staged_migration(h_work, s_tab, h_dst, d_tab, SCHEDULE, APPENDS, S, START,
                        lambda t, li, kv: vals[t - START, SAMPLE[li], kv])
    return dict(g=g, src=src, dst=dst, bt=bt, ctx=ctx, s_tab=s_tab, d_tab=d_tab, vals=vals, q=q, want_attn=want_attn,
                want_dst=h_dst, want_src_tail=h_work[:, :, s_tab[-1]], MB=MB, B=B)


def f64(t):
    return t.cpu().numpy().view(np.float16).astype(np.float64)


@pytest.mark.parametrize("policy", ["unthrottled", "budget_25gbps", "copy_engine"])
def test_migration_concurrent_with_the_decode_batch(env, scene, policy):
    H, llx = env
    sc = scene
    g, src, dst = sc["g"], sc["src"], sc["dst"]
    S, Hh, D, B, MB = g["block_size"], g["kv_heads"], g["head_dim"], sc["B"], sc["MB"]
    s_tab, d_tab = sc["s_tab"], sc["d_tab"]
    scale = 1.0 / float(np.sqrt(D))
    q = torch.from_numpy(sc["q"].view(np.int16)).cuda()
    d_bt = torch.from_numpy(sc["bt"]).cuda()
    d_ctx = torch.from_numpy(sc["ctx"].astype(np.int32)).cuda()
    dev_vals = torch.from_numpy(sc["vals"].view(np.int16)).cuda()
    tok_bytes = L * 2 * Hh * D * 2
    dst.view.fill_(SENT_I16)
    lo, hi = torch.cuda.Stream.priority_range()
    s_dec, s_mig = torch.cuda.Stream(priority=hi), torch.cuda.Stream(priority=lo)
    torch.cuda.synchronize()

    def attention(out, layer, stream):
        llx.decode_attention(src.pool, layer, q.data_ptr(), out.data_ptr(), d_bt.data_ptr(), d_ctx.data_ptr(), B, MB, scale, stream=stream)

    # the same launches alone (also grows the pool's attention workspace outside the concurrent region)
    alone = {l: torch.zeros_like(q) for l in SAMPLE}
    for l in SAMPLE:
        attention(alone[l], l, s_dec)
    s_dec.synchronize()
    for l in SAMPLE:
        err = np.abs(f64(alone[l]) - sc["want_attn"][l]).max()
        assert err <= TOL, f"layer {l} alone: max abs err {err}"

    stage_opts = {"unthrottled": None, "budget_25gbps": dict(bandwidth_gbps=25), "copy_engine": dict(route=llx.ROUTE_COPY_ENGINE)}[policy]
    final_opts = dict(route=llx.ROUTE_COPY_ENGINE) if policy == "copy_engine" else None
    rounds = {"unthrottled": 6, "budget_25gbps": 40, "copy_engine": 6}[policy]
    outs = [{l: torch.full_like(q, 0x7E00) for l in SAMPLE} for _ in range(rounds)]
    torch.cuda.synchronize()
    e_app = torch.cuda.Event()
    c0 = llx.counters()
    # migration stream: stages 0 and 1 now, the final stage once the appends are in
    llx.migrate_stage(src.pool, s_tab[:112], dst.pool, d_tab[:112], stream=s_mig, opts=stage_opts)
    llx.migrate_stage(src.pool, s_tab[112:126], dst.pool, d_tab[112:126], stream=s_mig, opts=stage_opts)
    # decode stream: attention rounds with the request's two appends in between
    t = START
    for r in range(rounds):
        for l in SAMPLE:
            attention(outs[r][l], l, s_dec)
        if r < len(APPENDS):
            llx.append_tokens(src.pool, s_tab, t, t + APPENDS[r], dev_vals.data_ptr() + (t - START) * tok_bytes, stream=s_dec)
            t += APPENDS[r]
            if r == len(APPENDS) - 1:
                e_app.record(s_dec)
                s_mig.wait_event(e_app)
                llx.migrate_stage(src.pool, s_tab[126:], dst.pool, d_tab[126:], stream=s_mig, opts=final_opts)
    torch.cuda.synchronize()
    c1 = llx.counters()
    if policy == "budget_25gbps":
        assert c1["copy_launches"] - c0["copy_launches"] > 3, "a budgeted stage is a chain of sliced launches"
    # ---- destination == oracle on the sampled layers (every word; sentinel outside the reserved blocks)
    for i, l in enumerate(SAMPLE):
        got = dst.host_layer(l)[0]
        if not np.array_equal(got, sc["want_dst"][i]):
            kv, b, e = np.argwhere(got != sc["want_dst"][i])[0]
            raise AssertionError(f"{policy}: layer {l} kv {kv} block {b} elem {e}: expected 0x{int(sc['want_dst'][i][kv, b, e]):04x} got 0x{int(got[kv, b, e]):04x}")
        tail = src.view[l, :, int(s_tab[-1])].cpu().numpy().view(np.uint16)
        assert np.array_equal(tail, sc["want_src_tail"][i]), f"{policy}: the source's tail block differs from the oracle's appends"
    # layers the host does not mirror: every migrated block equals its source block
    si = torch.from_numpy(s_tab.astype(np.int64)).cuda()
    di = torch.from_numpy(d_tab.astype(np.int64)).cuda()
    for l in range(L):
        assert torch.equal(dst.view[l].index_select(1, di), src.view[l].index_select(1, si)), l
    # ---- attention next to the migration: bit-identical to the launch alone, and within the tolerance of the oracle
    for r in range(rounds):
        for l in SAMPLE:
            assert torch.equal(outs[r][l], alone[l]), f"{policy}: round {r} layer {l}: attention changed next to the migration"
    for l in SAMPLE:
        assert np.abs(f64(outs[0][l]) - sc["want_attn"][l]).max() <= TOL
    # ---- resume equivalence: the migrated request attends identically on the destination
    q1 = torch.from_numpy(synth.queries_f16(9, 1, Hh, D).view(np.int16)).cuda()
    c2048 = torch.tensor([2048], dtype=torch.int32, device="cuda")
    for l in SAMPLE:
        o_s, o_d = torch.zeros_like(q1), torch.zeros_like(q1)
        bt_s = torch.from_numpy(s_tab.reshape(1, -1)).cuda()
        bt_d = torch.from_numpy(d_tab.reshape(1, -1)).cuda()
        llx.decode_attention(src.pool, l, q1.data_ptr(), o_s.data_ptr(), bt_s.data_ptr(), c2048.data_ptr(), 1, 128, scale)
        llx.decode_attention(dst.pool, l, q1.data_ptr(), o_d.data_ptr(), bt_d.data_ptr(), c2048.data_ptr(), 1, 128, scale)
        torch.cuda.synchronize()
        assert torch.equal(o_s, o_d), f"{policy}: layer {l}: attention on the destination differs from the source"
