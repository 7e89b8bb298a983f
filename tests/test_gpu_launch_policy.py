"""Launch policy is per call (llx_launch_opts) and stream capture is safe or refused.

PAPER.md:289-291: a migration must not slow the co-running requests (<= 1 %), so non-final stages run under a bandwidth
budget; the final stage IS the downtime, so it runs unthrottled; a source migrates requests
continuously.  Both policies are therefore live at once, on two streams, from two host threads."""
import statistics
import threading
import time

import numpy as np
import pytest
import torch

import synth
from oracle import kv_migration as om

pytestmark = pytest.mark.gpu

SENT = synth.SENTINEL_U16
SENT_I16 = int(np.array(SENT, np.uint16).view(np.int16))
# LLaMA-7B tiles (128 KiB, 8 MiB blocks) in pools small enough to mirror one layer at a time
G7 = dict(layers=32, kv_heads=32, head_dim=128, block_size=16, elem_bytes=2, num_blocks=300)


@pytest.fixture(scope="module")
def env():
    import gpu_harness as H
    import paper_2406_03243_b200 as llx
    llx.load()
    return H, llx


def test_budgeted_stage_and_unthrottled_final_stage_from_two_threads(env):
    """Thread A loops a 25 GB/s-budgeted 112-block stage (llx_migrate_stage_ex); thread B times 2-block final stages
    (llx_migrate_stage_wait).  Both bit-exact; B's median within 2x of its solo value; A's achieved rate within 10 % of
    its budget.  With process-global options (round 1) A's budget would have throttled B's final stage to milliseconds."""
    H, llx = env
    g = G7
    sample = [0, 31]
    src, dst_a, dst_b = H.DevPool(g), H.DevPool(g, fill=SENT), H.DevPool(g, fill=SENT)
    src.fill_device_random(77)
    src.fill_from_synth(0, 0, layers=sample)
    perm_s = synth.block_permutation(1, g["num_blocks"])
    perm_d = synth.block_permutation(2, g["num_blocks"])
    a_s, a_d = perm_s[:112], perm_d[:112]
    b_s, b_d = perm_s[112:114], perm_d[112:114]
    torch.cuda.synchronize()
    st_a, st_b = torch.cuda.Stream(), torch.cuda.Stream()
    budget = 25
    stage_bytes = 2 * 112 * src.pool.block_bytes                      # read + written

    def final_stage_us(reps):
        out = []
        for _ in range(reps):
            t0 = time.perf_counter_ns()
            llx.migrate_stage_wait(src.pool, b_s, dst_b.pool, b_d, stream=st_b)
            out.append((time.perf_counter_ns() - t0) / 1e3)
        return out

    final_stage_us(20)
    solo = statistics.median(final_stage_us(200))

    errors, a_ms, stop = [], [], threading.Event()

    def thread_a():
        try:
            torch.cuda.set_device(0)
            while not stop.is_set():
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(st_a)
                llx.migrate_stage(src.pool, a_s, dst_a.pool, a_d, stream=st_a, opts=dict(bandwidth_gbps=budget))
                e1.record(st_a)
                st_a.synchronize()
                a_ms.append(e0.elapsed_time(e1))
        except Exception as e:  # noqa: BLE001
            errors.append(repr(e))

    ta = threading.Thread(target=thread_a)
    ta.start()
    time.sleep(0.05)                                                   # A's first stage is in flight
    busy = []
    while len(a_ms) < 3 and not errors and len(busy) < 200000:         # B keeps issuing final stages while A streams
        busy += final_stage_us(100)
    stop.set()
    ta.join()
    assert not errors, errors
    with_a = statistics.median(busy)
    assert len(a_ms) >= 2
    achieved = stage_bytes / (statistics.median(a_ms) * 1e-3) / 1e9
    print(f"final stage solo {solo:.1f} us, next to a {budget} GB/s stage {with_a:.1f} us; budgeted stage achieved {achieved:.1f} GB/s")
    assert with_a <= 2.0 * solo, (solo, with_a)
    # and NEVER a whole stage: the budgeted copy keeps a CTA resident on every SM for ~75 ms; if it pinned the SMs'
    # L1/shared split at "all L1" (the driver's default for a kernel without shared memory) the final stage's bulk ring
    # would wait for the end of that stage on every SM (measured before LLX_OPT_COPY_SMEM_CARVEOUT_PCT: p90 75 ms)
    busy.sort()
    assert busy[int(0.99 * len(busy))] < 2000 and busy[-1] < 20000, (busy[int(0.99 * len(busy))], busy[-1])
    assert abs(achieved - budget) <= 0.10 * budget, achieved
    assert llx.get_option(llx.OPT_BANDWIDTH_GBPS) == 0                 # nobody touched the process defaults
    # bit-exact, both destinations, on the sampled layers (oracle) and on every layer (device gather)
    for l in sample:
        h_src = H.host_pool_from_synth(g, 0, 0, layers=[l])
        for dst, (s_ids, d_ids) in ((dst_a, (a_s, a_d)), (dst_b, (b_s, b_d))):
            h_dst = om.new_pool(1, g["num_blocks"], H.tile_elems(g), fill=SENT)
            om.migrate_stage(h_src, s_ids, h_dst, d_ids)
            H.assert_pool_equal(dst.host_layer(l), h_dst)
    for dst, (s_ids, d_ids) in ((dst_a, (a_s, a_d)), (dst_b, (b_s, b_d))):
        si, di = torch.from_numpy(s_ids.astype(np.int64)).cuda(), torch.from_numpy(d_ids.astype(np.int64)).cuda()
        for l in range(g["layers"]):
            assert torch.equal(dst.view[l].index_select(1, di), src.view[l].index_select(1, si))


def test_session_budget_applies_to_non_final_stages_only(env):
    """llx_migration_set_stage_opts: stage 0 of a session runs under the budget, the final stage at full speed."""
    H, llx = env
    g = G7
    src, dst = H.DevPool(g), H.DevPool(g, fill=SENT)
    src.fill_device_random(78)
    src.fill_from_synth(0, 0, layers=[7])
    nb = g["num_blocks"]
    src_mgr, dst_mgr = llx.BlockManager(nb), llx.BlockManager(nb)
    table = src_mgr.alloc(40)
    tokens = 39 * 16 + 5
    mig = llx.Migration(src.pool, src_mgr, dst.pool, dst_mgr, 16, 2)
    mig.set_stage_opts(dict(bandwidth_gbps=50))
    st = torch.cuda.Stream()
    st.wait_stream(torch.cuda.current_stream())
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
    ev[0].record(st)
    n0, fin0, ids0 = mig.stage(table, tokens, stream=st)
    ev[1].record(st)
    st.synchronize()
    ev[2].record(st)
    n1, fin1, ids1 = mig.stage(table, tokens, stream=st)
    ev[3].record(st)
    st.synchronize()
    assert (n0, fin0, n1, fin1) == (39, False, 1, True)               # the 39 full blocks, then the partly filled one
    t0, t1 = ev[0].elapsed_time(ev[1]), ev[2].elapsed_time(ev[3])
    rate0 = 2 * n0 * src.pool.block_bytes / (t0 * 1e-3) / 1e9
    rate1 = 2 * n1 * src.pool.block_bytes / (t1 * 1e-3) / 1e9
    print(f"session: stage 0 at {rate0:.1f} GB/s under a 50 GB/s budget, final stage {t1 * 1e3:.0f} us ({rate1:.0f} GB/s)")
    assert abs(rate0 - 50) <= 5 and t1 < 0.2           # one 8 MiB block under the budget would take 0.34 ms
    d_table = mig.commit(table)
    assert list(d_table) == list(ids0) + list(ids1)
    h_src = H.host_pool_from_synth(g, 0, 0, layers=[7])
    h_dst = om.new_pool(1, nb, H.tile_elems(g), fill=SENT)
    om.migrate_stage(h_src, table, h_dst, d_table)
    H.assert_pool_equal(dst.host_layer(7), h_dst)
    with pytest.raises(llx.LlxError) as e:
        mig2 = llx.Migration(src.pool, src_mgr, dst.pool, dst_mgr, 16, 2)
        mig2.stage([5, 5, 6], 40)                                      # a table that names a block twice cannot be committed
    assert e.value.name == "LLX_ERR_INVALID_ARG" and dst_mgr.num_free == nb - 40


# ---- CUDA graphs: captured where that is safe, refused (LLX_ERR_STATE) where it is not ------------------------------
G_LONG = dict(layers=8, kv_heads=8, head_dim=128, block_size=16, elem_bytes=2, num_blocks=800)      # 32 KiB tiles, 512 KiB blocks


def test_captured_long_stage_replays_on_other_streams_next_to_direct_launches(env):
    """A >= 64 MiB stage (the dynamic tail is active when it is launched directly) is captured on stream C and replayed
    on two other streams while the same kind of stage is launched directly on C.  In round 1 the captured launch kept C's
    claim counter: a replay running next to a direct launch shared it and chunks could be skipped silently.  Captured
    launches now run without the dynamic tail."""
    H, llx = env
    g = G_LONG
    nb = g["num_blocks"]
    src = H.DevPool(g)
    src.fill_device_random(5)
    dsts = [H.DevPool(g, fill=SENT) for _ in range(3)]                  # graph replay 1, graph replay 2, direct launches
    perm_s, perm_d = synth.block_permutation(61, nb), synth.block_permutation(62, nb)
    n = 256                                                             # ids still by value; 128 MiB payload = 4096 chunks of 32 KiB
    assert n * src.pool.block_bytes >= 64 << 20 and n * 2 * g["layers"] >= 148 * 16          # long stage with a tail worth claiming
    cap_st, r1, r2 = torch.cuda.Stream(), torch.cuda.Stream(), torch.cuda.Stream()
    for st in (cap_st, r1, r2):
        st.wait_stream(torch.cuda.current_stream())
    llx.migrate_stage(src.pool, perm_s[:n], dsts[2].pool, perm_d[:n], stream=cap_st)        # warm-up: first-use allocations
    cap_st.synchronize()
    dsts[2].view.fill_(SENT_I16)
    torch.cuda.synchronize()
    graphs = []
    for k in range(2):                                                  # one graph per destination pool
        gr = torch.cuda.CUDAGraph()
        with torch.cuda.graph(gr, stream=cap_st):
            llx.migrate_stage(src.pool, perm_s[:n], dsts[k].pool, perm_d[:n], stream=cap_st)
            llx.migrate_stage(src.pool, perm_s[n:2 * n], dsts[k].pool, perm_d[n:2 * n], stream=cap_st)
        graphs.append(gr)
    torch.cuda.synchronize()
    for d in dsts:
        assert bool((d.view == SENT_I16).all())                         # capturing ran nothing
    for rep in range(3):
        with torch.cuda.stream(r1):
            graphs[0].replay()
        with torch.cuda.stream(r2):
            graphs[1].replay()
        llx.migrate_stage(src.pool, perm_s[:n], dsts[2].pool, perm_d[:n], stream=cap_st)    # direct, dynamic tail on
        llx.migrate_stage(src.pool, perm_s[n:2 * n], dsts[2].pool, perm_d[n:2 * n], stream=cap_st)
    torch.cuda.synchronize()
    h_src = src.host()
    h_dst = om.new_pool(g["layers"], nb, H.tile_elems(g), fill=SENT)
    om.migrate_stage(h_src, perm_s[:2 * n], h_dst, perm_d[:2 * n])
    for d in dsts:
        H.assert_pool_equal(d.host(), h_dst)


def test_calls_that_cannot_be_captured_are_refused_and_leave_the_capture_valid(env):
    H, llx = env
    g = dict(synth.CONFIGS["tiny"], num_blocks=700)
    src, dst = H.DevPool(g), H.DevPool(g, fill=SENT)
    src.fill_from_synth(9, 0)
    h_src = H.host_pool_from_synth(g, 9, 0)
    s_ids, d_ids = synth.block_permutation(63, 700), synth.block_permutation(64, 700)
    pin = llx.PinnedStaging(llx.staging_bytes(src.pool, 4))
    dev_stg = torch.zeros(llx.staging_bytes(src.pool, 4), dtype=torch.uint8, device="cuda")
    st = torch.cuda.Stream()
    st.wait_stream(torch.cuda.current_stream())
    llx.migrate_stage(src.pool, s_ids[:3], dst.pool, d_ids[:3], stream=st)                   # warm-up
    st.synchronize()
    dst.view.fill_(SENT_I16)
    torch.cuda.synchronize()

    def refused(fn):
        with pytest.raises(llx.LlxError) as e:
            fn()
        assert e.value.name == "LLX_ERR_STATE", e.value

    gr = torch.cuda.CUDAGraph()
    with torch.cuda.graph(gr, stream=st):
        refused(lambda: llx.migrate_stage(src.pool, s_ids[:300], dst.pool, d_ids[:300], stream=st))          # ids through the pinned ring
        refused(lambda: llx.migrate_stage_wait(src.pool, s_ids[:2], dst.pool, d_ids[:2], stream=st))           # a blocking call
        refused(lambda: llx.pack(src.pool, s_ids[:4], pin.dev_alias, pin.nbytes, stream=st))                   # bounce buffers + copy engine
        refused(lambda: llx.migrate_via_host(src.pool, s_ids[:4], dst.pool, d_ids[:4], dev_stg.data_ptr(), dev_stg.numel(), stream=st))
        # what CAN be captured, in the same capture: it is still valid after the refusals
        llx.migrate_stage(src.pool, s_ids[:256], dst.pool, d_ids[:256], stream=st)                             # 256 pairs: ids by value
        llx.migrate_batch(src.pool, dst.pool, [0, 10, 44], s_ids[256:300], d_ids[256:300], stream=st)
        llx.pack(src.pool, s_ids[:4], dev_stg.data_ptr(), dev_stg.numel(), stream=st)                          # device staging buffer
    torch.cuda.synchronize()
    assert bool((dst.view == SENT_I16).all())
    other = torch.cuda.Stream()
    with torch.cuda.stream(other):
        gr.replay()
    other.synchronize()
    h_dst = om.new_pool(g["layers"], 700, H.tile_elems(g), fill=SENT)
    om.migrate_stage(h_src, s_ids[:300], h_dst, d_ids[:300])
    H.assert_pool_equal(dst.host(), h_dst)
    want = om.pack(h_src, s_ids[:4])
    assert np.array_equal(dev_stg.cpu().numpy().view(np.uint16).reshape(want.shape), want)
    pin.free()


# ---- a budgeted stage is a chain of short launches (LLX_OPT_PACED_SLICE_US) ------------------------------------------
@pytest.mark.parametrize("slice_us,unit_order,ids_by_value_max", [(1, 1, 256), (1, 0, 256), (1, 1, 0), (50, 1, 256)])
def test_sliced_budgeted_stage_is_bit_exact(env, slice_us, unit_order, ids_by_value_max):
    """Ragged 34,560-byte tiles (16 full 2 KiB chunks + a 1,792-byte tail per tile), 13 blocks, 40 GB/s: with tiny slices
    the stage becomes many launches over consecutive unit ranges; together they must copy every chunk exactly once."""
    H, llx = env
    g = dict(layers=3, kv_heads=9, head_dim=120, block_size=16, elem_bytes=2, num_blocks=40)
    src, dst = H.DevPool(g), H.DevPool(g, fill=SENT)
    src.fill_from_synth(5, 0)
    h_src = H.host_pool_from_synth(g, 5, 0)
    h_dst = om.new_pool(g["layers"], g["num_blocks"], H.tile_elems(g), fill=SENT)
    s_ids = synth.block_permutation(11, g["num_blocks"])[:13]
    d_ids = synth.block_permutation(12, g["num_blocks"])[:13]
    c0 = llx.counters()["copy_launches"]
    with llx.options(paced_slice_us=slice_us):
        llx.migrate_stage(src.pool, s_ids, dst.pool, d_ids, opts=dict(bandwidth_gbps=40, unit_order=unit_order, ids_by_value_max=ids_by_value_max))
    launches = llx.counters()["copy_launches"] - c0
    assert 2 <= launches <= 256, launches
    om.migrate_stage(h_src, s_ids, h_dst, d_ids)
    H.assert_pool_equal(dst.host(), h_dst)
    H.assert_pool_equal(src.host(), h_src)
    with llx.options(paced_slice_us=0):                                  # 0 = one launch for the whole stage
        c0 = llx.counters()["copy_launches"]
        llx.migrate_stage(src.pool, s_ids, dst.pool, d_ids, opts=dict(bandwidth_gbps=40))
        assert llx.counters()["copy_launches"] - c0 == 1
    H.assert_pool_equal(dst.host(), h_dst)


def test_overlapped_stages_are_bit_exact_and_complete_in_stream_order(env):
    """LLX_OPT_OVERLAP_PREV (llx_launch_opts.overlap_prev): a stage the caller declares independent of the previous
    kernel may START before that kernel has finished, but completion stays ordered.  A chain of stages over disjoint
    blocks — long ones with the dynamic tail (whose claim counter consecutive launches share), a short one right behind
    a long one (it could finish first if the deferred wait were dropped) and a batch launch (the stage of more than 256
    pairs, whose ids go through the pinned ring, is test_overlapped_stage_of_more_than_256_pairs below) — is enqueued back to back with the flag, then ONE event behind the last, smallest kernel is waited for: every
    byte of every stage must be there, equal to the oracle's, and the untouched blocks keep the sentinel."""
    H, llx = env
    g = G7
    sample = [0, 17, 31]
    src, dst = H.DevPool(g), H.DevPool(g, fill=SENT)
    src.fill_device_random(5)
    src.fill_from_synth(0, 0, layers=sample)
    perm_s = synth.block_permutation(11, g["num_blocks"])
    perm_d = synth.block_permutation(12, g["num_blocks"])
    cuts = [0, 112, 126, 128, 200, 264, 266, 267]                     # 112, 14, 2, 72 (batch), 64, 2, 1 blocks
    stream = torch.cuda.Stream()
    torch.cuda.synchronize()
    ov = dict(overlap_prev=1)
    for rep in range(3):                                                # the same chain three times: the counter is reused
        dst.view.fill_(SENT_I16)
        torch.cuda.synchronize()
        done = torch.cuda.Event()
        for k in range(len(cuts) - 1):
            a, b = cuts[k], cuts[k + 1]
            if b - a == 72:
                off = [0, 10, 10, 41, 72]                               # four requests, one of them empty
                llx.migrate_batch(src.pool, dst.pool, off, perm_s[a:b], perm_d[a:b], stream=stream, opts=ov)
            else:
                llx.migrate_stage(src.pool, perm_s[a:b], dst.pool, perm_d[a:b], stream=stream, opts=ov)
        done.record(stream)
        done.synchronize()                                              # NOT a device synchronize: only what the stream orders
        got = dst.view[sample].cpu().numpy().view(np.uint16)
        h_src = H.host_pool_from_synth(g, 0, 0, layers=sample)
        want = om.new_pool(len(sample), g["num_blocks"], src.te, fill=SENT)
        om.migrate_stage(h_src, perm_s[:cuts[-1]], want, perm_d[:cuts[-1]])
        H.assert_pool_equal(got, want)
    # layers the host does not mirror: every copied block equals its source block, element-wise on the device
    idx_s = torch.from_numpy(np.asarray(perm_s[:cuts[-1]], dtype=np.int64)).cuda()
    idx_d = torch.from_numpy(np.asarray(perm_d[:cuts[-1]], dtype=np.int64)).cuda()
    for l in range(g["layers"]):
        assert torch.equal(dst.view[l].index_select(1, idx_d), src.view[l].index_select(1, idx_s)), l


def test_overlapped_stage_of_more_than_256_pairs(env):
    """An overlapped stage whose id list does not fit the kernel parameters (> 256 pairs): the ids travel through the
    pinned ring and a device buffer, the copy of the ids is ordinary stream work in FRONT of the kernel.  Chain: a plain
    40-block stage, then 300 pairs with overlap_prev=1, then 8 pairs with overlap_prev=1; one event behind the last."""
    H, llx = env
    g = dict(G7, num_blocks=360)
    sample = [0, 13, 31]
    src, dst = H.DevPool(g), H.DevPool(g, fill=SENT)
    src.fill_device_random(15)
    src.fill_from_synth(0, 0, layers=sample)
    perm_s = synth.block_permutation(31, g["num_blocks"])
    perm_d = synth.block_permutation(32, g["num_blocks"])
    cuts = [0, 40, 340, 348]
    stream = torch.cuda.Stream()
    torch.cuda.synchronize()
    for rep in range(3):
        dst.view.fill_(SENT_I16)
        torch.cuda.synchronize()
        c0 = llx.counters()
        for k in range(3):
            a, b = cuts[k], cuts[k + 1]
            llx.migrate_stage(src.pool, perm_s[a:b], dst.pool, perm_d[a:b], stream=stream, opts=None if k == 0 else dict(overlap_prev=1))
        done = torch.cuda.Event()
        done.record(stream)
        done.synchronize()
        c1 = llx.counters()
        assert c1["id_uploads"] - c0["id_uploads"] == 1 and c1["copy_launches"] - c0["copy_launches"] == 3
        got = dst.view[sample].cpu().numpy().view(np.uint16)
        want = om.new_pool(len(sample), g["num_blocks"], src.te, fill=SENT)
        om.migrate_stage(H.host_pool_from_synth(g, 0, 0, layers=sample), perm_s[:cuts[-1]], want, perm_d[:cuts[-1]])
        H.assert_pool_equal(got, want)
    idx_s = torch.from_numpy(np.asarray(perm_s[:cuts[-1]], dtype=np.int64)).cuda()
    idx_d = torch.from_numpy(np.asarray(perm_d[:cuts[-1]], dtype=np.int64)).cuda()
    for l in range(g["layers"]):
        assert torch.equal(dst.view[l].index_select(1, idx_d), src.view[l].index_select(1, idx_s)), l


@pytest.mark.parametrize("middle", ["capped_stage", "append", "attention"])
def test_plain_launch_fences_the_start_of_an_overlapped_stage(env, middle):
    """llx.h, LLX_OPT_OVERLAP_PREV: an overlapped copy has to be independent of the launches back to the last PLAIN one
    only — what lies in front of that plain launch has completed when the copy starts, however small the plain launch is.
    Chain on one stream: A = a 64-block stage X -> Y capped at 4 CTAs (milliseconds, 144 SMs stay free); P = a plain launch
    that also leaves nearly every SM free (a 1-block stage capped at 2 CTAs / a 1-token append / a 1-sequence attention)
    and touches none of A's blocks; B = a full-width stage Y -> Z with overlap_prev=1 that reads what A wrote.  B is
    independent of P, as the contract asks, but not of A.  With kernels that let dependents launch BEFORE their own wait
    (round 2) P's CTAs released B at once, B found the free SMs and copied Y while A had written a fraction of it — with
    those kernels the capped-stage and append variants fail in the first repetitions (sentinel words in Z; the attention
    variant always held, llx_attn_partial waited first already); now P's CTAs release B only after A has completed.  Every word of Z
    is compared, 10 times with Y and Z invalidated in between."""
    H, llx = env
    g = dict(G7, num_blocks=160)
    X, Y, Z = H.DevPool(g), H.DevPool(g, fill=SENT), H.DevPool(g, fill=SENT)
    X.fill_device_random(19)
    perm_x = synth.block_permutation(41, g["num_blocks"])
    perm_y = synth.block_permutation(42, g["num_blocks"])
    perm_z = synth.block_permutation(43, g["num_blocks"])
    n = 64
    ax, ay, bz = perm_x[:n], perm_y[:n], perm_z[:n]
    # P's own blocks: outside everything A and B touch
    px, py = perm_x[n + 1:n + 2], perm_y[n + 1:n + 2]
    te_tok = g["kv_heads"] * g["head_dim"]
    vals = torch.zeros(g["layers"] * 2 * te_tok, dtype=torch.int16, device="cuda")
    q = torch.zeros(g["kv_heads"] * g["head_dim"], dtype=torch.int16, device="cuda")
    o = torch.zeros_like(q)
    bt = torch.tensor([int(px[0])], dtype=torch.int32, device="cuda")
    ctx = torch.tensor([16], dtype=torch.int32, device="cuda")
    i_x = torch.from_numpy(np.asarray(ax, dtype=np.int64)).cuda()
    i_z = torch.from_numpy(np.asarray(bz, dtype=np.int64)).cuda()
    want = [X.view[l].index_select(1, i_x) for l in range(g["layers"])]
    stream = torch.cuda.Stream()
    llx.decode_attention(X.pool, 0, q.data_ptr(), o.data_ptr(), bt.data_ptr(), ctx.data_ptr(), 1, 1, 1.0, stream=stream)  # workspace
    torch.cuda.synchronize()
    for rep in range(10):
        Y.view[:, :, :, ::256].fill_(SENT_I16)                          # one word per 512 B of every tile
        Z.view[:, :, :, ::256].fill_(SENT_I16)
        torch.cuda.synchronize()
        llx.migrate_stage(X.pool, ax, Y.pool, ay, stream=stream, opts=dict(max_ctas=4, copy_kernel=2))  # A
        if middle == "capped_stage":
            llx.migrate_stage(X.pool, px, Y.pool, py, stream=stream, opts=dict(max_ctas=2))            # P
        elif middle == "append":
            llx.append_tokens(X.pool, px, 3, 4, vals.data_ptr(), stream=stream)
        else:
            llx.decode_attention(X.pool, 0, q.data_ptr(), o.data_ptr(), bt.data_ptr(), ctx.data_ptr(), 1, 1, 1.0, stream=stream)
        llx.migrate_stage(Y.pool, ay, Z.pool, bz, stream=stream, opts=dict(overlap_prev=1))             # B reads what A wrote
        stream.synchronize()
        for l in range(g["layers"]):
            assert torch.equal(Z.view[l].index_select(1, i_z), want[l]), (rep, l)


def test_overlap_keeps_completion_transitive_behind_a_long_stage(env):
    """The property the deferred wait exists for: 'kernel N+1 has completed' implies 'kernel N has completed'.  A
    256-block stage (about 650 us) is followed by a ONE-block stage with overlap_prev=1 (about 10 us of work) and an
    event; as soon as the event has fired the long stage's LAST blocks are read back — they must already be complete.
    Repeated with fresh sentinel fills so that a stale pass cannot hide a miss.  Also: a stream-captured pair of
    overlapped stages replays bit-exactly (the flag touches no host state)."""
    H, llx = env
    g = dict(G7, num_blocks=600)
    src, dst = H.DevPool(g), H.DevPool(g, fill=SENT)
    src.fill_device_random(9)
    perm_s = synth.block_permutation(21, g["num_blocks"])
    perm_d = synth.block_permutation(22, g["num_blocks"])
    n_long = 256
    stream = torch.cuda.Stream()
    idx_s = torch.from_numpy(np.asarray(perm_s[:n_long + 1], dtype=np.int64)).cuda()
    idx_d = torch.from_numpy(np.asarray(perm_d[:n_long + 1], dtype=np.int64)).cuda()
    want = [src.view[l].index_select(1, idx_s) for l in (0, 31)]
    torch.cuda.synchronize()
    for rep in range(20):
        dst.view[:, :, :, ::512].fill_(SENT_I16)                        # cheap invalidation: one word per KiB of every tile
        torch.cuda.synchronize()
        ev = torch.cuda.Event()
        llx.migrate_stage(src.pool, perm_s[:n_long], dst.pool, perm_d[:n_long], stream=stream, opts=dict(ids_by_value_max=256))
        llx.migrate_stage(src.pool, perm_s[n_long:n_long + 1], dst.pool, perm_d[n_long:n_long + 1], stream=stream,
                          opts=dict(overlap_prev=1))
        ev.record(stream)
        ev.synchronize()
        check = torch.cuda.Stream()                                     # an unrelated stream: no implicit ordering helps
        with torch.cuda.stream(check):
            got = [dst.view[l].index_select(1, idx_d) for l in (0, 31)]
        check.synchronize()
        for gl, wl in zip(got, want):
            assert torch.equal(gl, wl), rep
    # capture: two overlapped stages in one graph, replayed on another stream
    a, b = perm_s[300:364], perm_s[364:380]
    da, db = perm_d[300:364], perm_d[364:380]
    cap = torch.cuda.Stream()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.stream(cap):
        llx.migrate_stage(src.pool, a, dst.pool, da, stream=cap, opts=dict(overlap_prev=1))     # warm-up outside the capture
        cap.synchronize()
        graph.capture_begin()
        llx.migrate_stage(src.pool, a, dst.pool, da, stream=cap, opts=dict(overlap_prev=1))
        llx.migrate_stage(src.pool, b, dst.pool, db, stream=cap, opts=dict(overlap_prev=1))
        graph.capture_end()
    dst.view.fill_(SENT_I16)
    torch.cuda.synchronize()
    with torch.cuda.stream(stream):
        graph.replay()
    stream.synchronize()
    i_s = torch.from_numpy(np.asarray(perm_s[300:380], dtype=np.int64)).cuda()
    i_d = torch.from_numpy(np.asarray(perm_d[300:380], dtype=np.int64)).cuda()
    for l in range(g["layers"]):
        assert torch.equal(dst.view[l].index_select(1, i_d), src.view[l].index_select(1, i_s)), l
    untouched = np.setdiff1d(np.arange(g["num_blocks"]), np.asarray(perm_d[300:380]))
    assert bool((dst.view[:, :, torch.from_numpy(untouched).cuda()] == SENT_I16).all())
