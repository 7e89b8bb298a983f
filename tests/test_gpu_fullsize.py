"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times (default options).

The pools are too large to mirror on the host (15.6 GiB / 71 GiB each), so — SURVEY.md §8(c) "verification
at scale" — layers are generated on the host from the seeded recipe ONE AT A TIME, replayed by the oracle and
compared with a readback of the same destination layer (all blocks: mapping P1 and sentinel P2): every layer
for configs[1], a sample of layers for the other configs, whose remaining layers are filled by a seeded device
generator and checked by properties that hold at any size (destination rows equal source rows under an independent torch gather; every untouched
destination block still holds the sentinel)."""
import numpy as np
import pytest
import torch

import synth
from oracle import kv_migration as om

pytestmark = pytest.mark.gpu
SENT = synth.SENTINEL_U16
SENT_I16 = int(np.array(SENT, dtype=np.uint16).view(np.int16))


@pytest.fixture(scope="module")
def env():
    import gpu_harness as H
    import paper_2406_03243_b200 as llx
    llx.load()
    return H, llx


def free_gib():
    import gc
    gc.collect()
    torch.cuda.empty_cache()
    free, _ = torch.cuda.mem_get_info()
    return free / 2**30


def check_untouched_and_mapping_on_device(src, dst, s_ids, d_ids, layers):
    """Properties on the device with torch indexing (independent of the library's kernels)."""
    s_idx = torch.from_numpy(np.asarray(s_ids, dtype=np.int64)).cuda()
    d_idx = torch.from_numpy(np.asarray(d_ids, dtype=np.int64)).cuda()
    mask = torch.ones(dst.nb, dtype=torch.bool, device="cuda")
    mask[d_idx] = False
    untouched = torch.nonzero(mask).flatten()
    for l in layers:
        for kv in range(2):
            assert torch.equal(dst.view[l, kv].index_select(0, d_idx), src.view[l, kv].index_select(0, s_idx)), (l, kv)
            assert bool((dst.view[l, kv].index_select(0, untouched) == SENT_I16).all()), (l, kv)


def test_llama7b_2048_tokens_three_stages_with_appends(env):
    """configs[1]: 2032 -> 2040 -> 2048 tokens, stages 112 / 14 / 2, 8-token appends between stages (A5).
    ALL 32 layers go through the oracle: each layer is generated from the seeded host recipe (A18), uploaded, and replayed
    by the oracle right away; what is kept per layer is the oracle's result for the rows it wrote (the 128 reserved
    destination blocks, the appended source block) after checking, in the oracle's own state, that nothing else changed —
    1 GiB for 32 layers instead of two 15.6 GiB host pools.  The device pools are then compared with that, every word."""
    H, llx = env
    g = synth.CONFIGS["llama7b"]
    if free_gib() < 50:
        pytest.skip("needs two 15.6 GiB pools and a snapshot of the source")
    L, S, te, nb = g["layers"], g["block_size"], H.tile_elems(g), g["num_blocks"]
    te_tok = g["kv_heads"] * g["head_dim"]
    src, dst = H.DevPool(g), H.DevPool(g, fill=SENT)
    s_tab = synth.block_permutation(1, nb)[:128]
    d_tab = synth.block_permutation(2, nb)[:128]
    schedule, appends, tokens = (112, 14, 2), (8, 8), 2032
    values = lambda t, l, kv: synth.append_values_f16(3, t, l, kv, te_tok)
    untouched = np.ones(nb, dtype=bool)
    untouched[d_tab] = False
    tail_block = int(s_tab[127])                                   # all 16 appended tokens land here (A5)

    want_dst_rows = np.empty((L, 2, 128, te), dtype=np.uint16)
    want_src_tail = np.empty((L, 2, te), dtype=np.uint16)
    for l in range(L):
        h_src = H.host_pool_from_synth(g, 0, 0, layers=[l])
        for kv in range(2):
            src.upload_slice(l, kv, h_src[0, kv])
        before = h_src[0][:, tail_block].copy()
        h_dst = om.new_pool(1, nb, te, fill=SENT)
        om.staged_migration(h_src, s_tab, h_dst, d_tab, schedule, appends, S, 2032, lambda t, _l, kv, l=l: values(t, l, kv))
        assert np.all(h_dst[0][:, untouched] == SENT)              # the oracle itself left every other block alone (P2)
        assert not np.array_equal(h_src[0][:, tail_block], before)  # and its appends did change the tail block
        want_dst_rows[l] = h_dst[0][:, d_tab]
        want_src_tail[l] = h_src[0][:, tail_block]
        del h_src, h_dst
    torch.cuda.synchronize()
    src_before = src.raw.clone()

    launches0 = llx.counters()["copy_launches"]
    m = 0
    for k, n in enumerate(schedule):
        llx.migrate_stage(src.pool, s_tab[m:m + n], dst.pool, d_tab[m:m + n])
        m += n
        if k < len(appends):
            vals = np.empty((appends[k], L, 2, te_tok), dtype=np.uint16)
            for j in range(appends[k]):
                for l in range(L):
                    for kv in range(2):
                        vals[j, l, kv] = values(tokens + j, l, kv)
            dev_vals = torch.from_numpy(vals.view(np.int16)).cuda()
            llx.append_tokens(src.pool, s_tab, tokens, tokens + appends[k], dev_vals.data_ptr())
            tokens += appends[k]
        # after EVERY stage: the blocks migrated so far equal their source blocks (device-side property, sampled layers)
        torch.cuda.synchronize()
        s_idx = torch.from_numpy(s_tab[:m].astype(np.int64)).cuda()
        d_idx = torch.from_numpy(d_tab[:m].astype(np.int64)).cuda()
        for l in (0, 17, 31):
            assert torch.equal(dst.view[l, 1].index_select(0, d_idx), src.view[l, 1].index_select(0, s_idx))
    assert tokens == 2048 and llx.counters()["copy_launches"] == launches0 + 3
    torch.cuda.synchronize()

    def verify():
        # destination: every word of every layer against the oracle
        for l in range(L):
            got = dst.host_layer(l)[0]
            rows = got[:, d_tab]
            if not np.array_equal(rows, want_dst_rows[l]):
                kv, i, e = np.argwhere(rows != want_dst_rows[l])[0]
                raise AssertionError(f"layer {l} kv {kv} block {d_tab[i]} elem {e}: expected 0x{int(want_dst_rows[l][kv, i, e]):04x} "
                                     f"got 0x{int(rows[kv, i, e]):04x}")
            assert np.all(got[:, untouched] == SENT), f"layer {l}: an unreserved destination block was written"
        # source: bit-identical to its state before the migration except the tail block, which holds the oracle's appends
        before_v = src_before.view(torch.int16).view(L, 2, nb, te)
        keep = torch.from_numpy(np.setdiff1d(np.arange(nb), [tail_block])).cuda()
        for l in range(L):
            assert torch.equal(src.view[l].index_select(1, keep), before_v[l].index_select(1, keep)), l
            assert np.array_equal(src.view[l, :, tail_block].cpu().numpy().view(np.uint16), want_src_tail[l]), l
        check_untouched_and_mapping_on_device(src, dst, s_tab, d_tab, range(L))

    verify()

    # The same request again exactly as bench.py issues it: nothing synchronised between the stages, stages 0 and 1
    # launched with llx_launch_opts.overlap_prev = 1 (they may start while the kernel before them drains), the appends
    # on the source's decode stream, the final stage waiting for them through an event.
    all_vals = np.empty((sum(appends), L, 2, te_tok), dtype=np.uint16)
    for j in range(sum(appends)):
        for l in range(L):
            for kv in range(2):
                all_vals[j, l, kv] = values(2032 + j, l, kv)
    dev_all = torch.from_numpy(all_vals.view(np.int16)).cuda()
    tok_bytes = L * 2 * te_tok * 2
    mig, dec = torch.cuda.Stream(), torch.cuda.Stream()
    ov = llx.LaunchOpts(overlap_prev=1)
    for rep in range(3):
        src.raw.copy_(src_before)
        dst.view.fill_(SENT_I16)
        torch.cuda.synchronize()
        e_app = torch.cuda.Event()
        t = 2032
        for a in appends:
            llx.append_tokens(src.pool, s_tab, t, t + a, dev_all.data_ptr() + (t - 2032) * tok_bytes, stream=dec)
            t += a
        e_app.record(dec)
        llx.migrate_stage(src.pool, s_tab[:112], dst.pool, d_tab[:112], stream=mig, opts=ov)
        llx.migrate_stage(src.pool, s_tab[112:126], dst.pool, d_tab[112:126], stream=mig, opts=ov)
        mig.wait_event(e_app)
        llx.migrate_stage(src.pool, s_tab[126:], dst.pool, d_tab[126:], stream=mig)
        mig.synchronize()
        if rep == 2:
            verify()
        else:
            check_untouched_and_mapping_on_device(src, dst, s_tab, d_tab, (0, 31))


@pytest.mark.parametrize("tokens", [256, 512, 1024, 2048, 4096, 8192])
def test_llama7b_length_sweep_ends_single_shot_vs_two_stage(env, tokens):
    """configs[2], every length of the sweep: single-shot copy == (n-2, 2) staged copy == oracle on sampled layers."""
    H, llx = env
    g = synth.CONFIGS["llama7b"]
    if free_gib() < 50:
        pytest.skip("needs three 15.6 GiB pools")
    n = tokens // g["block_size"]
    te = H.tile_elems(g)
    src, dst_a, dst_b = H.DevPool(g), H.DevPool(g, fill=SENT), H.DevPool(g, fill=SENT)
    src.fill_device_random(99)
    src.fill_from_synth(0, 0, layers=[5])
    s_tab = synth.block_permutation(40 + n, g["num_blocks"])[:n]
    d_tab = synth.block_permutation(50 + n, g["num_blocks"])[:n]
    llx.migrate_stage(src.pool, s_tab, dst_a.pool, d_tab)
    llx.migrate_stage(src.pool, s_tab[:n - 2], dst_b.pool, d_tab[:n - 2])
    llx.migrate_stage(src.pool, s_tab[n - 2:], dst_b.pool, d_tab[n - 2:])
    torch.cuda.synchronize()
    h_src = H.host_pool_from_synth(g, 0, 0, layers=[5])
    h_dst = om.new_pool(1, g["num_blocks"], te, fill=SENT)
    om.migrate_stage(h_src, s_tab, h_dst, d_tab)
    H.assert_pool_equal(dst_a.host_layer(5), h_dst)
    H.assert_pool_equal(dst_b.host_layer(5), h_dst)
    check_untouched_and_mapping_on_device(src, dst_a, s_tab, d_tab, range(0, g["layers"], 5))
    for l in range(0, g["layers"], 7):
        assert torch.equal(dst_a.view[l], dst_b.view[l])


def test_llama30b_batch_of_64_requests(env):
    """configs[3]: 64 requests, bounded-Pareto lengths (mean 512, [16, 8192]), one llx_migrate_batch launch."""
    H, llx = env
    g = dict(synth.CONFIGS["llama30b"])
    lens, nblk, seed_used = synth.batch_request_blocks(0, 64, g["block_size"], g["num_blocks"])
    total = int(nblk.sum())
    block_gib = 2 * g["layers"] * H.tile_elems(g) * 2 / 2**30
    # shrink both pools equally if two 3000-block pools (142.8 GiB) do not fit next to the workspace (recorded)
    nb = g["num_blocks"]
    while 2 * nb * block_gib > free_gib() - 6 and nb > total:
        nb -= 100
    if nb < total:
        pytest.skip(f"not enough device memory for {total} blocks per pool")
    g["num_blocks"] = nb
    te = H.tile_elems(g)
    src, dst = H.DevPool(g), H.DevPool(g, fill=SENT)
    src.fill_device_random(7)
    sample = [0, 59]
    src.fill_from_synth(0, 0, layers=sample)
    s_ids = synth.block_permutation(1, nb)[:total]
    d_ids = synth.block_permutation(2, nb)[:total]
    off = np.concatenate([[0], np.cumsum(nblk)]).astype(np.int32)
    c0 = llx.counters()
    llx.migrate_batch(src.pool, dst.pool, off, s_ids, d_ids)
    torch.cuda.synchronize()
    c1 = llx.counters()
    assert c1["copy_launches"] == c0["copy_launches"] + 1
    assert c1["bytes_moved"] - c0["bytes_moved"] == total * src.pool.block_bytes
    for l in sample:
        h_src = H.host_pool_from_synth(g, 0, 0, layers=[l])
        h_dst = om.new_pool(1, nb, te, fill=SENT)
        om.migrate_batch(h_src, h_dst, off, s_ids, d_ids)
        H.assert_pool_equal(dst.host_layer(l), h_dst)
    check_untouched_and_mapping_on_device(src, dst, s_ids, d_ids, range(0, g["layers"], 6))


def test_llama7b_2048_tokens_through_the_pinned_host_buffer(env):
    """bench.py's e2e leg: llx_migrate_via_host of the 128-block request with the library's own chunk schedule
    (64 MiB chunks), plus llx_pack / llx_unpack through the same 1 GiB pinned buffer."""
    H, llx = env
    g = synth.CONFIGS["llama7b"]
    if free_gib() < 34:
        pytest.skip("needs two 15.6 GiB pools")
    L, te = g["layers"], H.tile_elems(g)
    sample_layers = [0, 19, 31]
    src, dst = H.DevPool(g), H.DevPool(g, fill=SENT)
    src.fill_device_random(4321)
    src.fill_from_synth(0, 0, layers=sample_layers)
    s_tab = synth.block_permutation(1, g["num_blocks"])[:128]
    d_tab = synth.block_permutation(2, g["num_blocks"])[:128]
    nbytes = llx.staging_bytes(src.pool, 128)
    pin = llx.PinnedStaging(nbytes)
    st = torch.cuda.Stream()
    st.wait_stream(torch.cuda.current_stream())
    llx.migrate_via_host(src.pool, s_tab, dst.pool, d_tab, pin.dev_alias, nbytes, stream=st)
    st.synchronize()
    buf = pin.as_numpy().reshape(128, L, 2, te)
    for l in sample_layers:
        h_src = H.host_pool_from_synth(g, 0, 0, layers=[l])
        h_dst = om.new_pool(1, g["num_blocks"], te, fill=SENT)
        want = om.migrate_via_buffer(h_src, s_tab, h_dst, d_tab)
        H.assert_pool_equal(dst.host_layer(l), h_dst)
        assert np.array_equal(buf[:, l], want[:, 0])                 # the pinned buffer holds the fused blocks (A6)
    check_untouched_and_mapping_on_device(src, dst, s_tab, d_tab, range(L))
    # the same request once more through the other host leg (gather / scatter kernels + bounce buffers, 64 MiB chunks)
    d3 = synth.block_permutation(10, g["num_blocks"])
    d3 = d3[~np.isin(d3, d_tab)][:128]
    pin.as_numpy()[:] = 0
    llx.migrate_via_host(src.pool, s_tab, dst.pool, d3, pin.dev_alias, nbytes, stream=st, opts=dict(via_host_mode=3))
    st.synchronize()
    buf = pin.as_numpy().reshape(128, L, 2, te)
    for l in sample_layers[:1]:
        h_src = H.host_pool_from_synth(g, 0, 0, layers=[l])
        assert np.array_equal(buf[:, l], om.pack(h_src, s_tab)[:, 0])
    check_untouched_and_mapping_on_device(src, dst, np.concatenate([s_tab, s_tab]), np.concatenate([d_tab, d3]), range(0, L, 3))
    # the two halves on their own: pack into the buffer, unpack into other destination blocks
    d2 = synth.block_permutation(9, g["num_blocks"])
    d2 = d2[~np.isin(d2, np.concatenate([d_tab, d3]))][:128]
    pin.as_numpy()[:] = 0
    llx.pack(src.pool, s_tab, pin.dev_alias, nbytes, stream=st)
    llx.unpack(pin.dev_alias, nbytes, dst.pool, d2, stream=st)
    st.synchronize()
    check_untouched_and_mapping_on_device(src, dst, np.concatenate([s_tab, s_tab, s_tab]), np.concatenate([d_tab, d3, d2]), range(0, L, 5))
    pin.free()
