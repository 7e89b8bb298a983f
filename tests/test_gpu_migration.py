"""GPU-vs-oracle parity for the migration path (S3-S6, S8), bit-exact on uint16 views.  All calls go
through the C-ABI (paper_2406_03243_b200.binding -> libllx.so).  SURVEY.md §8(c) P1-P8 on the device."""
import numpy as np
import pytest
import torch

import synth
from oracle import kv_migration as om

pytestmark = pytest.mark.gpu

SENT = synth.SENTINEL_U16
TINY = synth.CONFIGS["tiny"]
# a tile of 34,560 bytes: two full 16 KiB chunks and a ragged 1,792-byte tail
RAGGED = dict(layers=3, kv_heads=9, head_dim=120, block_size=16, elem_bytes=2, num_blocks=40)
# a tile smaller than any chunk (1,008 bytes)
SMALLTILE = dict(layers=2, kv_heads=7, head_dim=24, block_size=3, elem_bytes=2, num_blocks=64)

KERNELS = [dict(copy_kernel=2), dict(copy_kernel=1), dict(copy_kernel=2, chunk_bytes=4096, ring_stages=2),
           dict(copy_kernel=1, chunk_bytes=2048), dict(copy_kernel=2, ids_by_value_max=0),
           dict(copy_kernel=1, ids_by_value_max=0), dict(copy_kernel=2, max_ctas=3), dict(copy_kernel=1, max_ctas=1),
           dict(bandwidth_gbps=40), dict(bandwidth_gbps=3000), dict(copy_kernel=2, unit_order=0), dict(copy_kernel=1, unit_order=0),
           dict(copy_kernel=2, l2_hint=3, rings_per_cta=2), dict(pdl=0),
           dict(copy_kernel=2, dynamic_tail_pct=30, max_ctas=2, chunk_bytes=1024),
           dict(copy_kernel=2, dynamic_tail_pct=100, max_ctas=3, chunk_bytes=512, ring_stages=3, rings_per_cta=2),
           dict(overlap_prev=1), dict(overlap_prev=1, copy_kernel=2, dynamic_tail_pct=50, max_ctas=2, chunk_bytes=1024),
           dict(overlap_prev=1, copy_kernel=1), dict(overlap_prev=1, pdl=0)]


@pytest.fixture(scope="module")
def env():
    import gpu_harness as H
    import paper_2406_03243_b200 as llx
    llx.load()
    return H, llx


def make(H, g, seed=0):
    src = H.DevPool(g)
    src.fill_from_synth(seed, 0)
    dst = H.DevPool(g, fill=SENT)
    h_src = H.host_pool_from_synth(g, seed, 0)
    h_dst = om.new_pool(g["layers"], g["num_blocks"], H.tile_elems(g), fill=SENT)
    return src, dst, h_src, h_dst


# ---- configs[0] "Tiny": 100-token request, 7 blocks, 2 stages (5 then 2); everything compared after every stage
@pytest.mark.parametrize("opts", KERNELS)
def test_tiny_two_stage_migration_bit_exact(env, opts):
    H, llx = env
    src, dst, h_src, h_dst = make(H, TINY)
    s_tab = synth.block_permutation(1, TINY["num_blocks"])[:7]
    d_tab = synth.block_permutation(2, TINY["num_blocks"])[:7]
    m = 0
    for n in (5, 2):                                    # the option set is THIS call's launch policy (llx_migrate_stage_ex)
        llx.migrate_stage(src.pool, s_tab[m:m + n], dst.pool, d_tab[m:m + n], opts=opts)
        om.migrate_stage(h_src, s_tab[m:m + n], h_dst, d_tab[m:m + n])
        m += n
        H.assert_pool_equal(dst.host(), h_dst)      # P1 mapping + P2 sentinel on every other block
        H.assert_pool_equal(src.host(), h_src)      # P3 source intact
    untouched = np.setdiff1d(np.arange(TINY["num_blocks"]), d_tab)
    assert np.all(dst.host()[:, :, untouched] == SENT)


@pytest.mark.parametrize("g", [RAGGED, SMALLTILE])
@pytest.mark.parametrize("opts", KERNELS)
@pytest.mark.parametrize("n", [1, 13])
def test_ragged_tiles_and_small_tiles(env, g, opts, n):
    H, llx = env
    src, dst, h_src, h_dst = make(H, g, seed=5)
    s_ids = synth.block_permutation(11, g["num_blocks"])[:n]
    d_ids = synth.block_permutation(12, g["num_blocks"])[:n]
    llx.migrate_stage(src.pool, s_ids, dst.pool, d_ids, opts=opts)
    om.migrate_stage(h_src, s_ids, h_dst, d_ids)
    H.assert_pool_equal(dst.host(), h_dst)
    H.assert_pool_equal(src.host(), h_src)


@pytest.mark.parametrize("opts", [dict(copy_kernel=1, chunk_bytes=2048), dict(bandwidth_gbps=40), dict(copy_kernel=2, max_ctas=3)])
def test_process_default_options_are_inherited_by_plain_calls(env, opts):
    """llx_set_option sets process DEFAULTS: a plain llx_migrate_stage (no llx_launch_opts) inherits them, and a call's
    own opts override them field by field."""
    H, llx = env
    src, dst, h_src, h_dst = make(H, RAGGED, seed=5)
    s_ids = synth.block_permutation(11, RAGGED["num_blocks"])[:13]
    d_ids = synth.block_permutation(12, RAGGED["num_blocks"])[:13]
    with llx.options(**opts):
        llx.migrate_stage(src.pool, s_ids[:6], dst.pool, d_ids[:6])
        llx.migrate_stage(src.pool, s_ids[6:], dst.pool, d_ids[6:], opts=dict(copy_kernel=2, bandwidth_gbps=0, max_ctas=0))
    om.migrate_stage(h_src, s_ids, h_dst, d_ids)
    H.assert_pool_equal(dst.host(), h_dst)
    with pytest.raises(llx.LlxError) as e:
        llx.migrate_stage(src.pool, s_ids, dst.pool, d_ids, opts=dict(chunk_bytes=100))      # not a multiple of 16
    assert e.value.name == "LLX_ERR_INVALID_ARG"
    bad = llx.LaunchOpts()
    bad.struct_size = 6
    with pytest.raises(llx.LlxError):
        llx.migrate_stage(src.pool, s_ids, dst.pool, d_ids, opts=bad)
    short = llx.LaunchOpts(copy_kernel=1, route=7)      # an older, shorter struct: fields beyond struct_size are not read
    short.struct_size = 16
    llx.migrate_stage(src.pool, s_ids, dst.pool, d_ids, opts=short)
    H.assert_pool_equal(dst.host(), h_dst)


def test_whole_pool_and_ids_through_the_ring(env):
    """n = num_blocks > 256: ids go through the pinned ring, every block moves, twice in a row (slot reuse)."""
    H, llx = env
    g = dict(TINY, num_blocks=700)
    src, dst, h_src, h_dst = make(H, g, seed=2)
    for rep in range(3):
        s_ids = synth.block_permutation(20 + rep, 700)
        d_ids = synth.block_permutation(30 + rep, 700)
        c0 = llx.counters()["id_uploads"]
        llx.migrate_stage(src.pool, s_ids, dst.pool, d_ids)
        assert llx.counters()["id_uploads"] == c0 + 1
        om.migrate_stage(h_src, s_ids, h_dst, d_ids)
        H.assert_pool_equal(dst.host(), h_dst)


def test_duplicate_source_ids_are_legal(env):
    H, llx = env
    src, dst, h_src, h_dst = make(H, TINY)
    llx.migrate_stage(src.pool, [9, 9, 9], dst.pool, [0, 100, 255])
    om.migrate_stage(h_src, [9, 9, 9], h_dst, [0, 100, 255])
    H.assert_pool_equal(dst.host(), h_dst)


def test_order_and_partition_invariance(env):                       # P6
    H, llx = env
    g = RAGGED
    src, dst_a, h_src, h_dst = make(H, g, seed=7)
    dst_b, dst_c = H.DevPool(g, fill=SENT), H.DevPool(g, fill=SENT)
    s_ids = synth.block_permutation(1, g["num_blocks"])[:17]
    d_ids = synth.block_permutation(2, g["num_blocks"])[:17]
    llx.migrate_stage(src.pool, s_ids, dst_a.pool, d_ids)
    p = np.random.default_rng(3).permutation(17)
    llx.migrate_stage(src.pool, s_ids[p], dst_b.pool, d_ids[p])
    for a, b in [(0, 1), (1, 9), (9, 17)]:
        llx.migrate_stage(src.pool, s_ids[a:b], dst_c.pool, d_ids[a:b])
    om.migrate_stage(h_src, s_ids, h_dst, d_ids)
    for d in (dst_a, dst_b, dst_c):
        H.assert_pool_equal(d.host(), h_dst)


def test_batch_equals_sequential_and_oracle(env):                   # P7, S5
    H, llx = env
    g = RAGGED
    src, dst, h_src, h_dst = make(H, g, seed=8)
    dst_seq = H.DevPool(g, fill=SENT)
    s_ids = synth.block_permutation(1, g["num_blocks"])[:30]
    d_ids = synth.block_permutation(2, g["num_blocks"])[:30]
    off = [0, 7, 7, 8, 21, 30]                                       # includes an empty request
    llx.migrate_batch(src.pool, dst.pool, off, s_ids, d_ids)
    for r in range(5):
        llx.migrate_stage(src.pool, s_ids[off[r]:off[r + 1]], dst_seq.pool, d_ids[off[r]:off[r + 1]])
    om.migrate_batch(h_src, h_dst, off, s_ids, d_ids)
    H.assert_pool_equal(dst.host(), h_dst)
    H.assert_pool_equal(dst_seq.host(), h_dst)
    llx.migrate_batch(src.pool, dst.pool, [0], [], [])               # R = 0
    llx.migrate_batch(src.pool, dst.pool, [0, 0, 0], [], [])         # only empty requests
    H.assert_pool_equal(dst.host(), h_dst)


@pytest.mark.parametrize("where", ["device", "pinned"])
@pytest.mark.parametrize("opts", [dict(), dict(copy_kernel=1), dict(copy_kernel=2), dict(via_host_mode=3), dict(via_host_mode=2)])
def test_pack_unpack_block_fusion(env, where, opts):                 # P5, S6
    H, llx = env
    g = RAGGED
    src, dst, h_src, h_dst = make(H, g, seed=9)
    n = 11
    s_ids = synth.block_permutation(1, g["num_blocks"])[:n]
    d_ids = synth.block_permutation(2, g["num_blocks"])[:n]
    nbytes = llx.staging_bytes(src.pool, n)
    assert nbytes == n * 2 * g["layers"] * src.pool.tile_bytes
    if where == "device":
        stg = torch.full((nbytes // 2,), 0x1111, dtype=torch.int16, device="cuda")
        ptr = stg.data_ptr()
    else:
        pin = llx.PinnedStaging(nbytes)
        pin.as_numpy()[:] = 0x1111
        ptr = pin.dev_alias
    llx.pack(src.pool, s_ids, ptr, nbytes, opts=opts)
    torch.cuda.synchronize()
    got = stg.cpu().numpy().view(np.uint16) if where == "device" else pin.as_numpy().copy()
    want = om.pack(h_src, s_ids)
    assert np.array_equal(got.reshape(want.shape), want)         # staging layout [i][l][kv][tile] (A6)
    llx.unpack(ptr, nbytes, dst.pool, d_ids, opts=opts)
    om.unpack(want, h_dst, d_ids)
    H.assert_pool_equal(dst.host(), h_dst)
    direct = H.DevPool(g, fill=SENT)
    llx.migrate_stage(src.pool, s_ids, direct.pool, d_ids)           # unpack(pack(.)) == migrate (P5)
    H.assert_pool_equal(direct.host(), h_dst)
    H.assert_pool_equal(src.host(), h_src)
    if where == "pinned":
        pin.free()


@pytest.mark.parametrize("where", ["device", "pinned", "pinned_zero_copy", "pinned_strided_ce", "pinned_bounce"])
@pytest.mark.parametrize("n,chunk", [(1, 0), (11, 0), (11, 1), (13, 4), (37, 5), (40, 64)])
def test_migrate_via_host_pipelined_route(env, where, n, chunk):    # S6: PAPER.md:235-237 in one call
    H, llx = env
    mode = {"pinned_zero_copy": 1, "pinned_strided_ce": 2, "pinned_bounce": 3}.get(where, 0)
    where = where.split("_")[0]
    g = RAGGED
    src, dst, h_src, h_dst = make(H, g, seed=10)
    s_ids = synth.block_permutation(5, g["num_blocks"])[:n]
    d_ids = synth.block_permutation(6, g["num_blocks"])[:n]
    nbytes = llx.staging_bytes(src.pool, n)
    if where == "device":
        stg = torch.full((nbytes // 2,), 0x2222, dtype=torch.int16, device="cuda")
        ptr = stg.data_ptr()
    else:
        pin = llx.PinnedStaging(nbytes)
        pin.as_numpy()[:] = 0x2222
        ptr = pin.dev_alias
    st = torch.cuda.Stream()
    st.wait_stream(torch.cuda.current_stream())
    o = dict(via_host_mode=mode)
    llx.migrate_via_host(src.pool, s_ids, dst.pool, d_ids, ptr, nbytes, chunk_blocks=chunk, stream=st, opts=o)
    if n == 37:      # a second migration right behind the first reuses the bounce buffers and events
        llx.migrate_via_host(src.pool, s_ids[::-1], dst.pool, d_ids[::-1], ptr, nbytes, chunk_blocks=chunk + 1, stream=st, opts=o)
        llx.migrate_via_host(src.pool, s_ids, dst.pool, d_ids, ptr, nbytes, chunk_blocks=chunk, stream=st, opts=o)
    # work enqueued on the caller's stream afterwards must see the complete migration (the call joins its side stream)
    with torch.cuda.stream(st):
        after = dst.view.clone()
    st.synchronize()
    want_buf = om.migrate_via_buffer(h_src, s_ids, h_dst, d_ids)
    H.assert_pool_equal(after.cpu().numpy().view(np.uint16), h_dst)
    got = stg.cpu().numpy().view(np.uint16) if where == "device" else pin.as_numpy().copy()
    assert np.array_equal(got.reshape(want_buf.shape), want_buf)
    H.assert_pool_equal(src.host(), h_src)
    if where == "pinned":
        pin.free()


def test_migrate_via_host_argument_errors(env):
    H, llx = env
    src, dst, h_src, h_dst = make(H, TINY)
    stg = torch.empty(llx.staging_bytes(src.pool, 2), dtype=torch.uint8, device="cuda")
    launches = llx.counters()["kernel_launches"]
    for name, fn in [
        ("LLX_ERR_STAGING_TOO_SMALL", lambda: llx.migrate_via_host(src.pool, [0, 1, 2], dst.pool, [0, 1, 2], stg.data_ptr(), stg.numel())),
        ("LLX_ERR_DUPLICATE_DST", lambda: llx.migrate_via_host(src.pool, [0, 1], dst.pool, [3, 3], stg.data_ptr(), stg.numel())),
        ("LLX_ERR_BLOCK_OUT_OF_RANGE", lambda: llx.migrate_via_host(src.pool, [0, 999], dst.pool, [3, 4], stg.data_ptr(), stg.numel())),
        ("LLX_ERR_ALIAS", lambda: llx.migrate_via_host(src.pool, [0], dst.pool, [3], dst.raw.data_ptr(), dst.raw.numel())),
        ("LLX_ERR_ALIAS", lambda: llx.migrate_via_host(src.pool, [0], src.pool, [3], stg.data_ptr(), stg.numel())),
    ]:
        with pytest.raises(llx.LlxError) as e:
            fn()
        assert e.value.name == name, e.value
    llx.migrate_via_host(src.pool, [], dst.pool, [], stg.data_ptr(), stg.numel())
    assert llx.counters()["kernel_launches"] == launches
    H.assert_pool_equal(dst.host(), h_dst)


def test_staged_with_appends_equals_oracle_and_single_shot(env):     # P4, S1, S8 on the Tiny shape
    H, llx = env
    g = TINY
    S, te_tok = g["block_size"], g["kv_heads"] * g["head_dim"]
    src, dst, h_src, h_dst = make(H, g)
    s_tab = synth.block_permutation(1, g["num_blocks"])[:7]
    d_tab = synth.block_permutation(2, g["num_blocks"])[:7]
    values = lambda t, l, kv: synth.append_values_f16(3, t, l, kv, te_tok)
    tokens, m = 97, 0
    for k, (n, app) in enumerate([(5, 3), (2, 0)]):
        if k == 1:                                                   # S1: the library's planner names the final stage
            assert llx.plan_stage(tokens, m, S, 2) == om.plan_stage(tokens, m, S, 2) == (n, True)
        llx.migrate_stage(src.pool, s_tab[m:m + n], dst.pool, d_tab[m:m + n])
        m += n
        if app:
            vals = np.stack([np.stack([np.stack([values(t, l, kv) for kv in range(2)]) for l in range(g["layers"])])
                             for t in range(tokens, tokens + app)])          # [t][l][kv][H*D]
            dev_vals = torch.from_numpy(vals.view(np.int16)).cuda()
            llx.append_tokens(src.pool, s_tab, tokens, tokens + app, dev_vals.data_ptr())
            tokens += app
    final_tokens = om.staged_migration(h_src, s_tab, h_dst, d_tab, (5, 2), (3,), S, 97, values)
    assert final_tokens == tokens == 100
    H.assert_pool_equal(src.host(), h_src)                          # appends landed in exactly the oracle's slots
    H.assert_pool_equal(dst.host(), h_dst)
    single = om.new_pool(g["layers"], g["num_blocks"], H.tile_elems(g), SENT)
    om.migrate_stage(h_src, s_tab, single, d_tab)
    H.assert_pool_equal(dst.host(), single)                         # P4


def test_library_owned_pool_upload_download_fill(env):
    H, llx = env
    g = SMALLTILE
    te = H.tile_elems(g)
    a = llx.pool_create(g["layers"], g["kv_heads"], g["head_dim"], g["block_size"], llx.F16, g["num_blocks"])
    b = llx.pool_create(g["layers"], g["kv_heads"], g["head_dim"], g["block_size"], llx.F16, 80)   # other num_blocks: legal
    assert a.tile_bytes == te * 2 and a.num_blocks == 64 and b.nbytes == 80 * a.block_bytes
    h_src = H.host_pool_from_synth(g, 4, 0)
    for l in range(g["layers"]):
        for kv in range(2):
            a.upload(l, kv, 0, h_src[l, kv])
    b.fill_u16(SENT)
    h_dst = om.new_pool(g["layers"], 80, te, fill=SENT)
    s_ids, d_ids = [63, 0, 5, 17], [79, 64, 1, 0]
    llx.migrate_stage(a, s_ids, b, d_ids)
    om.migrate_stage(h_src, s_ids, h_dst, d_ids)
    torch.cuda.synchronize()
    for l in range(g["layers"]):
        for kv in range(2):
            got = b.download(l, kv, 0, 80)
            torch.cuda.synchronize()
            assert np.array_equal(got, h_dst[l, kv])
            assert np.array_equal(a.download(l, kv, 3, 5), h_src[l, kv, 3:8])
    a.destroy()
    b.destroy()


def test_argument_errors_change_no_byte(env):
    H, llx = env
    src, dst, h_src, h_dst = make(H, TINY)
    other = H.DevPool(RAGGED, fill=SENT)
    launches = llx.counters()["kernel_launches"]

    def err(name, fn):
        with pytest.raises(llx.LlxError) as e:
            fn()
        assert e.value.name == name, e.value

    err("LLX_ERR_BLOCK_OUT_OF_RANGE", lambda: llx.migrate_stage(src.pool, [0, 256], dst.pool, [1, 2]))
    err("LLX_ERR_BLOCK_OUT_OF_RANGE", lambda: llx.migrate_stage(src.pool, [0, 1], dst.pool, [1, -1]))
    err("LLX_ERR_DUPLICATE_DST", lambda: llx.migrate_stage(src.pool, [0, 1], dst.pool, [4, 4]))
    err("LLX_ERR_ALIAS", lambda: llx.migrate_stage(src.pool, [0], src.pool, [1]))
    err("LLX_ERR_GEOMETRY_MISMATCH", lambda: llx.migrate_stage(src.pool, [0], other.pool, [1]))
    err("LLX_ERR_INVALID_ARG", lambda: llx.migrate_batch(src.pool, dst.pool, [0, 2, 1, 3], [0, 1, 2], [0, 1, 2]))
    err("LLX_ERR_DUPLICATE_DST", lambda: llx.migrate_batch(src.pool, dst.pool, [0, 1, 2], [0, 1], [7, 7]))
    stg = torch.empty(llx.staging_bytes(src.pool, 2), dtype=torch.uint8, device="cuda")
    err("LLX_ERR_STAGING_TOO_SMALL", lambda: llx.pack(src.pool, [0, 1, 2], stg.data_ptr(), stg.numel()))
    err("LLX_ERR_STAGING_TOO_SMALL", lambda: llx.unpack(stg.data_ptr(), stg.numel(), dst.pool, [0, 1, 2]))
    err("LLX_ERR_ALIAS", lambda: llx.pack(src.pool, [0], src.raw.data_ptr(), src.raw.numel()))
    err("LLX_ERR_INVALID_ARG", lambda: llx.append_tokens(src.pool, [1, 2], 30, 40, stg.data_ptr()))
    alias = llx.pool_wrap(src.raw.data_ptr(), src.raw.numel(), TINY["layers"], TINY["kv_heads"], TINY["head_dim"],
                          TINY["block_size"], llx.F16, TINY["num_blocks"])
    err("LLX_ERR_ALIAS", lambda: llx.migrate_stage(src.pool, [0], alias, [1]))       # distinct handle, same memory
    err("LLX_ERR_INVALID_ARG", lambda: llx.pool_wrap(src.raw.data_ptr(), 100, 2, 4, 64, 16, llx.F16, 256))
    err("LLX_ERR_INVALID_ARG", lambda: llx.pool_wrap(src.raw.data_ptr() + 2, 1 << 20, 1, 1, 8, 1, llx.F16, 4))
    llx.migrate_stage(src.pool, [], dst.pool, [])                                   # n == 0: OK, no launch
    assert llx.counters()["kernel_launches"] == launches
    H.assert_pool_equal(dst.host(), h_dst)
    H.assert_pool_equal(src.host(), h_src)


def test_migration_on_a_side_stream_concurrent_with_default_stream(env):
    H, llx = env
    src, dst, h_src, h_dst = make(H, TINY)
    side = torch.cuda.Stream(priority=0)
    side.wait_stream(torch.cuda.current_stream())
    s_ids = synth.block_permutation(1, 256)[:100]
    d_ids = synth.block_permutation(2, 256)[:100]
    for a in range(0, 100, 10):
        llx.migrate_stage(src.pool, s_ids[a:a + 10], dst.pool, d_ids[a:a + 10], stream=side)
    side.synchronize()
    om.migrate_stage(h_src, s_ids, h_dst, d_ids)
    H.assert_pool_equal(dst.host(), h_dst)


def test_migration_session_handshake_drives_the_copies(env):        # NEXT-3: PAPER.md:142 around S1/S3/S4/S8
    """A whole live migration through llx_migration_*: planner + PRE-ALLOC + copy per stage, appends in between,
    commit; destination content equals the oracle's staged migration, block bookkeeping equals oracle.handshake."""
    from oracle import handshake as oh
    H, llx = env
    g = TINY
    S, te_tok, nb = g["block_size"], g["kv_heads"] * g["head_dim"], g["num_blocks"]
    src, dst, h_src, h_dst = make(H, g)
    values = lambda t, l, kv: synth.append_values_f16(3, t, l, kv, te_tok)
    src_mgr, dst_mgr = llx.BlockManager(nb), llx.BlockManager(nb)
    o_src, o_dst = oh.BlockManager(nb), oh.BlockManager(nb)
    dst_mgr.alloc(9), o_dst.allocate(9)                              # the destination already serves other requests
    table = src_mgr.alloc(7)
    o_table = o_src.allocate(7)
    assert list(table) == o_table
    mig = llx.Migration(src.pool, src_mgr, dst.pool, dst_mgr, S, 2)
    o_mig = oh.Migration(o_src, o_dst, S, 2)
    st = torch.cuda.Stream()
    st.wait_stream(torch.cuda.current_stream())
    tokens, schedule = 97, []
    while mig.state not in (llx.MIG_FINAL_COPYING,):
        n, fin, ids = mig.stage(table, tokens, stream=st)
        o = o_mig.stage(tokens)
        assert (n, fin, list(ids)) == (o[0], o[1], o[3])
        schedule.append(n)
        if not fin:                                                  # decoding continues: 3 more tokens
            vals = np.stack([np.stack([np.stack([values(t, l, kv) for kv in range(2)]) for l in range(g["layers"])])
                             for t in range(tokens, tokens + 3)])
            dev_vals = torch.from_numpy(vals.view(np.int16)).cuda()
            st.wait_stream(torch.cuda.current_stream())
            llx.append_tokens(src.pool, table, tokens, tokens + 3, dev_vals.data_ptr(), stream=st)
            tokens += 3
    st.synchronize()
    d_table = mig.commit(table)
    assert list(d_table) == o_mig.commit(o_table) and mig.state == llx.MIG_COMMITTED
    assert (src_mgr.num_free, dst_mgr.num_free) == (o_src.num_free(), o_dst.num_free()) == (nb, nb - 9 - 7)
    assert schedule == [6, 1] and tokens == 100
    om.staged_migration(h_src, np.array(o_table), h_dst, np.array(d_table), schedule, (3,), S, 97, values)
    H.assert_pool_equal(dst.host(), h_dst)
    H.assert_pool_equal(src.host(), h_src)


def test_migration_session_abort_releases_reservation_and_touches_nothing_else(env):
    H, llx = env
    g = TINY
    nb = g["num_blocks"]
    src, dst, h_src, h_dst = make(H, g)
    src_mgr, dst_mgr = llx.BlockManager(nb), llx.BlockManager(nb)
    table = src_mgr.alloc(7)
    mig = llx.Migration(src.pool, src_mgr, dst.pool, dst_mgr, g["block_size"], 2)
    n, fin, ids = mig.stage(table, 97)
    assert (n, fin) == (6, False) and dst_mgr.num_free == nb - 6
    n2, _, _ = mig.stage(table, 100, llx.REQ_FINISHED)              # the request produced EOS during stage 0
    assert n2 == 0 and mig.state == llx.MIG_ABORTED and mig.abort_reason == llx.ABORT_FINISHED
    assert dst_mgr.num_free == nb and src_mgr.num_free == nb - 7     # reservation released, source keeps its blocks
    om.migrate_stage(h_src, table[:6], h_dst, ids)                   # A10/A25: no byte rollback
    H.assert_pool_equal(dst.host(), h_dst)
    # destination out of space: PRE-ALLOC fails, nothing is copied
    small = llx.BlockManager(nb)
    small.alloc(nb - 3)
    launches = llx.counters()["kernel_launches"]
    mig2 = llx.Migration(src.pool, src_mgr, dst.pool, small, g["block_size"], 2)
    assert mig2.stage(table, 97)[0] == 0 and mig2.abort_reason == llx.ABORT_NO_SPACE and small.num_free == 3
    assert llx.counters()["kernel_launches"] == launches
    wrong = llx.BlockManager(nb + 1)
    with pytest.raises(llx.LlxError) as e:
        llx.Migration(src.pool, src_mgr, dst.pool, wrong, g["block_size"], 2)
    assert e.value.name == "LLX_ERR_GEOMETRY_MISMATCH"


@pytest.mark.parametrize("opts", [dict(), dict(copy_kernel=1), dict(copy_kernel=2, max_ctas=5), dict(bandwidth_gbps=500)])
def test_migrate_stage_wait_returns_after_completion(env, opts):     # S4: the final stage as one blocking call
    H, llx = env
    g = RAGGED
    src, dst, h_src, h_dst = make(H, g, seed=12)
    torch.cuda.synchronize()
    st, other = torch.cuda.Stream(), torch.cuda.Stream()
    for rep in range(4):                                             # flag slots and sequence numbers are reused
        s_ids = synth.block_permutation(60 + rep, g["num_blocks"])[:9]
        d_ids = synth.block_permutation(70 + rep, g["num_blocks"])[:9]
        llx.migrate_stage(src.pool, s_ids[:6], dst.pool, d_ids[:6], stream=st, opts=opts)        # earlier stage, not synchronised
        llx.migrate_stage_wait(src.pool, s_ids[6:], dst.pool, d_ids[6:], stream=st, opts=opts)
        with torch.cuda.stream(other):                               # no synchronize of `st`: the call itself waited
            snap = dst.view.clone()
        other.synchronize()
        om.migrate_stage(h_src, s_ids, h_dst, d_ids)
        H.assert_pool_equal(snap.cpu().numpy().view(np.uint16), h_dst)
    llx.migrate_stage_wait(src.pool, [], dst.pool, [], stream=st)    # n == 0
    with pytest.raises(llx.LlxError) as e:
        llx.migrate_stage_wait(src.pool, [0, 1], dst.pool, [3, 3], stream=st)
    assert e.value.name == "LLX_ERR_DUPLICATE_DST"
    H.assert_pool_equal(dst.host(), h_dst)


@pytest.mark.parametrize("opts", KERNELS)
def test_guard_bands_around_pools_and_staging_stay_intact(env, opts):
    """compute-sanitizer is closed on this pool of machines, so out-of-bounds writes are looked for directly:
    pools and the staging buffer sit between 64 KiB guard bands that must keep their pattern."""
    H, llx = env
    g = RAGGED
    L, nb, te = g["layers"], g["num_blocks"], H.tile_elems(g)
    guard = 64 << 10
    nbytes = llx.pool_bytes_for(L, g["kv_heads"], g["head_dim"], g["block_size"], llx.F16, nb)
    n = 7
    stg_bytes = n * 2 * L * te * 2
    bufs = []
    for size in (nbytes, nbytes, stg_bytes):
        raw = torch.full((size + 2 * guard,), 0x5A, dtype=torch.uint8, device="cuda")
        bufs.append(raw)
    src = llx.pool_wrap(bufs[0].data_ptr() + guard, nbytes, L, g["kv_heads"], g["head_dim"], g["block_size"], llx.F16, nb)
    dst = llx.pool_wrap(bufs[1].data_ptr() + guard, nbytes, L, g["kv_heads"], g["head_dim"], g["block_size"], llx.F16, nb)
    bufs[0][guard:guard + nbytes] = torch.randint(0, 255, (nbytes,), dtype=torch.uint8, device="cuda")
    ids_s = np.array([0, nb - 1, 1, nb - 2, 5, 17, 3])               # first and last blocks of every slice
    ids_d = np.array([nb - 1, 0, nb - 2, 1, 9, 2, 30])
    llx.migrate_stage(src, ids_s, dst, ids_d, opts=opts)
    llx.pack(src, ids_s, bufs[2].data_ptr() + guard, stg_bytes, opts=opts)
    # unpack READS what pack wrote: it is never declared independent of the kernel before it
    llx.unpack(bufs[2].data_ptr() + guard, stg_bytes, dst, ids_d, opts={k: v for k, v in opts.items() if k != "overlap_prev"})
    llx.migrate_via_host(src, ids_s, dst, ids_d, bufs[2].data_ptr() + guard, stg_bytes, chunk_blocks=3, opts=opts)
    torch.cuda.synchronize()
    for raw, size in zip(bufs, (nbytes, nbytes, stg_bytes)):
        assert bool((raw[:guard] == 0x5A).all()) and bool((raw[guard + size:] == 0x5A).all()), "guard band overwritten"
    sv = bufs[0][guard:guard + nbytes].view(torch.int16).view(L, 2, nb, te)
    dv = bufs[1][guard:guard + nbytes].view(torch.int16).view(L, 2, nb, te)
    assert bool(torch.equal(dv[:, :, torch.from_numpy(ids_d).cuda()], sv[:, :, torch.from_numpy(ids_s).cuda()]))


@pytest.mark.parametrize("n", [255, 256, 257])
def test_ids_by_value_boundary(env, n):
    """256 pairs still travel in the kernel parameters, 257 go through the pinned id ring."""
    H, llx = env
    g = dict(TINY, num_blocks=300)
    src, dst, h_src, h_dst = make(H, g, seed=3)
    s_ids = synth.block_permutation(80, 300)[:n]
    d_ids = synth.block_permutation(81, 300)[:n]
    c0 = llx.counters()["id_uploads"]
    llx.migrate_stage(src.pool, s_ids, dst.pool, d_ids)
    assert llx.counters()["id_uploads"] - c0 == (1 if n > 256 else 0)
    om.migrate_stage(h_src, s_ids, h_dst, d_ids)
    H.assert_pool_equal(dst.host(), h_dst)


def test_default_launch_shape_with_dynamic_tail_on_a_mid_size_stage(env):
    """A stage long enough (>= 64 MiB, >= 16 chunks per ring) that the DEFAULT options take the one-CTA-per-SM ring
    with the dynamic tail; three launches back to back on one stream share the self-resetting claim counter."""
    H, llx = env
    g = dict(layers=4, kv_heads=8, head_dim=128, block_size=16, elem_bytes=2, num_blocks=700)      # 32 KiB tiles
    src = H.DevPool(g)
    src.fill_device_random(21)
    dst = H.DevPool(g, fill=SENT)
    st = torch.cuda.Stream()
    st.wait_stream(torch.cuda.current_stream())
    perm_s, perm_d = synth.block_permutation(90, 700), synth.block_permutation(91, 700)
    for a, b in ((0, 330), (330, 660), (660, 700)):                 # 330 blocks = 82.5 MiB: 2640 chunks of 32 KiB over 148 rings
        llx.migrate_stage(src.pool, perm_s[a:b], dst.pool, perm_d[a:b], stream=st)
    st.synchronize()
    h_src = src.host()
    h_dst = om.new_pool(g["layers"], 700, H.tile_elems(g), fill=SENT)
    om.migrate_stage(h_src, perm_s, h_dst, perm_d)
    H.assert_pool_equal(dst.host(), h_dst)


@pytest.mark.parametrize("heads", [5, 9, 10, 13, 17, 26])          # 20, 36, 40, 52 (a TP=4 rank of LLaMA-30B), 68, 104 KiB tiles
def test_long_stage_of_tiles_that_are_no_multiple_of_32k_is_split_into_equal_chunks(env, heads):
    """>= 64 MiB of tiles whose size is not a multiple of 32 KiB: the default launch shape cuts every tile into m equal chunks
    (13-31 KiB, the last one a few bytes shorter) with 3-6 ring stages.  A second, overlapped stage and a
    pack / unpack round trip of the same shape follow; every word against the oracle."""
    H, llx = env
    te_bytes = 16 * heads * 128 * 2
    n = (70 << 20) // (2 * 2 * te_bytes) + 1
    g = dict(layers=2, kv_heads=heads, head_dim=128, block_size=16, elem_bytes=2, num_blocks=2 * n + 20)
    src = H.DevPool(g)
    src.fill_device_random(40 + heads)
    dst = H.DevPool(g, fill=SENT)
    assert 2 * g["layers"] * src.pool.tile_bytes * n >= 64 << 20
    nb = g["num_blocks"]
    ps, pd = synth.block_permutation(5, nb), synth.block_permutation(6, nb)
    st = torch.cuda.Stream()
    st.wait_stream(torch.cuda.current_stream())
    llx.migrate_stage(src.pool, ps[:n], dst.pool, pd[:n], stream=st)
    stg = torch.empty(llx.staging_bytes(src.pool, n), dtype=torch.uint8, device="cuda")
    llx.pack(src.pool, ps[n:2 * n], stg.data_ptr(), stg.numel(), stream=st, opts=dict(overlap_prev=1))
    llx.unpack(stg.data_ptr(), stg.numel(), dst.pool, pd[n:2 * n], stream=st)
    st.synchronize()
    h_src = src.host()
    h_dst = om.new_pool(g["layers"], nb, H.tile_elems(g), fill=SENT)
    om.migrate_stage(h_src, ps[:2 * n], h_dst, pd[:2 * n])
    H.assert_pool_equal(dst.host(), h_dst)
    assert np.array_equal(stg.cpu().numpy().view(np.uint16).reshape(n, g["layers"], 2, -1), om.pack(h_src, ps[n:2 * n]))


def test_two_host_threads_on_two_streams(env):
    """llx.h, "Threads": data calls may be issued from several host threads at once on distinct streams.  Two threads migrate different requests
    between the same pools at the same time: long id lists (pinned id ring), pinned-host pack (shared bounce
    buffers) and the blocking final-stage call (flag slots)."""
    import threading
    H, llx = env
    g = dict(TINY, num_blocks=1400)
    src, dst, h_src, h_dst = make(H, g, seed=6)
    torch.cuda.synchronize()
    perm_s, perm_d = synth.block_permutation(7, 1400), synth.block_permutation(8, 1400)
    errors, packs = [], {}

    def worker(tid):
        try:
            torch.cuda.set_device(0)
            st = torch.cuda.Stream()
            lo = tid * 700
            pin = llx.PinnedStaging(llx.staging_bytes(src.pool, 40))
            for it in range(12):
                a = lo + (it % 2) * 300
                llx.migrate_stage(src.pool, perm_s[a:a + 300], dst.pool, perm_d[a:a + 300], stream=st)      # 300 > 256: id ring
                llx.pack(src.pool, perm_s[lo + 600:lo + 640], pin.dev_alias, pin.nbytes, stream=st)
                llx.migrate_stage_wait(src.pool, perm_s[lo + 640:lo + 700], dst.pool, perm_d[lo + 640:lo + 700], stream=st)
            st.synchronize()
            packs[tid] = pin.as_numpy().copy()
            pin.free()
        except Exception as e:  # noqa: BLE001
            errors.append(repr(e))

    ts = [threading.Thread(target=worker, args=(i,)) for i in range(2)]
    for t in ts:
        t.start()
    for t in ts:
        t.join()
    assert not errors, errors
    for tid in range(2):
        lo = tid * 700
        om.migrate_stage(h_src, perm_s[lo:lo + 600], h_dst, perm_d[lo:lo + 600])
        om.migrate_stage(h_src, perm_s[lo + 640:lo + 700], h_dst, perm_d[lo + 640:lo + 700])
        want = om.pack(h_src, perm_s[lo + 600:lo + 640])
        assert np.array_equal(packs[tid].reshape(want.shape), want)
    H.assert_pool_equal(dst.host(), h_dst)


@pytest.mark.parametrize("dtype_name,elem", [("U8", 1), ("BF16", 2)])
def test_other_element_types_are_bit_copied(env, dtype_name, elem):
    """Migration is dtype-agnostic: only the element size enters (tile_bytes).  One-byte elements halve the tile."""
    H, llx = env
    g = dict(layers=3, kv_heads=5, head_dim=48, block_size=16, num_blocks=50)
    dt = getattr(llx, dtype_name)
    te_bytes = g["block_size"] * g["kv_heads"] * g["head_dim"] * elem              # 3840 or 7680 bytes
    nbytes = llx.pool_bytes_for(g["layers"], g["kv_heads"], g["head_dim"], g["block_size"], dt, 50)
    assert nbytes == 50 * 2 * g["layers"] * te_bytes
    rs = torch.randint(0, 256, (nbytes,), dtype=torch.uint8, device="cuda")
    rd = torch.full((nbytes,), 0xAD, dtype=torch.uint8, device="cuda")
    src = llx.pool_wrap(rs.data_ptr(), nbytes, g["layers"], g["kv_heads"], g["head_dim"], g["block_size"], dt, 50)
    dst = llx.pool_wrap(rd.data_ptr(), nbytes, g["layers"], g["kv_heads"], g["head_dim"], g["block_size"], dt, 50)
    assert src.tile_bytes == te_bytes
    s_ids, d_ids = synth.block_permutation(1, 50)[:9], synth.block_permutation(2, 50)[:9]
    llx.migrate_stage(src, s_ids, dst, d_ids)
    torch.cuda.synchronize()
    # oracle on 16-bit words: a one-byte pool is viewed as half as many uint16 per tile (a bit copy either way)
    h_src = rs.cpu().numpy().view(np.uint16).reshape(g["layers"], 2, 50, te_bytes // 2)
    h_dst = np.full_like(h_src, 0xADAD)
    om.migrate_stage(h_src, s_ids, h_dst, d_ids)
    got = rd.cpu().numpy().view(np.uint16).reshape(h_dst.shape)
    H.assert_pool_equal(got, h_dst)
    other_dt = llx.F16 if elem == 1 else llx.U8                      # same shape, other element size
    extra = torch.empty(llx.pool_bytes_for(g["layers"], g["kv_heads"], g["head_dim"], g["block_size"], other_dt, 50),
                        dtype=torch.uint8, device="cuda")
    other = llx.pool_wrap(extra.data_ptr(), extra.numel(), g["layers"], g["kv_heads"], g["head_dim"], g["block_size"], other_dt, 50)
    with pytest.raises(llx.LlxError) as e:
        llx.migrate_stage(src, [0], other, [1])
    assert e.value.name == "LLX_ERR_GEOMETRY_MISMATCH"


@pytest.mark.parametrize("heads,blocks", [(2, 1500), (4, 800), (8, 420)])     # 4 KiB, 8 KiB, 16 KiB tiles
def test_long_stage_of_small_tiles_uses_several_ctas_per_sm(env, heads, blocks):
    """>= 64 MiB of small tiles: the default launch shape takes 4 / 2 / 1 CTAs per SM (chunk = tile) with the dynamic tail."""
    H, llx = env
    g = dict(layers=8, kv_heads=heads, head_dim=64, block_size=16, elem_bytes=2, num_blocks=blocks)
    src = H.DevPool(g)
    src.fill_device_random(31 + heads)
    dst = H.DevPool(g, fill=SENT)
    n = blocks - 100
    assert 2 * g["layers"] * src.pool.tile_bytes * n >= 64 << 20
    s_ids, d_ids = synth.block_permutation(3, blocks)[:n], synth.block_permutation(4, blocks)[:n]
    st = torch.cuda.Stream()
    st.wait_stream(torch.cuda.current_stream())
    llx.migrate_stage(src.pool, s_ids, dst.pool, d_ids, stream=st)
    llx.migrate_stage(src.pool, s_ids[:50], dst.pool, d_ids[:50], stream=st)       # a short stage right behind it
    st.synchronize()
    h_src = src.host()
    h_dst = om.new_pool(g["layers"], blocks, H.tile_elems(g), fill=SENT)
    om.migrate_stage(h_src, s_ids, h_dst, d_ids)
    H.assert_pool_equal(dst.host(), h_dst)


def test_stages_are_stream_capturable_into_a_cuda_graph(env):
    """Stages of <= 256 pairs carry their ids in the kernel parameters and touch no host state at launch, so a whole
    staged migration (copies + appends) can be captured once and replayed (first-use allocations happen in a warm-up)."""
    H, llx = env
    g = TINY
    S, te_tok = g["block_size"], g["kv_heads"] * g["head_dim"]
    src, dst, h_src, h_dst = make(H, g)
    s_tab = synth.block_permutation(1, g["num_blocks"])[:7]
    d_tab = synth.block_permutation(2, g["num_blocks"])[:7]
    values = lambda t, l, kv: synth.append_values_f16(3, t, l, kv, te_tok)
    vals = np.stack([np.stack([np.stack([values(t, l, kv) for kv in range(2)]) for l in range(g["layers"])]) for t in range(97, 100)])
    dev_vals = torch.from_numpy(vals.view(np.int16)).cuda()
    st = torch.cuda.Stream()
    st.wait_stream(torch.cuda.current_stream())

    def staged():
        llx.migrate_stage(src.pool, s_tab[:5], dst.pool, d_tab[:5], stream=st)
        llx.append_tokens(src.pool, s_tab, 97, 100, dev_vals.data_ptr(), stream=st)
        llx.migrate_stage(src.pool, s_tab[5:], dst.pool, d_tab[5:], stream=st)

    staged()                                                         # warm-up outside the capture
    st.synchronize()
    dst.view.fill_(int(np.array(SENT, np.uint16).view(np.int16)))
    torch.cuda.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=st):
        staged()
    torch.cuda.synchronize()
    assert bool((dst.view == int(np.array(SENT, np.uint16).view(np.int16))).all())      # capturing ran nothing
    graph.replay()
    graph.replay()
    torch.cuda.synchronize()
    om.staged_migration(h_src, s_tab, h_dst, d_tab, (5, 2), (3,), S, 97, values)
    H.assert_pool_equal(dst.host(), h_dst)
    H.assert_pool_equal(src.host(), h_src)
