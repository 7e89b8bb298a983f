"""SURVEY NEXT-2 as far as ONE GPU allows (PAPER.md:235 §5, :254 §6.1, :285 §6.2).

(a) The cross-GPU ROUTE (kernel choice, launch shape and addressing that `llx_migrate_stage` takes when the destination
    pool lives on another GPU) executed on one device through llx_launch_opts.route = LLX_ROUTE_PEER, bit-exact against
    the oracle over the option matrix.  What this cannot show is the NVLink transfer itself and the peer-access set-up:
    the real two-GPU test below stays and skips on a one-GPU box.
(b) The tensor-parallel sharding claim of SURVEY §8(e): LLaMA-30B on 4 GPUs keeps heads [13r, 13r+13) of
    every tile on rank r, rank r of the source instance migrates to rank r of the destination with no cross-rank
    exchange, and the four rank-local results together ARE the unsharded 52-head migration the oracle
    computes."""
import numpy as np
import pytest
import torch

import synth
from oracle import kv_migration as om

pytestmark = pytest.mark.gpu

SENT = synth.SENTINEL_U16
RAGGED = dict(layers=3, kv_heads=9, head_dim=120, block_size=16, elem_bytes=2, num_blocks=40)      # 34,560-byte tiles
SMALLTILE = dict(layers=2, kv_heads=7, head_dim=24, block_size=3, elem_bytes=2, num_blocks=64)     # 1,008-byte tiles

PEER_OPTS = [dict(), dict(chunk_bytes=2048), dict(ids_by_value_max=0), dict(max_ctas=1), dict(unit_order=0), dict(pdl=0),
             dict(bandwidth_gbps=40), dict(max_ctas=7, chunk_bytes=512)]


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


@pytest.mark.parametrize("g", [RAGGED, SMALLTILE])
@pytest.mark.parametrize("opts", PEER_OPTS)
def test_peer_route_on_one_device_is_bit_exact(env, g, opts):
    H, llx = env
    src, dst, h_src, h_dst = make(H, g, seed=21)
    s_ids = synth.block_permutation(31, g["num_blocks"])[:17]
    d_ids = synth.block_permutation(32, g["num_blocks"])[:17]
    o = dict(opts, route=llx.ROUTE_PEER)
    st = torch.cuda.Stream()
    st.wait_stream(torch.cuda.current_stream())
    llx.migrate_stage(src.pool, s_ids[:11], dst.pool, d_ids[:11], stream=st, opts=o)
    llx.migrate_batch(src.pool, dst.pool, [0, 2, 2, 6], s_ids[11:], d_ids[11:], stream=st, opts=o)
    st.synchronize()
    om.migrate_stage(h_src, s_ids, h_dst, d_ids)
    H.assert_pool_equal(dst.host(), h_dst)
    H.assert_pool_equal(src.host(), h_src)


@pytest.mark.parametrize("g", [RAGGED, SMALLTILE])
def test_copy_engine_route_is_bit_exact(env, g):
    """LLX_ROUTE_COPY_ENGINE: no kernel at all, one pitched transfer per block; stage, batch, the blocking final stage
    and a stream capture (memcpy nodes) — all bit-exact, and not one llx kernel launched."""
    H, llx = env
    src, dst, h_src, h_dst = make(H, g, seed=24)
    s_ids = synth.block_permutation(35, g["num_blocks"])[:19]
    d_ids = synth.block_permutation(36, g["num_blocks"])[:19]
    o = dict(route=llx.ROUTE_COPY_ENGINE)
    st = torch.cuda.Stream()
    st.wait_stream(torch.cuda.current_stream())
    c0 = llx.counters()
    llx.migrate_stage(src.pool, s_ids[:9], dst.pool, d_ids[:9], stream=st, opts=o)
    llx.migrate_batch(src.pool, dst.pool, [0, 3, 3, 6], s_ids[9:15], d_ids[9:15], stream=st, opts=o)
    llx.migrate_stage_wait(src.pool, s_ids[15:17], dst.pool, d_ids[15:17], stream=st, opts=o)
    c1 = llx.counters()
    assert c1["kernel_launches"] == c0["kernel_launches"] and c1["bytes_moved"] - c0["bytes_moved"] == 17 * src.pool.block_bytes
    gr = torch.cuda.CUDAGraph()
    with torch.cuda.graph(gr, stream=st):
        llx.migrate_stage(src.pool, s_ids[17:], dst.pool, d_ids[17:], stream=st, opts=o)
    gr.replay()
    torch.cuda.synchronize()
    om.migrate_stage(h_src, s_ids, h_dst, d_ids)
    H.assert_pool_equal(dst.host(), h_dst)
    H.assert_pool_equal(src.host(), h_src)


def test_copy_engine_route_refuses_a_budget_and_counts_bytes(env):
    """llx.h, LLX_ROUTE_COPY_ENGINE: the copy engines cannot be paced or capped, so a call that asks for both the route and
    a bandwidth budget / CTA cap (per call, or inherited from the process defaults) is refused before anything is enqueued
    instead of running unthrottled.  The copy-engine host legs (llx_pack / llx_unpack mode 2) count their bytes like the
    pool-to-pool route; an explicit copy_kernel makes llx_migrate_via_host take its kernel route (as llx_pack does)."""
    H, llx = env
    g = RAGGED
    src, dst, h_src, h_dst = make(H, g, seed=25)
    s_ids = synth.block_permutation(37, g["num_blocks"])[:6]
    d_ids = synth.block_permutation(38, g["num_blocks"])[:6]
    for bad in (dict(bandwidth_gbps=25), dict(max_ctas=4)):
        with pytest.raises(llx.LlxError) as e:
            llx.migrate_stage(src.pool, s_ids, dst.pool, d_ids, opts=dict(route=llx.ROUTE_COPY_ENGINE, **bad))
        assert e.value.name == "LLX_ERR_INVALID_ARG" and "LLX_ROUTE_COPY_ENGINE" in str(e.value)
        with pytest.raises(llx.LlxError):
            llx.migrate_batch(src.pool, dst.pool, [0, 6], s_ids, d_ids, opts=dict(route=llx.ROUTE_COPY_ENGINE, **bad))
    with llx.options(bandwidth_gbps=25):                                  # inherited from the process default
        with pytest.raises(llx.LlxError):
            llx.migrate_stage(src.pool, s_ids, dst.pool, d_ids, opts=dict(route=llx.ROUTE_COPY_ENGINE))
    torch.cuda.synchronize()
    H.assert_pool_equal(dst.host(), h_dst)                                # refused: not a byte moved
    nbytes = llx.staging_bytes(src.pool, 6)
    pin = llx.PinnedStaging(nbytes)
    c0 = llx.counters()
    llx.pack(src.pool, s_ids, pin.dev_alias, nbytes, opts=dict(via_host_mode=2))
    llx.unpack(pin.dev_alias, nbytes, dst.pool, d_ids, opts=dict(via_host_mode=2))
    c1 = llx.counters()
    assert c1["kernel_launches"] == c0["kernel_launches"] and c1["bytes_moved"] - c0["bytes_moved"] == 2 * nbytes
    torch.cuda.synchronize()
    om.migrate_stage(h_src, s_ids, h_dst, d_ids)
    H.assert_pool_equal(dst.host(), h_dst)
    # explicit copy_kernel: llx_migrate_via_host runs its kernels (pack into / unpack from the bounce buffers)
    s2 = synth.block_permutation(37, g["num_blocks"])[6:12]
    d2 = synth.block_permutation(38, g["num_blocks"])[6:12]
    c0 = llx.counters()
    llx.migrate_via_host(src.pool, s2, dst.pool, d2, pin.dev_alias, nbytes)                      # auto: copy engines only
    c1 = llx.counters()
    assert c1["kernel_launches"] == c0["kernel_launches"]
    llx.migrate_via_host(src.pool, s2, dst.pool, d2, pin.dev_alias, nbytes, opts=dict(copy_kernel=1))
    c2 = llx.counters()
    assert c2["copy_launches"] - c1["copy_launches"] >= 2
    torch.cuda.synchronize()
    om.migrate_stage(h_src, s2, h_dst, d2)
    H.assert_pool_equal(dst.host(), h_dst)
    pin.free()


def test_peer_route_long_id_list_and_blocking_final_stage(env):
    """> 256 pairs through the (per-device) id ring on the peer route, then the blocking final-stage call, which falls
    back to the stream synchronize because the peer route's kernel carries no completion flag."""
    H, llx = env
    g = dict(synth.CONFIGS["tiny"], num_blocks=700)
    src, dst, h_src, h_dst = make(H, g, seed=22)
    s_ids, d_ids = synth.block_permutation(33, 700), synth.block_permutation(34, 700)
    o = dict(route=llx.ROUTE_PEER)
    up0 = llx.counters()["id_uploads"]
    llx.migrate_stage(src.pool, s_ids[:690], dst.pool, d_ids[:690], opts=o)
    assert llx.counters()["id_uploads"] == up0 + 1
    llx.migrate_stage_wait(src.pool, s_ids[690:], dst.pool, d_ids[690:], opts=o)
    other = torch.cuda.Stream()
    with torch.cuda.stream(other):                                     # no synchronize: the call itself waited
        snap = dst.view.clone()
    other.synchronize()
    om.migrate_stage(h_src, s_ids, h_dst, d_ids)
    H.assert_pool_equal(snap.cpu().numpy().view(np.uint16), h_dst)


def test_peer_route_option_is_validated_and_counted(env):
    """The route option is validated, counted like any other copy launch, and changes no byte of the result."""
    H, llx = env
    src, dst, h_src, h_dst = make(H, RAGGED, seed=23)
    c0 = llx.counters()
    llx.migrate_stage(src.pool, [0, 1, 2], dst.pool, [5, 6, 7], opts=dict(route=llx.ROUTE_PEER))
    c1 = llx.counters()
    assert c1["copy_launches"] == c0["copy_launches"] + 1 and c1["bytes_moved"] - c0["bytes_moved"] == 3 * src.pool.block_bytes
    with pytest.raises(llx.LlxError) as e:
        llx.migrate_stage(src.pool, [0], dst.pool, [1], opts=dict(route=5))
    assert e.value.name == "LLX_ERR_INVALID_ARG"
    om.migrate_stage(h_src, [0, 1, 2], h_dst, [5, 6, 7])
    H.assert_pool_equal(dst.host(), h_dst)


# ---- (b) tensor-parallel sharding: 52 KV heads = 4 ranks x 13 -----------------------------------------------------
TP, H_FULL, D, S, L30 = 4, 52, 128, 16, 60


def test_llama30b_tp4_rank_local_migration_equals_unsharded_oracle(env):
    """Four rank pairs (kv_heads = 13, 52 KiB tiles, all 60 layers) on four streams at once.  The oracle migrates the
    UNSHARDED 52-head pools; rank r's destination pool must equal the oracle's result restricted to heads [13r, 13r+13),
    sentinel blocks included.  Block tables are shared by the ranks (one logical table per request)."""
    H, llx = env
    nb_src, nb_dst, n = 56, 48, 23
    Hr = H_FULL // TP
    te_full = S * H_FULL * D
    g_rank = dict(layers=L30, kv_heads=Hr, head_dim=D, block_size=S, elem_bytes=2)
    # the unsharded source pool of the oracle (seeded, one slice at a time) and its destination
    h_src = np.empty((L30, 2, nb_src, te_full), dtype=np.uint16)
    for l in range(L30):
        for kv in range(2):
            h_src[l, kv] = synth.slice_values_f16(5, 0, l, kv, nb_src, te_full)
    h_dst = om.new_pool(L30, nb_dst, te_full, fill=SENT)

    def shard(full, nb, r):        # heads [13r, 13r+13) of every slot of every tile: what rank r holds
        return np.ascontiguousarray(full.reshape(L30, 2, nb, S, H_FULL, D)[:, :, :, :, r * Hr:(r + 1) * Hr, :]).reshape(L30, 2, nb, S * Hr * D)

    src_r = [H.DevPool(g_rank, num_blocks=nb_src) for _ in range(TP)]
    dst_r = [H.DevPool(g_rank, num_blocks=nb_dst, fill=SENT) for _ in range(TP)]
    assert src_r[0].pool.tile_bytes == 52 * 1024
    for r in range(TP):
        src_r[r].view.copy_(torch.from_numpy(shard(h_src, nb_src, r).view(np.int16)))
    s_tab = synth.block_permutation(41, nb_src)[:n]
    d_tab = synth.block_permutation(42, nb_dst)[:n]
    streams = [torch.cuda.Stream() for _ in range(TP)]
    torch.cuda.synchronize()
    # rank r -> rank r, two stages each (21 blocks, then the final 2), all ranks in flight at once, no exchange between them
    for r in range(TP):
        llx.migrate_stage(src_r[r].pool, s_tab[:n - 2], dst_r[r].pool, d_tab[:n - 2], stream=streams[r])
    for r in range(TP):
        llx.migrate_stage(src_r[r].pool, s_tab[n - 2:], dst_r[r].pool, d_tab[n - 2:], stream=streams[r])
    torch.cuda.synchronize()
    om.staged_migration(h_src, s_tab, h_dst, d_tab, (n - 2, 2), (), S, n * S, None)
    for r in range(TP):
        H.assert_pool_equal(dst_r[r].host(), shard(h_dst, nb_dst, r))
        H.assert_pool_equal(src_r[r].host(), shard(h_src, nb_src, r))
    # and the four shards put back together are the oracle's unsharded destination
    whole = np.empty((L30, 2, nb_dst, S, H_FULL, D), dtype=np.uint16)
    for r in range(TP):
        whole[:, :, :, :, r * Hr:(r + 1) * Hr, :] = dst_r[r].host().reshape(L30, 2, nb_dst, S, Hr, D)
    assert np.array_equal(whole.reshape(h_dst.shape), h_dst)


def test_destination_pool_on_a_peer_gpu(env):                       # the real thing; needs two GPUs (skipped on a 1-GPU box)
    H, llx = env
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs with peer access: NVLink transfer unmeasured on hardware in this run")
    g = RAGGED
    src, _, h_src, h_dst = make(H, g, seed=14)
    with torch.cuda.device(1):
        dst = H.DevPool(g, fill=SENT)
    s_ids = synth.block_permutation(1, g["num_blocks"])[:13]
    d_ids = synth.block_permutation(2, g["num_blocks"])[:13]
    llx.migrate_stage(src.pool, s_ids, dst.pool, d_ids)              # kernel on device 0 stores into device 1's pool
    torch.cuda.synchronize(0)
    om.migrate_stage(h_src, s_ids, h_dst, d_ids)
    with torch.cuda.device(1):
        H.assert_pool_equal(dst.host(), h_dst)
    # both directions with > 256 pairs: the id ring is per device
    g2 = dict(synth.CONFIGS["tiny"], num_blocks=400)
    a = H.DevPool(g2)
    a.fill_from_synth(3, 0)
    with torch.cuda.device(1):
        b = H.DevPool(g2)
        b.fill_from_synth(3, 1)
        b2 = H.DevPool(g2, fill=SENT)
    a2 = H.DevPool(g2, fill=SENT)
    ids_s, ids_d = synth.block_permutation(5, 400)[:300], synth.block_permutation(6, 400)[:300]
    llx.migrate_stage(a.pool, ids_s, b2.pool, ids_d)                 # 0 -> 1
    with torch.cuda.device(1):
        llx.migrate_stage(b.pool, ids_s, a2.pool, ids_d)             # 1 -> 0
    torch.cuda.synchronize(0)
    torch.cuda.synchronize(1)
    ha, hb = H.host_pool_from_synth(g2, 3, 0), H.host_pool_from_synth(g2, 3, 1)
    want_b2, want_a2 = om.new_pool(2, 400, H.tile_elems(g2), SENT), om.new_pool(2, 400, H.tile_elems(g2), SENT)
    om.migrate_stage(ha, ids_s, want_b2, ids_d)
    om.migrate_stage(hb, ids_s, want_a2, ids_d)
    H.assert_pool_equal(a2.host(), want_a2)
    with torch.cuda.device(1):
        H.assert_pool_equal(b2.host(), want_b2)
