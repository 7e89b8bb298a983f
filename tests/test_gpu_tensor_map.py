"""The tensor-map copy kernel (llx_copy_tma: cp.async.bulk.tensor.4d, one box = one block in several (layer, K|V) slices)
against the oracle.  It serves pool-to-pool stages of small tiles (<= 16 KiB: TP-sharded or GQA caches, Tiny), selected with
copy_kernel = 3 (the default stays the 1-D ring, which ties it once its depth is right: DESIGN.md section 5.1b).  Same definition as every other route (PAPER.md:134,
:237): dst[l][kv][dst_ids[i]] = src[l][kv][src_ids[i]], whole tiles, everything else untouched."""
import numpy as np
import pytest
import torch

import synth
from oracle import kv_migration as om

pytestmark = pytest.mark.gpu
SENT = synth.SENTINEL_U16
SENT_I16 = int(np.array(SENT, np.uint16).view(np.int16))

TINY = dict(synth.CONFIGS["tiny"], num_blocks=400)                                                  # 8 KiB tiles, 4 slices: box of 4
G_ROWS5 = dict(layers=3, kv_heads=5, head_dim=64, block_size=16, elem_bytes=2, num_blocks=350)      # 10 KiB = 5 rows of 2 KiB, box of 3
G_ONE_ROW = dict(layers=4, kv_heads=3, head_dim=40, block_size=8, elem_bytes=2, num_blocks=500)     # 1920 B = one row, box of 8
G_ROWS6 = dict(layers=5, kv_heads=3, head_dim=112, block_size=16, elem_bytes=2, num_blocks=330)     # 10.5 KiB = 6 rows of 1792 B, box of 2
G_16K = dict(layers=6, kv_heads=4, head_dim=128, block_size=16, elem_bytes=2, num_blocks=340)       # 16 KiB tiles, box of 2
GEOMS = [TINY, G_ROWS5, G_ONE_ROW, G_ROWS6, G_16K]
OPTS = [dict(copy_kernel=3), dict(copy_kernel=3, unit_order=0), dict(copy_kernel=3, ids_by_value_max=0),
        dict(copy_kernel=3, dynamic_tail_pct=50, max_ctas=3), dict(copy_kernel=3, overlap_prev=1, ring_stages=2),
        dict(copy_kernel=3, rings_per_cta=2, ring_stages=3, l2_hint=3, pdl=0)]


@pytest.fixture(scope="module")
def env():
    import gpu_harness as H
    import paper_2406_03243_b200 as llx
    llx.load()
    return H, llx


def pools(H, g, seed):
    src = H.DevPool(g)
    src.fill_from_synth(seed, 0)
    dst = H.DevPool(g, fill=SENT)
    return src, dst, H.host_pool_from_synth(g, seed, 0), om.new_pool(g["layers"], g["num_blocks"], H.tile_elems(g), fill=SENT)


@pytest.mark.parametrize("g", GEOMS)
@pytest.mark.parametrize("opts", OPTS)
def test_tensor_map_kernel_matches_the_oracle(env, g, opts):
    """Stages of 1, 13 and 300 pairs (the last through the pinned id ring), the first and the last block of the pool among
    them, one after the other into disjoint destination blocks; every word of both pools compared after each."""
    H, llx = env
    src, dst, h_src, h_dst = pools(H, g, seed=9)
    nb = g["num_blocks"]
    ps = np.concatenate([[0, nb - 1], np.setdiff1d(synth.block_permutation(31, nb), [0, nb - 1], assume_unique=True)])
    pd = np.concatenate([[nb - 1, 0], np.setdiff1d(synth.block_permutation(32, nb), [0, nb - 1], assume_unique=True)])
    m = 0
    for n in (1, 13, 300):
        llx.migrate_stage(src.pool, ps[m:m + n], dst.pool, pd[m:m + n], opts=opts)
        om.migrate_stage(h_src, ps[m:m + n], h_dst, pd[m:m + n])
        m += n
        H.assert_pool_equal(dst.host(), h_dst)
        H.assert_pool_equal(src.host(), h_src)


def test_tensor_map_kernel_batch_capture_and_guard_bands(env):
    """One batch launch of four requests; the same stage captured into a CUDA graph and replayed on another stream; pools
    between 64 KiB guard bands that must keep their pattern (a box that strayed outside the pool would hit them)."""
    H, llx = env
    g = G_ROWS5
    L, nb, te = g["layers"], g["num_blocks"], H.tile_elems(g)
    nbytes = llx.pool_bytes_for(L, g["kv_heads"], g["head_dim"], g["block_size"], llx.F16, nb)
    guard = 64 << 10
    raws = [torch.full((nbytes + 2 * guard,), 0x5A, dtype=torch.uint8, device="cuda") for _ in range(2)]
    wrap = lambda r: llx.pool_wrap(r.data_ptr() + guard, nbytes, L, g["kv_heads"], g["head_dim"], g["block_size"], llx.F16, nb, keepalive=r)
    src, dst = wrap(raws[0]), wrap(raws[1])
    sv = raws[0][guard:guard + nbytes].view(torch.int16).view(L, 2, nb, te)
    dv = raws[1][guard:guard + nbytes].view(torch.int16).view(L, 2, nb, te)
    h_src = H.host_pool_from_synth(g, 4, 0)
    sv.copy_(torch.from_numpy(h_src.view(np.int16)))
    dv.fill_(SENT_I16)
    h_dst = om.new_pool(L, nb, te, fill=SENT)
    ps, pd = synth.block_permutation(41, nb), synth.block_permutation(42, nb)
    off = [0, 10, 10, 41, 72]
    llx.migrate_batch(src, dst, off, ps[:72], pd[:72], opts=dict(copy_kernel=3))
    om.migrate_batch(h_src, h_dst, off, ps[:72], pd[:72])
    torch.cuda.synchronize()
    H.assert_pool_equal(dv.cpu().numpy().view(np.uint16), h_dst)
    cap, other = torch.cuda.Stream(), torch.cuda.Stream()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.stream(cap):
        graph.capture_begin()
        llx.migrate_stage(src, ps[72:200], dst, pd[72:200], stream=cap, opts=dict(copy_kernel=3))
        graph.capture_end()
    with torch.cuda.stream(other):
        graph.replay()
    other.synchronize()
    om.migrate_stage(h_src, ps[72:200], h_dst, pd[72:200])
    H.assert_pool_equal(dv.cpu().numpy().view(np.uint16), h_dst)
    H.assert_pool_equal(sv.cpu().numpy().view(np.uint16), h_src)
    for raw in raws:
        assert bool((raw[:guard] == 0x5A).all()) and bool((raw[guard + nbytes:] == 0x5A).all()), "guard band overwritten"


@pytest.mark.parametrize("opts", [None, dict(copy_kernel=3)])
def test_long_stage_of_16k_tiles_by_the_default_ring_and_by_the_tensor_map_kernel(env, opts):
    """>= 64 MiB of 16 KiB tiles with the default options (1-D ring, one CTA per SM, 5 stages of 16 KiB) and with the
    tensor-map kernel (boxes of two tiles, 3 stages); an overlapped short stage right behind it.  Pools of different
    sizes (A21)."""
    H, llx = env
    g = dict(layers=16, kv_heads=4, head_dim=128, block_size=16, elem_bytes=2, num_blocks=900)
    src = H.DevPool(g)
    src.fill_device_random(77)
    dst = H.DevPool(g, num_blocks=1000, fill=SENT)
    n = 800
    assert 2 * g["layers"] * src.pool.tile_bytes * n >= 64 << 20
    s_ids, d_ids = synth.block_permutation(3, 900)[:n + 20], synth.block_permutation(4, 1000)[:n + 20]
    st = torch.cuda.Stream()
    st.wait_stream(torch.cuda.current_stream())
    llx.migrate_stage(src.pool, s_ids[:n], dst.pool, d_ids[:n], stream=st, opts=opts)
    llx.migrate_stage(src.pool, s_ids[n:], dst.pool, d_ids[n:], stream=st, opts=dict(overlap_prev=1))
    st.synchronize()
    h_src = src.host()
    h_dst = om.new_pool(g["layers"], 1000, H.tile_elems(g), fill=SENT)
    om.migrate_stage(h_src, s_ids, h_dst, d_ids)
    H.assert_pool_equal(dst.host(), h_dst)


def test_tensor_map_kernel_is_refused_where_it_does_not_apply(env):
    H, llx = env
    big = dict(layers=2, kv_heads=9, head_dim=120, block_size=16, elem_bytes=2, num_blocks=40)      # 33.75 KiB tiles
    odd = dict(layers=2, kv_heads=7, head_dim=24, block_size=3, elem_bytes=2, num_blocks=64)        # 1008 B: no box of 128-byte multiples
    for g in (big, odd):
        src, dst = H.DevPool(g), H.DevPool(g, fill=SENT)
        with pytest.raises(llx.LlxError) as e:
            llx.migrate_stage(src.pool, [1, 2], dst.pool, [3, 4], opts=dict(copy_kernel=3))
        assert e.value.name == "LLX_ERR_INVALID_ARG"
        llx.migrate_stage(src.pool, [1, 2], dst.pool, [3, 4])                                       # the default route serves it
        torch.cuda.synchronize()
        assert bool((dst.view[:, :, [0, 1, 2, 5]] == SENT_I16).all())
    src, dst = H.DevPool(TINY), H.DevPool(TINY, fill=SENT)
    stg = torch.zeros(llx.staging_bytes(src.pool, 2), dtype=torch.uint8, device="cuda")
    with pytest.raises(llx.LlxError):                                                                # one side is a staging buffer
        llx.pack(src.pool, [1, 2], stg.data_ptr(), stg.numel(), opts=dict(copy_kernel=3))
    with pytest.raises(llx.LlxError):
        llx.migrate_stage(src.pool, [1, 2], dst.pool, [3, 4], opts=dict(copy_kernel=4))
