"""Seeded fuzz of the migration entry points against the oracle: random pool geometries (tile sizes from 16 bytes to
~100 KiB, any multiple of 16), random scattered ids, random launch policies — every kernel (1-D ring, tensor-map boxes
where a box exists, register-staged copy, paced, copy engine), chunk sizes, ring depths, CTA caps, unit orders, the
dynamic tail on tiny stages, overlapped stages.  After every case the WHOLE destination pool, the source pool and (for
pack) the staging buffer are compared with the oracle's, word for word."""
import numpy as np
import pytest
import torch

import synth
from oracle import kv_migration as om

pytestmark = pytest.mark.gpu
SENT = synth.SENTINEL_U16


@pytest.fixture(scope="module")
def env():
    import gpu_harness as H
    import paper_2406_03243_b200 as llx
    llx.load()
    return H, llx


def random_geometry(rng):
    while True:
        elem = int(rng.choice([1, 2]))
        g = dict(layers=int(rng.integers(1, 6)), kv_heads=int(rng.integers(1, 14)), head_dim=int(rng.choice([8, 16, 24, 40, 64, 96, 128])),
                 block_size=int(rng.integers(1, 33)), elem_bytes=elem, num_blocks=int(rng.integers(3, 90)))
        tile = g["block_size"] * g["kv_heads"] * g["head_dim"] * elem
        if tile % 16 == 0 and tile * 2 * g["layers"] * g["num_blocks"] <= (24 << 20):
            return g, tile


def random_policy(rng, tile):
    kind = int(rng.integers(0, 9))
    if kind == 0:
        return None
    if kind == 1:
        return dict(copy_kernel=1, chunk_bytes=int(rng.choice([16, 256, 2048, 16384])), unit_order=int(rng.integers(0, 2)))
    if kind == 2:
        chunk = int(rng.choice([16, 48, 1024, 4096, 13312, 32768, 65536]))
        return dict(copy_kernel=2, chunk_bytes=chunk, ring_stages=int(rng.integers(2, 7)), rings_per_cta=int(rng.integers(1, 3)),
                    unit_order=int(rng.integers(0, 2)), overlap_prev=int(rng.integers(0, 2)))
    if kind == 3:
        return dict(copy_kernel=2, chunk_bytes=int(rng.choice([64, 512, 8192])), max_ctas=int(rng.integers(1, 9)),
                    dynamic_tail_pct=int(rng.choice([0, 20, 60, 100])), dynamic_tail_batch=int(rng.integers(1, 6)), ring_stages=3)
    if kind == 4:
        return dict(bandwidth_gbps=int(rng.choice([1, 30, 700, 5000])))
    if kind == 5:
        return dict(route=int(rng.choice([1, 2])))
    if kind == 6:
        return dict(copy_kernel=3, ring_stages=int(rng.integers(2, 5)), overlap_prev=int(rng.integers(0, 2)))       # refused where no box exists
    if kind == 7:
        return dict(ids_by_value_max=0, pdl=int(rng.integers(0, 2)), l2_hint=int(rng.integers(0, 4)))
    return dict(overlap_prev=1)


@pytest.mark.parametrize("seed", range(6))
def test_random_geometries_ids_and_policies_against_the_oracle(env, seed):
    H, llx = env
    rng = np.random.default_rng(1000 + seed)
    for case in range(12):
        g, tile = random_geometry(rng)
        dtype = llx.U8 if g["elem_bytes"] == 1 else llx.F16
        L, nb = g["layers"], g["num_blocks"]
        words = tile // 2
        h_src = rng.integers(0, 65536, size=(L, 2, nb, words), dtype=np.uint16)
        h_dst = om.new_pool(L, nb, words, fill=SENT)
        nbytes = llx.pool_bytes_for(L, g["kv_heads"], g["head_dim"], g["block_size"], dtype, nb)
        assert nbytes == h_src.nbytes
        # both pools sit between 8 KiB guard bands (compute-sanitizer is closed on this pool of machines): a copy that
        # strayed outside a pool — a box, a chunk, a remainder — would hit them
        GUARD = 8192
        raw_s = torch.full((nbytes + 2 * GUARD,), 0x5A, dtype=torch.uint8, device="cuda")
        raw_d = torch.full((nbytes + 2 * GUARD,), 0x5A, dtype=torch.uint8, device="cuda")
        d_src = raw_s[GUARD:GUARD + nbytes].view(torch.int16)
        d_dst = raw_d[GUARD:GUARD + nbytes].view(torch.int16)
        d_src.copy_(torch.from_numpy(h_src.view(np.int16).reshape(-1)))
        d_dst.copy_(torch.from_numpy(h_dst.view(np.int16).reshape(-1)))
        src = llx.pool_wrap(d_src.data_ptr(), nbytes, L, g["kv_heads"], g["head_dim"], g["block_size"], dtype, nb, keepalive=raw_s)
        dst = llx.pool_wrap(d_dst.data_ptr(), nbytes, L, g["kv_heads"], g["head_dim"], g["block_size"], dtype, nb, keepalive=raw_d)
        stream = torch.cuda.Stream()
        stream.wait_stream(torch.cuda.current_stream())
        free_dst = list(rng.permutation(nb))
        for step in range(int(rng.integers(1, 5))):
            n = int(rng.integers(0, min(len(free_dst), nb) + 1))
            s_ids = rng.integers(0, nb, size=n).astype(np.int32) if rng.random() < 0.3 else rng.permutation(nb)[:n].astype(np.int32)
            d_ids = np.array([free_dst.pop() for _ in range(n)], dtype=np.int32)       # disjoint across the steps: overlap_prev is legal
            opts = random_policy(rng, tile)
            what = int(rng.integers(0, 3))
            label = (seed, case, step, g, n, opts, what)
            try:
                if what == 0:
                    llx.migrate_stage(src, s_ids, dst, d_ids, stream=stream, opts=opts)
                elif what == 1:
                    cuts = np.sort(rng.integers(0, n + 1, size=int(rng.integers(0, 4))))
                    off = np.concatenate([[0], cuts, [n]]).astype(np.int32)
                    llx.migrate_batch(src, dst, off, s_ids, d_ids, stream=stream, opts=opts)
                else:
                    o2 = None if opts is None else {k: v for k, v in opts.items() if k not in ("overlap_prev", "route")}
                    stg = torch.zeros(max(llx.staging_bytes(src, n), 16), dtype=torch.uint8, device="cuda")
                    stream.wait_stream(torch.cuda.current_stream())
                    llx.pack(src, s_ids, stg.data_ptr(), stg.numel(), stream=stream, opts=o2)
                    llx.unpack(stg.data_ptr(), stg.numel(), dst, d_ids, stream=stream, opts=o2)
                    stream.synchronize()
                    if n:
                        got = stg.cpu().numpy()[:n * 2 * L * tile].view(np.uint16).reshape(n, L, 2, words)
                        assert np.array_equal(got, om.pack(h_src, s_ids)), label
            except llx.LlxError as e:
                # the tensor-map kernel where no box exists (or a side is a staging buffer), a ring that does not fit: refused
                # BEFORE anything is launched — the pools must be exactly as they were
                assert e.name == "LLX_ERR_INVALID_ARG" and opts is not None and (opts.get("copy_kernel") in (2, 3)), (label, str(e))
                free_dst.extend(int(x) for x in d_ids)
                stream.synchronize()
                assert np.array_equal(d_dst.cpu().numpy().view(np.uint16), h_dst.reshape(-1)), label
                continue
            om.migrate_stage(h_src, s_ids, h_dst, d_ids)
            stream.synchronize()
            assert np.array_equal(d_dst.cpu().numpy().view(np.uint16), h_dst.reshape(-1)), label
            assert np.array_equal(d_src.cpu().numpy().view(np.uint16), h_src.reshape(-1)), label
            for raw in (raw_s, raw_d):
                assert bool((raw[:GUARD] == 0x5A).all()) and bool((raw[GUARD + nbytes:] == 0x5A).all()), ("guard band overwritten", label)
