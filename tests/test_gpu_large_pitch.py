"""Pools whose slice stride num_blocks*tile_bytes exceeds the pitch limit of a pitched transfer (cudaDevAttrMaxPitch,
2^31-1 bytes): the copy-engine routes (llx_migrate_via_host's default host leg, LLX_OPT_VIA_HOST_MODE=2 of llx_pack /
llx_unpack, LLX_ROUTE_COPY_ENGINE) issue one cudaMemcpy2DAsync per block with that stride as the pitch, which CUDA
refuses there.  A LLaMA-7B-shaped pool reaches the limit at 16384 blocks (128 GiB); a one-layer pool
with the same 128 KiB tiles reaches it with 4.3 GB, which is what this test allocates twice.

The pools are far too large to mirror on the host, so the oracle runs on COMPACT pools that hold only the blocks the
test uses (index mapping only); the device pools are compared block by block with them, the staging buffer word for
word, and the neighbours of every written block must keep the sentinel."""
import numpy as np
import pytest
import torch

import synth
from oracle import kv_migration as om

pytestmark = pytest.mark.gpu

SENT = synth.SENTINEL_U16
SENT_I16 = int(np.array(SENT, np.uint16).view(np.int16))
G = dict(layers=1, kv_heads=32, head_dim=128, block_size=16, elem_bytes=2, num_blocks=16400)   # stride 2.15e9 B > 2^31-1
N = 12


@pytest.fixture(scope="module")
def env():
    import gpu_harness as H
    import paper_2406_03243_b200 as llx
    llx.load()
    return H, llx


@pytest.fixture(scope="module")
def pools(env):
    H, llx = env
    assert G["num_blocks"] * H.tile_elems(G) * 2 > 2**31 - 1
    src, dst = H.DevPool(G, fill=SENT), H.DevPool(G, fill=SENT)
    rng = np.random.default_rng(7)
    # first, last and the blocks around the 2 GiB offset of a slice, plus random ones; distinct
    s_ids = np.unique(np.concatenate([[0, 16383, 16384, 16399], rng.integers(1, 16383, 40)]))[:N].astype(np.int32)
    s_ids = np.concatenate([s_ids[:N - 3], [16383, 16384, 16399]]).astype(np.int32)
    assert len(set(s_ids.tolist())) == N
    d_ids = np.array([16399, 5, 16384, 9000, 1, 16385, 77, 12000, 3, 16000, 8191, 8192], dtype=np.int32)
    h_src = np.empty((1, 2, N, src.te), dtype=np.uint16)                 # compact: block i of it is block s_ids[i] of the pool
    for kv in range(2):
        h_src[0, kv] = synth.slice_values_f16(50, 0, 0, kv, N, src.te)
        src.view[0, kv, torch.from_numpy(s_ids.astype(np.int64)).cuda()] = torch.from_numpy(h_src[0, kv].view(np.int16)).cuda()
    torch.cuda.synchronize()
    return src, dst, s_ids, d_ids, h_src


def check(H, src, dst, s_ids, d_ids, h_src, staging_u16=None):
    """dst blocks d_ids == oracle on compact pools; neighbours untouched; src intact; staging == the oracle's buffer."""
    compact = np.arange(N, dtype=np.int32)
    h_dst = om.new_pool(1, N, src.te, fill=SENT)
    want_buf = om.migrate_via_buffer(h_src, compact, h_dst, compact)
    torch.cuda.synchronize()
    di = torch.from_numpy(d_ids.astype(np.int64)).cuda()
    si = torch.from_numpy(s_ids.astype(np.int64)).cuda()
    for kv in range(2):
        got = dst.view[0, kv, di].cpu().numpy().view(np.uint16)
        assert np.array_equal(got, h_dst[0, kv]), f"kv={kv}"
        assert np.array_equal(src.view[0, kv, si].cpu().numpy().view(np.uint16), h_src[0, kv])
    written = set(d_ids.tolist())
    near = sorted({b for d in d_ids.tolist() for b in (d - 1, d + 1) if 0 <= b < G["num_blocks"] and b not in written})
    ni = torch.tensor(near, dtype=torch.int64, device="cuda")
    assert bool((dst.view[0, :, ni] == SENT_I16).all()), "a block next to a destination block was written"
    if staging_u16 is not None:
        assert np.array_equal(np.asarray(staging_u16).reshape(want_buf.shape), want_buf)


def reset(dst, d_ids):
    dst.view[0, :, torch.from_numpy(d_ids.astype(np.int64)).cuda()] = SENT_I16
    torch.cuda.synchronize()


@pytest.mark.parametrize("mode", [0, 2, 3], ids=["auto", "copy_engine", "bounce"])
def test_migrate_via_host_on_pools_beyond_the_pitch_limit(env, pools, mode):
    H, llx = env
    src, dst, s_ids, d_ids, h_src = pools
    reset(dst, d_ids)
    nbytes = llx.staging_bytes(src.pool, N)
    pin = llx.PinnedStaging(nbytes)
    pin.as_numpy()[:] = 0x2222
    st = torch.cuda.Stream()
    llx.migrate_via_host(src.pool, s_ids, dst.pool, d_ids, pin.dev_alias, nbytes, stream=st, opts=dict(via_host_mode=mode))
    st.synchronize()
    check(H, src, dst, s_ids, d_ids, h_src, pin.as_numpy().copy())
    pin.free()


def test_pack_unpack_copy_engine_mode_beyond_the_pitch_limit(env, pools):
    H, llx = env
    src, dst, s_ids, d_ids, h_src = pools
    reset(dst, d_ids)
    nbytes = llx.staging_bytes(src.pool, N)
    pin = llx.PinnedStaging(nbytes)
    pin.as_numpy()[:] = 0x2222
    st = torch.cuda.Stream()
    llx.pack(src.pool, s_ids, pin.dev_alias, nbytes, stream=st, opts=dict(via_host_mode=2))
    llx.unpack(pin.dev_alias, nbytes, dst.pool, d_ids, stream=st, opts=dict(via_host_mode=2))
    st.synchronize()
    check(H, src, dst, s_ids, d_ids, h_src, pin.as_numpy().copy())
    pin.free()


@pytest.mark.parametrize("route", ["copy_engine", "kernel"])
def test_pool_to_pool_beyond_the_pitch_limit(env, pools, route):
    """LLX_ROUTE_COPY_ENGINE tile by tile, and the ordinary kernel route on the same pools (64-bit slice strides)."""
    H, llx = env
    src, dst, s_ids, d_ids, h_src = pools
    reset(dst, d_ids)
    st = torch.cuda.Stream()
    llx.migrate_stage(src.pool, s_ids, dst.pool, d_ids, stream=st,
                      opts=dict(route=llx.ROUTE_COPY_ENGINE) if route == "copy_engine" else None)
    st.synchronize()
    check(H, src, dst, s_ids, d_ids, h_src)
