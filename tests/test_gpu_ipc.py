"""SURVEY NEXT-2, the part one GPU can run for real: the destination instance is ANOTHER PROCESS.
The child process plays the destination instance: it owns its pool (llx_pool_create), exports a handle
(llx_pool_ipc_export) and later checks its own pool against the oracle.  The parent plays the source instance: it opens
the handle (llx_pool_ipc_open) and migrates a request into the other process's KV cache in two stages.  With two GPUs
the same code stores across NVLink (the mapping enables peer access); on one GPU the two instances share the device."""
import multiprocessing as mp
import os
import sys

import numpy as np
import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
G = dict(layers=3, kv_heads=9, head_dim=120, block_size=16, elem_bytes=2, num_blocks=40)     # ragged 34,560-byte tiles
N = 17


def _ids():
    import synth
    return synth.block_permutation(51, G["num_blocks"])[:N], synth.block_permutation(52, G["num_blocks"])[:N]


def _fnv1a(b: bytes) -> int:
    """The handle's last word as llx.h describes it (32-bit FNV-1a of the 92 bytes in front of it)."""
    x = 2166136261
    for c in b:
        x = ((x ^ c) * 16777619) & 0xFFFFFFFF
    return x


def destination_instance(conn, device):
    """Runs in the child: owns the destination pool; never calls a copy itself."""
    try:
        sys.path.insert(0, ROOT)
        import torch
        import paper_2406_03243_b200 as llx
        import synth
        from oracle import kv_migration as om
        torch.cuda.set_device(device)
        llx.load()
        te = G["block_size"] * G["kv_heads"] * G["head_dim"]
        dst = llx.pool_create(G["layers"], G["kv_heads"], G["head_dim"], G["block_size"], llx.F16, G["num_blocks"])
        dst.fill_u16(synth.SENTINEL_U16)
        llx.synchronize()
        conn.send(llx.pool_ipc_export(dst))
        assert conn.recv() == "migrated"                      # the source's commit message
        got = np.empty((G["layers"], 2, G["num_blocks"], te), dtype=np.uint16)
        for l in range(G["layers"]):
            for kv in range(2):
                got[l, kv] = dst.download(l, kv, 0, G["num_blocks"])
        llx.synchronize()
        h_src = np.empty_like(got)
        for l in range(G["layers"]):
            for kv in range(2):
                h_src[l, kv] = synth.slice_values_f16(31, 0, l, kv, G["num_blocks"], te)
        want = om.new_pool(G["layers"], G["num_blocks"], te, fill=synth.SENTINEL_U16)
        s_ids, d_ids = _ids()
        om.migrate_stage(h_src, s_ids, want, d_ids)
        conn.send("equal" if np.array_equal(got, want) else f"{int((got != want).sum())} words differ from the oracle")
        dst.destroy()
    except Exception as e:  # noqa: BLE001
        conn.send("error: " + repr(e))


def test_migration_into_another_process_pool():
    import torch
    import gpu_harness as H
    import paper_2406_03243_b200 as llx
    import synth
    llx.load()
    dst_device = 1 if torch.cuda.device_count() > 1 else 0     # a second GPU if there is one: the NVLink route
    ctx = mp.get_context("spawn")
    here, there = ctx.Pipe()
    child = ctx.Process(target=destination_instance, args=(there, dst_device))
    child.start()
    try:
        handle = here.recv()
        assert isinstance(handle, bytes) and len(handle) == llx.IPC_HANDLE_BYTES, handle
        src = H.DevPool(G)
        src.fill_from_synth(31, 0)
        # a damaged handle is refused by its checksum; a handle that names a larger pool than the exporter allocated,
        # with a checksum made to match (a stale or forged handle), is refused against the size of the real mapping
        flipped = bytearray(handle)
        flipped[64 + 4 + 20] ^= 0x40                            # num_blocks: 40 -> 104
        with pytest.raises(llx.LlxError) as e:
            llx.pool_ipc_open(bytes(flipped))
        assert e.value.name == "LLX_ERR_INVALID_ARG" and "checksum" in str(e.value)
        flipped[92:96] = _fnv1a(bytes(flipped[:92])).to_bytes(4, "little")
        with pytest.raises(llx.LlxError) as e:
            llx.pool_ipc_open(bytes(flipped))
        assert e.value.name == "LLX_ERR_INVALID_ARG" and "allocation has" in str(e.value), str(e.value)
        assert _fnv1a(handle[:92]).to_bytes(4, "little") == handle[92:96]
        dst = llx.pool_ipc_open(handle)
        assert dst.num_blocks == G["num_blocks"] and dst.tile_bytes == src.pool.tile_bytes
        s_ids, d_ids = _ids()
        st = torch.cuda.Stream()
        st.wait_stream(torch.cuda.current_stream())
        llx.migrate_stage(src.pool, s_ids[:N - 2], dst, d_ids[:N - 2], stream=st)
        llx.migrate_stage_wait(src.pool, s_ids[N - 2:], dst, d_ids[N - 2:], stream=st)     # the final stage: returns when the bytes have landed
        here.send("migrated")
        verdict = here.recv()
        assert verdict == "equal", verdict
        with pytest.raises(llx.LlxError):
            llx.pool_ipc_export(src.pool)                      # a wrapped pool cannot be exported
        with pytest.raises(llx.LlxError):
            llx.pool_ipc_open(b"\0" * llx.IPC_HANDLE_BYTES)    # not a handle
        dst.destroy()
    finally:
        child.join(timeout=120)
        if child.is_alive():
            child.kill()
    assert child.exitcode == 0
