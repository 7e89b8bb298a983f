"""Writes the input and expected files of tests/c/abi_gpu.c (the C client that moves data through the ABI).
Calls only `synth` (seeded inputs) and `oracle` (expected values): nothing here comes from the CUDA path.

    python tests/golden/make_abi_gpu_case.py OUTDIR

Files (little-endian, raw): ids.bin      int32: n, src_ids[n], dst_ids[n], dst2_ids[n]
                            src.bin      uint16[L][2][num_blocks][tile_elems]   the source pool (BASELINE configs[0] "Tiny", seed 0)
                            staging.bin  uint16[n][L][2][tile_elems]            oracle.pack of the request (block fusion)
                            dst.bin      uint16[L][2][num_blocks][tile_elems]   the destination after stage (5) + final stage (2)
                                                                                 and oracle.unpack of the buffer into dst2_ids
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import synth  # noqa: E402
from oracle import kv_migration as om  # noqa: E402


def main(outdir: str) -> None:
    g = synth.CONFIGS["tiny"]
    L, nb = g["layers"], g["num_blocks"]
    te = g["block_size"] * g["kv_heads"] * g["head_dim"]
    src = np.empty((L, 2, nb, te), dtype=np.uint16)
    for l in range(L):
        for kv in range(2):
            src[l, kv] = synth.slice_values_f16(0, 0, l, kv, nb, te)
    dst = om.new_pool(L, nb, te, fill=synth.SENTINEL_U16)
    n = 7
    s_ids = synth.block_permutation(1, nb)[:n]
    perm_d = synth.block_permutation(2, nb)
    d_ids, d2_ids = perm_d[:n], perm_d[n:2 * n]
    om.migrate_stage(src, s_ids[:5], dst, d_ids[:5])
    om.migrate_stage(src, s_ids[5:], dst, d_ids[5:])
    buf = om.pack(src, s_ids)
    om.unpack(buf, dst, d2_ids)
    os.makedirs(outdir, exist_ok=True)
    np.concatenate([[n], s_ids, d_ids, d2_ids]).astype("<i4").tofile(os.path.join(outdir, "ids.bin"))
    src.astype("<u2").tofile(os.path.join(outdir, "src.bin"))
    buf.astype("<u2").tofile(os.path.join(outdir, "staging.bin"))
    dst.astype("<u2").tofile(os.path.join(outdir, "dst.bin"))


if __name__ == "__main__":
    main(sys.argv[1])
