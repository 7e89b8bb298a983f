"""Oracle: stage-wise migration of a paged KV cache.  Plain definition, NumPy, no tricks.

Pool state (reading A1 in DESIGN.md): one array per serving instance

    POOL : uint16[L][2][num_blocks][S*H*D]        kv index 0 = K, 1 = V

i.e. per layer and per K|V a dense tensor [num_blocks, S, H, D] of 16-bit
elements held as raw bit patterns — migration is a bit copy, so floats are never
interpreted here.  One row POOL[l][kv][b] is the paper's "block" (PAPER.md:237:
"key or value tensors of 16 tokens in each layer", 128 KB for 16-bit LLaMA-7B).

The loops below are the definition written out in the paper's order (block,
then layer, then K|V); there is no blocking, fusion or reordering.
"""
from __future__ import annotations

import numpy as np


# --------------------------------------------------------------------------
# Geometry (§5 Block fusion)
# --------------------------------------------------------------------------
def tile_bytes(kv_heads: int, head_dim: int, block_size: int, elem_bytes: int) -> int:
    """Bytes of one block = K *or* V of `block_size` tokens of ONE layer."""
    return block_size * kv_heads * head_dim * elem_bytes


def tiles_for_tokens(num_tokens: int, layers: int, block_size: int) -> int:
    """Number of such blocks a sequence of `num_tokens` occupies: ceil(tokens/S) * layers * 2
    ("a sequence of 1k tokens translates to 4k such blocks (32 layers)")."""
    return -(-num_tokens // block_size) * layers * 2


def new_pool(layers: int, num_blocks: int, tile_elems: int, fill: int | None = None) -> np.ndarray:
    pool = np.empty((layers, 2, num_blocks, tile_elems), dtype=np.uint16)
    if fill is not None:
        pool[...] = np.uint16(fill)
    return pool


def _check_ids(ids, num_blocks: int, what: str) -> np.ndarray:
    ids = np.asarray(ids, dtype=np.int64).reshape(-1)
    if ids.size and (ids.min() < 0 or ids.max() >= num_blocks):
        raise IndexError(f"{what} block id out of range [0,{num_blocks})")
    return ids


# --------------------------------------------------------------------------
# One stage (PAPER.md:134 "copy the KV cache blocks"; :142 reserved dst blocks)
# --------------------------------------------------------------------------
def migrate_stage(src: np.ndarray, src_block_ids, dst: np.ndarray, dst_block_ids) -> None:
    """for i<n, l<L, kv<2:  DST[l][kv][dst_ids[i]][:] = SRC[l][kv][src_ids[i]][:]

    Whole blocks are copied, including unused token slots of a partly filled last
    block (reading A2).  Duplicate destination ids are rejected (reading A8): the
    destination reserves distinct blocks.  Duplicate source ids are legal.
    """
    if src is dst:
        raise ValueError("source and destination are the same pool")
    if src.shape[0] != dst.shape[0] or src.shape[1] != 2 or dst.shape[1] != 2 or src.shape[3] != dst.shape[3]:
        raise ValueError("geometry mismatch")
    s_ids = _check_ids(src_block_ids, src.shape[2], "src")
    d_ids = _check_ids(dst_block_ids, dst.shape[2], "dst")
    if s_ids.size != d_ids.size:
        raise ValueError("src/dst id lists differ in length")
    if np.unique(d_ids).size != d_ids.size:
        raise ValueError("duplicate destination block id")
    layers = src.shape[0]
    for i in range(s_ids.size):
        for l in range(layers):
            for kv in range(2):
                dst[l, kv, d_ids[i], :] = src[l, kv, s_ids[i], :]


def migrate_batch(src: np.ndarray, dst: np.ndarray, req_offsets, src_block_ids, dst_block_ids) -> None:
    """R requests: request r owns pairs [req_offsets[r], req_offsets[r+1]) of the flat id lists.

    Defined as R successive `migrate_stage` calls (the source migrates
    its chosen requests one after another); destination ids must be distinct across
    the whole batch (each request's blocks are reserved separately).
    """
    off = np.asarray(req_offsets, dtype=np.int64).reshape(-1)
    s_ids = np.asarray(src_block_ids, dtype=np.int64).reshape(-1)
    d_ids = np.asarray(dst_block_ids, dtype=np.int64).reshape(-1)
    if off.size < 1 or off[0] != 0 or np.any(np.diff(off) < 0) or off[-1] != s_ids.size or s_ids.size != d_ids.size:
        raise ValueError("bad req_offsets")
    if np.unique(d_ids).size != d_ids.size:
        raise ValueError("duplicate destination block id across the batch")
    for r in range(off.size - 1):
        a, b = int(off[r]), int(off[r + 1])
        if b > a:
            migrate_stage(src, s_ids[a:b], dst, d_ids[a:b])


# --------------------------------------------------------------------------
# Block fusion: gather into / scatter from ONE contiguous buffer
# --------------------------------------------------------------------------
def pack(src: np.ndarray, src_block_ids) -> np.ndarray:
    """BUF : uint16[n][L][2][S*H*D];  BUF[i][l][kv][:] = SRC[l][kv][src_ids[i]][:]   (layout: reading A6)"""
    s_ids = _check_ids(src_block_ids, src.shape[2], "src")
    layers, _, _, te = src.shape
    buf = np.empty((s_ids.size, layers, 2, te), dtype=np.uint16)
    for i in range(s_ids.size):
        for l in range(layers):
            for kv in range(2):
                buf[i, l, kv, :] = src[l, kv, s_ids[i], :]
    return buf


def unpack(buf: np.ndarray, dst: np.ndarray, dst_block_ids) -> None:
    """DST[l][kv][dst_ids[i]][:] = BUF[i][l][kv][:]"""
    d_ids = _check_ids(dst_block_ids, dst.shape[2], "dst")
    layers, _, _, te = dst.shape
    if buf.shape != (d_ids.size, layers, 2, te):
        raise ValueError("staging buffer shape mismatch")
    if np.unique(d_ids).size != d_ids.size:
        raise ValueError("duplicate destination block id")
    for i in range(d_ids.size):
        for l in range(layers):
            for kv in range(2):
                dst[l, kv, d_ids[i], :] = buf[i, l, kv, :]


# --------------------------------------------------------------------------
# Append-only growth while decoding continues
# --------------------------------------------------------------------------
def append_tokens(pool: np.ndarray, block_table, t0: int, t1: int, block_size: int, values) -> None:
    """Write the K and V vectors of tokens t0..t1-1 into their slots.

    Token t lives in logical block t // S, slot t % S; a slot is H*D consecutive
    elements of the block row.  `values(t, l, kv)` returns uint16[H*D].  Nothing
    written earlier is modified ("leaving the parameters generated by previous
    iterations remain constant").
    """
    layers, _, _, te = pool.shape
    token_elems = te // block_size
    table = np.asarray(block_table, dtype=np.int64)
    for t in range(t0, t1):
        b = int(table[t // block_size])
        s = t % block_size
        for l in range(layers):
            for kv in range(2):
                pool[l, kv, b, s * token_elems:(s + 1) * token_elems] = values(t, l, kv)


def staged_migration(src, src_table, dst, dst_table, schedule, appends, block_size, num_tokens, values) -> int:
    """Fig. 6: stage k copies logical blocks [m, m+n_k); after stage k
    (k < len(appends)) the source decodes `appends[k]` more tokens.  Returns the final token count."""
    src_table = np.asarray(src_table)
    dst_table = np.asarray(dst_table)
    m = 0
    for k, n in enumerate(schedule):
        migrate_stage(src, src_table[m:m + n], dst, dst_table[m:m + n])
        m += n
        if k < len(appends):
            append_tokens(src, src_table, num_tokens, num_tokens + appends[k], block_size, values)
            num_tokens += appends[k]
    return num_tokens


def migrate_via_buffer(src: np.ndarray, src_block_ids, dst: np.ndarray, dst_block_ids) -> np.ndarray:
    """The paper's transfer route written out: the request's blocks are fused into one
    contiguous buffer (`pack`), the buffer is what travels, and the destination scatters it into its reserved
    blocks (`unpack`).  Returns the buffer.  The final DST equals `migrate_stage` (pin P5)."""
    if src is dst:
        raise ValueError("source and destination are the same pool")
    s_ids = _check_ids(src_block_ids, src.shape[2], "src")
    d_ids = _check_ids(dst_block_ids, dst.shape[2], "dst")
    if s_ids.size != d_ids.size:
        raise ValueError("src/dst id lists differ in length")
    if np.unique(d_ids).size != d_ids.size:
        raise ValueError("duplicate destination block id")
    buf = pack(src, s_ids)
    unpack(buf, dst, d_ids)
    return buf


# --------------------------------------------------------------------------
# Stage planning (readings A3, A4 in DESIGN.md)
# --------------------------------------------------------------------------
def plan_stage(num_tokens: int, blocks_migrated: int, block_size: int, last_stage_max_blocks: int):
    """Which logical blocks [m, m+n) the next stage takes, and whether it is the final one.

    A non-final stage copies "the KV cache blocks of completed iterations"
     that can no longer change: the full blocks [m, num_tokens // S).
    When at most `last_stage_max_blocks` blocks remain, the stage is final: the
    request is drained and "the remaining block" is copied.
    """
    if num_tokens < 0 or blocks_migrated < 0 or block_size <= 0 or last_stage_max_blocks < 1:
        raise ValueError("bad arguments")
    total = -(-num_tokens // block_size)
    full = num_tokens // block_size
    if blocks_migrated > total:
        raise ValueError("more blocks migrated than the request has")
    remaining = total - blocks_migrated
    if remaining <= last_stage_max_blocks:
        return remaining, True
    return full - blocks_migrated, False


def stage_sizes(n0: int, copy_blocks_per_s: float, decode_tokens_per_s: float, block_size: int, max_stages: int = 64):
    """Stage-size recurrence behind "the number of new blocks is typically small"
    and "the migration only takes two stages":

        time of stage k  = n_k / c ;  tokens decoded meanwhile = r * n_k / c
        n_{k+1} = ceil(n_k * r / (c * S))          (c = copy rate blocks/s, r = decode tokens/s)

    stops when a stage is a single block (that stage is the final one)."""
    out = [int(n0)]
    while out[-1] > 1 and len(out) < max_stages:
        nxt = int(np.ceil(out[-1] * decode_tokens_per_s / (copy_blocks_per_s * block_size)))
        out.append(max(1, nxt))
    return out
