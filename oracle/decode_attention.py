"""Oracle: paged decode attention in float64 (one query token per sequence).

The paper relies on the standard attention over the KV cache (PAPER.md:74-80,
ref [59]) read from dynamically allocated blocks (PagedAttention).
Readings (A14): MHA (q heads = KV heads), scale 1/sqrt(D), no mask
other than t < ctx_len, ctx_len includes the current token, no positional term.

    per sequence b, head h:   s_t = (q . k_t) / sqrt(D)         t < ctx_len[b]
                              p_t = exp(s_t - max s) / sum_t exp(s_t - max s)
                              o   = sum_t p_t v_t

K and V are gathered token by token through the block table, up-converting the
stored fp16 BIT PATTERNS to float64 exactly; the output is NOT re-quantised.
"""
from __future__ import annotations

import numpy as np


def _f64(bits: np.ndarray) -> np.ndarray:
    return np.ascontiguousarray(bits).view(np.float16).astype(np.float64)


def decode_attention_fp64(pool: np.ndarray, layer: int, q_bits: np.ndarray, block_tables: np.ndarray,
                          ctx_lens: np.ndarray, block_size: int, kv_heads: int, head_dim: int,
                          scale: float | None = None) -> np.ndarray:
    """pool: uint16[L][2][num_blocks][S*H*D]; q_bits: uint16[B,H,D]; block_tables: int[B,max_blocks];
    ctx_lens: int[B].  Returns float64[B,H,D]."""
    S, H, D = block_size, kv_heads, head_dim
    B = q_bits.shape[0]
    if scale is None:
        scale = 1.0 / np.sqrt(float(D))
    q = _f64(q_bits).reshape(B, H, D)
    out = np.zeros((B, H, D), dtype=np.float64)
    for b in range(B):
        n = int(ctx_lens[b])
        k = np.empty((n, H, D), dtype=np.float64)
        v = np.empty((n, H, D), dtype=np.float64)
        for t in range(n):
            blk = int(block_tables[b, t // S])
            slot = t % S
            k[t] = _f64(pool[layer, 0, blk].reshape(S, H, D)[slot])
            v[t] = _f64(pool[layer, 1, blk].reshape(S, H, D)[slot])
        for h in range(H):
            s = (k[:, h, :] @ q[b, h]) * scale          # [n]
            p = np.exp(s - s.max())
            p = p / p.sum()
            out[b, h] = p @ v[:, h, :]
    return out
