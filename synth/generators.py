"""Seeded input generators (NumPy only).  See synth/__init__.py for the rules.

Every generator is a pure function of its integer seeds, so the oracle run and
the CUDA run of a test see byte-identical inputs, and a big pool can be
regenerated one (layer, K|V) slice at a time during verification instead of
being mirrored on the host.
"""
from __future__ import annotations

import math

import numpy as np

#: fp16 bit pattern the destination pool is pre-filled with (BASELINE.json configs[0]).
#: 0x7BAD is a finite fp16 (62880.0), not a NaN; comparisons are on bits anyway.
SENTINEL_U16 = 0x7BAD

#: Shapes named by BASELINE.json `configs` — plain numbers only, no derived sizes.
CONFIGS = {
    # configs[0]
    "tiny": dict(layers=2, kv_heads=4, head_dim=64, block_size=16, elem_bytes=2, num_blocks=256),
    # configs[1], [2], [4]  (LLaMA-7B: 32 layers, 32 KV heads, head_dim 128)
    "llama7b": dict(layers=32, kv_heads=32, head_dim=128, block_size=16, elem_bytes=2, num_blocks=2000),
    # configs[3]  (LLaMA-30B: 60 layers, 52 KV heads, head_dim 128)
    "llama30b": dict(layers=60, kv_heads=52, head_dim=128, block_size=16, elem_bytes=2, num_blocks=3000),
}


def _rng(*key: int) -> np.random.Generator:
    return np.random.default_rng([int(k) & 0xFFFFFFFF for k in key])


def slice_values_f16(seed: int, pool_id: int, layer: int, kv: int, num_blocks: int, tile_elems: int) -> np.ndarray:
    """One (layer, K|V) slice of a pool: uint16 view of fp16 values U[-1,1).

    float32 uniform -> *2-1 -> round-to-nearest-even fp16.  Independent sub-seed
    per (seed, pool_id, layer, kv) so slices can be regenerated one at a time.
    Returns uint16[num_blocks, tile_elems] (the fp16 bit patterns).
    """
    r = _rng(seed, pool_id, layer, kv, 0xA11CE)
    x = r.random((num_blocks, tile_elems), dtype=np.float32)
    x *= 2.0
    x -= 1.0
    return x.astype(np.float16).view(np.uint16)


def block_permutation(seed: int, num_blocks: int) -> np.ndarray:
    """Seeded permutation of range(num_blocks) as int32: prefixes are unique, scattered ids."""
    return _rng(seed, 0xB10C).permutation(num_blocks).astype(np.int32)


def append_values_f16(seed: int, token_index: int, layer: int, kv: int, token_elems: int) -> np.ndarray:
    """K or V vector (all heads) of one newly decoded token, uint16 fp16 bits, U[-1,1)."""
    r = _rng(seed, token_index, layer, kv, 0xA99E)
    x = r.random(token_elems, dtype=np.float32) * 2.0 - 1.0
    return x.astype(np.float16).view(np.uint16)


def context_lengths(seed: int, batch: int, lo: int, hi: int) -> np.ndarray:
    """Context lengths uniform on the integers {lo..hi} (inclusive), int32[batch]."""
    return _rng(seed, 0xC7).integers(lo, hi + 1, size=batch).astype(np.int32)


def queries_f16(seed: int, batch: int, heads: int, head_dim: int) -> np.ndarray:
    """Decode queries, one token per sequence: uint16 fp16 bits [batch, heads, head_dim], U[-1,1)."""
    r = _rng(seed, 0x9)
    x = r.random((batch, heads, head_dim), dtype=np.float32) * 2.0 - 1.0
    return x.astype(np.float16).view(np.uint16)


# ----------------------------------------------------------------------------
# Power-law request lengths (stand-in for PAPER.md Table 1, "Gen" rows).
# ----------------------------------------------------------------------------
def _bounded_pareto_mean(alpha: float, lo: float, hi: float) -> float:
    if abs(alpha - 1.0) < 1e-12:
        return (math.log(hi) - math.log(lo)) / (1.0 / lo - 1.0 / hi)
    c = lo**alpha / (1.0 - (lo / hi) ** alpha)
    return c * alpha / (alpha - 1.0) * (lo ** (1.0 - alpha) - hi ** (1.0 - alpha))


def bounded_pareto_alpha(mean: float, lo: float, hi: float) -> float:
    """Shape alpha of the bounded Pareto on [lo, hi] whose continuous mean is `mean` (bisection)."""
    a, b = 1e-6, 8.0  # mean is decreasing in alpha
    for _ in range(200):
        mid = 0.5 * (a + b)
        if _bounded_pareto_mean(mid, lo, hi) > mean:
            a = mid
        else:
            b = mid
    return 0.5 * (a + b)


def bounded_pareto_quantile(u, alpha: float, lo: float, hi: float):
    """Inverse CDF x(u) = ((1-u) lo^-a + u hi^-a)^(-1/a) of the bounded Pareto."""
    u = np.asarray(u, dtype=np.float64)
    return ((1.0 - u) * lo ** (-alpha) + u * hi ** (-alpha)) ** (-1.0 / alpha)


def bounded_pareto_lengths(seed: int, count: int, mean: float = 512.0, lo: int = 16, hi: int = 8192) -> np.ndarray:
    """`count` request lengths (tokens), int32, bounded-Pareto with the given mean, clamped to [lo, hi]."""
    alpha = bounded_pareto_alpha(mean, lo, hi)
    u = _rng(seed, 0x1E46).random(count)
    x = np.floor(bounded_pareto_quantile(u, alpha, lo, hi)).astype(np.int64)
    return np.clip(x, lo, hi).astype(np.int32)


def batch_request_blocks(seed: int, count: int, block_size: int, pool_blocks: int,
                         mean: float = 512.0, lo: int = 16, hi: int = 8192):
    """Lengths for a batch whose total block demand fits `pool_blocks` (configs[3]).

    Advances the seed by +1 until sum(ceil(len/block_size)) <= pool_blocks and
    returns (lengths int32[count], blocks_per_request int32[count], seed_used).
    """
    s = seed
    while True:
        lens = bounded_pareto_lengths(s, count, mean, lo, hi)
        nblk = (lens.astype(np.int64) + block_size - 1) // block_size
        if int(nblk.sum()) <= pool_blocks:
            return lens, nblk.astype(np.int32), s
        s += 1
