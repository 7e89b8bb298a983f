"""Pins for oracle/kv_migration.py (SURVEY.md §8(c) P1–P9, P12).  CPU only.

The oracle is compared with (a) tests/brute.py — pure-Python element loops on nested lists,
(b) the numbers the paper prints (tests/golden/), (c) invariants fixed by the paper's statement
(append-only ⇒ staged == single-shot; reserved blocks only; source keeps running ⇒ unchanged).
"""
import os

import numpy as np
import pytest

import brute
import synth
from oracle import kv_migration as om

GOLD = os.path.join(os.path.dirname(__file__), "golden")
SENT = synth.SENTINEL_U16

MICRO = dict(layers=2, kv_heads=1, head_dim=8, block_size=4, num_blocks=8)        # SURVEY P8 micro-pool
SMALL = dict(layers=3, kv_heads=2, head_dim=4, block_size=4, num_blocks=12)


def make_pools(g, seed=0):
    te = g["block_size"] * g["kv_heads"] * g["head_dim"]
    src = om.new_pool(g["layers"], g["num_blocks"], te)
    for l in range(g["layers"]):
        for kv in range(2):
            src[l, kv] = synth.slice_values_f16(seed, 0, l, kv, g["num_blocks"], te)
    dst = om.new_pool(g["layers"], g["num_blocks"], te, fill=SENT)
    return src, dst


def read_golden(name):
    out = {}
    for line in open(os.path.join(GOLD, name)):
        line = line.strip()
        if line and not line.startswith("#"):
            k, v = [x.strip() for x in line.split("=")]
            out[k] = int(v)
    return out


# ---- P12: the paper's printed block arithmetic -----------------------------
def test_geometry_matches_paper_example():
    g = read_golden("paper_block_arithmetic.txt")
    assert om.tile_bytes(g["kv_heads"], g["head_dim"], g["block_size_tokens"], g["elem_bytes"]) \
        == g["block_bytes_K_or_V_one_layer"] == 128 * 1024
    assert om.tiles_for_tokens(g["sequence_tokens"], g["layers"], g["block_size_tokens"]) \
        == g["blocks_for_sequence"] == 4096
    # ragged length: 100 tokens = 7 blocks of 16 (BASELINE.json configs[0]) ; 2 layers * 2 * 7
    assert om.tiles_for_tokens(100, 2, 16) == 28


# ---- P1/P2/P3/P8: one stage against brute force ------------------------------------------
@pytest.mark.parametrize("g", [MICRO, SMALL])
@pytest.mark.parametrize("n", [0, 1, 3, 8])
def test_stage_equals_bruteforce(g, n):
    src, dst = make_pools(g)
    src0 = src.copy()
    s_ids = synth.block_permutation(1, g["num_blocks"])[:n]
    d_ids = synth.block_permutation(2, g["num_blocks"])[:n]
    bs, bd = brute.pool_from_numpy(src), brute.pool_from_numpy(dst)
    om.migrate_stage(src, s_ids, dst, d_ids)
    brute.migrate_stage(bs, s_ids, bd, d_ids)
    assert dst.tolist() == bd                                   # P8 (implies P1)
    assert np.array_equal(src, src0) and src.tolist() == bs     # P3 source intact
    untouched = np.setdiff1d(np.arange(g["num_blocks"]), d_ids)
    assert np.all(dst[:, :, untouched, :] == SENT)              # P2 sentinel
    for i in range(n):                                          # P1 mapping, stated directly
        assert np.array_equal(dst[:, :, d_ids[i], :], src0[:, :, s_ids[i], :])


def test_direction_and_index_mistakes_are_detectable():
    """A swapped operand, a transposed (l,kv) or an off-by-one id must change the result the pins check."""
    g = MICRO
    src, dst = make_pools(g)
    s_ids = np.array([5, 0, 3], dtype=np.int32)
    d_ids = np.array([1, 7, 2], dtype=np.int32)
    om.migrate_stage(src, s_ids, dst, d_ids)
    assert not np.array_equal(dst[0, 0, 1], src[0, 1, 5])       # K is not V
    assert not np.array_equal(dst[0, 0, 1], src[1, 0, 5])       # layer 0 is not layer 1
    assert not np.array_equal(dst[0, 0, 1], src[0, 0, 0])       # pair i is not pair i+1
    assert np.array_equal(dst[1, 1, 7], src[1, 1, 0])


def test_duplicate_src_allowed_duplicate_dst_rejected_and_ranges():
    src, dst = make_pools(MICRO)
    om.migrate_stage(src, [3, 3], dst, [0, 1])                  # prefix-shared source block: legal
    assert np.array_equal(dst[:, :, 0], src[:, :, 3]) and np.array_equal(dst[:, :, 1], src[:, :, 3])
    with pytest.raises(ValueError):
        om.migrate_stage(src, [1, 2], dst, [4, 4])
    with pytest.raises(IndexError):
        om.migrate_stage(src, [8], dst, [0])
    with pytest.raises(IndexError):
        om.migrate_stage(src, [0], dst, [-1])
    with pytest.raises(ValueError):
        om.migrate_stage(src, [0], src, [1])


# ---- P6: order invariance and arbitrary partition into calls -----------------------------
def test_order_and_partition_invariance():
    g = SMALL
    src, dst_a = make_pools(g)
    _, dst_b = make_pools(g)
    _, dst_c = make_pools(g)
    s_ids = synth.block_permutation(1, g["num_blocks"])[:9]
    d_ids = synth.block_permutation(2, g["num_blocks"])[:9]
    om.migrate_stage(src, s_ids, dst_a, d_ids)
    p = np.random.default_rng(7).permutation(9)
    om.migrate_stage(src, s_ids[p], dst_b, d_ids[p])
    for a, b in [(0, 2), (2, 3), (3, 9)]:
        om.migrate_stage(src, s_ids[a:b], dst_c, d_ids[a:b])
    assert np.array_equal(dst_a, dst_b) and np.array_equal(dst_a, dst_c)


# ---- P7: batch == sequential, against brute force ----------------------------------------
def test_batch_equals_sequential_and_bruteforce():
    g = SMALL
    src, dst = make_pools(g)
    _, dst_seq = make_pools(g)
    s_ids = synth.block_permutation(1, g["num_blocks"])[:10]
    d_ids = synth.block_permutation(2, g["num_blocks"])[:10]
    off = [0, 3, 3, 4, 10]                                      # includes an empty request
    om.migrate_batch(src, dst, off, s_ids, d_ids)
    for r in range(4):
        om.migrate_stage(src, s_ids[off[r]:off[r + 1]], dst_seq, d_ids[off[r]:off[r + 1]])
    bs, bd = brute.pool_from_numpy(src), brute.pool_from_numpy(om.new_pool(g["layers"], g["num_blocks"], dst.shape[3], SENT))
    brute.migrate_stage(bs, s_ids, bd, d_ids)
    assert np.array_equal(dst, dst_seq) and dst.tolist() == bd
    with pytest.raises(ValueError):
        om.migrate_batch(src, dst, [0, 2, 1, 10], s_ids, d_ids)
    with pytest.raises(ValueError):
        om.migrate_batch(src, dst, [0, 5, 10], s_ids, np.r_[d_ids[:9], d_ids[0]])


# ---- P5: block fusion round trip ----------------------------------------------------------
def test_pack_unpack_roundtrip_and_layout():
    g = SMALL
    src, dst = make_pools(g)
    _, dst_direct = make_pools(g)
    s_ids = synth.block_permutation(1, g["num_blocks"])[:5]
    d_ids = synth.block_permutation(2, g["num_blocks"])[:5]
    buf = om.pack(src, s_ids)
    assert buf.shape == (5, g["layers"], 2, src.shape[3])
    assert buf.reshape(-1).tolist() == brute.pack(brute.pool_from_numpy(src), s_ids)   # flat layout [i][l][kv][e]
    om.unpack(buf, dst, d_ids)
    om.migrate_stage(src, s_ids, dst_direct, d_ids)
    assert np.array_equal(dst, dst_direct)
    bd = brute.pool_from_numpy(om.new_pool(g["layers"], g["num_blocks"], src.shape[3], SENT))
    brute.unpack(buf.reshape(-1).tolist(), bd, d_ids)
    assert dst.tolist() == bd
    # identity table on a contiguous pool: pack is a pure axis reorder of the pool
    ident = np.arange(g["num_blocks"])
    assert np.array_equal(om.pack(src, ident), np.transpose(src, (2, 0, 1, 3)))
    # a prefix of the buffer is the pack of a prefix of the table (stages concatenate, reading A6)
    assert np.array_equal(om.pack(src, s_ids[:2]), buf[:2])


def test_migrate_via_buffer_equals_bruteforce_stage():
    """PAPER.md:235-237 route (fuse -> send buffer -> scatter) against the brute-force stage and brute-force pack."""
    for g in (MICRO, SMALL):
        src, dst = make_pools(g)
        s_ids = synth.block_permutation(3, g["num_blocks"])[:6]
        d_ids = synth.block_permutation(4, g["num_blocks"])[:6]
        bs = brute.pool_from_numpy(src)
        bd = brute.pool_from_numpy(dst)
        brute.migrate_stage(bs, s_ids, bd, d_ids)
        buf = om.migrate_via_buffer(src, s_ids, dst, d_ids)
        assert dst.tolist() == bd
        assert buf.reshape(-1).tolist() == brute.pack(bs, s_ids)
        with pytest.raises(ValueError):
            om.migrate_via_buffer(src, [0, 1], dst, [2, 2])


# ---- P4: append-only => staged migration == single-shot copy of the FINAL state ----------
def _values(seed, te_tok):
    return lambda t, l, kv: synth.append_values_f16(seed, t, l, kv, te_tok)


@pytest.mark.parametrize("schedule,appends,start_tokens", [
    ((5, 2), (3,), 97),             # Tiny-like: 7 blocks, 97 -> 100 tokens
    ((4, 2, 1), (2, 2), 24),        # block_size 4: 24 -> 26 -> 28 tokens = 7 blocks
])
def test_staged_equals_single_shot_of_final_state(schedule, appends, start_tokens):
    g = dict(SMALL)
    S = 16 if start_tokens > 50 else 4
    g["block_size"] = S
    g["num_blocks"] = 12
    src, dst = make_pools(g)
    te_tok = g["kv_heads"] * g["head_dim"]
    nblk = sum(schedule)
    s_tab = synth.block_permutation(1, g["num_blocks"])[:nblk]
    d_tab = synth.block_permutation(2, g["num_blocks"])[:nblk]
    src_brute = brute.pool_from_numpy(src)
    final_tokens = om.staged_migration(src, s_tab, dst, d_tab, schedule, appends, S, start_tokens, _values(3, te_tok))
    assert final_tokens == start_tokens + sum(appends)
    assert -(-final_tokens // S) == nblk
    # brute-force replay of the appends on an independent copy gives the final source state
    for t in range(start_tokens, final_tokens):
        brute.append_token(src_brute, s_tab, t, S, te_tok, _values(3, te_tok))
    assert src.tolist() == src_brute
    single = om.new_pool(g["layers"], g["num_blocks"], src.shape[3], SENT)
    om.migrate_stage(src, s_tab, single, d_tab)
    assert np.array_equal(dst, single)                         # P4
    # and the append really changed the late blocks (so a premature copy would have been caught)
    early = om.new_pool(g["layers"], g["num_blocks"], src.shape[3], SENT)
    src_initial, _ = make_pools(g)
    om.migrate_stage(src_initial, s_tab, early, d_tab)
    assert not np.array_equal(early, single)


def test_append_touches_only_its_slots():
    g = SMALL
    src, _ = make_pools(g)
    before = src.copy()
    te_tok = g["kv_heads"] * g["head_dim"]
    tab = [7, 2, 9]
    om.append_tokens(src, tab, 5, 7, g["block_size"], _values(3, te_tok))      # tokens 5,6 -> block 2 (logical 1), slots 1,2
    diff = np.argwhere(src != before)
    assert set(diff[:, 2].tolist()) == {2}
    assert diff[:, 3].min() >= 1 * te_tok and diff[:, 3].max() < 3 * te_tok
    assert np.array_equal(src[1, 1, 2, te_tok:2 * te_tok], synth.append_values_f16(3, 5, 1, 1, te_tok))


# ---- S1 planning: readings A3/A4 and P9 ----------------------------------------------------
def test_plan_stage_rules():
    S = 16
    # 2032 tokens = 127 full blocks, nothing migrated: non-final stage takes all full blocks
    assert om.plan_stage(2032, 0, S, 2) == (127, False)
    # 8 tokens later: block 127 is partly filled, 1 block remains -> final
    assert om.plan_stage(2040, 127, S, 2) == (1, True)
    # partially filled tail is never taken by a non-final stage
    assert om.plan_stage(100, 0, S, 2) == (6, False)
    assert om.plan_stage(100, 6, S, 2) == (1, True)
    assert om.plan_stage(100, 5, S, 2) == (2, True)
    # short request: single final stage
    assert om.plan_stage(20, 0, S, 2) == (2, True)
    assert om.plan_stage(0, 0, S, 2) == (0, True)
    with pytest.raises(ValueError):
        om.plan_stage(16, 2, S, 2)
    # invariant for every state: a non-final stage never includes the block being appended to
    for tokens in range(0, 200):
        for m in range(0, -(-tokens // S) + 1):
            n, final = om.plan_stage(tokens, m, S, 2)
            assert n >= 0 and m + n <= -(-tokens // S)
            if not final:
                assert (m + n) * S <= tokens and n >= 1
            else:
                assert m + n == -(-tokens // S)


def test_stage_size_recurrence_two_stages():
    """"the migration only takes two stages, which is the minimum", because copying is much
    faster than decoding.  Closed form: with rho = c*S/r >= n0 the second stage is a single block."""
    # paper-like rates: 64 Gb/s link = 8 GB/s over 8 MiB blocks ~ 950 blocks/s; ~15 tokens/s decode (65 ms/step, :287)
    for n0 in (16, 64, 128, 512):
        assert om.stage_sizes(n0, 950.0, 15.4, 16) == [n0, 1]
    # slow copier: rho = 4 -> geometric shrink by 4 each stage (ceil)
    assert om.stage_sizes(64, 4.0, 16.0, 16) == [64, 16, 4, 1]
    assert om.stage_sizes(1, 1.0, 1.0, 16) == [1]
