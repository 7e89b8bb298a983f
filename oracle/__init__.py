"""CPU oracle for the Llumnix KV-cache live-migration hot path.  TEST INFRASTRUCTURE ONLY.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` /
`--impl reference` legs may import this package.  It shares no code with the
CUDA path (`paper_2406_03243_b200/`): no common kernels, headers, helpers,
tables or constants; neither imports the other.  Inputs come from `synth/`,
passed in as arrays by the caller.

What it computes, and the passage each part follows (all `PAPER.md:<line>`):

* `kv_migration.migrate_stage`   — one migration stage: the blocks of the request
  named by (src_block_ids, dst_block_ids) are copied whole, every layer, K and V
  (§4.2 live migration; block = K or V of `block_size` tokens of
  one layer, §5 "Block fusion"; destination blocks are reserved
  before the stage, §4.2 handshake).
* `kv_migration.migrate_batch`   — the same for many requests (the source llumlet
  migrates requests one after another, §4.4.3).
* `kv_migration.pack` / `unpack` — block fusion: gather into / scatter from ONE
  contiguous buffer (§5 "Block fusion"; buffer is what the
  transport sends, §5 "KV cache transfer").
* `kv_migration.append_tokens`   — the append-only growth of the cache while
  decoding continues (§4.2).
* `kv_migration.staged_migration`— stage 0..N with decoding in between (Fig. 6,
  PAPER.md:134).
* `kv_migration.plan_stage`, `stage_sizes` — which logical blocks a stage takes
   and the shrinking-stage recurrence behind "only takes two
  stages" (§6.2).
* `handshake.BlockManager`, `handshake.Migration`, `handshake.run_script` — the migration
  handshake of Figure 7 (§4.2): PRE-ALLOC before each stage, the source's
  check after each stage, abort and release, commit.
* `policy.calc_freeness`, `policy.pair_instances`, `policy.migration_order` — Algorithm 1
  (virtual usage and freeness) and the pairing rule of §4.4.3.
* `policy.plan_migration_batch` — one migration round of one (source, destination) pair as one batch: migration
  order, the source-state threshold and all-or-nothing PRE-ALLOC (PAPER.md:225 + :142; reading A31 in DESIGN.md).
* `policy.BudgetController` — the bandwidth budget of non-final stages chosen from observed decode steps so that their
  slowdown stays at a target (PAPER.md:289-291 states the bound, not a mechanism: reading A34 in DESIGN.md).
* `decode_attention.decode_attention_fp64` — standard KV-cache attention for one
  decode token per sequence, read through the block table (§2).

Parity pins (tests/test_oracle_*.py, `-m "not gpu"`): every function above is
pinned to something other than itself — pure-Python element-loop brute force on
micro pools (P1–P8), the paper's printed block arithmetic (P12,
tests/golden/paper_block_arithmetic.txt), closed-form special cases and
`torch.nn.functional.scaled_dot_product_attention` in float64 (P11), and the
closed form of the stage recurrence (P9); the handshake is pinned to the message
sequence the paper narrates (tests/golden/paper_handshake_fig7.txt), block conservation,
leak freedom at every abort point and the commit bookkeeping in closed form
(tests/test_oracle_handshake.py); Algorithm 1 is pinned to the meaning the paper gives
freeness (decode iterations left, by brute-force simulation), to the printed capacity
13,616 tokens / target load 1,600 tokens (tests/golden/paper_priority_headroom.txt) and to
the rule-by-rule special cases; the batch round to a closed form for equal requests, hand-computed special cases and
an independent brute-force restatement (tests/test_oracle_policy.py); `stage_sizes` also to an exact-rational time-stepped
simulation that shares nothing with the recurrence (tests/test_abi.py); `BudgetController` to the closed-form fixed point of an
affine cost, B* = (target - a) / b, reached from either side, to hand-computed single adjustments, to its limits (floor above
the target -> minimum; no cost -> doubling up to the maximum) and to one outlier per window (tests/test_oracle_policy.py).
Nothing here is "parity unpinned".
"""
