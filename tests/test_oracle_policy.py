"""Pins for oracle/policy.py (Algorithm 1; §4.4.3) and the C routines
llx_calc_freeness / llx_pair_instances / llx_migration_order against it.  CPU only."""
import math
import os

import numpy as np
import pytest

from oracle import policy as op

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def golden():
    out = {}
    for line in open(os.path.join(GOLD, "paper_priority_headroom.txt")):
        if line.strip() and not line.startswith("#"):
            k, v = [x.strip() for x in line.split("=")]
            out[k] = int(v)
    return out


def running(u, p=0):
    return op.Req(physical_usage=float(u), priority=p)


# ---- what the metric MEANS: "how many iterations the batch can still run for" ----
def test_freeness_counts_the_decode_iterations_left_bruteforce():
    rng = np.random.default_rng(0)
    for _ in range(200):
        B = int(rng.integers(1, 20))
        usage = [int(x) for x in rng.integers(1, 500, B)]
        M = int(sum(usage) + rng.integers(0, 2000))
        F, total = op.calc_freeness(op.Instance(M=M, requests=[running(u) for u in usage], headroom_for_priority=[0.0]))
        assert total == sum(usage)
        k, used = 0, sum(usage)               # brute force: every iteration appends one token per running request
        while used + B <= M:
            used += B
            k += 1
        assert k == math.floor(F)


# ---- execution priority: the headroom keeps the REAL load under the target --------
def test_headroom_makes_the_instance_overloaded_exactly_above_the_target_load():
    g = golden()
    M, target = g["instance_capacity_tokens"], g["high_priority_target_load_tokens"]
    headroom = [0.0, float(M - target)]
    for k_high in (1, 2, 5):
        for real_load in (target - 200, target - 1, target, target + 1, target + 500):
            per = real_load // (k_high + 3)
            usages = [per] * (k_high + 3)
            usages[0] += real_load - sum(usages)
            reqs = [running(u, 1) for u in usages[:k_high]] + [running(u, 0) for u in usages[k_high:]]
            F, total = op.calc_freeness(op.Instance(M=M, requests=reqs, headroom_for_priority=headroom))
            assert total == pytest.approx(real_load + (M - target))          # the headroom is divided, not multiplied (line 10)
            assert (F < 0) == (real_load > target)
    # without a high-priority request nobody gets the headroom
    F, total = op.calc_freeness(op.Instance(M=M, requests=[running(100), running(200)], headroom_for_priority=headroom))
    assert total == 300 and F == (M - 300) / 2


def test_queuing_fake_and_terminating_rules():
    inst = op.Instance(M=1000.0, headroom_for_priority=[0.0], requests=[
        running(300), running(100),
        op.Req(is_queuing=True, is_head_of_line=True, demand=700.0),          # line 4: its real demand
        op.Req(is_queuing=True, demand=900.0)])                                # line 5 (A27): 0
    F, total = op.calc_freeness(inst)
    assert total == 1100.0 and F == -50.0                                      # negative: "treat such instances as overloaded"
    inst.is_terminating = True                                                 # lines 12-13, 7
    F, total = op.calc_freeness(inst)
    assert F == -math.inf and total == math.inf
    assert op.calc_virtual_usage(op.Req(is_fake=True), inst) == math.inf
    F, total = op.calc_freeness(op.Instance(M=500.0, requests=[], headroom_for_priority=[0.0]))
    assert (F, total) == (500.0, 0.0)                                          # A28
    F, _ = op.calc_freeness(op.Instance(M=500.0, headroom_for_priority=[0.0],
                                        requests=[op.Req(is_queuing=True, is_head_of_line=True, demand=600.0)]))
    assert F == -100.0


def test_pairing_and_order_rules():
    g = golden()
    lo, hi = g["scale_up_below_freeness"], g["scale_down_above_freeness"]
    F = [5.0, 80.0, -3.0, 70.0, 20.0, -math.inf, 61.0, 9.0]
    pairs = op.pair_instances(F, lo, hi)
    assert pairs == [(5, 1), (2, 3), (0, 6)]                  # lowest with highest, repeatedly; 7 (F=9) finds no partner
    assert op.pair_instances([20.0, 30.0], lo, hi) == []
    assert op.pair_instances([1.0, 1.0, 90.0, 90.0], lo, hi) == [(0, 2), (1, 3)]          # ties: lower index first
    assert op.migration_order([1, 0, 0, 1, 0], [5, 9, 3, 2, 3]) == [2, 4, 1, 3, 0]      # low priority, then short


# ---- the C routines against the oracle ---------------------------------------------------------
@pytest.fixture(scope="module")
def llx():
    from paper_2406_03243_b200 import build
    build.build()
    import paper_2406_03243_b200 as m
    m.load()
    return m


def as_tuple(r: op.Req):
    return (r.is_queuing, r.is_head_of_line, r.is_fake, r.priority, r.demand, r.physical_usage)


def test_c_freeness_equals_oracle_on_seeded_instances(llx):
    rng = np.random.default_rng(3)
    for case in range(500):
        P = int(rng.integers(1, 4))
        headroom = [0.0] + [float(rng.integers(0, 5000)) for _ in range(P - 1)]
        reqs = []
        for i in range(int(rng.integers(0, 25))):
            if rng.random() < 0.25:
                reqs.append(op.Req(is_queuing=True, is_head_of_line=bool(rng.random() < 0.3), priority=int(rng.integers(0, P)),
                                   demand=float(rng.integers(1, 3000))))
            else:
                reqs.append(op.Req(priority=int(rng.integers(0, P)), physical_usage=float(rng.integers(1, 3000))))
        term = bool(rng.random() < 0.1)
        M = float(rng.integers(1000, 20000))
        want = op.calc_freeness(op.Instance(M=M, requests=reqs, headroom_for_priority=headroom, is_terminating=term))
        got = llx.calc_freeness([as_tuple(r) for r in reqs], M, headroom, term)
        for w, g_ in zip(want, got):
            assert (w == g_) or abs(w - g_) <= 1e-9 * max(1.0, abs(w)), (case, want, got)
    with pytest.raises(llx.LlxError):
        llx.calc_freeness([(0, 0, 0, 3, 0.0, 1.0)], 10.0, [0.0])             # priority out of range


def test_c_pairing_and_order_equal_oracle(llx):
    rng = np.random.default_rng(4)
    for case in range(300):
        n = int(rng.integers(0, 40))
        F = [float(x) for x in rng.integers(-50, 120, n)]                   # integers: many ties
        if n and rng.random() < 0.3:
            F[int(rng.integers(0, n))] = -math.inf
        assert llx.pair_instances(F, 10.0, 60.0) == op.pair_instances(F, 10.0, 60.0), (case, F)
        pr = [int(x) for x in rng.integers(0, 2, n)]
        sl = [int(x) for x in rng.integers(1, 20, n)]
        assert llx.migration_order(pr, sl) == op.migration_order(pr, sl)
    with pytest.raises(llx.LlxError):
        llx.pair_instances([1.0, 2.0], 60.0, 10.0)                           # overlapping thresholds
