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


# ---- one migration round as one batch (reading A31, PAPER.md:225 + :142) ---------------------------------
def random_source(rng, P=2, max_reqs=14, nb_pool=400):
    """A seeded source instance: requests, sequence lengths, disjoint block tables (usage unit: blocks)."""
    reqs, seq, tables = [], [], []
    free = list(rng.permutation(nb_pool))
    hol_given = False
    for _ in range(int(rng.integers(0, max_reqs))):
        if rng.random() < 0.2:
            hol = (not hol_given) and bool(rng.random() < 0.6)
            hol_given |= hol
            reqs.append(op.Req(is_queuing=True, is_head_of_line=hol, priority=int(rng.integers(0, P)),
                               demand=float(rng.integers(1, 60))))
            seq.append(int(rng.integers(1, 900)))
            tables.append([])
        else:
            nb = int(rng.integers(1, 30))
            t = [int(free.pop()) for _ in range(nb)]
            reqs.append(op.Req(priority=int(rng.integers(0, P)), physical_usage=float(nb)))
            seq.append(int(rng.integers((nb - 1) * 16 + 1, nb * 16 + 1)))
            tables.append(t)
    return reqs, seq, tables


def test_batch_plan_closed_form_for_equal_requests():
    """B running requests of u blocks each, nothing queuing, no headroom: after k requests have left,
    F_k = M/(B-k) - u, so the round takes k* = the smallest k with F_k >= T, i.e. max(0, ceil(B - M/(T+u)))
    (and everything when even one remaining request keeps F below T: then B = 1 by A28 once all are gone)."""
    from oracle import handshake as oh
    for B, u, M, T in [(8, 10, 100, 5.0), (8, 10, 100, 15.0), (5, 4, 40, 2.0), (6, 7, 20, 1.0), (3, 9, 100, 0.5), (4, 10, 30, 40.0)]:
        inst = op.Instance(M=float(M), requests=[running(u) for _ in range(B)], headroom_for_priority=[0.0])
        tables = [list(range(r * u, (r + 1) * u)) for r in range(B)]
        dst = oh.BlockManager(1000)
        chosen, off, s_ids, d_ids = op.plan_migration_batch(inst, [u * 16] * B, tables, T, dst)
        k_star = max(0, math.ceil(B - M / (T + u)))
        if k_star >= B:                       # all running requests gone: B := 1 (A28), F = M >= T unless T > M
            k_star = B
        assert len(chosen) == k_star, (B, u, M, T, chosen)
        assert chosen == list(range(k_star))                          # equal priority and length: index order
        assert off == [u * i for i in range(k_star + 1)]
        assert s_ids == [b for r in chosen for b in tables[r]]
        assert d_ids == list(range(u * k_star)) and dst.num_free() == 1000 - u * k_star    # A23: a fresh manager hands out 0,1,2,...


def test_batch_plan_special_cases():
    from oracle import handshake as oh
    reqs = [running(10, 1), running(30, 0), running(5, 0), op.Req(is_queuing=True, is_head_of_line=True, demand=50.0), running(5, 0)]
    seq, tables = [160, 480, 70, 800, 80], [list(range(0, 10)), list(range(10, 40)), list(range(40, 45)), [], list(range(45, 50))]
    inst = op.Instance(M=80.0, requests=reqs, headroom_for_priority=[0.0, 20.0])
    # sum V = 10+20 + 30 + 5 + 50 + 5 = 120 -> F = -40/4 = -10: a source for any threshold above -10
    assert op.calc_freeness(inst)[0] == -10.0
    dst = oh.BlockManager(100)
    assert op.plan_migration_batch(inst, seq, tables, -10.0, dst) == ([], [0], [], [])        # F is not BELOW the threshold
    # lower priority first, then shorter: 2 (70 tokens), 4 (80), 1 (480), and the high-priority request 0 last
    chosen, off, s_ids, d_ids = op.plan_migration_batch(inst, seq, tables, 1e9, dst)
    assert chosen == [2, 4, 1, 0] and off == [0, 5, 10, 40, 50] and d_ids == list(range(50))
    assert s_ids == tables[2] + tables[4] + tables[1] + tables[0] and dst.num_free() == 50
    # threshold 0: after 2 leaves F = (80-115)/3, after 4: (80-110)/2 = -15, after 1: (80-80)/1 = 0 -> stop before request 0
    dst = oh.BlockManager(100)
    assert op.plan_migration_batch(inst, seq, tables, 0.0, dst)[0] == [2, 4, 1]
    # the destination runs out: all-or-nothing per request, the first misfit ends the round (nothing of it is reserved)
    dst = oh.BlockManager(100)
    dst.allocate(70)                                                    # 30 free: 5 + 5 fit, the 30-block request does not
    chosen, off, s_ids, d_ids = op.plan_migration_batch(inst, seq, tables, 1e9, dst)
    assert chosen == [2, 4] and dst.num_free() == 20 and d_ids == list(range(70, 80))
    dst = oh.BlockManager(100)
    assert op.plan_migration_batch(inst, seq, tables, 1e9, dst, dst_reserve_blocks=91)[0] == [2]      # 9 usable: only 5 fit
    # a terminating instance is drained whatever the threshold (fake request: F = -inf)
    inst.is_terminating = True
    dst = oh.BlockManager(100)
    assert op.plan_migration_batch(inst, seq, tables, -1e300, dst)[0] == [2, 4, 1, 0]


def brute_batch_plan(reqs, seq, tables, M, headroom, term, T, dst_free):
    """Independent restatement of A31 from the paper's sentences, without oracle.policy: plain tuples and loops."""
    here = [i for i in range(len(reqs))]
    cand = [i for i in range(len(reqs)) if not reqs[i].is_queuing]
    # "prefers the requests with lower priorities and shorter sequence lengths": repeated selection of the minimum
    ordered = []
    while cand:
        best = cand[0]
        for i in cand[1:]:
            if (reqs[i].priority, seq[i], i) < (reqs[best].priority, seq[best], best):
                best = i
        ordered.append(best)
        cand.remove(best)
    taken = []
    for r in ordered:
        run = [i for i in here if not reqs[i].is_queuing]
        V = 0.0
        for i in here:
            q = reqs[i]
            if q.is_queuing:
                V += q.demand if q.is_head_of_line else 0.0
            else:
                V += q.physical_usage + headroom[q.priority] / sum(1 for j in run if reqs[j].priority == q.priority)
        F = -math.inf if term else (M - V) / max(1, len(run))
        if F >= T or len(tables[r]) > dst_free:
            break
        dst_free -= len(tables[r])
        taken.append(r)
        here.remove(r)
    return taken


def test_batch_plan_equals_bruteforce_restatement_and_c(llx):
    from oracle import handshake as oh
    rng = np.random.default_rng(11)
    nonempty = 0
    for case in range(400):
        P = int(rng.integers(1, 3))
        headroom = [0.0] + [float(rng.integers(0, 80))] * (P - 1)
        reqs, seq, tables = random_source(rng, P)
        used = sum(len(t) for t in tables)
        M = float(rng.integers(max(1, used // 2), used + 120))
        term = bool(rng.random() < 0.1)
        T = float(rng.integers(-20, 40))
        nb_dst, taken_before, reserve = 300, int(rng.integers(0, 300)), int(rng.integers(0, 20))
        o_dst, c_dst = oh.BlockManager(nb_dst), llx.BlockManager(nb_dst)
        o_dst.allocate(taken_before), c_dst.alloc(taken_before)
        inst = op.Instance(M=M, requests=reqs, headroom_for_priority=headroom, is_terminating=term)
        want = op.plan_migration_batch(inst, seq, tables, T, o_dst, reserve)
        assert want[0] == brute_batch_plan(reqs, seq, tables, M, headroom, term, T, nb_dst - taken_before - reserve), case
        got = llx.plan_migration_batch([as_tuple(r) for r in reqs], seq, M, headroom, T, tables, c_dst, reserve, term)
        assert got[0] == want[0] and list(got[1]) == want[1] and list(got[2]) == want[2] and list(got[3]) == want[3], case
        assert c_dst.num_free == o_dst.num_free() == nb_dst - taken_before - len(want[3])
        assert len(set(want[3])) == len(want[3])
        nonempty += bool(want[0])
    assert nonempty > 100


def test_c_batch_plan_argument_errors_reserve_nothing(llx):
    l = llx.lib()
    import ctypes as C
    mgr = llx.BlockManager(50)
    reqs = [(0, 0, 0, 0, 0.0, 10.0), (0, 0, 0, 0, 0.0, 10.0)]
    assert llx.plan_migration_batch(reqs, [100, 100], 5.0, [0.0], 100.0, [[1, 2, 3], [4, 5]], mgr)[0] == [0, 1]
    assert mgr.num_free == 45
    # outputs too small: LLX_ERR_INVALID_ARG, *n_pairs tells the size needed, nothing reserved
    arr = (llx.binding.ReqInfo * 2)(*[llx.binding.ReqInfo(*[int(x) for x in r[:4]], r[4], r[5]) for r in reqs])
    i32 = lambda v: (C.c_int32 * len(v))(*v)
    hr = (C.c_double * 1)(0.0)
    chosen, ro, so, do = i32([0, 0]), i32([0, 0, 0]), i32([0] * 4), i32([0] * 4)
    nc, npairs = C.c_int(), C.c_int()
    rc = l.llx_plan_migration_batch(arr, i32([100, 100]), 2, 5.0, hr, 1, 0, 100.0, i32([0, 3, 5]), i32([1, 2, 3, 4, 5]),
                                    mgr.handle, 0, chosen, C.byref(nc), ro, so, do, 4, C.byref(npairs))
    assert rc == -1 and npairs.value == 5 and mgr.num_free == 45
    rc = l.llx_plan_migration_batch(arr, i32([100, 100]), 2, 5.0, hr, 1, 0, 100.0, i32([0, 3, 2]), i32([1, 2, 3, 4, 5]),
                                    mgr.handle, 0, chosen, C.byref(nc), ro, so, do, 4, C.byref(npairs))
    assert rc == -1 and mgr.num_free == 45                                      # offsets decrease


# ---- the budget controller (reading A34): pinned by what it must achieve on plants with a known answer ----------
def _drive(ctl, cost, base_ms=5.0, rounds=40, noise=None):
    """Alternate `window` steps without a migration and `window` steps with one whose slowdown is cost(budget)."""
    rng = np.random.default_rng(3)
    for _ in range(rounds):
        for migrating in (False, True):
            for _ in range(ctl.window):
                t = base_ms * (1.0 + (cost(ctl.gbps()) if migrating else 0.0))
                if noise:
                    t *= 1.0 + noise * float(rng.standard_normal())
                ctl.observe(t, migrating)
    return ctl.gbps()


def test_budget_controller_finds_the_budget_where_the_cost_equals_the_target():
    """Affine plant s(B) = a + b*B (what DESIGN.md section 5.2a measures: a floor from the write turn-arounds plus a share
    of the DRAM bytes).  The fixed point is B* = (t - a) / b; the rule must reach it from either side."""
    from oracle.policy import BudgetController
    t = 0.01
    for a, b in ((0.0, 0.0004), (0.004, 0.00025), (0.007, 0.00025), (0.002, 0.00002)):
        star = (t - a) / b
        for start in (1, 8, 64, 400):
            ctl = BudgetController(1.0, 1, 1000, start, 8)
            got = _drive(ctl, lambda B: a + b * B)
            assert abs(got - star) <= max(1.0, 0.03 * star), (a, b, start, got, star)
    # the measured sustained-decoding curve of DESIGN.md section 5.2a (12 -> 1.0 %, 25 -> 1.5 %, 50 -> 2.2 %, 100 -> 3.35 %),
    # linearly interpolated: the 1 % budget is 12 GB/s
    xs, ys = [0, 12, 25, 50, 100, 200, 400], [0.0, 0.010, 0.015, 0.022, 0.0335, 0.0585, 0.0865]
    ctl = BudgetController(1.0, 1, 1000, 100, 8)
    assert abs(_drive(ctl, lambda B: float(np.interp(B, xs, ys))) - 12) <= 1


def test_budget_controller_limits_and_single_steps():
    from oracle.policy import BudgetController
    # a floor above the target: the budget goes to its minimum and stays there
    ctl = BudgetController(1.0, 5, 1000, 200, 4)
    assert _drive(ctl, lambda B: 0.02 + 0.0001 * B) == 5
    # no measurable cost: doubles at every adjustment up to the maximum
    ctl = BudgetController(1.0, 1, 300, 10, 4)
    seen = []
    for _ in range(7):
        for m in (False, True):
            for _ in range(4):
                ctl.observe(5.0, m)
        seen.append(ctl.gbps())
    assert seen == [20, 40, 80, 160, 300, 300, 300]
    # one adjustment, by hand: slowdown 2 % at target 1 % halves; 1 % keeps; 0.5 % doubles; 10 % is clamped to a half
    for slow, want in ((0.02, 50), (0.01, 100), (0.005, 200), (0.10, 50), (0.0125, 80)):
        ctl = BudgetController(1.0, 1, 1000, 100, 4)
        for _ in range(4):
            ctl.observe(4.0, False)
        for _ in range(4):
            ctl.observe(4.0 * (1.0 + slow), True)
        assert ctl.gbps() == want and abs(ctl.last_slowdown_pct - 100 * slow) < 1e-9 and ctl.adjustments == 1
    # medians: one wild step among eight does not move the decision; steps with a migration before any baseline are dropped
    ctl = BudgetController(1.0, 1, 1000, 100, 8)
    for k in range(8):
        ctl.observe(40.0 if k == 3 else 4.0, True)
    assert ctl.adjustments == 0
    for k in range(8):
        ctl.observe(9.0 if k == 5 else 4.0, False)
    for k in range(8):
        ctl.observe(30.0 if k == 2 else 4.04, True)
    assert ctl.gbps() == 100 and ctl.adjustments == 1
    # with 1 % noise on every step the rule still settles within 35 % of the fixed point (B* = 40)
    ctl = BudgetController(1.0, 1, 1000, 300, 16)
    got = _drive(ctl, lambda B: 0.00025 * B, rounds=60, noise=0.002)
    assert 26 <= got <= 54, got
    for bad in ((0.0, 1, 10, 5, 8), (1.0, 0, 10, 5, 8), (1.0, 5, 4, 5, 8), (1.0, 1, 10, 11, 8), (1.0, 1, 10, 5, 1)):
        with pytest.raises(ValueError):
            BudgetController(*bad)


def test_library_budget_controller_equals_the_oracle_on_seeded_step_sequences():
    """llx_budget_ctl_* (C++) against oracle.policy.BudgetController: the same budget and the same slowdown estimate
    after EVERY observation of 200 seeded sequences (random parameters, step times, migrating flags, outliers)."""
    import paper_2406_03243_b200 as llx
    from oracle.policy import BudgetController
    rng = np.random.default_rng(11)
    for case in range(200):
        target = float(rng.choice([0.5, 1.0, 2.0, 5.0]))
        lo = int(rng.integers(1, 20))
        hi = int(rng.integers(lo, 2000))
        start = int(rng.integers(lo, hi + 1))
        window = int(rng.integers(2, 20))
        a, b = BudgetController(target, lo, hi, start, window), llx.BudgetController(target, lo, hi, start, window)
        base = float(rng.uniform(0.5, 20.0))
        slope = float(rng.uniform(0.0, 0.001))
        for _ in range(int(rng.integers(10, 400))):
            mig = bool(rng.random() < 0.5)
            t = base * (1.0 + (slope * a.gbps() if mig else 0.0)) * float(rng.uniform(0.97, 1.03))
            if rng.random() < 0.03:
                t *= 5.0
            assert a.observe(t, mig) == b.observe(t, mig) == b.gbps, case
            assert a.adjustments == b.adjustments
            assert (math.isnan(a.last_slowdown_pct) and math.isnan(b.last_slowdown_pct)) or a.last_slowdown_pct == b.last_slowdown_pct
    with pytest.raises(llx.LlxError):
        llx.BudgetController(0.0, 1, 10, 5, 8)
    with pytest.raises(llx.LlxError):
        llx.BudgetController(1.0, 1, 10, 5, 8).observe(float("nan"), True)
    with pytest.raises(llx.LlxError):
        llx.BudgetController(1.0, 1, 10, 5, 8).observe(-1.0, False)
    assert llx.lib().llx_budget_ctl_gbps(None) == -1 and llx.lib().llx_budget_ctl_adjustments(None) == -1
