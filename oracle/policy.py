"""Oracle: Llumnix's virtual usage / freeness calculation (Algorithm 1) and the
migration pairing policy built on it (§4.4.3).  TEST INFRASTRUCTURE ONLY — the
algorithm in the paper's order and notation, plain Python, fp64.  Shares no code with
paper_2406_03243_b200/csrc/llx_coord.cu.

Algorithm 1 as printed (line numbers are the paper's; the extracted text lost lines 2-5's layout,
the prose fixes them: "directly uses its real demand (line 4)", "a fake request with a virtual usage
of infinity (line 7)", "adding such a headroom on the physical usage (line 8)", "this headroom is
divided among them (line 10)"):

     1  Function CalcVirtualUsage(req, instance):
     2    if req.isQueuing then
     3      if req.isHeadOfLine then
     4        return req.demand
     5      return 0
     6    if req.isFake then
     7      return inf
     8    return req.physicalUsage + GetHeadroom(req.priority, instance)
     9  Function GetHeadroom(p, instance):
    10    return headroomForPriority[p] / instance.numRequests[p]
    11  Function CalcFreeness(instance):
    12    if instance.isTerminating then
    13      AddFakeReq(instance.requests)
    14    totalVirtualUsages = 0
    15    for req in instance.requests do
    16      totalVirtualUsages += CalcVirtualUsage(req, instance)
    17    freeness = (instance.M - totalVirtualUsages) / instance.B
    18    return freeness

Readings (A27-A30):
  A27  line 5 (lost in extraction): a queuing request that is not head-of-line has virtual usage 0
       ("For the head-of-line queuing request ... we assign a positive virtual usage").
  A28  B = number of running requests ("the batch size ... the number of new tokens per iteration",
       PAPER.md:223); an instance with no running request uses B = 1 so that F stays finite.
  A29  numRequests[p] counts the RUNNING requests of priority p (the ones that receive headroom).
  A30  pairing: sources are instances with F < src_below, destinations those with F > dst_above; the
       lowest-F source is paired with the highest-F destination, repeatedly, until one set is empty
       (PAPER.md:225); ties broken by the lower instance index.  Requests to migrate: lower priority
       first, then shorter sequence, then lower index ("prefers the requests with lower
       priorities and shorter sequence lengths").
  A31  one migration round of one (source, destination) pair, taken as ONE batch ("The llumlet of each
       source instance then starts to migrate requests to the destination continuously, until it is no longer set in
       the source state"): the source offers its RUNNING requests in `migration_order`; before each request it
       recomputes its own freeness over the requests it still has and stops once F >= src_below (it would no longer be
       chosen as a source); the request's blocks are pre-allocated on the destination all-or-nothing;
       the first request the destination cannot hold ends the round.  The paper re-evaluates the thresholds "in the
       next round"; evaluating them after every request is the same rule at the finest round length.
"""
from __future__ import annotations

import math
from dataclasses import dataclass


@dataclass
class Req:
    is_queuing: bool = False
    is_head_of_line: bool = False
    is_fake: bool = False
    priority: int = 0
    demand: float = 0.0
    physical_usage: float = 0.0


@dataclass
class Instance:
    M: float                                # total memory, in the unit of the usages (tokens or blocks)
    requests: list
    headroom_for_priority: list             # per priority class; 0 for the normal class
    is_terminating: bool = False


def num_requests(instance: Instance, p: int) -> int:
    return sum(1 for r in instance.requests if not r.is_queuing and not r.is_fake and r.priority == p)   # A29


def get_headroom(p: int, instance: Instance) -> float:                      # lines 9-10
    return instance.headroom_for_priority[p] / num_requests(instance, p)


def calc_virtual_usage(req: Req, instance: Instance) -> float:             # lines 1-8
    if req.is_queuing:
        if req.is_head_of_line:
            return req.demand
        return 0.0
    if req.is_fake:
        return math.inf
    return req.physical_usage + get_headroom(req.priority, instance)


def calc_freeness(instance: Instance):                                      # lines 11-18
    """-> (freeness, total virtual usage)"""
    requests = list(instance.requests)
    if instance.is_terminating:
        requests.append(Req(is_fake=True))
    total = 0.0
    for req in requests:
        total += calc_virtual_usage(req, instance)
    B = sum(1 for r in instance.requests if not r.is_queuing and not r.is_fake)
    if B == 0:
        B = 1                                                               # A28
    return (instance.M - total) / B, total


def pair_instances(freeness, src_below: float, dst_above: float):
    """list of (source index, destination index)."""
    src = sorted((i for i, f in enumerate(freeness) if f < src_below), key=lambda i: (freeness[i], i))
    dst = sorted((i for i, f in enumerate(freeness) if f > dst_above), key=lambda i: (-freeness[i], i))
    return list(zip(src, dst))


def migration_order(priority, seq_len):
    """request indices in the order the source llumlet offers them for migration."""
    return sorted(range(len(priority)), key=lambda i: (priority[i], seq_len[i], i))


def plan_migration_batch(instance: Instance, seq_len, block_tables, src_below: float, dst_mgr, dst_reserve_blocks: int = 0):
    """One migration round of one (source, destination) pair (reading A31).  `block_tables[r]` is request r's block
    table on the source (empty for queuing requests); `dst_mgr` is the destination's oracle.handshake.BlockManager.
    Returns (chosen request indices in the order taken, req_offsets, src_ids, dst_ids) — the arguments of
    oracle.kv_migration.migrate_batch.  The destination blocks are reserved in `dst_mgr`."""
    requests = list(instance.requests)
    remaining = list(range(len(requests)))                      # the requests the source still has
    order = migration_order([r.priority for r in requests], seq_len)
    chosen, req_offsets, src_ids, dst_ids = [], [0], [], []
    for r in order:
        if requests[r].is_queuing or requests[r].is_fake:
            continue                                            # no KV cache on this instance: nothing to migrate
        still_here = Instance(instance.M, [requests[i] for i in remaining], instance.headroom_for_priority,
                              instance.is_terminating)
        F, _ = calc_freeness(still_here)
        if not F < src_below:
            break                                               # "no longer set in the source state"
        table = [int(b) for b in block_tables[r]]
        if len(table) > dst_mgr.num_free() - dst_reserve_blocks:
            break                                               # PRE-ALLOC would fail: abort, the round ends
        ids = dst_mgr.allocate(len(table))                      # PRE-ALLOC, all or nothing
        chosen.append(r)
        src_ids += table
        dst_ids += ids
        req_offsets.append(len(src_ids))
        remaining.remove(r)
    return chosen, req_offsets, src_ids, dst_ids


# --------------------------------------------------------------------------
# Bandwidth budget of the non-final stages, chosen from the decode steps the engine observes
# ("nearly zero (up to 1%) overhead" on the co-running requests).
# The paper states the bound, not a mechanism — on its hardware the copy is too slow to matter.  Reading A34
# (DESIGN.md): a multiplicative feedback rule on medians of observed step times.
# --------------------------------------------------------------------------
def _median(xs):
    s = sorted(xs)
    n = len(s)
    return s[n // 2] if n % 2 else (s[n // 2 - 1] + s[n // 2]) / 2.0


class BudgetController:
    """budget <- clamp(budget * f, min, max) every `window` steps observed WITH a migration in flight, where
        s = median(those steps) / median(the last 2*window steps observed WITHOUT one) - 1     (the slowdown)
        f = 2                      if s <= target / 4      (cost within noise of zero: probe upwards)
            clamp(target / s, 1/2, 2)   otherwise
    Steps with a migration are dropped until at least one step without has been seen."""

    def __init__(self, target_pct: float, min_gbps: int, max_gbps: int, start_gbps: int, window: int):
        if not (target_pct > 0 and 1 <= min_gbps <= start_gbps <= max_gbps and 2 <= window <= 256):
            raise ValueError("bad arguments")
        self.target = target_pct / 100.0
        self.lo, self.hi, self.window = float(min_gbps), float(max_gbps), window
        self.budget = float(start_gbps)
        self.base, self.mig = [], []
        self.last_slowdown_pct = math.nan
        self.adjustments = 0

    def gbps(self) -> int:
        return int(math.floor(self.budget + 0.5))

    def observe(self, step_ms: float, migrating: bool) -> int:
        if not (step_ms > 0 and math.isfinite(step_ms)):
            raise ValueError("step_ms")
        if not migrating:
            self.base.append(step_ms)
            if len(self.base) > 2 * self.window:
                self.base.pop(0)
            return self.gbps()
        if not self.base:
            return self.gbps()
        self.mig.append(step_ms)
        if len(self.mig) >= self.window:
            s = _median(self.mig) / _median(self.base) - 1.0
            f = 2.0 if s <= self.target / 4.0 else min(2.0, max(0.5, self.target / s))
            self.budget = min(self.hi, max(self.lo, self.budget * f))
            self.last_slowdown_pct = 100.0 * s
            self.adjustments += 1
            self.mig = []
        return self.gbps()
