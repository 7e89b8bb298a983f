"""Pins for oracle/handshake.py (Figure 7) and the C++ coordinator against it.  CPU only:
the coordinator runs without pools (no copy is enqueued), so the whole handshake is host logic."""
import itertools
import os

import numpy as np
import pytest

from oracle import handshake as oh
from oracle import kv_migration as om

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def golden_sequence():
    return [l.strip() for l in open(os.path.join(GOLD, "paper_handshake_fig7.txt")) if l.strip() and not l.startswith("#")]


def kinds(log):
    return [m[0] if m[0] != "COPY" else f"COPY {m[3]}" for m in log]


def fresh(nb_src=40, nb_dst=40, req_blocks=9):
    src, dst = oh.BlockManager(nb_src), oh.BlockManager(nb_dst)
    table = src.allocate(req_blocks)
    return src, dst, table


# ---- the paper's narrated two-stage sequence ---------------------------------------------------
def test_two_stage_message_sequence_matches_the_paper():
    S = 4
    src, dst, table = fresh(req_blocks=8)                # room for 32 tokens
    mig = oh.run_script(src, dst, table, S, 1, 30, [dict(append=1), dict(), dict()])   # 30 -> 31 tokens
    assert mig.state == oh.COMMITTED
    assert kinds(mig.log) == golden_sequence()
    # stage 0 took the 7 full blocks of 30 tokens; the final stage the block that was being appended to
    assert [m for m in mig.log if m[0] == "COPY"] == [("COPY", 0, 7, "stage"), ("COPY", 7, 8, "final")]


def test_final_only_when_few_blocks_remain():
    src, dst, table = fresh(req_blocks=2)
    mig = oh.run_script(src, dst, table, 4, 2, 7, [dict(), dict()])
    assert kinds(mig.log) == ["PRE_ALLOC", "OK", "COPY final", "RELEASE_SRC", "COMMIT"]


# ---- conservation and the commit bookkeeping in closed form -------------------------------------
@pytest.mark.parametrize("start,appends,S,last", [(30, (3,), 4, 1), (97, (3,), 16, 2), (2032, (8,), 16, 2), (5, (), 4, 2)])
def test_commit_bookkeeping_closed_form(start, appends, S, last):
    total_tokens = start + sum(appends)
    nblk = -(-total_tokens // S)
    src, dst = oh.BlockManager(nblk + 50), oh.BlockManager(nblk + 7)
    table = src.allocate(nblk)
    f_src, f_dst = src.num_free(), dst.num_free()
    script = [dict(append=a) for a in appends] + [dict()] * 4
    mig = oh.run_script(src, dst, table, S, last, start, script)
    assert mig.state == oh.COMMITTED and mig.final_tokens == total_tokens
    assert mig.blocks_migrated == nblk
    assert src.num_free() == f_src + nblk            # "the source releases its local blocks"
    assert dst.num_free() == f_dst - nblk            # the destination keeps what it reserved
    assert len(set(mig.dst_table)) == nblk and all(not dst.is_free[b] for b in mig.dst_table)
    assert all(src.is_free[b] for b in table)


# ---- every abort point: no leak on the destination, source untouched -----------------------------
def all_scripts(rounds):
    opts = [dict(), dict(status=oh.FINISHED), dict(status=oh.PREEMPTED), dict(status=oh.PEER_FAILED), dict(dst_takes=100)]
    for combo in itertools.product(range(len(opts)), repeat=rounds):
        yield [dict(opts[c], append=2) for c in combo]


def test_every_abort_point_is_leak_free():
    S, last = 4, 1
    n_commit = n_abort = 0
    for script in all_scripts(4):
        src, dst, table = fresh(nb_src=30, nb_dst=12, req_blocks=10)
        f_src, f_dst = src.num_free(), dst.num_free()
        mig = oh.run_script(src, dst, table, S, last, 26, script)
        held = len(mig.taken_by_dst)
        if mig.state == oh.ABORTED:
            n_abort += 1
            assert dst.num_free() == f_dst - held, (script, mig.log)       # everything reserved was given back (A25)
            assert src.num_free() == f_src and not any(src.is_free[b] for b in table)
            assert mig.dst_table == [] and mig.log[-1][0] == "ABORT"
        elif mig.state == oh.COMMITTED:
            n_commit += 1
            assert dst.num_free() == f_dst - held - mig.blocks_migrated
            assert src.num_free() == f_src + mig.blocks_migrated
        # conservation on both sides at the end
        assert sum(dst.is_free) == dst.num_free() and sum(src.is_free) == src.num_free()
    assert n_commit > 0 and n_abort > 0


def test_abort_reasons_and_no_space_is_all_or_nothing():
    src, dst, table = fresh(nb_dst=5, req_blocks=9)
    mig = oh.Migration(src, dst, 4, 1)
    assert mig.stage(30) is None and mig.state == oh.ABORTED and mig.abort_reason == "no_space"
    assert dst.num_free() == 5                                   # A24: nothing was reserved
    assert mig.log == [("PRE_ALLOC", 7), ("ABORT", "no_space")]
    with pytest.raises(RuntimeError):
        mig.stage(30)


def test_block_manager_policy_A23():
    m = oh.BlockManager(6)
    assert m.allocate(3) == [0, 1, 2] and m.allocate(0) == []
    m.release([1, 0])
    assert m.allocate(3) == [0, 1, 3]                            # last released first, then the untouched ones
    assert m.allocate(3) is None and m.num_free() == 2
    with pytest.raises(ValueError):
        m.release([4])                                           # still free
    with pytest.raises(ValueError):
        m.release([0, 0])
    with pytest.raises(IndexError):
        m.release([6])


# ---- the C++ coordinator (libllx.so, no device needed) against the oracle --------------------------
@pytest.fixture(scope="module")
def llx():
    from paper_2406_03243_b200 import build
    build.build()
    import paper_2406_03243_b200 as m
    m.load()
    return m


STATUS = {oh.RUNNING: 0, oh.FINISHED: 1, oh.PREEMPTED: 2, oh.PEER_FAILED: 3}
STATE = {oh.READY: 0, oh.COPYING: 1, oh.FINAL_COPYING: 2, oh.COMMITTED: 3, oh.ABORTED: 4}
REASON = {None: 0, oh.FINISHED: 1, oh.PREEMPTED: 2, oh.PEER_FAILED: 3, "no_space": 4}


def drive_c(llx, nb_src, nb_dst, req_blocks, S, last, start_tokens, script):
    """The same script as oracle.handshake.run_script, through the C ABI."""
    src, dst = llx.BlockManager(nb_src), llx.BlockManager(nb_dst)
    table = src.alloc(req_blocks)
    mig = llx.Migration(None, src, None, dst, S, last)
    tokens, taken, trace, dst_table = start_tokens, [], [], None
    for rnd in script:
        j = rnd.get("dst_takes", 0)
        if j:
            try:
                taken += list(dst.alloc(j))
            except llx.LlxError as e:
                assert e.name == "LLX_ERR_NO_SPACE"
        st = STATUS[rnd.get("status", oh.RUNNING)]
        if mig.state == llx.MIG_FINAL_COPYING:
            dst_table = mig.commit(table[:-(-tokens // S)], st)
        else:
            n, fin, ids = mig.stage(table, tokens, st)
            if mig.state != llx.MIG_ABORTED:
                trace.append((n, fin, list(ids)))
                if not fin:
                    tokens += rnd.get("append", 0)
        if mig.state in (llx.MIG_COMMITTED, llx.MIG_ABORTED):
            break
    return dict(state=mig.state, reason=mig.abort_reason, migrated=mig.blocks_migrated, stages=mig.stages,
                src_free=src.num_free, dst_free=dst.num_free, trace=trace, dst_table=None if dst_table is None else list(dst_table),
                tokens=tokens, src=src, dst=dst, table=table)


def test_coordinator_matches_oracle_on_every_script(llx):
    S, last = 4, 1
    for script in all_scripts(4):
        o_src, o_dst, o_table = fresh(nb_src=30, nb_dst=12, req_blocks=10)
        o = oh.run_script(o_src, o_dst, o_table, S, last, 26, script)
        c = drive_c(llx, 30, 12, 10, S, last, 26, script)
        assert c["state"] == STATE[o.state], (script, o.log)
        assert c["reason"] == REASON[o.abort_reason]
        assert c["migrated"] == o.blocks_migrated and c["tokens"] == o.final_tokens
        assert c["src_free"] == o_src.num_free() and c["dst_free"] == o_dst.num_free()
        o_copies = [m for m in o.log if m[0] == "COPY"]
        assert [(m[2] - m[1], m[3] == "final") for m in o_copies] == [(n, f) for n, f, _ in c["trace"]]
        assert c["stages"] == len(o_copies)
        if o.state == oh.COMMITTED:
            assert c["dst_table"] == o.dst_table           # same free-list policy (A23) => same ids


def test_coordinator_matches_oracle_on_seeded_random_scripts(llx):
    rng = np.random.default_rng(7)
    for case in range(300):
        S = int(rng.choice([1, 4, 16]))
        last = int(rng.integers(1, 4))
        start = int(rng.integers(1, 40 * S))
        rounds = int(rng.integers(1, 6))
        script = []
        for _ in range(rounds + 2):
            r = dict(append=int(rng.integers(0, 3 * S)))
            u = rng.random()
            if u < 0.08:
                r["status"] = [oh.FINISHED, oh.PREEMPTED, oh.PEER_FAILED][int(rng.integers(0, 3))]
            elif u < 0.2:
                r["dst_takes"] = int(rng.integers(1, 30))
            script.append(r)
        req_blocks = -(-(start + sum(r["append"] for r in script)) // S)
        nb_src, nb_dst = req_blocks + int(rng.integers(0, 5)), int(rng.integers(1, req_blocks + 20))
        o_src, o_dst = oh.BlockManager(nb_src), oh.BlockManager(nb_dst)
        o_table = o_src.allocate(req_blocks)
        o = oh.run_script(o_src, o_dst, o_table, S, last, start, script)
        c = drive_c(llx, nb_src, nb_dst, req_blocks, S, last, start, script)
        assert (c["state"], c["reason"], c["migrated"], c["tokens"]) == \
            (STATE[o.state], REASON[o.abort_reason], o.blocks_migrated, o.final_tokens), (case, script, o.log)
        assert c["src_free"] == o_src.num_free() and c["dst_free"] == o_dst.num_free()
        if o.state == oh.COMMITTED:
            assert c["dst_table"] == o.dst_table
            assert len(set(c["dst_table"])) == len(c["dst_table"]) == -(-c["tokens"] // S)


def test_coordinator_block_manager_and_state_errors(llx):
    m = llx.BlockManager(6)
    assert list(m.alloc(3)) == [0, 1, 2] and m.num_free == 3 and m.num_blocks == 6
    m.release([1, 0])
    assert list(m.alloc(3)) == [0, 1, 3]
    with pytest.raises(llx.LlxError) as e:
        m.alloc(3)
    assert e.value.name == "LLX_ERR_NO_SPACE" and m.num_free == 2
    for bad, name in (([4], "LLX_ERR_INVALID_ARG"), ([0, 0], "LLX_ERR_INVALID_ARG"), ([6], "LLX_ERR_BLOCK_OUT_OF_RANGE")):
        free = m.num_free
        with pytest.raises(llx.LlxError) as e:
            m.release(bad)
        assert e.value.name == name and m.num_free == free      # a failed release changes nothing
    a, b = llx.BlockManager(8), llx.BlockManager(8)
    t = a.alloc(3)
    with pytest.raises(llx.LlxError) as e:
        llx.Migration(None, a, None, a, 4, 1)
    assert e.value.name == "LLX_ERR_ALIAS"
    g = llx.Migration(None, a, None, b, 4, 1)
    with pytest.raises(llx.LlxError) as e:
        g.commit(t)                                              # no final stage yet
    assert e.value.name == "LLX_ERR_STATE"
    with pytest.raises(llx.LlxError):
        g.stage(t[:1], 12)                                       # table too short for the stage
    assert b.num_free == 8 and g.state == llx.MIG_READY
    g.stage(t, 12)
    assert g.state == llx.MIG_FINAL_COPYING or g.state == llx.MIG_COPYING
    g.abort(llx.ABORT_PEER_FAILED)
    assert g.state == llx.MIG_ABORTED and b.num_free == 8
    with pytest.raises(llx.LlxError) as e:
        g.abort()
    assert e.value.name == "LLX_ERR_STATE"
    g2 = llx.Migration(None, a, None, b, 4, 1)
    g2.stage(t, 12)
    del g2                                                       # destroying an open session releases its reservation
    import gc
    gc.collect()
    assert b.num_free == 8
