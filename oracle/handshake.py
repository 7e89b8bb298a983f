"""Oracle: the migration handshake of Llumnix §4.2 (Figure 7) and the block
reservation it drives.  TEST INFRASTRUCTURE ONLY — plain Python, one statement per sentence
of the paper, no cleverness.  Shares no code with the C++ coordinator in
paper_2406_03243_b200/csrc/llx_coord.cu.

The passage, sentence by sentence, and where it lives below:

  (a) "Before each stage, the source instance issues a pre-allocate request with the number
      of blocks to migrate"                                              -> msg PRE_ALLOC(n)
  (b) "The destination will try to allocate and reserve the blocks; if it succeeds or fails,
      the destination will notify the source to proceed or abort the migration and clean
      the states, respectively."                                          -> msg OK | ABORT(no_space)
  (c) "after each stage, the source instance also checks whether the request being migrated
      has completed or been preempted — if it has, the source will notify the destination to
      abort and release the reserved blocks; otherwise the source will go ahead to the next
      stage."                                                             -> msg ABORT(finished|preempted)
  (d) "The source or destination will also abort the migration if the other side fails."
                                                                          -> msg ABORT(peer_failed)
  (e) "After the final stage finishes, the source releases its local blocks and notifies the
      destination to commit the migration and resume the execution of the request."
                                                                          -> msg RELEASE_SRC, COMMIT

Which blocks a stage takes is §4.2's stage rule, i.e. oracle.kv_migration.plan_stage.

Readings where the paper is silent (A23-A26):
  A23  free-list policy of an instance's block manager: a stack; a fresh manager hands out
       0,1,2,...; released ids are pushed in the order given and handed out again last-in-first-out.
  A24  pre-allocation is all-or-nothing: a failed PRE_ALLOC reserves nothing.
  A25  "clean the states": every block the destination reserved for THIS migration (all earlier
       stages included) goes back to its free list; the source keeps its blocks and the request
       keeps running there (or is already gone, in case (c)).  No bytes are rolled back.
  A26  the check of (c) also runs before the first stage and once more after the final copy,
       before the source releases its blocks: a request that finished during the final copy is
       aborted, not committed.

Pins (tests/test_oracle_handshake.py): the message sequence the paper narrates for the normal
two-stage case (tests/golden/paper_handshake_fig7.txt), block conservation at every step, leak
freedom after every abort point, the commit bookkeeping in closed form, exhaustive enumeration of
all abort points on small cases.
"""
from __future__ import annotations

from oracle.kv_migration import plan_stage

RUNNING, FINISHED, PREEMPTED, PEER_FAILED = "running", "finished", "preempted", "peer_failed"
READY, COPYING, FINAL_COPYING, COMMITTED, ABORTED = "ready", "copying", "final_copying", "committed", "aborted"


class BlockManager:
    """One instance's free list (reading A23)."""

    def __init__(self, num_blocks: int):
        self.num_blocks = num_blocks
        self.free = list(range(num_blocks - 1, -1, -1))     # a stack whose pops give 0, 1, 2, ...
        self.is_free = [True] * num_blocks

    def num_free(self) -> int:
        return len(self.free)

    def allocate(self, n: int):
        """All-or-nothing (A24): n ids, or None when fewer than n blocks are free."""
        if n < 0:
            raise ValueError("n < 0")
        if n > len(self.free):
            return None
        ids = [self.free.pop() for _ in range(n)]
        for b in ids:
            self.is_free[b] = False
        return ids

    def release(self, ids) -> None:
        ids = [int(b) for b in ids]
        for b in ids:
            if b < 0 or b >= self.num_blocks:
                raise IndexError("block id out of range")
        if len(set(ids)) != len(ids) or any(self.is_free[b] for b in ids):
            raise ValueError("double free")
        for b in ids:
            self.is_free[b] = True
            self.free.append(b)


class Migration:
    """The source-side driver of one request's migration; `log` is the message trace."""

    def __init__(self, src_mgr: BlockManager, dst_mgr: BlockManager, block_size: int, last_stage_max_blocks: int):
        self.src_mgr, self.dst_mgr = src_mgr, dst_mgr
        self.S, self.last = block_size, last_stage_max_blocks
        self.state = READY
        self.blocks_migrated = 0
        self.dst_table: list[int] = []          # blocks reserved on the destination so far, in logical order
        self.abort_reason = None
        self.log: list[tuple] = []

    def _abort(self, reason: str) -> None:
        # (b)/(c)/(d) + A25: release everything reserved for this migration; source untouched
        self.log.append(("ABORT", reason))
        self.dst_mgr.release(self.dst_table)
        self.dst_table = []
        self.abort_reason = reason
        self.state = ABORTED

    def stage(self, num_tokens: int, status: str = RUNNING):
        """One round: check (c)/(d), plan, PRE_ALLOC (a)/(b); returns
        (n, is_final, logical_range, dst_ids) of the copy to perform, or None after an abort."""
        if self.state not in (READY, COPYING):
            raise RuntimeError(f"stage() in state {self.state}")
        if status != RUNNING:
            self._abort(status)
            return None
        n, is_final = plan_stage(num_tokens, self.blocks_migrated, self.S, self.last)
        self.log.append(("PRE_ALLOC", n))
        ids = self.dst_mgr.allocate(n)
        if ids is None:
            self._abort("no_space")
            return None
        self.log.append(("OK",))
        lo = self.blocks_migrated
        self.dst_table += ids
        self.blocks_migrated += n
        self.state = FINAL_COPYING if is_final else COPYING
        self.log.append(("COPY", lo, lo + n, "final" if is_final else "stage"))
        return n, is_final, (lo, lo + n), ids

    def commit(self, src_table, status: str = RUNNING):
        """(e): after the final copy.  Returns the destination block table, or None after an abort (A26)."""
        if self.state != FINAL_COPYING:
            raise RuntimeError(f"commit() in state {self.state}")
        if status != RUNNING:
            self._abort(status)
            return None
        src_table = [int(b) for b in src_table]
        if len(src_table) != self.blocks_migrated:
            raise ValueError("source block table does not match the blocks migrated")
        self.log.append(("RELEASE_SRC", len(src_table)))
        self.src_mgr.release(src_table)
        self.log.append(("COMMIT",))
        self.state = COMMITTED
        return list(self.dst_table)

    def abort(self, reason: str = PEER_FAILED) -> None:
        """(d): either side may abort at any time before the commit."""
        if self.state in (COMMITTED, ABORTED):
            raise RuntimeError(f"abort() in state {self.state}")
        self._abort(reason)


def run_script(src_mgr, dst_mgr, src_table, block_size, last_stage_max_blocks, start_tokens, script):
    """Drive one migration from a script of what happens around it.  `script` is a list of per-round
    dicts, consumed one per stage() / commit() call:
        {"status": RUNNING|FINISHED|PREEMPTED|PEER_FAILED,   # what the source sees at this check
         "append": k,                                         # tokens decoded during this stage's copy
         "dst_takes": j}                                      # blocks the destination's own requests grab first
    The request's source blocks `src_table` cover ceil(tokens/S) blocks at any time (the caller pre-reserved
    them, as the block manager of the engine does when a token spills into a new block).
    Returns the Migration (state, log, dst_table) — the source table is released on commit."""
    mig = Migration(src_mgr, dst_mgr, block_size, last_stage_max_blocks)
    tokens = start_tokens
    taken_by_dst: list[int] = []
    for rnd in script:
        j = rnd.get("dst_takes", 0)
        if j:
            got = dst_mgr.allocate(j)
            if got is not None:
                taken_by_dst += got
        status = rnd.get("status", RUNNING)
        if mig.state == FINAL_COPYING:
            total = -(-tokens // block_size)
            mig.commit(src_table[:total], status)
        else:
            r = mig.stage(tokens, status)
            if r is not None and not r[1]:
                tokens += rnd.get("append", 0)
        if mig.state in (COMMITTED, ABORTED):
            break
    mig.final_tokens = tokens
    mig.taken_by_dst = taken_by_dst
    return mig
