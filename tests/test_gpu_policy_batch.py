"""SURVEY NEXT-4 wired to the hot path: Algorithm 1 and the pairing rule decide WHICH
requests move between WHICH instances, llx_plan_migration_batch turns that into the argument list of llx_migrate_batch
(PRE-ALLOC on the destination's block manager), and ONE launch per (source, destination) pair moves the
bytes.  The same round is played by the oracle (oracle.policy + oracle.handshake.BlockManager +
oracle.kv_migration.migrate_batch); decisions, block ids and every byte of every pool must agree."""
import numpy as np
import pytest
import torch

import synth
from oracle import handshake as oh
from oracle import kv_migration as om
from oracle import policy as op

pytestmark = pytest.mark.gpu

SENT = synth.SENTINEL_U16
G = dict(layers=3, kv_heads=4, head_dim=64, block_size=16, elem_bytes=2, num_blocks=160)     # 8 KiB tiles
HEADROOM = [0.0, 30.0]          # blocks; priority 1 = high
SRC_BELOW, DST_ABOVE = 4.0, 12.0


@pytest.fixture(scope="module")
def env():
    import gpu_harness as H
    import paper_2406_03243_b200 as llx
    llx.load()
    return H, llx


def as_tuple(r: op.Req):
    return (r.is_queuing, r.is_head_of_line, r.is_fake, r.priority, r.demand, r.physical_usage)


def seeded_cluster(seed, K, nb):
    """K instances with seeded running / queuing / high-priority requests.  Usage unit: blocks.  The load is skewed on
    purpose (even instances heavy, odd ones light) so that both candidate sets of PAPER.md:225 are non-empty."""
    rng = np.random.default_rng(seed)
    cluster = []
    for k in range(K):
        heavy = k % 2 == 0
        o_mgr = oh.BlockManager(nb)
        reqs, seq, tables = [], [], []
        for _ in range(int(rng.integers(7, 11)) if heavy else int(rng.integers(1, 3))):
            nblk = int(rng.integers(4, 22)) if heavy else int(rng.integers(2, 8))
            t = o_mgr.allocate(nblk)
            if t is None:
                break
            reqs.append(op.Req(priority=int(rng.random() < 0.25), physical_usage=float(nblk)))
            seq.append(int(rng.integers((nblk - 1) * 16 + 1, nblk * 16 + 1)))
            tables.append(t)
        if heavy:                                        # a queue behind a full instance (Fig. 9b)
            reqs.append(op.Req(is_queuing=True, is_head_of_line=True, demand=float(rng.integers(10, 40))))
            seq.append(int(rng.integers(100, 600)))
            tables.append([])
            reqs.append(op.Req(is_queuing=True, demand=float(rng.integers(10, 40))))
            seq.append(int(rng.integers(100, 600)))
            tables.append([])
        cluster.append(dict(reqs=reqs, seq=seq, tables=tables, o_mgr=o_mgr))
    return cluster


@pytest.mark.parametrize("seed,K,terminating", [(0, 4, None), (1, 6, None), (2, 5, 3), (3, 4, 0)])
def test_policy_output_feeds_one_batch_launch_per_pair(env, seed, K, terminating):
    H, llx = env
    nb, te = G["num_blocks"], H.tile_elems(G)
    cluster = seeded_cluster(seed, K, nb)
    # every instance: a device pool with its own seeded content + an llx block manager in the same state as the oracle's
    for k, inst in enumerate(cluster):
        inst["pool"] = H.DevPool(G)
        inst["pool"].fill_from_synth(100 + seed, k)
        inst["h_pool"] = H.host_pool_from_synth(G, 100 + seed, k)
        inst["mgr"] = llx.BlockManager(nb)
        used = nb - inst["o_mgr"].num_free()
        assert list(inst["mgr"].alloc(used)) == list(range(used))                   # A23: both hand out 0, 1, 2, ...
        inst["term"] = terminating == k
    M = float(nb)

    # ---- Algorithm 1 per instance, both sides
    F_c, F_o = [], []
    for inst in cluster:
        f, _ = llx.calc_freeness([as_tuple(r) for r in inst["reqs"]], M, HEADROOM, inst["term"])
        fo, _ = op.calc_freeness(op.Instance(M=M, requests=inst["reqs"], headroom_for_priority=HEADROOM, is_terminating=inst["term"]))
        F_c.append(f)
        F_o.append(fo)
    assert F_c == F_o
    # ---- pairing
    pairs = llx.pair_instances(F_c, SRC_BELOW, DST_ABOVE)
    assert pairs == op.pair_instances(F_o, SRC_BELOW, DST_ABOVE) and len(pairs) >= 1

    # ---- per pair: plan the round, PRE-ALLOC on the destination, ONE llx_migrate_batch launch on the pair's stream
    streams = [torch.cuda.Stream() for _ in pairs]
    for st in streams:
        st.wait_stream(torch.cuda.current_stream())
    moved_pairs, launches0 = 0, llx.counters()["copy_launches"]
    plans = []
    for (s, d), st in zip(pairs, streams):
        src, dst = cluster[s], cluster[d]
        chosen, off, s_ids, d_ids = llx.plan_migration_batch([as_tuple(r) for r in src["reqs"]], src["seq"], M, HEADROOM, SRC_BELOW,
                                                             src["tables"], dst["mgr"], dst_reserve_blocks=8, is_terminating=src["term"])
        o_plan = op.plan_migration_batch(op.Instance(M=M, requests=src["reqs"], headroom_for_priority=HEADROOM, is_terminating=src["term"]),
                                         src["seq"], src["tables"], SRC_BELOW, dst["o_mgr"], dst_reserve_blocks=8)
        assert (chosen, list(off), list(s_ids), list(d_ids)) == (o_plan[0], o_plan[1], o_plan[2], o_plan[3]), (s, d)
        assert dst["mgr"].num_free == dst["o_mgr"].num_free()
        llx.migrate_batch(src["pool"].pool, dst["pool"].pool, off, s_ids, d_ids, stream=st)
        om.migrate_batch(src["h_pool"], dst["h_pool"], o_plan[1], o_plan[2], o_plan[3])
        moved_pairs += len(s_ids)
        plans.append((s, d, chosen, s_ids, d_ids))
    assert llx.counters()["copy_launches"] - launches0 == sum(1 for p in plans if len(p[3]))      # one launch per pair
    assert moved_pairs > 0
    torch.cuda.synchronize()

    # ---- commit: the source releases the blocks of the requests that left, both sides
    for s, d, chosen, s_ids, d_ids in plans:
        if len(s_ids):
            cluster[s]["mgr"].release(s_ids)
            cluster[s]["o_mgr"].release(list(s_ids))
        assert cluster[s]["mgr"].num_free == cluster[s]["o_mgr"].num_free()
        # the moved requests' KV on the destination equals what they had on the source, request by request
        p = 0
        for r in chosen:
            n = len(cluster[s]["tables"][r])
            got = cluster[d]["pool"].host()[:, :, d_ids[p:p + n]]
            assert np.array_equal(got, cluster[s]["h_pool"][:, :, cluster[s]["tables"][r]])
            p += n
    # ---- every byte of every pool (destinations received exactly the oracle's blocks, nothing else changed anywhere)
    for inst in cluster:
        H.assert_pool_equal(inst["pool"].host(), inst["h_pool"])


def test_plan_with_a_full_destination_moves_nothing_and_launches_nothing(env):
    H, llx = env
    nb = G["num_blocks"]
    src, dst = H.DevPool(G), H.DevPool(G, fill=SENT)
    src.fill_from_synth(7, 0)
    dst_mgr = llx.BlockManager(nb)
    dst_mgr.alloc(nb - 3)
    reqs = [(0, 0, 0, 0, 0.0, 10.0), (0, 0, 0, 0, 0.0, 6.0)]
    launches = llx.counters()["kernel_launches"]
    chosen, off, s_ids, d_ids = llx.plan_migration_batch(reqs, [150, 90], 10.0, [0.0], 5.0, [list(range(10)), list(range(10, 16))], dst_mgr)
    assert chosen == [] and list(off) == [0] and dst_mgr.num_free == 3
    llx.migrate_batch(src.pool, dst.pool, off, s_ids, d_ids)
    torch.cuda.synchronize()
    assert llx.counters()["kernel_launches"] == launches
    assert bool((dst.view == int(np.array(SENT, np.uint16).view(np.int16))).all())
