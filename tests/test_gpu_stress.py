"""A short soak: three host threads on their own streams issue a random mix of migration calls (all entry points,
a random launch policy PER CALL — llx_launch_opts — so the threads run different launch shapes side by side) for a few
seconds; after every call the touched destination blocks must equal their source blocks (torch gather on the device,
independent of the library).  90 s of the same loop (88,000 calls) ran clean on a B200 while this was written."""
import os
import threading
import time

import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu

NB = 3000
SECONDS = float(os.environ.get("LLX_STRESS_SECONDS", "4"))        # per geometry; a longer soak: LLX_STRESS_SECONDS=120 python -m pytest tests/test_gpu_stress.py -m gpu


@pytest.mark.parametrize("heads", [8, 13])                         # 32 KiB tiles (3 x 32 KiB ring) and 52 KiB tiles (equal chunks of 13 KiB, 6 stages)
def test_random_mix_of_calls_from_three_threads(heads):
    import paper_2406_03243_b200 as llx
    llx.load()
    G = dict(layers=4, kv_heads=heads, head_dim=128, block_size=16)
    te = G["block_size"] * G["kv_heads"] * G["head_dim"]

    def pool():
        nbytes = llx.pool_bytes_for(G["layers"], G["kv_heads"], G["head_dim"], G["block_size"], llx.F16, NB)
        raw = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
        return raw, llx.pool_wrap(raw.data_ptr(), nbytes, G["layers"], G["kv_heads"], G["head_dim"], G["block_size"],
                                  llx.F16, NB, keepalive=raw)

    src_raw, src = pool()
    src_raw.view(torch.int16).copy_(torch.randint(-30000, 30000, (src_raw.numel() // 2,), dtype=torch.int16, device="cuda"))
    sv = src_raw.view(torch.int16).view(G["layers"], 2, NB, te)
    torch.cuda.synchronize()
    errors, counts = [], []
    t_end = time.time() + SECONDS

    def worker(tid):
        try:
            torch.cuda.set_device(0)
            rng = np.random.default_rng(tid)
            st = torch.cuda.Stream()
            dst_raw, dst = pool()
            dv = dst_raw.view(torch.int16).view(G["layers"], 2, NB, te)
            pin = llx.PinnedStaging(llx.staging_bytes(src, 300))
            it = 0
            while time.time() < t_end:
                it += 1
                n = int(rng.choice([1, 2, 7, 40, 255, 256, 257, 300, 700, 1500]))
                s_ids = rng.permutation(NB)[:n].astype(np.int32)
                d_ids = rng.permutation(NB)[:n].astype(np.int32)
                kind = int(rng.integers(0, 6))
                opts = [None, dict(), dict(copy_kernel=1), dict(dynamic_tail_pct=30), dict(max_ctas=int(rng.integers(1, 400))),
                        dict(exact_residency=0), dict(bandwidth_gbps=int(rng.integers(2000, 6000))),
                        dict(route=llx.ROUTE_PEER), dict(overlap_prev=1), dict(overlap_prev=1, dynamic_tail_pct=30)][int(rng.integers(0, 10))]
                overlap = bool(opts) and opts.get("overlap_prev") == 1
                if kind <= 2 and overlap and n >= 2:
                    # two stages over disjoint halves, the second one allowed to start while the first drains
                    h = n // 2
                    llx.migrate_stage(src, s_ids[:h], dst, d_ids[:h], stream=st, opts=opts)
                    llx.migrate_stage(src, s_ids[h:], dst, d_ids[h:], stream=st, opts=opts)
                elif kind <= 2:
                    llx.migrate_stage(src, s_ids, dst, d_ids, stream=st, opts=opts)
                elif kind == 3:
                    llx.migrate_stage_wait(src, s_ids, dst, d_ids, stream=st, opts=opts)
                else:
                    n = min(n, 300)
                    s_ids, d_ids = s_ids[:n], d_ids[:n]
                    if kind == 4:
                        llx.migrate_via_host(src, s_ids, dst, d_ids, pin.dev_alias, pin.nbytes,
                                             chunk_blocks=int(rng.integers(0, 60)), stream=st, opts=opts)
                    else:
                        llx.pack(src, s_ids, pin.dev_alias, pin.nbytes, stream=st, opts=opts)
                        # unpack READS what pack wrote: never declared independent of it
                        llx.unpack(pin.dev_alias, pin.nbytes, dst, d_ids, stream=st, opts=None if overlap else opts)
                st.synchronize()
                si = torch.from_numpy(s_ids.astype(np.int64)).cuda()
                di = torch.from_numpy(d_ids.astype(np.int64)).cuda()
                for l in range(G["layers"]):
                    for kv in range(2):
                        if not torch.equal(dv[l, kv].index_select(0, di), sv[l, kv].index_select(0, si)):
                            errors.append((tid, it, kind, n, opts, l, kv))
                            return
            counts.append(it)
            pin.free()
        except Exception as e:  # noqa: BLE001
            errors.append((tid, repr(e)))

    ts = [threading.Thread(target=worker, args=(i,)) for i in range(3)]
    for t in ts:
        t.start()
    for t in ts:
        t.join()
    assert not errors, errors
    assert len(counts) == 3 and min(counts) > 20
    # per-call policies leave the process defaults alone
    assert [llx.get_option(o) for o in (llx.OPT_COPY_KERNEL, llx.OPT_MAX_CTAS, llx.OPT_DYNAMIC_TAIL_PCT, llx.OPT_EXACT_RESIDENCY,
                                        llx.OPT_BANDWIDTH_GBPS)] == [0, 0, 6, 1, 0]
