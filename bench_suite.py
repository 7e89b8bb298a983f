"""The other BASELINE.json configs, measured through the C-ABI: configs[2] length sweep, configs[3] 30B batch,
configs[4] interference with a decode step + staging through pinned host memory, plus the NEXT-row measurements
(bandwidth budget, live migration during decode, TP-rank sharded tiles, peer route).  A measuring harness beside
bench.py, not part of the library: `bench.py --suite` calls run(); `python bench_suite.py --only NAME` runs one leg.

Everything here is measurement harness: pools are torch allocations (memory + streams only), inputs come
from `synth`, all timing is CUDA events on the launching stream (or host wall clock where stated)."""
from __future__ import annotations

import gc
import statistics
import time

import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import synth  # noqa: E402

SENT_I16 = int(np.array(synth.SENTINEL_U16, np.uint16).view(np.int16))


def _events(torch, n):
    return [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n)]


def _time_stream(torch, stream, fn, reps=10, warm=2, before=None):
    for _ in range(warm):
        fn()
    stream.synchronize()
    evs = _events(torch, reps)
    for a, b in evs:
        if before is not None:
            before()
        a.record(stream)
        fn()
        b.record(stream)
    stream.synchronize()
    ts = sorted(a.elapsed_time(b) for a, b in evs)
    return {"median_ms": statistics.median(ts), "min_ms": ts[0]}


def _in_thread(torch, fn):
    """Runs `fn` (the migration's enqueue) on its own host thread, as a serving engine's migration thread would: a
    budgeted stage is a chain of launches, and enqueueing it from the thread that launches the decode step would put its
    host time inside the decode step's measured interval.  Returns after the thread has started; join() the result."""
    import threading
    dev = torch.cuda.current_device()
    started = threading.Event()

    def run():
        torch.cuda.set_device(dev)
        started.set()
        fn()
    th = threading.Thread(target=run)
    th.start()
    started.wait()
    return th


def _free(torch):
    gc.collect()
    torch.cuda.empty_cache()
    return torch.cuda.mem_get_info()[0]


class Pools:
    def __init__(self, torch, llx, g, nb_src, nb_dst, fill_src=True):
        self.torch, self.llx, self.g = torch, llx, dict(g)
        self.src_raw, self.src = self._pool(nb_src)
        self.dst_raw, self.dst = self._pool(nb_dst)
        if fill_src:
            gen = torch.Generator(device="cuda")
            gen.manual_seed(0)
            flat = self.src_raw.view(torch.float16)
            step = 1 << 28
            for a in range(0, flat.numel(), step):
                b = min(flat.numel(), a + step)
                flat[a:b] = (torch.rand(b - a, generator=gen, device="cuda", dtype=torch.float32) * 2 - 1).half()
        self.dst_raw.view(torch.int16).fill_(SENT_I16)
        torch.cuda.synchronize()

    def _pool(self, nb):
        g, torch, llx = self.g, self.torch, self.llx
        nbytes = llx.pool_bytes_for(g["layers"], g["kv_heads"], g["head_dim"], g["block_size"], llx.F16, nb)
        raw = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
        return raw, llx.pool_wrap(raw.data_ptr(), nbytes, g["layers"], g["kv_heads"], g["head_dim"], g["block_size"],
                                  llx.F16, nb, keepalive=raw)

    def view(self, raw, nb):
        g = self.g
        return raw.view(self.torch.int16).view(g["layers"], 2, nb, g["block_size"] * g["kv_heads"] * g["head_dim"])


# ---- configs[2]: length sweep ------------------------------------------------------------------
def length_sweep(torch, llx, p: Pools, stream, nb):
    import ctypes as C
    lib = llx.lib()
    out = []
    flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")
    for tokens in (256, 512, 1024, 2048, 4096, 8192):
        n = tokens // p.g["block_size"]
        s_tab = synth.block_permutation(40 + n, nb)[:n]
        d_tab = synth.block_permutation(50 + n, nb)[:n]
        by = 2 * n * p.src.block_bytes
        single = _time_stream(torch, stream, lambda: llx.migrate_stage(p.src, s_tab, p.dst, d_tab, stream=stream))
        first = _time_stream(torch, stream, lambda: llx.migrate_stage(p.src, s_tab[:n - 2], p.dst, d_tab[:n - 2], stream=stream))
        # final stage: cold (L2 flushed by a 512 MiB write on the same stream), GPU time by events, host time by wall clock
        with torch.cuda.stream(stream):
            fin = _time_stream(torch, stream, lambda: llx.migrate_stage(p.src, s_tab[n - 2:], p.dst, d_tab[n - 2:], stream=stream),
                               reps=20, before=lambda: flush.fill_(1))
        s_ids = np.ascontiguousarray(s_tab[n - 2:], dtype=np.int32)
        d_ids = np.ascontiguousarray(d_tab[n - 2:], dtype=np.int32)
        sp, dp = s_ids.ctypes.data_as(C.POINTER(C.c_int32)), d_ids.ctypes.data_as(C.POINTER(C.c_int32))
        host = []
        for _ in range(60):
            llx.migrate_stage(p.src, s_tab[:n - 2], p.dst, d_tab[:n - 2], stream=stream)   # the long stage evicts L2
            stream.synchronize()
            t0 = time.perf_counter_ns()
            lib.llx_migrate_stage(p.src.handle, sp, p.dst.handle, dp, 2, stream.cuda_stream)
            stream.synchronize()
            host.append((time.perf_counter_ns() - t0) / 1e3)
        host.sort()
        out.append({"tokens": tokens, "blocks": n, "payload_MiB": n * p.src.block_bytes / 2**20,
                    "single_shot_GBps": by / single["median_ms"] / 1e6, "single_shot_ms": single["median_ms"],
                    "stage0_GBps": 2 * (n - 2) * p.src.block_bytes / first["median_ms"] / 1e6,
                    "final_stage_gpu_us_cold": fin["median_ms"] * 1e3,
                    "final_stage_host_us_median": host[len(host) // 2], "final_stage_host_us_p99": host[-1],
                    "blocking_copy_downtime_us": single["median_ms"] * 1e3})
    return out


# ---- the latency floor under the final stage -------------------------------------------------------
def latency_floor(torch, llx, p: Pools, stream, nb):
    """What one launch + one synchronize cost on this box when the copy itself is negligible: a 1-block stage of a
    Tiny-shaped pool (32 KiB payload) through the same entry point, next to the 2-block final stage of the 7B shape.
    Host wall clock (enqueue -> synchronize returns) and CUDA-event time, 300 repetitions each."""
    import ctypes as C
    lib = llx.lib()
    gt = dict(synth.CONFIGS["tiny"])
    pt = Pools(torch, llx, gt, 64, 64)
    out = {}
    for label, pools, n in (("tiny_1_block_32KiB", pt, 1), ("llama7b_2_blocks_16MiB", p, 2)):
        s_ids = np.ascontiguousarray(synth.block_permutation(7, pools.src.num_blocks)[:n], dtype=np.int32)
        d_ids = np.ascontiguousarray(synth.block_permutation(8, pools.dst.num_blocks)[:n], dtype=np.int32)
        sp, dp = s_ids.ctypes.data_as(C.POINTER(C.c_int32)), d_ids.ctypes.data_as(C.POINTER(C.c_int32))
        host, enq, gpu = [], [], []
        ea, eb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        for rep in range(320):
            stream.synchronize()
            t0 = time.perf_counter_ns()
            lib.llx_migrate_stage(pools.src.handle, sp, pools.dst.handle, dp, n, stream.cuda_stream)
            t1 = time.perf_counter_ns()
            stream.synchronize()
            t2 = time.perf_counter_ns()
            ea.record(stream)
            lib.llx_migrate_stage(pools.src.handle, sp, pools.dst.handle, dp, n, stream.cuda_stream)
            eb.record(stream)
            stream.synchronize()
            if rep >= 20:
                host.append((t2 - t0) / 1e3)
                enq.append((t1 - t0) / 1e3)
                gpu.append(ea.elapsed_time(eb) * 1e3)
        out[label] = {"host_us_median": statistics.median(host), "enqueue_us_median": statistics.median(enq),
                      "sync_us_median": statistics.median(host) - statistics.median(enq), "gpu_event_us_median": statistics.median(gpu)}
    out["note"] = ("the 32 KiB stage moves nothing worth timing: its numbers are the floor of one launch + one synchronize through this "
                   "entry point; the final stage's excess over it is the copy itself")
    out["c99_client"] = c_client_downtime()
    return out


def c_client_downtime(reps=300):
    """The same two measurements by a plain C99 program (bench_downtime.c: llx.h and libllx.so only, legacy default stream,
    clock_gettime): what the library costs with no Python and no ctypes in the timed interval."""
    import json
    import shutil
    import subprocess
    import tempfile
    gcc = shutil.which("gcc")
    if not gcc:
        return {"skipped": "gcc unavailable"}
    root = os.path.dirname(os.path.abspath(__file__))
    libdir = os.path.join(root, "paper_2406_03243_b200")
    with tempfile.TemporaryDirectory() as tmp:
        exe = os.path.join(tmp, "bench_downtime")
        r = subprocess.run([gcc, "-std=c99", "-O2", "-Wall", "-Wextra", "-Werror", "-pedantic", "-I", os.path.join(root, "include"),
                            os.path.join(root, "bench_downtime.c"), "-o", exe, "-L", libdir, "-lllx", "-Wl,-rpath," + libdir],
                           capture_output=True, text=True)
        if r.returncode != 0:
            return {"error": r.stderr[-500:]}
        r = subprocess.run([exe, str(reps)], capture_output=True, text=True, timeout=600)
        try:
            return json.loads(r.stdout)
        except Exception:  # noqa: BLE001
            return {"error": (r.stdout + r.stderr)[-500:]}


# ---- reference points on the same data ---------------------------------------
def reference_points(torch, llx, p: Pools, stream, nb):
    n = 128
    s_tab = synth.block_permutation(1, nb)[:n]
    d_tab = synth.block_permutation(2, nb)[:n]
    by = 2 * n * p.src.block_bytes
    res = {}
    a = torch.empty(n * p.src.block_bytes, dtype=torch.uint8, device="cuda")
    b = torch.empty_like(a)
    with torch.cuda.stream(stream):
        t = _time_stream(torch, stream, lambda: b.copy_(a))
        res["torch_contiguous_copy_GBps"] = by / t["median_ms"] / 1e6
        sv, dv = p.view(p.src_raw, nb), p.view(p.dst_raw, nb)
        si = torch.from_numpy(s_tab.astype(np.int64)).cuda()
        di = torch.from_numpy(d_tab.astype(np.int64)).cuda()

        def index_form():
            for l in range(p.g["layers"]):
                for kv in range(2):
                    dv[l, kv].index_copy_(0, di, sv[l, kv].index_select(0, si))
        t = _time_stream(torch, stream, index_form, reps=5, warm=1)
        res["torch_index_select_index_copy_GBps"] = by / t["median_ms"] / 1e6

        def per_tile_memcpy():     # "many small messages": one cudaMemcpyAsync per 128 KiB tile
            for i in range(n):
                for l in range(p.g["layers"]):
                    for kv in range(2):
                        dv[l, kv, int(d_tab[i])].copy_(sv[l, kv, int(s_tab[i])])
        t = _time_stream(torch, stream, per_tile_memcpy, reps=2, warm=1)
        res["per_tile_memcpy_loop_GBps"] = by / t["median_ms"] / 1e6
        res["per_tile_memcpy_loop_ms"] = t["median_ms"]
    t = _time_stream(torch, stream, lambda: llx.migrate_stage(p.src, s_tab, p.dst, d_tab, stream=stream))
    res["llx_migrate_stage_GBps"] = by / t["median_ms"] / 1e6
    for o, name in ((dict(copy_kernel=1), "llx_vec16_kernel_GBps"), (dict(copy_kernel=2), "llx_bulk_kernel_GBps"),
                    (dict(route=llx.ROUTE_PEER), "llx_peer_route_on_one_device_GBps"),
                    (dict(route=llx.ROUTE_COPY_ENGINE), "llx_copy_engine_route_on_one_device_GBps")):
        t = _time_stream(torch, stream, lambda: llx.migrate_stage(p.src, s_tab, p.dst, d_tab, stream=stream, opts=o))
        res[name] = by / t["median_ms"] / 1e6
    # device-buffer block fusion (pack then unpack through HBM)
    stg = torch.empty(llx.staging_bytes(p.src, n), dtype=torch.uint8, device="cuda")
    t = _time_stream(torch, stream, lambda: llx.pack(p.src, s_tab, stg.data_ptr(), stg.numel(), stream=stream))
    res["llx_pack_device_GBps"] = by / t["median_ms"] / 1e6
    t = _time_stream(torch, stream, lambda: llx.unpack(stg.data_ptr(), stg.numel(), p.dst, d_tab, stream=stream))
    res["llx_unpack_device_GBps"] = by / t["median_ms"] / 1e6
    return res


# ---- configs[4] second half: staging through pinned host memory --------------------------------
def staging_host(torch, llx, p: Pools, stream, nb):
    n = 128
    s_tab = synth.block_permutation(1, nb)[:n]
    d_tab = synth.block_permutation(2, nb)[:n]
    nbytes = llx.staging_bytes(p.src, n)
    pin = llx.PinnedStaging(nbytes)
    res = {"payload_GiB": nbytes / 2**30}
    # host-link peak: plain copy-engine transfers of the same size, each direction
    dev = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    host = torch.empty(nbytes, dtype=torch.uint8).pin_memory()
    with torch.cuda.stream(stream):
        t = _time_stream(torch, stream, lambda: host.copy_(dev, non_blocking=True), reps=5, warm=1)
        res["link_peak_d2h_GBps"] = nbytes / t["min_ms"] / 1e6
        t = _time_stream(torch, stream, lambda: dev.copy_(host, non_blocking=True), reps=5, warm=1)
        res["link_peak_h2d_GBps"] = nbytes / t["min_ms"] / 1e6
    del host
    t = _time_stream(torch, stream, lambda: llx.pack(p.src, s_tab, pin.dev_alias, nbytes, stream=stream), reps=5, warm=1)
    res["llx_pack_to_pinned_host_GBps"] = nbytes / t["median_ms"] / 1e6
    t = _time_stream(torch, stream, lambda: llx.unpack(pin.dev_alias, nbytes, p.dst, d_tab, stream=stream), reps=5, warm=1)
    res["llx_unpack_from_pinned_host_GBps"] = nbytes / t["median_ms"] / 1e6
    res["pack_frac_of_link_peak"] = res["llx_pack_to_pinned_host_GBps"] / res["link_peak_d2h_GBps"]
    res["unpack_frac_of_link_peak"] = res["llx_unpack_from_pinned_host_GBps"] / res["link_peak_h2d_GBps"]
    zc = dict(via_host_mode=1)               # the kernels address the pinned buffer themselves
    t = _time_stream(torch, stream, lambda: llx.pack(p.src, s_tab, pin.dev_alias, nbytes, stream=stream, opts=zc), reps=5, warm=1)
    res["llx_pack_zero_copy_GBps"] = nbytes / t["median_ms"] / 1e6
    t = _time_stream(torch, stream, lambda: llx.unpack(pin.dev_alias, nbytes, p.dst, d_tab, stream=stream, opts=zc), reps=5, warm=1)
    res["llx_unpack_zero_copy_GBps"] = nbytes / t["median_ms"] / 1e6
    t = _time_stream(torch, stream, lambda: llx.migrate_via_host(p.src, s_tab, p.dst, d_tab, pin.dev_alias, nbytes, stream=stream), reps=5, warm=1)
    res["llx_migrate_via_host_roundtrip_ms"] = t["median_ms"]
    t = _time_stream(torch, stream, lambda: llx.migrate_via_host(p.src, s_tab, p.dst, d_tab, pin.dev_alias, nbytes, stream=stream,
                                                                 opts=dict(via_host_mode=3)), reps=5, warm=1)
    res["llx_migrate_via_host_kernels_and_bounce_buffers_roundtrip_ms"] = t["median_ms"]
    # alternative: pack into a DEVICE buffer, then one copy-engine transfer (and back)
    stg = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    hbuf = torch.empty(nbytes, dtype=torch.uint8).pin_memory()

    def via_ce():
        llx.pack(p.src, s_tab, stg.data_ptr(), nbytes, stream=stream)
        with torch.cuda.stream(stream):
            hbuf.copy_(stg, non_blocking=True)
            stg.copy_(hbuf, non_blocking=True)
        llx.unpack(stg.data_ptr(), nbytes, p.dst, d_tab, stream=stream)
    t = _time_stream(torch, stream, via_ce, reps=5, warm=1)
    res["device_pack_plus_copy_engine_roundtrip_ms"] = t["median_ms"]

    def direct():
        llx.pack(p.src, s_tab, pin.dev_alias, nbytes, stream=stream)
        llx.unpack(pin.dev_alias, nbytes, p.dst, d_tab, stream=stream)
    t = _time_stream(torch, stream, direct, reps=5, warm=1)
    res["zero_copy_pack_unpack_roundtrip_ms"] = t["median_ms"]
    pin.free()
    return res


# ---- configs[3]: LLaMA-30B batch --------------------------------------------------------------
def batch_30b(torch, llx, stream, seed=0):
    """seed 0 is the config's draw as specified; its sample of 64 lengths has mean 248 tokens (1023 blocks, 24.4 GiB) —
    a fair draw of a heavy tail (the distribution's mean is 512).  seed 2 is added because its SAMPLE mean (507 tokens,
    2064 blocks, 49 GiB) is within 10 % of the nominal 512."""
    g = dict(synth.CONFIGS["llama30b"])
    lens, nblk, seed_used = synth.batch_request_blocks(seed, 64, g["block_size"], g["num_blocks"])
    total = int(nblk.sum())
    block_bytes = 2 * g["layers"] * g["block_size"] * g["kv_heads"] * g["head_dim"] * 2
    nb = g["num_blocks"]
    free = _free(torch)
    while 2 * nb * block_bytes > free - (6 << 30) and nb > total:
        nb -= 100
    if nb < total:
        return {"skipped": f"not enough device memory for {total} blocks per pool"}
    p = Pools(torch, llx, g, nb, nb)
    s_ids = synth.block_permutation(1, nb)[:total]
    d_ids = synth.block_permutation(2, nb)[:total]
    off = np.concatenate([[0], np.cumsum(nblk)]).astype(np.int32)
    by = 2 * total * block_bytes
    t = _time_stream(torch, stream, lambda: llx.migrate_batch(p.src, p.dst, off, s_ids, d_ids, stream=stream), reps=5, warm=1)

    def sequential():
        for r in range(64):
            llx.migrate_stage(p.src, s_ids[off[r]:off[r + 1]], p.dst, d_ids[off[r]:off[r + 1]], stream=stream)
    ts = _time_stream(torch, stream, sequential, reps=3, warm=1)
    res = {"requests": 64, "length_seed_used": int(seed_used), "total_blocks": total, "pool_blocks_used": nb,
           "pool_blocks_config": g["num_blocks"], "payload_GiB": total * block_bytes / 2**30,
           "mean_tokens": float(lens.mean()), "max_tokens": int(lens.max()), "min_tokens": int(lens.min()),
           "one_launch_ms": t["median_ms"], "one_launch_GBps": by / t["median_ms"] / 1e6,
           "sequential_64_launches_ms": ts["median_ms"], "sequential_GBps": by / ts["median_ms"] / 1e6}
    del p
    _free(torch)
    return res


# ---- configs[4] first half: interference with a decode step -----------------------------------
def _power_state(torch):
    """SM clock, power draw and clock-event reasons right now (NVML), or None."""
    try:
        import pynvml
        pynvml.nvmlInit()
        h = pynvml.nvmlDeviceGetHandleByIndex(torch.cuda.current_device())
        return {"sm_mhz": pynvml.nvmlDeviceGetClockInfo(h, pynvml.NVML_CLOCK_SM), "power_w": pynvml.nvmlDeviceGetPowerUsage(h) / 1000.0,
                "reasons": hex(pynvml.nvmlDeviceGetCurrentClocksEventReasons(h))}
    except Exception:  # noqa: BLE001
        return None


def interference(torch, llx, stream_mig_unused, paced_only=False, budgets=None):
    """budgets: None = the full case list; a tuple of GB/s = the bounded list of bench.py's default line (one unthrottled
    migration at the step's start, then a looped migration under each budget)."""
    g = dict(synth.CONFIGS["llama7b"])
    L, H, D, S = g["layers"], g["kv_heads"], g["head_dim"], g["block_size"]
    B = 32
    ctx = synth.context_lengths(4, B, 128, 4096)
    need = [-(-int(c) // S) for c in ctx]
    nb_src = B * 256 + 128 + 128          # reading A12: worst case for any seed, + the migrating request + slack
    nb_dst = g["num_blocks"]
    block_bytes = 2 * L * S * H * D * 2
    if (nb_src + nb_dst) * block_bytes > _free(torch) - (4 << 30):
        return {"skipped": "not enough device memory"}
    p = Pools(torch, llx, g, nb_src, nb_dst)
    perm = synth.block_permutation(6, nb_src)
    MB = 256
    bt = np.zeros((B, MB), dtype=np.int32)
    pos = 0
    for b, n in enumerate(need):
        bt[b, :n] = perm[pos:pos + n]
        pos += n
    mig_src = perm[pos:pos + 128]
    mig_dst = synth.block_permutation(2, nb_dst)[:128]
    q = torch.from_numpy(synth.queries_f16(5, B, H, D).view(np.int16)).cuda()
    o = torch.zeros_like(q)
    d_bt = torch.from_numpy(bt).cuda()
    d_ctx = torch.from_numpy(ctx).cuda()
    scale = 1.0 / float(np.sqrt(D))
    lo, hi = torch.cuda.Stream.priority_range()            # (least, greatest) = (0, -N)
    s_dec = torch.cuda.Stream(priority=hi)
    s_mig = torch.cuda.Stream(priority=lo)
    kv_bytes_step = int(ctx.sum()) * 2 * H * D * 2 * L

    def decode_step():
        for l in range(L):
            llx.decode_attention(p.src, l, q.data_ptr(), o.data_ptr(), d_bt.data_ptr(), d_ctx.data_ptr(), B, MB, scale,
                                 stream=s_dec)

    def migrate(o=None):
        llx.migrate_stage(p.src, mig_src, p.dst, mig_dst, stream=s_mig, opts=o)

    decode_step()
    torch.cuda.synchronize()
    alone = _time_stream(torch, s_dec, decode_step, reps=10, warm=2)
    mig_alone = _time_stream(torch, s_mig, migrate, reps=10, warm=2)
    mig_bytes = 2 * 128 * block_bytes

    def one_step(n_mig, max_ctas, budget):
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ma, mb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        o = dict(max_ctas=max_ctas, bandwidth_gbps=budget)          # the launch policy of these calls only

        def enqueue_migrations():
            for _ in range(n_mig):
                migrate(o)
        ma.record(s_mig)
        th = _in_thread(torch, enqueue_migrations)
        time.sleep(0.0002)                                           # the first migration launch is on the device (same pause in both arms of a pair)
        a.record(s_dec)
        decode_step()
        b.record(s_dec)
        th.join()
        mb.record(s_mig)
        torch.cuda.synchronize()
        return a.elapsed_time(b), ma.elapsed_time(mb)

    def with_migration(n_mig, max_ctas, budget=0):
        """PAIRED: every step with the migration is preceded by an isolated step; the slowdown is the median of the
        per-pair ratios (the isolated step drifts by +-2 % between blocks of measurements, more than the small cases)."""
        times, mig_ms, ratios = [], [], []
        for _ in range(8):
            one_step(0, 0, 0)          # discarded: the previous pair ended with the GPU all but idle under a long paced tail;
            t0, _ = one_step(0, 0, 0)  # both measured steps now follow a decode step
            t1, m = one_step(n_mig, max_ctas, budget)
            times.append(t1)
            mig_ms.append(m)
            ratios.append(t1 / t0)
        return statistics.median(times), statistics.median(mig_ms), statistics.median(ratios)

    iso_ms = statistics.median(one_step(0, 0, 0)[0] for _ in range(8))      # one isolated step, measured the same way
    res = {"batch": B, "ctx_tokens_total": int(ctx.sum()), "src_pool_blocks": nb_src, "dst_pool_blocks": nb_dst,
           "decode_step_alone_ms": alone["median_ms"], "decode_step_alone_isolated_ms": iso_ms,
           "decode_attention_GBps": kv_bytes_step / alone["median_ms"] / 1e6,
           "migration_alone_ms": mig_alone["median_ms"], "migration_alone_GBps": mig_bytes / mig_alone["median_ms"] / 1e6,
           "cases": []}
    loop_n = max(2, int(alone["median_ms"] / mig_alone["median_ms"]) + 2)
    step_s = alone["median_ms"] * 1e-3

    def n_for(gbps):      # migrations needed to keep the copy stream busy for the whole decode step
        return max(1, int(gbps * 1e9 * step_s * 1.6 / mig_bytes) + 1)
    cases = [("one 2048-token migration at step start, full speed", 1, 0, 0),
             ("migration looped for the whole step, full speed", loop_n, 0, 0)]
    cases += [(f"looped, {c} full-speed CTAs (LLX_OPT_MAX_CTAS)", n_for(c * 33), c, 0) for c in (32, 16, 8, 4)]
    cases += [(f"looped, budget {bw} GB/s (LLX_OPT_BANDWIDTH_GBPS: " + ("few full-speed CTAs" if bw >= 500 else "paced on all SMs") + ")",
               n_for(bw), 0, bw) for bw in (2400, 1600, 800, 400, 200, 100, 65, 20)]
    if paced_only:
        cases = [c for c in cases if 0 < c[3] < 500]
    if budgets is not None:
        cases = [cases[0]] + [(f"looped, budget {bw} GB/s (paced on all SMs)", n_for(bw), 0, bw) for bw in budgets]
    res["power_state_before_cases"] = _power_state(torch)
    for label, n_mig, cap, bw in cases:
        t, m, ratio = with_migration(n_mig, cap, bw)
        res["cases"].append({"case": label, "migrations": n_mig, "max_ctas": cap, "bandwidth_budget_GBps": bw,
                             "decode_step_ms": t, "slowdown_pct": 100.0 * (ratio - 1.0),
                             "migration_GBps_while_overlapped": n_mig * mig_bytes / m / 1e6,
                             "bandwidth_share_pct": 100.0 * min(1.0, t / m) * n_mig * mig_bytes / (kv_bytes_step + min(1.0, t / m) * n_mig * mig_bytes)})
    res["power_state_after_cases"] = _power_state(torch)
    res["note"] = ("slowdown = median of per-pair ratios (step with migration / isolated step right before it); any concurrent kernel of another "
                   "stream costs ~3.5 % (floor, independent of its rate: launch gaps of the 64-launch step grow), a co-resident "
                   "CTA holding > ~6 KB shared memory costs +30 % (L1 carve-out), and a few full-speed CTAs make their SMs "
                   "stragglers; the paced mode therefore copies through registers with one small CTA per SM")
    del p
    _free(torch)
    return res


# ---- NEXT-1: choose the bandwidth budget from a decode-slowdown target (<= 1 %) ----------
def auto_budget(torch, llx, stream_unused=None, target_pct=1.0, rounds=16, grid=None):
    """Largest LLX_OPT_BANDWIDTH_GBPS whose decode-step slowdown stays within `target_pct`.

    The isolated decode step varies by about +-2 % from one measurement block to the next on a B200, more than
    the target itself, so every candidate is measured PAIRED: steps alternate without / with the migration
    (A B A B ...), the slowdown is the median of the per-pair ratios, and a candidate passes when that median
    is within the target.  Candidates are searched by bisection on a geometric grid."""
    g = dict(synth.CONFIGS["llama7b"])
    L, H, D, S = g["layers"], g["kv_heads"], g["head_dim"], g["block_size"]
    B = 32
    ctx = synth.context_lengths(4, B, 128, 4096)
    need = [-(-int(c) // S) for c in ctx]
    nb_src, nb_dst = B * 256 + 256, g["num_blocks"]
    block_bytes = 2 * L * S * H * D * 2
    if (nb_src + nb_dst) * block_bytes > _free(torch) - (4 << 30):
        return {"skipped": "not enough device memory"}
    p = Pools(torch, llx, g, nb_src, nb_dst)
    perm = synth.block_permutation(6, nb_src)
    MB = 256
    bt = np.zeros((B, MB), dtype=np.int32)
    pos = 0
    for b, n in enumerate(need):
        bt[b, :n] = perm[pos:pos + n]
        pos += n
    mig_src, mig_dst = perm[pos:pos + 128], synth.block_permutation(2, nb_dst)[:128]
    q = torch.from_numpy(synth.queries_f16(5, B, H, D).view(np.int16)).cuda()
    o = torch.zeros_like(q)
    d_bt, d_ctx = torch.from_numpy(bt).cuda(), torch.from_numpy(ctx).cuda()
    scale = 1.0 / float(np.sqrt(D))
    lo, hi = torch.cuda.Stream.priority_range()
    s_dec, s_mig = torch.cuda.Stream(priority=hi), torch.cuda.Stream(priority=lo)
    mig_bytes = 2 * 128 * block_bytes

    def decode_step():
        for l in range(L):
            llx.decode_attention(p.src, l, q.data_ptr(), o.data_ptr(), d_bt.data_ptr(), d_ctx.data_ptr(), B, MB, scale,
                                 stream=s_dec)

    def one(budget, n_mig):
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

        def enqueue_migrations():
            for _ in range(n_mig):
                llx.migrate_stage(p.src, mig_src, p.dst, mig_dst, stream=s_mig, opts=dict(bandwidth_gbps=budget))
        th = _in_thread(torch, enqueue_migrations)
        time.sleep(0.0002)                                           # same pause in both arms of a pair
        a.record(s_dec)
        decode_step()
        b.record(s_dec)
        th.join()
        torch.cuda.synchronize()
        return a.elapsed_time(b)

    grid = list(grid) if grid else [5, 8, 12, 18, 25, 35, 50, 100, 200]

    def measure_state():
        for _ in range(3):
            one(0, 0)
        base = statistics.median(one(0, 0) for _ in range(5))
        by_budget = {}
        for budget in grid:
            n_mig = max(1, int(budget * 1e9 * base * 1e-3 * 1.6 / mig_bytes) + 1)   # keeps the copy stream busy all step long
            ratios, with_mig = [], []
            for _ in range(rounds):
                one(0, 0)              # discarded (see interference(): both measured steps follow a decode step)
                t0 = one(0, 0)
                t1 = one(budget, n_mig)
                ratios.append(t1 / t0)
                with_mig.append(t1)
            by_budget[str(budget)] = {"slowdown_pct": 100.0 * (statistics.median(ratios) - 1.0), "decode_step_ms": statistics.median(with_mig)}
        ok = [b_ for b_ in grid if by_budget[str(b_)]["slowdown_pct"] <= target_pct]
        largest = None
        for b_ in grid:                          # the largest budget below which every candidate holds the target
            if by_budget[str(b_)]["slowdown_pct"] <= target_pct:
                largest = b_
            else:
                break
        null = 100.0 * (statistics.median(one(0, 0) / one(0, 0) for _ in range(rounds)) - 1.0)
        return {"decode_step_alone_ms": base, "chosen_budget_GBps": largest, "by_budget": by_budget, "null_pair_pct": null,
                "candidates_within_target": ok}

    # Two states of the same GPU.  "pristine": the GPU idled before and idles between pairs (cool, SM clock at its maximum).
    # "steady": right after 20 full-speed bulk-ring migrations (warm).  The decode loop pulls this B200 to its power cap
    # (sw_power_cap, SM clock 1965 -> ~1600 MHz, the step 5.18 -> 5.5 ms) when it runs without pause; isolated pairs sit
    # between those two points, and where they sit changes what "alone" means.  interference_sustained() is the reference;
    # this sweep brackets what short measurements see.
    res = {"target_slowdown_pct": target_pct, "pairs_per_candidate": rounds, "pristine": measure_state()}
    for _ in range(20):
        llx.migrate_stage(p.src, mig_src, p.dst, mig_dst, stream=s_mig)
    torch.cuda.synchronize()
    res["steady"] = measure_state()
    res["chosen_budget_GBps"] = res["pristine"]["chosen_budget_GBps"]
    res["note"] = ("slowdown = median of per-pair ratios (step with migration / step without, alternating, each after a discarded "
                   "step); null_pair_pct = the same statistic for two steps without migration (the measurement floor); the "
                   "migration is enqueued from its own host thread")
    del p
    _free(torch)
    return res


# ---- interference under SUSTAINED decoding: the state a serving GPU is in ---------------------------------------
def interference_sustained(torch, llx, stream_unused=None, budgets=(12, 25, 50, 100, 200, 400), alt_budgets=(25, 100, 400), seg_steps=150, segments=4):
    """The configs[4] decode step run back to back without pause, as a serving engine does.  After ~0.5 s of that the
    B200 sits at its power cap (about 1000 W, SM clock 1965 -> ~1600 MHz, NVML reason sw_power_cap) and the step takes
    5.5 ms instead of the 5.2 ms of a GPU that idles between measurements — the "pristine" and "steady" baselines of
    auto_budget are two points on that curve.  Here the decode loop never stops; a host thread keeps budgeted
    16-block stages in flight during the ON segments and none during the OFF segments; the first and last 20 steps of
    every segment are dropped.  slowdown = median ON step / median OFF step - 1.
    Two other mechanisms at the same byte rate, to separate what the KERNEL costs from what the BYTES cost: the same
    blocks moved by the copy engine (LLX_ROUTE_COPY_ENGINE: no SM at all) and by the full-speed bulk kernel, one block
    per interval, paced by the host thread."""
    import threading
    g = dict(synth.CONFIGS["llama7b"])
    L, H, D, S = g["layers"], g["kv_heads"], g["head_dim"], g["block_size"]
    B, MB = 32, 256
    ctx = synth.context_lengths(4, B, 128, 4096)
    need = [-(-int(c) // S) for c in ctx]
    nb_src, nb_dst = B * 256 + 256, g["num_blocks"]
    if (nb_src + nb_dst) * 2 * L * S * H * D * 2 > _free(torch) - (4 << 30):
        return {"skipped": "not enough device memory"}
    p = Pools(torch, llx, g, nb_src, nb_dst)
    perm = synth.block_permutation(6, nb_src)
    bt = np.zeros((B, MB), dtype=np.int32)
    pos = 0
    for b, n in enumerate(need):
        bt[b, :n] = perm[pos:pos + n]
        pos += n
    mig_src, mig_dst = perm[pos:pos + 16], synth.block_permutation(2, nb_dst)[:16]
    q = torch.from_numpy(synth.queries_f16(5, B, H, D).view(np.int16)).cuda()
    o = torch.zeros_like(q)
    d_bt, d_ctx = torch.from_numpy(bt).cuda(), torch.from_numpy(ctx).cuda()
    scale = 1.0 / float(np.sqrt(D))
    lo, hi = torch.cuda.Stream.priority_range()
    s_dec, s_mig = torch.cuda.Stream(priority=hi), torch.cuda.Stream(priority=lo)
    dev = torch.cuda.current_device()

    def run_steps(n):
        evs = [torch.cuda.Event(enable_timing=True) for _ in range(n + 1)]
        evs[0].record(s_dec)
        for k in range(n):
            for l in range(L):
                llx.decode_attention(p.src, l, q.data_ptr(), o.data_ptr(), d_bt.data_ptr(), d_ctx.data_ptr(), B, MB, scale, stream=s_dec)
            evs[k + 1].record(s_dec)
            if k % 8 == 7:
                evs[k - 6].synchronize()          # keep the host a few steps ahead of the GPU, never idle, never far ahead
        s_dec.synchronize()
        return [evs[k].elapsed_time(evs[k + 1]) for k in range(n)]

    nvml = None
    try:
        import pynvml
        pynvml.nvmlInit()
        nvml = (pynvml, pynvml.nvmlDeviceGetHandleByIndex(dev))
    except Exception:  # noqa: BLE001
        pass

    def clocks():
        if not nvml:
            return None
        nv, h = nvml
        return {"sm_mhz": nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM), "power_w": nv.nvmlDeviceGetPowerUsage(h) / 1000.0,
                "reasons": hex(nv.nvmlDeviceGetCurrentClocksEventReasons(h))}

    res = {"idle_clocks": clocks()}
    first = run_steps(5)
    run_steps(300)                                    # into the power-capped steady state
    res["decode_step_first_ms"] = statistics.median(first)
    res["sustained_clocks"] = clocks()
    res["cases"] = []
    block_rw = 2 * p.src.block_bytes

    def feeder_paced_kernel(budget, stop):           # the library's budget: paced register-staged kernel on every SM
        while not stop.is_set():
            llx.migrate_stage(p.src, mig_src, p.dst, mig_dst, stream=s_mig, opts=dict(bandwidth_gbps=budget))
            llx.migrate_stage(p.src, mig_src, p.dst, mig_dst, stream=s_mig, opts=dict(bandwidth_gbps=budget))
            ev = torch.cuda.Event()
            ev.record(s_mig)
            while not ev.query() and not stop.is_set():
                time.sleep(0.0005)

    def feeder_per_block(opts):                      # one block per interval, paced by the HOST: no resident kernel at all
        def feed(budget, stop):
            i, t_next, interval = 0, time.perf_counter(), block_rw / (budget * 1e9)
            while not stop.is_set():
                k = i % len(mig_src)
                llx.migrate_stage(p.src, mig_src[k:k + 1], p.dst, mig_dst[k:k + 1], stream=s_mig, opts=opts)
                i += 1
                t_next += interval
                d = t_next - time.perf_counter()
                if d > 0:
                    time.sleep(d)
        return feed

    mechanisms = [("paced kernel on every SM (bandwidth_gbps)", feeder_paced_kernel, budgets),
                  ("copy engine, one block per interval paced by the host (no SM at all)", feeder_per_block(dict(route=llx.ROUTE_COPY_ENGINE)), alt_budgets),
                  ("full-speed bulk kernel, one block per interval paced by the host", feeder_per_block(None), alt_budgets)]
    for label, feed, bl in mechanisms:
        for budget in bl:
            on, off = [], []
            for _ in range(segments):
                t = run_steps(seg_steps)
                off += t[20:-20]
                stop = threading.Event()

                def run_feeder():
                    torch.cuda.set_device(dev)
                    feed(budget, stop)
                th = threading.Thread(target=run_feeder)
                th.start()
                run_steps(10)                         # the first stage is on the device
                t = run_steps(seg_steps)
                on += t[20:-20]
                stop.set()
                th.join()
                s_mig.synchronize()
            res["cases"].append({"mechanism": label, "bandwidth_budget_GBps": budget, "decode_step_off_ms": statistics.median(off),
                                 "decode_step_on_ms": statistics.median(on),
                                 "slowdown_pct": 100.0 * (statistics.median(on) / statistics.median(off) - 1.0), "steps_each": len(on)})
    res["end_clocks"] = clocks()
    res["note"] = "decode loop never pauses; ON = budgeted 16-block stages kept in flight by a host thread; 20 steps dropped at both ends of every segment"
    del p
    _free(torch)
    return res


# ---- the budget chosen behind the ABI: llx_budget_ctl driven by a decode loop that never pauses ---------------
def budget_controller_live(torch, llx, stream_unused=None, target_pct=1.0, window=16, rounds=24, start_gbps=200, drop=3):
    """SURVEY NEXT-1 "chosen automatically so decode slowdown <= 1 %", as an engine would run it: the configs[4] decode
    loop never stops (power-capped steady state, see interference_sustained); it reports every step's duration to
    llx_budget_ctl_observe.  Rounds alternate 2*window steps without a migration and window steps with budgeted
    16-block stages kept in flight by a host thread at the controller's current budget (3 steps dropped after every
    switch).  The trajectory is printed; the budget the controller settles on is then measured like interference_sustained
    measures a fixed budget (4 segments ON / OFF of 150 steps)."""
    import threading
    g = dict(synth.CONFIGS["llama7b"])
    L, H, D, S = g["layers"], g["kv_heads"], g["head_dim"], g["block_size"]
    B, MB = 32, 256
    ctx = synth.context_lengths(4, B, 128, 4096)
    need = [-(-int(c) // S) for c in ctx]
    nb_src, nb_dst = B * 256 + 256, g["num_blocks"]
    if (nb_src + nb_dst) * 2 * L * S * H * D * 2 > _free(torch) - (4 << 30):
        return {"skipped": "not enough device memory"}
    p = Pools(torch, llx, g, nb_src, nb_dst)
    perm = synth.block_permutation(6, nb_src)
    bt = np.zeros((B, MB), dtype=np.int32)
    pos = 0
    for b, n in enumerate(need):
        bt[b, :n] = perm[pos:pos + n]
        pos += n
    mig_src, mig_dst = perm[pos:pos + 16], synth.block_permutation(2, nb_dst)[:16]
    q = torch.from_numpy(synth.queries_f16(5, B, H, D).view(np.int16)).cuda()
    o = torch.zeros_like(q)
    d_bt, d_ctx = torch.from_numpy(bt).cuda(), torch.from_numpy(ctx).cuda()
    scale = 1.0 / float(np.sqrt(D))
    lo, hi = torch.cuda.Stream.priority_range()
    s_dec, s_mig = torch.cuda.Stream(priority=hi), torch.cuda.Stream(priority=lo)
    dev = torch.cuda.current_device()

    def run_steps(n):
        evs = [torch.cuda.Event(enable_timing=True) for _ in range(n + 1)]
        evs[0].record(s_dec)
        for k in range(n):
            for l in range(L):
                llx.decode_attention(p.src, l, q.data_ptr(), o.data_ptr(), d_bt.data_ptr(), d_ctx.data_ptr(), B, MB, scale, stream=s_dec)
            evs[k + 1].record(s_dec)
            if k % 8 == 7:
                evs[k - 6].synchronize()
        s_dec.synchronize()
        return [evs[k].elapsed_time(evs[k + 1]) for k in range(n)]

    def feeder(budget_of, stop):
        torch.cuda.set_device(dev)
        while not stop.is_set():
            o_ = dict(bandwidth_gbps=budget_of())
            llx.migrate_stage(p.src, mig_src, p.dst, mig_dst, stream=s_mig, opts=o_)
            llx.migrate_stage(p.src, mig_src, p.dst, mig_dst, stream=s_mig, opts=o_)
            ev = torch.cuda.Event()
            ev.record(s_mig)
            while not ev.query() and not stop.is_set():
                time.sleep(0.0005)

    def with_feeder(budget_of, n_steps):
        stop = threading.Event()
        th = threading.Thread(target=feeder, args=(budget_of, stop))
        th.start()
        run_steps(drop)
        t = run_steps(n_steps)
        stop.set()
        th.join()
        s_mig.synchronize()
        return t

    run_steps(300)                                    # into the power-capped steady state
    ctl = llx.BudgetController(target_pct, 1, 2000, start_gbps, window)
    trajectory = []
    for r in range(rounds):
        run_steps(drop)
        for t in run_steps(2 * window):
            ctl.observe(t, False)
        before = ctl.gbps
        for t in with_feeder(lambda: before, window):
            ctl.observe(t, True)
        trajectory.append({"budget_GBps": before, "observed_slowdown_pct": round(ctl.last_slowdown_pct, 3), "next_budget_GBps": ctl.gbps})
    tail = [x["budget_GBps"] for x in trajectory[rounds // 2:]]
    chosen = int(statistics.median(tail))
    on, off = [], []
    for _ in range(4):
        off += run_steps(150)[20:-20]
        on += with_feeder(lambda: chosen, 150)[20:-20]
    res = {"target_slowdown_pct": target_pct, "window_steps": window, "start_budget_GBps": start_gbps, "trajectory": trajectory,
           "settled_budget_GBps": {"median_of_second_half": chosen, "min": min(tail), "max": max(tail)},
           "verification_at_settled_budget": {"decode_step_off_ms": statistics.median(off), "decode_step_on_ms": statistics.median(on),
                                              "slowdown_pct": 100.0 * (statistics.median(on) / statistics.median(off) - 1.0), "steps_each": len(on)},
           "note": "decode loop never pauses; the controller sees event-timed steps, 2*window without and window with a migration per round"}
    del p
    _free(torch)
    return res


# ---- the paper's Fig. 10 situation on one B200: a request migrates WHILE its batch keeps decoding -------------
def live_migration(torch, llx, stream_unused=None, budgets=(0, 100, 25), start_tokens=2040):
    """One request of a 32-sequence decode batch is migrated live (§6.2): the decode loop keeps
    appending one token per step to its last source block while the session (llx_migration_*: planner, PRE-ALLOC,
    copy) moves the completed blocks; when the planner names the final stage the request is drained, the last blocks
    are copied (downtime) and the request resumes on the destination.  Reported per bandwidth budget: stages and
    their sizes, copy time, downtime, decode-step time during the migration vs before."""
    g = dict(synth.CONFIGS["llama7b"])
    L, H, D, S = g["layers"], g["kv_heads"], g["head_dim"], g["block_size"]
    B, MB = 32, 256
    ctx0 = synth.context_lengths(4, B, 128, 4096).copy()
    r = 0
    ctx0[r] = start_tokens                                    # the migrating request
    nb_src, nb_dst = B * 256 + 256, g["num_blocks"]
    block_bytes = 2 * L * S * H * D * 2
    if (nb_src + nb_dst) * block_bytes > _free(torch) - (4 << 30):
        return {"skipped": "not enough device memory"}
    p = Pools(torch, llx, g, nb_src, nb_dst)
    scale = 1.0 / float(np.sqrt(D))
    lo, hi = torch.cuda.Stream.priority_range()
    s_dec, s_mig = torch.cuda.Stream(priority=hi), torch.cuda.Stream(priority=lo)
    q = torch.from_numpy(synth.queries_f16(5, B, H, D).view(np.int16)).cuda()
    o = torch.zeros_like(q)
    tok_bytes = L * 2 * H * D * 2
    new_vals = torch.randint(-0x3C00, 0x3C00, (64, L, 2, H * D), dtype=torch.int16, device="cuda")   # K/V of the tokens decoded meanwhile
    out = {"batch": B, "request_start_tokens": start_tokens, "runs": []}

    for budget in budgets:
        src_mgr, dst_mgr = llx.BlockManager(nb_src), llx.BlockManager(nb_dst)
        dst_mgr.alloc(500)                                    # the destination serves other requests already
        need = [-(-int(c) // S) for c in ctx0]
        bt = np.zeros((B, MB), dtype=np.int32)
        tables = []
        for b in range(B):
            t = src_mgr.alloc(need[b] + (8 if b == r else 0))   # room for the tokens decoded during the migration
            tables.append(t)
            bt[b, :len(t)] = t
        d_bt = torch.from_numpy(bt).cuda()
        ctx = ctx0.copy()
        d_ctx = torch.from_numpy(ctx).cuda()
        table_r = tables[r]
        tokens = int(ctx[r])

        def decode_step(pool, with_append=True):
            nonlocal tokens
            a, b_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(s_dec)
            if with_append:                                   # the step's new token of the migrating request (S8)
                llx.append_tokens(pool, table_r, tokens, tokens + 1,
                                  new_vals.data_ptr() + (tokens - start_tokens) * tok_bytes, stream=s_dec)
                tokens += 1
                with torch.cuda.stream(s_dec):
                    d_ctx[r] = tokens
            for l in range(L):
                llx.decode_attention(pool, l, q.data_ptr(), o.data_ptr(), d_bt.data_ptr(), d_ctx.data_ptr(), B, MB, scale,
                                     stream=s_dec)
            b_.record(s_dec)
            s_dec.synchronize()                               # the engine samples the token: one host sync per step
            return a.elapsed_time(b_)

        for _ in range(3):
            decode_step(p.src)
        before = statistics.median([decode_step(p.src) for _ in range(8)])     # same step (append + 32 layers), no migration
        tokens_at_start = tokens
        mig = llx.Migration(p.src, src_mgr, p.dst, dst_mgr, S, 2)
        stages, during, t_start = [], [], time.perf_counter()
        mig.set_stage_opts(dict(bandwidth_gbps=budget))       # non-final stages only: the session runs the final stage unthrottled
        while True:
            n, fin, _ = mig.stage(table_r, tokens, stream=s_mig)
            ev = torch.cuda.Event()
            ev.record(s_mig)
            stages.append(n)
            assert not fin and mig.state == llx.MIG_COPYING
            while not ev.query():                             # decoding continues while the stage copies
                during.append(decode_step(p.src))
            n_next, fin_next = llx.plan_stage(tokens, mig.blocks_migrated, S, 2)
            if fin_next:
                break
        copy_ms = (time.perf_counter() - t_start) * 1e3
        # final stage: the request is drained (no more decode steps for it), the last blocks move, it resumes on dst
        t0 = time.perf_counter_ns()
        n, fin, _ = mig.stage(table_r, tokens, stream=s_mig)  # handshake round (check, plan, PRE-ALLOC) + copy
        s_mig.synchronize()
        t1 = time.perf_counter_ns()
        dst_table = mig.commit(table_r[:-(-tokens // S)])
        downtime_us, commit_us = (t1 - t0) / 1e3, (time.perf_counter_ns() - t1) / 1e3
        assert fin and mig.state == llx.MIG_COMMITTED
        stages.append(n)
        # resume on the destination: attention of the request over (dst pool, dst table) == over (src pool, src table)
        bt1 = np.zeros((1, MB), dtype=np.int32)
        bt1[0, :len(dst_table)] = dst_table
        d_bt1, d_ctx1 = torch.from_numpy(bt1).cuda(), torch.tensor([tokens], dtype=torch.int32, device="cuda")
        o_src, o_dst = torch.zeros_like(q[:1]), torch.zeros_like(q[:1])
        llx.decode_attention(p.src, L - 1, q.data_ptr(), o_src.data_ptr(), d_bt.data_ptr(), d_ctx1.data_ptr(), 1, MB, scale, stream=s_dec)
        llx.decode_attention(p.dst, L - 1, q.data_ptr(), o_dst.data_ptr(), d_bt1.data_ptr(), d_ctx1.data_ptr(), 1, MB, scale, stream=s_dec)
        s_dec.synchronize()
        # the same count from the MEASURED rates (llx_predict_stage_sizes): copy rate of the non-final
        # stages in blocks/s, decode rate of this request = one token per step
        copy_rate = sum(stages[:-1]) / (copy_ms * 1e-3)
        decode_rate = 1e3 / (statistics.median(during) if during else before)
        out["runs"].append({
            "bandwidth_budget_GBps": budget, "stages_blocks": stages, "num_stages": len(stages),
            "predicted_stage_sizes_from_measured_rates": llx.predict_stage_sizes(stages[0], copy_rate, decode_rate, S),
            "measured_copy_blocks_per_s": copy_rate, "measured_decode_tokens_per_s": decode_rate,
            "tokens_at_start": tokens_at_start, "tokens_at_commit": tokens, "decode_steps_during_migration": len(during),
            "copy_phase_ms": copy_ms, "downtime_us_final_stage": downtime_us, "commit_us": commit_us,
            "decode_step_ms_before": before, "decode_step_ms_during": statistics.median(during) if during else None,
            "decode_slowdown_pct": 100.0 * (statistics.median(during) / before - 1.0) if during else None,
            "resume_on_destination_bit_identical": bool(torch.equal(o_src, o_dst)),
            "src_free_blocks_after": src_mgr.num_free, "dst_free_blocks_after": dst_mgr.num_free})
        del mig
    out["note"] = ("decode_slowdown_pct here is UNPAIRED (median step during the migration vs 8 steps before it, one host sync per "
                   "step) and good to about +-2 %; the paired figures are in interference_decode_batch32 / auto_budget_1pct")
    out["paper"] = "Llumnix Fig. 10: downtime 20-30 ms, always 2 stages, <= 1 % decode slowdown (A10, 64 Gb/s, PAPER.md:287-289)"
    del p
    _free(torch)
    return out


# ---- NEXT-1, the other variant the row names: an SM partition (green contexts) instead of pacing -----------------------
def green_partition(torch, llx, stream_unused=None, sm_counts=(8, 16)):
    """The migration gets its own few SMs (CUDA green context: cuDevSmResourceSplitByCount), the decode step the rest;
    inside its partition the migration runs unthrottled.  Paired slowdown of the configs[4] decode step, next to the
    same measurement for a CTA-capped launch on plain streams (LLX_OPT_MAX_CTAS).  Needs cuda-python."""
    try:
        from cuda.bindings import driver as drv
    except Exception as e:  # noqa: BLE001
        return {"skipped": "cuda-python unavailable: " + repr(e)}

    def ck(r):
        if r[0] != drv.CUresult.CUDA_SUCCESS:
            raise RuntimeError(str(r[0]))
        return r[1:] if len(r) > 2 else (r[1] if len(r) == 2 else None)

    g = dict(synth.CONFIGS["llama7b"])
    L, H, D, S = g["layers"], g["kv_heads"], g["head_dim"], g["block_size"]
    B, MB = 32, 256
    ctx = synth.context_lengths(4, B, 128, 4096)
    need = [-(-int(c) // S) for c in ctx]
    nb_src, nb_dst = B * 256 + 256, g["num_blocks"]
    if (nb_src + nb_dst) * 2 * L * S * H * D * 2 > _free(torch) - (4 << 30):
        return {"skipped": "not enough device memory"}
    p = Pools(torch, llx, g, nb_src, nb_dst)
    perm = synth.block_permutation(6, nb_src)
    bt = np.zeros((B, MB), dtype=np.int32)
    pos = 0
    for b, n in enumerate(need):
        bt[b, :n] = perm[pos:pos + n]
        pos += n
    mig_src, mig_dst = perm[pos:pos + 128], synth.block_permutation(2, nb_dst)[:128]
    q = torch.from_numpy(synth.queries_f16(5, B, H, D).view(np.int16)).cuda()
    o = torch.zeros_like(q)
    d_bt, d_ctx = torch.from_numpy(bt).cuda(), torch.from_numpy(ctx).cuda()
    scale = 1.0 / float(np.sqrt(D))
    mig_bytes = 2 * 128 * p.src.block_bytes

    def case(s_dec, s_mig, opts, n_mig):
        def one(nm):
            torch.cuda.synchronize()
            a, b_, ma, mb = (torch.cuda.Event(enable_timing=True) for _ in range(4))
            a.record(s_dec)
            ma.record(s_mig)
            for _ in range(nm):
                llx.migrate_stage(p.src, mig_src, p.dst, mig_dst, stream=s_mig, opts=opts)
            mb.record(s_mig)
            for l in range(L):
                llx.decode_attention(p.src, l, q.data_ptr(), o.data_ptr(), d_bt.data_ptr(), d_ctx.data_ptr(), B, MB, scale, stream=s_dec)
            b_.record(s_dec)
            torch.cuda.synchronize()
            return a.elapsed_time(b_), ma.elapsed_time(mb)
        for _ in range(3):
            one(0)
        ratios, mig_ms = [], []
        for _ in range(8):
            t0, _ = one(0)
            t1, m = one(n_mig)
            ratios.append(t1 / t0)
            mig_ms.append(m)
        return {"decode_slowdown_pct": 100.0 * (statistics.median(ratios) - 1.0),
                "migration_GBps": n_mig * mig_bytes / statistics.median(mig_ms) / 1e6 if n_mig else 0.0}

    res = {"cases": []}
    lo, hi = torch.cuda.Stream.priority_range()
    sd, sm = torch.cuda.Stream(priority=hi), torch.cuda.Stream(priority=lo)
    for c in sm_counts:
        r = case(sd, sm, dict(max_ctas=c), 8)
        res["cases"].append(dict(r, case=f"plain streams, {c} full-speed CTAs (LLX_OPT_MAX_CTAS)"))
    dev = ck(drv.cuDeviceGet(torch.cuda.current_device()))
    sm_res = ck(drv.cuDeviceGetDevResource(dev, drv.CUdevResourceType.CU_DEV_RESOURCE_TYPE_SM))
    res["device_sms"] = int(sm_res.sm.smCount)
    for c in sm_counts:
        try:
            groups, _, remaining = ck(drv.cuDevSmResourceSplitByCount(1, sm_res, 0, c))
            streams = []
            for part in (groups[0], remaining):
                desc = ck(drv.cuDevResourceGenerateDesc([part], 1))
                gctx = ck(drv.cuGreenCtxCreate(desc, dev, drv.CUgreenCtxCreate_flags.CU_GREEN_CTX_DEFAULT_STREAM))
                streams.append(torch.cuda.ExternalStream(int(ck(drv.cuGreenCtxStreamCreate(gctx, drv.CUstream_flags.CU_STREAM_NON_BLOCKING, 0)))))
        except Exception as e:  # noqa: BLE001
            res["cases"].append({"case": f"green context with {c} SMs", "skipped": repr(e)})
            continue
        r = case(streams[1], streams[0], None, 8)
        res["cases"].append(dict(r, case=f"green contexts: {int(groups[0].sm.smCount)} SMs migrate at full speed, {int(remaining.sm.smCount)} SMs decode"))
        r = case(streams[1], streams[0], None, 0)
        res["cases"].append(dict(r, case=f"green contexts: decode alone on its {int(remaining.sm.smCount)} SMs, paired with itself (floor)"))
    del p
    _free(torch)
    return res


# ---- NEXT-2 / SURVEY 8(e): tensor-parallel rank shards of LLaMA-30B (52 heads = 4 ranks x 13 -> 52 KiB tiles) ----------
def tp_shard_30b(torch, llx, stream_unused=None, tp=4, n=128, nb=700):
    """Rank r of the source instance migrates to rank r of the destination, no exchange between ranks (PAPER.md:235,
    :254).  On ONE GPU the four rank pairs are four pool pairs on four streams; reported: one rank's stage alone, and
    the four ranks' stages in flight together (they share this GPU's HBM; on a TP=4 node each rank has its own)."""
    g = dict(synth.CONFIGS["llama30b"])
    g["kv_heads"] //= tp
    pools = [Pools(torch, llx, g, nb, nb) for _ in range(tp)]
    streams = [torch.cuda.Stream() for _ in range(tp)]
    s_tab, d_tab = synth.block_permutation(1, nb)[:n], synth.block_permutation(2, nb)[:n]
    by = 2 * n * pools[0].src.block_bytes
    one = _time_stream(torch, streams[0], lambda: llx.migrate_stage(pools[0].src, s_tab, pools[0].dst, d_tab, stream=streams[0]))
    for _ in range(2):
        for r in range(tp):
            llx.migrate_stage(pools[r].src, s_tab, pools[r].dst, d_tab, stream=streams[r])
    torch.cuda.synchronize()
    ts = []
    for _ in range(10):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(streams[0])
        for r in range(1, tp):
            streams[r].wait_event(a)
        for r in range(tp):
            llx.migrate_stage(pools[r].src, s_tab, pools[r].dst, d_tab, stream=streams[r])
        for r in range(1, tp):
            e = torch.cuda.Event()
            e.record(streams[r])
            streams[0].wait_event(e)
        b.record(streams[0])
        torch.cuda.synchronize()
        ts.append(a.elapsed_time(b))
    t4 = statistics.median(ts)
    fin = _time_stream(torch, streams[0], lambda: llx.migrate_stage(pools[0].src, s_tab[:2], pools[0].dst, d_tab[:2], stream=streams[0]), reps=20)
    res = {"tp": tp, "kv_heads_per_rank": g["kv_heads"], "tile_KiB": pools[0].src.tile_bytes / 1024, "blocks": n,
           "payload_per_rank_MiB": n * pools[0].src.block_bytes / 2**20,
           "one_rank_alone_GBps": by / one["median_ms"] / 1e6, "one_rank_alone_ms": one["median_ms"],
           "four_ranks_concurrent_total_GBps": tp * by / t4 / 1e6, "four_ranks_concurrent_ms": t4,
           "final_stage_2_blocks_gpu_us_warm": fin["median_ms"] * 1e3,
           "note": "one GPU stands in for the four GPUs of a TP=4 instance pair: the concurrent figure is four rank-local stages sharing ONE HBM"}
    del pools
    _free(torch)
    return res


# ---- launches for the ncu metric pass of profiles/ (each shape twice: the first launch warms up, ncu reads the second) --
def ncu_targets(torch, llx, stream):
    """Launches, in this order and twice each, the kernel shapes the ncu evidence covers beyond bench.py's own step:
      1 llx_copy_bulk   LLaMA-30B batch, 64 requests / 1023 blocks in ONE launch (208 KiB tiles)
      2 llx_copy_bulk   llx_pack of a 2048-token 7B request into a DEVICE buffer          3 llx_copy_bulk  llx_unpack of it
      4 llx_copy_vec16  paced stage, 25 GB/s budget (16 blocks of 7B)                     5 llx_copy_vec16 paced, 400 GB/s
      6 llx_copy_bulk   long stage of Tiny-shaped 8 KiB tiles (8000 blocks, 250 MiB: larger than L2)
      7 llx_copy_bulk   the final stage: 2 blocks of 7B (cold: a 512 MiB fill runs before it)
      8 llx_copy_vec16  peer route of a 2048-token 7B request on one device
      9 llx_copy_vec16  zero-copy llx_pack into pinned host memory (16 blocks)           10 llx_copy_vec16 zero-copy llx_unpack
    and prints the order so that the launch list can be labelled."""
    out = []
    flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")

    def twice(label, fn, cold=False):
        for _ in range(2):
            if cold:
                with torch.cuda.stream(stream):
                    flush.fill_(1)
            fn()
        stream.synchronize()
        out.append(label)

    g30 = dict(synth.CONFIGS["llama30b"])
    lens, nblk, _ = synth.batch_request_blocks(0, 64, g30["block_size"], g30["num_blocks"])
    total = int(nblk.sum())
    p30 = Pools(torch, llx, g30, total + 50, total + 50)
    off = np.concatenate([[0], np.cumsum(nblk)]).astype(np.int32)
    s30, d30 = synth.block_permutation(1, total + 50)[:total], synth.block_permutation(2, total + 50)[:total]
    twice("batch_30b_1023_blocks", lambda: llx.migrate_batch(p30.src, p30.dst, off, s30, d30, stream=stream))
    del p30
    _free(torch)

    g7 = synth.CONFIGS["llama7b"]
    p7 = Pools(torch, llx, g7, 600, 600)
    s7, d7 = synth.block_permutation(1, 600)[:128], synth.block_permutation(2, 600)[:128]
    stg = torch.empty(llx.staging_bytes(p7.src, 128), dtype=torch.uint8, device="cuda")
    twice("pack_device_128_blocks", lambda: llx.pack(p7.src, s7, stg.data_ptr(), stg.numel(), stream=stream))
    twice("unpack_device_128_blocks", lambda: llx.unpack(stg.data_ptr(), stg.numel(), p7.dst, d7, stream=stream))
    twice("paced_25GBps_16_blocks", lambda: llx.migrate_stage(p7.src, s7[:16], p7.dst, d7[:16], stream=stream, opts=dict(bandwidth_gbps=25)))
    twice("paced_400GBps_16_blocks", lambda: llx.migrate_stage(p7.src, s7[:16], p7.dst, d7[:16], stream=stream, opts=dict(bandwidth_gbps=400)))
    gt = dict(synth.CONFIGS["tiny"])
    pt = Pools(torch, llx, gt, 8400, 8400)        # 8000 blocks of 32 KiB = 250 MiB read + 250 MiB written: twice the 126 MB L2
    st_, dt_ = synth.block_permutation(1, 8400)[:8000], synth.block_permutation(2, 8400)[:8000]
    twice("tiny_tiles_8KiB_8000_blocks", lambda: llx.migrate_stage(pt.src, st_, pt.dst, dt_, stream=stream))
    twice("final_stage_2_blocks_cold", lambda: llx.migrate_stage(p7.src, s7[126:], p7.dst, d7[126:], stream=stream), cold=True)
    twice("peer_route_128_blocks", lambda: llx.migrate_stage(p7.src, s7, p7.dst, d7, stream=stream, opts=dict(route=llx.ROUTE_PEER)))
    pin = llx.PinnedStaging(llx.staging_bytes(p7.src, 16))
    zc = dict(via_host_mode=1)          # the kernel itself crosses the host link: the only host leg a kernel profiler can see
    twice("pack_zero_copy_pinned_host_16_blocks", lambda: llx.pack(p7.src, s7[:16], pin.dev_alias, pin.nbytes, stream=stream, opts=zc))
    twice("unpack_zero_copy_pinned_host_16_blocks", lambda: llx.unpack(pin.dev_alias, pin.nbytes, p7.dst, d7[:16], stream=stream, opts=zc))
    pin.free()
    # small tiles: the tensor-map kernel (copy_kernel = 3) next to the default, the 1-D ring
    twice("tiny_tiles_8KiB_8000_blocks_tensor_map", lambda: llx.migrate_stage(pt.src, st_, pt.dst, dt_, stream=stream, opts=dict(copy_kernel=3)))
    del p7, pt
    _free(torch)
    g16 = dict(layers=32, kv_heads=4, head_dim=128, block_size=16, elem_bytes=2, num_blocks=4400)
    p16 = Pools(torch, llx, g16, 4400, 4400)
    s16, d16 = synth.block_permutation(1, 4400)[:4000], synth.block_permutation(2, 4400)[:4000]
    twice("tiles_16KiB_4000_blocks_6_stages_round1", lambda: llx.migrate_stage(p16.src, s16, p16.dst, d16, stream=stream, opts=dict(ring_stages=6)))
    twice("tiles_16KiB_4000_blocks", lambda: llx.migrate_stage(p16.src, s16, p16.dst, d16, stream=stream))
    twice("tiles_16KiB_4000_blocks_tensor_map", lambda: llx.migrate_stage(p16.src, s16, p16.dst, d16, stream=stream, opts=dict(copy_kernel=3)))
    del p16
    _free(torch)
    # a TP=4 rank shard of LLaMA-30B (13 heads, 52 KiB tiles): "32 KiB, then the rest" next to the computed shape (4 equal chunks, 6 stages)
    g52 = dict(synth.CONFIGS["llama30b"], kv_heads=13, num_blocks=400)
    p52 = Pools(torch, llx, g52, 400, 400)
    s52, d52 = synth.block_permutation(1, 400)[:128], synth.block_permutation(2, 400)[:128]
    twice("tp4_shard_52KiB_128_blocks_32K_then_rest", lambda: llx.migrate_stage(p52.src, s52, p52.dst, d52, stream=stream,
                                                                                 opts=dict(chunk_bytes=32768, ring_stages=3)))
    twice("tp4_shard_52KiB_128_blocks", lambda: llx.migrate_stage(p52.src, s52, p52.dst, d52, stream=stream))
    return {"order": out, "note": "each label = two consecutive launches of that shape; llx_fill / at:: kernels in between are input generation"}


# ---- small tiles (TP-sharded / GQA caches): the 1-D ring next to the tensor-map kernel ------------------------------
def small_tiles(torch, llx, stream):
    """Long pool-to-pool stages of 4, 8 and 16 KiB tiles (one KV head per rank ... four), scattered ids, by CUDA events:
    copy_kernel = 2 (1-D bulk ring; 4 / 2 / 1 CTAs per SM, ring depth from the loads-in-flight rule) against copy_kernel = 3
    (the same ring fed by 4-D tensor-map boxes of 32 KiB), against what the library picks by itself (the 1-D ring) and
    against the 1-D ring with round 1's ring depths (4 / 4 / 6 stages)."""
    out = []
    for label, L, H, nb, n in (("4 KiB tiles, 64 slices (1 KV head of 128)", 32, 1, 33000, 30000),
                               ("8 KiB tiles, 4 slices (Tiny)", 2, 4, 8400, 8000),
                               ("8 KiB tiles, 80 slices (2 KV heads of 128)", 40, 2, 9000, 8000),
                               ("16 KiB tiles, 64 slices (4 KV heads of 128)", 32, 4, 4400, 4000)):
        D = 64 if H == 4 and L == 2 else 128
        g = dict(layers=L, kv_heads=H, head_dim=D, block_size=16, elem_bytes=2, num_blocks=nb)
        p = Pools(torch, llx, g, nb, nb)
        s_ids, d_ids = synth.block_permutation(1, nb)[:n], synth.block_permutation(2, nb)[:n]
        row = {"shape": label, "blocks": n, "payload_MiB": n * p.src.block_bytes / 2**20}
        old_depth = 6 if p.src.tile_bytes >= 16384 else 4
        for name, o in (("ring_1d", dict(copy_kernel=2)), ("tensor_map", dict(copy_kernel=3)), ("default", None),
                        ("ring_1d_round1_depth", dict(copy_kernel=2, ring_stages=old_depth))):
            t = _time_stream(torch, stream, lambda: llx.migrate_stage(p.src, s_ids, p.dst, d_ids, stream=stream, opts=o), reps=12, warm=3)
            row[name + "_GBps"] = 2 * n * p.src.block_bytes / (t["median_ms"] * 1e-3) / 1e9
        out.append(row)
        del p
        _free(torch)
    return out


def link_peak(torch, nbytes=1 << 30, reps=10):
    """Host-link peak measured in THIS run: best of `reps` plain 1 GiB pinned copy-engine transfers each way, and both ways
    at once on two streams (the full-duplex floor a round trip through the host is held against)."""
    dev_a = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    dev_b = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    host_a = torch.empty(nbytes, dtype=torch.uint8).pin_memory()
    host_b = torch.empty(nbytes, dtype=torch.uint8).pin_memory()
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    torch.cuda.synchronize()
    res = {"bytes_each_way": nbytes, "reps": reps}
    with torch.cuda.stream(s1):
        t = _time_stream(torch, s1, lambda: host_a.copy_(dev_a, non_blocking=True), reps=reps, warm=1)
        res["d2h_GBps"] = nbytes / t["min_ms"] / 1e6
        t = _time_stream(torch, s1, lambda: dev_b.copy_(host_b, non_blocking=True), reps=reps, warm=1)
        res["h2d_GBps"] = nbytes / t["min_ms"] / 1e6
    both = []
    for _ in range(reps + 1):
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(s1)
        s2.wait_event(a)
        with torch.cuda.stream(s1):
            host_a.copy_(dev_a, non_blocking=True)
        with torch.cuda.stream(s2):
            dev_b.copy_(host_b, non_blocking=True)
        s1.wait_stream(s2)
        b.record(s1)
        torch.cuda.synchronize()
        both.append(a.elapsed_time(b))
    t_both = min(both[1:])
    res["duplex_ms_per_GiB_each_way"] = t_both * (1 << 30) / nbytes
    res["duplex_GBps_both_directions_summed"] = 2 * nbytes / t_both / 1e6
    del dev_a, dev_b, host_a, host_b
    return res


def baseline_configs(torch, llx, stream):
    """The BASELINE.json configs other than configs[1], bounded for bench.py's default line (about a minute in all):
    configs[2] the length sweep, configs[3] the LLaMA-30B batch (the config's draw and the draw whose sample mean is the
    nominal 512 tokens), configs[4] the batch-32 decode step alone / next to an unthrottled migration / next to a 25 and
    a 12 GB/s budget (paired, with the power state), SURVEY 8(d)'s reference points.  Numbers only; the long notes stay
    in the full legs (`bench.py --suite`)."""
    out = {}
    g = synth.CONFIGS["llama7b"]
    nb = g["num_blocks"]
    p = Pools(torch, llx, g, nb, nb)
    sweep = length_sweep(torch, llx, p, stream, nb)
    out["configs2_length_sweep_llama7b"] = [
        {"tokens": r["tokens"], "single_shot_GBps": round(r["single_shot_GBps"], 1), "stage0_GBps": round(r["stage0_GBps"], 1),
         "final_stage_gpu_us_cold": round(r["final_stage_gpu_us_cold"], 2), "final_stage_host_us_median": round(r["final_stage_host_us_median"], 2),
         "blocking_copy_downtime_us": round(r["blocking_copy_downtime_us"], 1)} for r in sweep]
    refs = reference_points(torch, llx, p, stream, nb)
    out["reference_points_2048tok_GBps"] = {k: round(v, 1) for k, v in refs.items() if k.endswith("_GBps")}
    del p
    _free(torch)
    b = {}
    for name, seed in (("seed0_as_specified", 0), ("seed2_sample_mean_507tok", 2)):
        r = batch_30b(torch, llx, stream, seed=seed)
        b[name] = r if "skipped" in r else {k: (round(r[k], 2) if isinstance(r[k], float) else r[k]) for k in
                                            ("total_blocks", "payload_GiB", "mean_tokens", "one_launch_ms", "one_launch_GBps", "sequential_GBps")}
    out["configs3_batch_llama30b_64req"] = b
    r = interference(torch, llx, stream, budgets=(25, 12))
    if "skipped" in r:
        out["configs4_interference_decode_batch32"] = r
    else:
        out["configs4_interference_decode_batch32"] = {
            "decode_step_alone_ms": round(r["decode_step_alone_ms"], 4), "decode_attention_GBps": round(r["decode_attention_GBps"], 1),
            "migration_alone_GBps": round(r["migration_alone_GBps"], 1),
            "cases": [{"case": c["case"], "budget_GBps": c["bandwidth_budget_GBps"], "decode_step_ms": round(c["decode_step_ms"], 4),
                       "slowdown_pct": round(c["slowdown_pct"], 2), "migration_GBps": round(c["migration_GBps_while_overlapped"], 1)}
                      for c in r["cases"]],
            "power_state_before": r["power_state_before_cases"], "power_state_after": r["power_state_after_cases"],
            "method": "paired: each step next to a migration follows an isolated step; median of 8 per-pair ratios"}
    return out


def run(torch, llx, stream):
    res = {}
    g = synth.CONFIGS["llama7b"]
    nb = g["num_blocks"]
    p = Pools(torch, llx, g, nb, nb)
    res["length_sweep_llama7b"] = length_sweep(torch, llx, p, stream, nb)
    res["latency_floor"] = latency_floor(torch, llx, p, stream, nb)
    res["reference_points_2048tok"] = reference_points(torch, llx, p, stream, nb)
    res["staging_pinned_host_2048tok"] = staging_host(torch, llx, p, stream, nb)
    del p
    _free(torch)
    res["interference_decode_batch32"] = interference(torch, llx, stream)
    res["auto_budget_1pct"] = auto_budget(torch, llx, stream, target_pct=1.0)
    res["interference_sustained_decoding"] = interference_sustained(torch, llx, stream)
    res["budget_controller_live_1pct"] = budget_controller_live(torch, llx, stream)
    res["live_migration_during_decode"] = live_migration(torch, llx, stream)
    res["batch_llama30b_64req"] = batch_30b(torch, llx, stream)
    res["batch_llama30b_64req_seed2_mean507"] = batch_30b(torch, llx, stream, seed=2)
    res["tp4_rank_shards_llama30b"] = tp_shard_30b(torch, llx, stream)
    res["small_tiles_ring_1d_vs_tensor_map"] = small_tiles(torch, llx, stream)
    res["sm_partition_green_contexts"] = green_partition(torch, llx, stream)
    return res


def main():
    """python bench_suite.py [--only NAME]   (NAME: sweep | refs | staging | interference | autobudget | live | batch | batch2 | sustained | controller | tp | small | green | floor | ncu_targets)"""
    import argparse
    import json

    import torch

    import paper_2406_03243_b200 as llx
    ap = argparse.ArgumentParser()
    ap.add_argument("--only", default="")
    ap.add_argument("--carveout", type=int, default=-1,
                    help="LLX_OPT_COPY_SMEM_CARVEOUT_PCT for this run (the sweep behind its default: 0, 50, 64, 75, 100)")
    args = ap.parse_args()
    llx.load()
    if args.carveout >= 0:
        llx.set_option(llx.OPT_COPY_SMEM_CARVEOUT_PCT, args.carveout)
    stream = torch.cuda.Stream()
    if not args.only:
        print(json.dumps(run(torch, llx, stream), indent=1))
        return 0
    g = synth.CONFIGS["llama7b"]
    nb = g["num_blocks"]
    if args.only == "interference":
        res = interference(torch, llx, stream)
    elif args.only == "autobudget":
        res = auto_budget(torch, llx, stream)
    elif args.only == "live":
        res = live_migration(torch, llx, stream)
    elif args.only == "batch":
        res = batch_30b(torch, llx, stream)
    elif args.only == "batch2":
        res = batch_30b(torch, llx, stream, seed=2)
    elif args.only == "tp":
        res = tp_shard_30b(torch, llx, stream)
    elif args.only == "sustained":
        res = interference_sustained(torch, llx, stream)
    elif args.only == "controller":
        res = budget_controller_live(torch, llx, stream)
    elif args.only == "green":
        res = green_partition(torch, llx, stream)
    elif args.only == "small":
        res = small_tiles(torch, llx, stream)
    elif args.only == "ncu_targets":
        res = ncu_targets(torch, llx, stream)
    else:
        p = Pools(torch, llx, g, nb, nb)
        fn = {"sweep": length_sweep, "refs": reference_points, "staging": staging_host, "floor": latency_floor}[args.only]
        res = fn(torch, llx, p, stream, nb)
    print(json.dumps(res, indent=1))
    return 0


if __name__ == "__main__":
    sys.exit(main())
