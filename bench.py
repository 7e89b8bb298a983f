#!/usr/bin/env python
"""bench.py — KV-cache live-migration throughput on B200 (BASELINE.json metric).

One STEP = one pass of the hot path over BASELINE.json configs[1] (LLaMA-7B shape): a 2048-token request
(128 scattered blocks of 8 MiB) migrated between two 2000-block pools in 3 stages (112, 14, then the 2
final blocks) with 8 new tokens appended to the source between stages — S1 planning check, S3 stages,
S8 appends and the S4 final stage, all through the C-ABI (libllx.so).  The copies run on the migration
stream, the appends on a second "decode" stream, as in the paper ("continues the computation at the same
time"; "another CUDA stream"): a stage waits for an append only when it reads
the appended block, i.e. the final stage does.  Both streams lie inside the event-bracketed region; nothing
is removed from the step (`--serial-appends` puts the appends back on the migration stream for comparison).

    value     GB/s, bytes read + written by the three stage copies / device time of the whole step
              (pools resident in HBM; CUDA events on the launching stream; max over ranks)
    e2e       the same request migrated THROUGH HOST BUFFERS: llx_migrate_via_host moves it into a pinned host staging
              buffer (D2H) and out of it into the destination's blocks (H2D), both directions of the link at once — the
              paper's GPU->CPU buffer->GPU route.  Default host leg: one pitched copy-engine transfer
              per block (no kernel); the gather/scatter-kernel route through bounce buffers and the plain
              llx_pack -> llx_unpack pair are reported beside it
    roofline  the dominant kernel (stage 0: 112 blocks, 1.75 GiB of traffic) against the measured HBM peak
    cpu_baseline / --impl reference   the NumPy oracle timed on the host cores on a bounded sample

`--suite` adds the other BASELINE.json configs (length sweep, 30B batch, interference + staging) as
extra JSON lines on stderr and in gpurun_out/suite.json; the ONE stdout line keeps the contract.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import synth  # noqa: E402

METRIC = "kv_migration_gbps_rd_plus_wr"
UNIT = "GB/s"
WORKLOAD = "llama7b_2048tok_3stage_112_14_2"
SCHEDULE, APPENDS, START_TOKENS = (112, 14, 2), (8, 8), 2032
NOMINAL_HBM_GBS = 8000.0
FALLBACK_HBM_GBS = 6650.0       # B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent


# --------------------------------------------------------------------------------------------
# clocks: sampled with NVML in a thread DURING the timed regions
# --------------------------------------------------------------------------------------------
class ClockSampler:
    REASONS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap",
               0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting", 0x10: "sync_boost"}

    def __init__(self, index: int):
        self.samples, self.windows, self._stop, self.ok = [], [], threading.Event(), False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            phys = int(vis.split(",")[index]) if vis and vis.split(",")[index].isdigit() else index
            self.h = pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception as e:  # noqa: BLE001
            self.err = repr(e)
        self.t = threading.Thread(target=self._run, daemon=True)

    def _run(self):
        nv = self.nv
        while not self._stop.is_set():
            try:
                mhz = nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:  # noqa: BLE001
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                self.samples.append((time.perf_counter(), mhz, r))
            except Exception:  # noqa: BLE001
                pass
            time.sleep(0.01)

    def start(self):
        if self.ok:
            self.t.start()

    def window(self, t0, t1):
        self.windows.append((t0, t1))

    def stop(self) -> dict:
        if not self.ok:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "error": getattr(self, "err", "")}
        self._stop.set()
        self.t.join(timeout=2)
        inside = [(m, r) for (t, m, r) in self.samples if any(a <= t <= b for a, b in self.windows)]
        use = inside if inside else [(m, r) for (_, m, r) in self.samples]
        bits = 0
        for _, r in use:
            bits |= r
        reasons = sorted(n for b, n in self.REASONS.items() if bits & b)
        return {"sm_mhz": statistics.median([m for m, _ in use]) if use else None, "sm_max_mhz": self.max_mhz,
                "reasons": reasons, "samples_in_timed_regions": len(inside), "samples": len(self.samples)}


def profiled_traffic(launch="stage0_112_blocks"):
    """dram__bytes_read.sum + dram__bytes_write.sum of the dominant kernel, per launch, from the newest committed
    `ncu --set full` capture (profiles/rNN_copy_bulk_traffic.csv; its `commit` column names the commit the capture
    was taken at — a run does not re-measure it)."""
    import csv
    import glob
    for path in sorted(glob.glob(os.path.join(ROOT, "profiles", "r*_copy_bulk_traffic.csv")), reverse=True):
        try:
            with open(path) as f:
                for row in csv.DictReader(f):
                    if row["launch"] == launch:
                        return {"bytes": int(row["dram_bytes_read"]) + int(row["dram_bytes_write"]),
                                "source": os.path.relpath(path, ROOT) + " (ncu --set full)",
                                "commit": row.get("commit") or "round-1 capture (before the kernel-shape commits d0dd35d, ccc79b2, 2c0d0bf)"}
        except Exception:  # noqa: BLE001
            continue
    return {"bytes": None, "source": None, "commit": None}


def measured_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, torch copy_ rd+wr)"
    except Exception:  # noqa: BLE001
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


# --------------------------------------------------------------------------------------------
# the oracle on the host cores (cpu_baseline leg and --impl reference)
# --------------------------------------------------------------------------------------------
def oracle_sample_setup(pool_blocks=160):
    """configs[1]'s request (128 scattered blocks, LLaMA-7B tiles) inside two host pools shrunk to
    `pool_blocks` blocks so that they fit host RAM (2 x 1.25 GiB); same schedule and appends."""
    from oracle import kv_migration as om
    g = synth.CONFIGS["llama7b"]
    te = g["block_size"] * g["kv_heads"] * g["head_dim"]
    src = om.new_pool(g["layers"], pool_blocks, te)
    for l in range(g["layers"]):
        # seeded fp16 bit patterns; one slice generated and rolled per layer to keep the setup short
        base = synth.slice_values_f16(0, 0, l, 0, pool_blocks, te)
        src[l, 0] = base
        src[l, 1] = np.roll(base, 1, axis=0)
    dst = om.new_pool(g["layers"], pool_blocks, te, fill=synth.SENTINEL_U16)
    s_tab = synth.block_permutation(1, pool_blocks)[:128]
    d_tab = synth.block_permutation(2, pool_blocks)[:128]
    te_tok = g["kv_heads"] * g["head_dim"]
    vals = np.empty((16, g["layers"], 2, te_tok), dtype=np.uint16)      # the appended tokens: the generator the tests use
    for t in range(16):
        for l in range(g["layers"]):
            for kv in range(2):
                vals[t, l, kv] = synth.append_values_f16(3, START_TOKENS + t, l, kv, te_tok)
    values = lambda t, l, kv: vals[t - START_TOKENS, l, kv]
    return om, g, src, dst, s_tab, d_tab, values


def oracle_step(ctx):
    om, g, src, dst, s_tab, d_tab, values = ctx
    t0 = time.perf_counter()
    om.staged_migration(src, s_tab, dst, d_tab, SCHEDULE, APPENDS, g["block_size"], START_TOKENS, values)
    return time.perf_counter() - t0


def step_bytes(g) -> int:
    block_bytes = 2 * g["layers"] * g["block_size"] * g["kv_heads"] * g["head_dim"] * g["elem_bytes"]
    return 2 * sum(SCHEDULE) * block_bytes          # read + written


def attention_oracle_sample() -> dict:
    """oracle.decode_attention.decode_attention_fp64 timed on ONE sequence of 2048 context tokens, one layer, LLaMA-7B heads
    (a bounded sample of configs[4]'s decode batch: 32 sequences, 128..4096 tokens, 32 layers)."""
    from oracle.decode_attention import decode_attention_fp64
    g = synth.CONFIGS["llama7b"]
    S, H, D = g["block_size"], g["kv_heads"], g["head_dim"]
    nb, te = 128, S * H * D
    pool = np.empty((1, 2, nb, te), dtype=np.uint16)
    for kv in range(2):
        pool[0, kv] = synth.slice_values_f16(4, 0, 0, kv, nb, te)
    q = synth.queries_f16(5, 1, H, D)
    bt = synth.block_permutation(6, nb)[:nb].reshape(1, nb).astype(np.int32)
    ctx = np.array([nb * S], dtype=np.int32)
    t0 = time.perf_counter()
    decode_attention_fp64(pool, 0, q, bt, ctx, S, H, D)
    dt = time.perf_counter() - t0
    return {"kind": "oracle", "cores": 1, "sample": "one sequence of 2048 context tokens, one layer, 32 heads x 128 dims (fp64)",
            "ms": dt * 1e3, "context_tokens_per_s": nb * S / dt}


def cpu_baseline(budget_s=12.0) -> dict:
    ctx = oracle_sample_setup()
    g = ctx[1]
    times = [oracle_step(ctx)]
    while sum(times) < budget_s and len(times) < 50:
        times.append(oracle_step(ctx))
    t = statistics.median(times)
    # the final stage alone on the host (context for the paper's downtime figure)
    om, _, src, dst, s_tab, d_tab, _ = ctx
    fin = []
    for _ in range(5):
        t0 = time.perf_counter()
        om.migrate_stage(src, s_tab[-SCHEDULE[-1]:], dst, d_tab[-SCHEDULE[-1]:])
        fin.append(time.perf_counter() - t0)
    # block fusion on the host: the oracle's pack and unpack of the whole 128-block request
    t0 = time.perf_counter()
    buf = om.pack(src, s_tab)
    t_pack = time.perf_counter() - t0
    t0 = time.perf_counter()
    om.unpack(buf, dst, d_tab)
    t_unpack = time.perf_counter() - t0
    del buf
    return {"value": step_bytes(g) / t / 1e9, "unit": UNIT, "cores": 1, "kind": "oracle",
            "host_cores_available": len(os.sched_getaffinity(0)),
            "final_stage_ms": statistics.median(fin) * 1e3, "pack_ms": t_pack * 1e3, "unpack_ms": t_unpack * 1e3,
            "attention_oracle": attention_oracle_sample(),
            "sample": f"the whole configs[1] step (128 blocks, stages 112/14/2, 2 appends of 8 tokens) inside two "
                      f"160-block host pools instead of 2000-block ones; {len(times)} repetitions, median; "
                      f"oracle.kv_migration.staged_migration as it stands (NumPy row copies, single thread)",
            "ms_per_step": t * 1e3}


def cpu_baseline_all_cores(budget_s=8.0) -> dict:
    """The oracle as it stands over a thread pool: one task per layer (the oracle's pool shape keeps K and V of a layer
    together), `host_cores_available` threads; NumPy's row copies release the GIL.  Same sample as cpu_baseline."""
    from concurrent.futures import ThreadPoolExecutor
    om, g, src, dst, s_tab, d_tab, values = oracle_sample_setup()
    cores = len(os.sched_getaffinity(0))
    L = g["layers"]

    def one_layer(l):
        om.staged_migration(src[l:l + 1], s_tab, dst[l:l + 1], d_tab, SCHEDULE, APPENDS, g["block_size"], START_TOKENS,
                            lambda t, _l, kv: values(t, l, kv))

    times = []
    with ThreadPoolExecutor(max_workers=cores) as ex:
        while sum(times) < budget_s and len(times) < 50:
            t0 = time.perf_counter()
            list(ex.map(one_layer, range(L)))
            times.append(time.perf_counter() - t0)
    t = statistics.median(times)
    return {"value": step_bytes(g) / t / 1e9, "unit": UNIT, "cores": min(cores, L), "kind": "oracle",
            "host_cores_available": cores, "ms_per_step": t * 1e3,
            "sample": f"the cpu_baseline sample; oracle.kv_migration.staged_migration per layer over a pool of {cores} threads "
                      f"({L} tasks), {len(times)} repetitions, median"}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    ctx = oracle_sample_setup()
    g = ctx[1]
    for _ in range(args.warmup):
        oracle_step(ctx)
    steps = min(args.steps, 2000)       # ~0.13 s per step: the default 1000 steps take about two minutes
    t0 = time.perf_counter()
    for _ in range(steps):
        oracle_step(ctx)
    dt = (time.perf_counter() - t0) / steps
    val = step_bytes(g) / dt / 1e9
    sample = ("configs[1] step (128 blocks, stages 112/14/2, appends 8+8) inside two 160-block host pools; "
              f"{steps} timed steps after {args.warmup} warm-up steps")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
        "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "u16", "data": "synthetic",
        "config": {"workload": WORKLOAD, "pools": "2 x 160 host blocks (sample)", "note": "CPU oracle, host memory"},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))
    return 0


# --------------------------------------------------------------------------------------------
# the llx arm
# --------------------------------------------------------------------------------------------
class Workload:
    """Two LLaMA-7B-shaped pools on the current device and the configs[1] request."""

    def __init__(self, torch, llx, cfg="llama7b", num_blocks=None, src_blocks=None, overlap=True):
        g = dict(synth.CONFIGS[cfg])
        if num_blocks:
            g["num_blocks"] = num_blocks
        self.g, self.torch, self.llx = g, torch, llx
        L, H, D, S = g["layers"], g["kv_heads"], g["head_dim"], g["block_size"]
        self.nb_dst = g["num_blocks"]
        self.nb_src = src_blocks or g["num_blocks"]
        self.te = S * H * D
        self.src_raw, self.src = self._pool(self.nb_src)
        self.dst_raw, self.dst = self._pool(self.nb_dst)
        # seeded synthetic fill on the device: fp16 U[-1,1) (input generation, not part of the path)
        gen = torch.Generator(device="cuda")
        gen.manual_seed(0)
        flat = self.src_raw.view(torch.float16)
        step = 1 << 28
        for a in range(0, flat.numel(), step):
            b = min(flat.numel(), a + step)
            flat[a:b] = (torch.rand(b - a, generator=gen, device="cuda", dtype=torch.float32) * 2 - 1).half()
        self.dst_raw.view(torch.int16).fill_(int(np.array(synth.SENTINEL_U16, np.uint16).view(np.int16)))
        # two requests of 128 scattered blocks each: consecutive steps migrate them alternately ("the llumlet ... starts
        # to migrate requests to the destination continuously") — every step is one whole configs[1] request
        ps, pd = synth.block_permutation(1, self.nb_src), synth.block_permutation(2, self.nb_dst)
        self.s_tabs, self.d_tabs = (ps[:128], ps[128:256]), (pd[:128], pd[128:256])
        self.s_tab, self.d_tab = self.s_tabs[0], self.d_tabs[0]
        te_tok = H * D
        vals = np.empty((16, L, 2, te_tok), dtype=np.uint16)
        for t in range(16):
            for l in range(L):
                for kv in range(2):
                    vals[t, l, kv] = synth.append_values_f16(3, START_TOKENS + t, l, kv, te_tok)
        self.append_host = torch.from_numpy(vals.view(np.int16)).pin_memory()
        self.append_dev = self.append_host.cuda()
        self.e_mid = (torch.cuda.Event(), torch.cuda.Event())
        self.e_app = (torch.cuda.Event(), torch.cuda.Event())
        # Non-final stages are declared independent of the kernel before them (llx_launch_opts.overlap_prev): stage 0 reads
        # and writes other blocks than the previous request's final stage, stage 1 other blocks than stage 0, and full
        # blocks are never written again.  Completion order on the stream is unchanged.  The final stage
        # keeps plain stream order (it reads the block the appends wrote).
        self.stage_opts = llx.LaunchOpts(overlap_prev=1) if overlap else None
        self.k, self.primed = 0, False
        torch.cuda.synchronize()

    def _pool(self, nb):
        g, torch, llx = self.g, self.torch, self.llx
        nbytes = llx.pool_bytes_for(g["layers"], g["kv_heads"], g["head_dim"], g["block_size"], llx.F16, nb)
        raw = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
        return raw, llx.pool_wrap(raw.data_ptr(), nbytes, g["layers"], g["kv_heads"], g["head_dim"], g["block_size"],
                                  llx.F16, nb, keepalive=raw)

    def reset_fork(self):
        """The next step forks its decode-stream work from the migration stream AT ITS START (first step of a timed region)."""
        self.primed = False

    def step(self, stream, dec=None, ev=None):
        """One pass of the path over the next request: stage 0, append, stage 1, append, final stage.
        dec is None: everything on `stream`, in that order.  Otherwise the appends run on the decode stream `dec`
        concurrently with stages 0 and 1, which do not read the appended block; the final stage, which does, waits for
        them (e_app).  Ordering of the decode stream against the migration stream: the appends of step k start after the
        event e_mid(k-1), recorded on the migration stream just before the final stage of step k-1 — i.e. after the final
        stage of step k-2, the last reader of THIS request's tail block (steps alternate between two requests).  The wait
        and the record share one stream boundary, so stage 0 -> stage 1 and final -> next stage 0 stay adjacent kernels
        (programmatic dependent launch).  The first step of a timed region forks at its own start instead (reset_fork).
        ev: optional {name: (start, end)} timing events around "stage0", "stage1", "final" (on `stream`) and "appends"."""
        llx, g = self.llx, self.g
        r = self.k % 2
        s_tab, d_tab = self.s_tabs[r], self.d_tabs[r]
        tokens, m = START_TOKENS, 0
        vptr = self.append_dev.data_ptr()
        tok_bytes = g["layers"] * 2 * g["kv_heads"] * g["head_dim"] * 2
        names = ("stage0", "stage1", "final")
        if dec is not None:
            if not self.primed:
                self.e_mid[1 - r].record(stream)
                self.primed = True
            dec.wait_event(self.e_mid[1 - r])
            if ev is not None and "appends" in ev:
                ev["appends"][0].record(dec)
            for a in APPENDS:
                llx.append_tokens(self.src, s_tab, tokens, tokens + a, vptr + (tokens - START_TOKENS) * tok_bytes, stream=dec)
                tokens += a
            if ev is not None and "appends" in ev:
                ev["appends"][1].record(dec)
            self.e_app[r].record(dec)
        for k, n in enumerate(SCHEDULE):
            if dec is not None and k == len(SCHEDULE) - 1:
                stream.wait_event(self.e_app[r])           # the final stage reads the block the appends wrote
                self.e_mid[r].record(stream)               # the next step's appends (other request) may start from here
            if ev is not None and names[k] in ev:
                ev[names[k]][0].record(stream)
            llx.migrate_stage(self.src, s_tab[m:m + n], self.dst, d_tab[m:m + n], stream=stream,
                              opts=self.stage_opts if k < len(SCHEDULE) - 1 else None)
            if ev is not None and names[k] in ev:
                ev[names[k]][1].record(stream)
            m += n
            if dec is None and k < len(APPENDS):
                llx.append_tokens(self.src, s_tab, tokens, tokens + APPENDS[k],
                                  vptr + (tokens - START_TOKENS) * tok_bytes, stream=stream)
                tokens += APPENDS[k]
        self.k += 1
        return tokens


def dist_setup(torch, n_gpus):
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    return world, rank, local


def run_llx(args):
    import torch

    import paper_2406_03243_b200 as llx
    from paper_2406_03243_b200 import replicas
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the llx path has no CPU fallback")
    llx.load()
    world, rank, local = dist_setup(torch, args.gpus)
    peak, peak_src = measured_peak()

    w = Workload(torch, llx, overlap=not args.no_overlap and not args.serial_appends)
    g = w.g
    assert llx.plan_stage(START_TOKENS + sum(APPENDS), sum(SCHEDULE[:-1]), g["block_size"], 2) == (SCHEDULE[-1], True)
    stream = torch.cuda.Stream()
    stream.wait_stream(torch.cuda.current_stream())
    dec = None if args.serial_appends else torch.cuda.Stream()      # the source's decode stream (appends)
    sampler = ClockSampler(local)
    sampler.start()

    # ---- device-resident throughput -----------------------------------------------------
    for _ in range(args.warmup):
        w.step(stream, dec)
    stream.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    replicas.barrier()
    torch.cuda.synchronize()
    c0 = llx.counters()
    tw0 = time.perf_counter()
    w.reset_fork()
    e0.record(stream)
    for k in range(args.steps):
        w.step(stream, dec)
    e1.record(stream)              # behind the last final stage, which waited for the decode stream's appends
    stream.synchronize()
    tw1 = time.perf_counter()
    replicas.barrier()
    torch.cuda.synchronize()
    c1 = llx.counters()
    sampler.window(tw0, tw1)
    ms_local = e0.elapsed_time(e1) / args.steps
    ms_step = replicas.max_over_ranks(ms_local)
    total_bytes = replicas.sum_over_ranks(step_bytes(g))
    value = total_bytes / (ms_step * 1e-3) / 1e9
    launches = c1["kernel_launches"] - c0["kernel_launches"]

    # dominant kernel (stage 0) timed on its own events, in the same step sequence (second pass: the event
    # records would otherwise sit between the kernels of the pass that defines `value`)
    k_steps = min(args.steps, 200)
    mk = lambda: (torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
    pairs = [mk() for _ in range(k_steps)]
    tw0 = time.perf_counter()
    for k in range(k_steps):
        w.step(stream, dec, {"stage0": pairs[k]})
    stream.synchronize()
    sampler.window(tw0, time.perf_counter())
    stage0_ms = statistics.mean(a.elapsed_time(b) for a, b in pairs)
    stage0_bytes = 2 * SCHEDULE[0] * w.src.block_bytes
    achieved = stage0_bytes / (stage0_ms * 1e-3) / 1e9

    # where the step's time goes: every kernel of the step on its own events (third pass; events between the kernels
    # cost the PDL overlap, so the parts sum to slightly MORE than ms_per_step — the difference is reported, not hidden)
    parts = {k: [mk() for _ in range(k_steps)] for k in ("stage0", "stage1", "final") + (("appends",) if dec is not None else ())}
    whole = [mk() for _ in range(k_steps)]
    for k in range(k_steps):
        whole[k][0].record(stream)
        w.step(stream, dec, {name: evs[k] for name, evs in parts.items()})
        whole[k][1].record(stream)
    stream.synchronize()
    mean_us = lambda evs: 1e3 * statistics.mean(a.elapsed_time(b) for a, b in evs)
    breakdown = {name + "_us": mean_us(evs) for name, evs in parts.items()}
    breakdown["step_with_events_us"] = mean_us(whole)
    breakdown["step_us"] = ms_local * 1e3
    breakdown["ideal_at_measured_peak_us"] = step_bytes(g) / peak / 1e3
    breakdown["stage_kernels_sum_us"] = breakdown["stage0_us"] + breakdown["stage1_us"] + breakdown["final_us"]
    breakdown["outside_stage_kernels_us"] = breakdown["step_us"] - breakdown["stage_kernels_sum_us"]
    breakdown["appends"] = ("on the decode stream, concurrent with stages 0 and 1; the final stage waits for them" if dec is not None
                            else "serialised on the migration stream between the stages")

    # the same 128 blocks as ONE stage (what a blocking copy would do; north_star's "2048-token request")
    ss = [mk() for _ in range(min(args.steps, 100))]
    for _ in range(3):
        llx.migrate_stage(w.src, w.s_tab, w.dst, w.d_tab, stream=stream)
    for a, b in ss:
        a.record(stream)
        llx.migrate_stage(w.src, w.s_tab, w.dst, w.d_tab, stream=stream)
        b.record(stream)
    stream.synchronize()
    single_ms = statistics.mean(a.elapsed_time(b) for a, b in ss)
    single_shot = {"GBps": step_bytes(g) / (single_ms * 1e-3) / 1e9, "ms": single_ms,
                   "frac_of_nominal_8TBps": step_bytes(g) / (single_ms * 1e-3) / 1e9 / NOMINAL_HBM_GBS,
                   "frac_of_measured_peak": step_bytes(g) / (single_ms * 1e-3) / 1e9 / peak}

    # the step as round 1 defined it: every stage in plain stream order, the appends serialised between the
    # stages on the migration stream — so that rounds stay comparable
    saved_opts, w.stage_opts = w.stage_opts, None
    r1_steps = min(args.steps, 200)
    for _ in range(5):
        w.step(stream, None)
    stream.synchronize()
    r0, r1 = mk()
    r0.record(stream)
    for _ in range(r1_steps):
        w.step(stream, None)
    r1.record(stream)
    stream.synchronize()
    w.stage_opts = saved_opts
    r1_ms = r0.elapsed_time(r1) / r1_steps
    round1_def = {"ms_per_step": r1_ms, "value": step_bytes(g) / (r1_ms * 1e-3) / 1e9, "steps": r1_steps,
                  "definition": "plain stream order, appends between the stages on the migration stream (bench.py --serial-appends)"}

    # ---- end to end through pinned host buffers (block fusion path) -----------------------
    # llx_migrate_via_host: gather -> pinned host buffer -> scatter, chunked so that both directions of the
    # host link are busy at once; the sequential llx_pack -> llx_unpack pair is timed beside it.
    n = sum(SCHEDULE)
    stg_bytes = llx.staging_bytes(w.src, n)
    pin = llx.PinnedStaging(stg_bytes)
    e2e_steps = max(3, min(args.steps, 10))

    def via_host():
        llx.migrate_via_host(w.src, w.s_tab, w.dst, w.d_tab, pin.dev_alias, stg_bytes, stream=stream)

    def via_host_kernels():      # LLX_OPT_VIA_HOST_MODE = 3: gather / scatter kernels + bounce buffers, the copy engine crosses the link
        llx.migrate_via_host(w.src, w.s_tab, w.dst, w.d_tab, pin.dev_alias, stg_bytes, stream=stream, opts=dict(via_host_mode=3))

    def pack_unpack():
        llx.pack(w.src, w.s_tab, pin.dev_alias, stg_bytes, stream=stream)       # device -> pinned host
        llx.unpack(pin.dev_alias, stg_bytes, w.dst, w.d_tab, stream=stream)     # pinned host -> device

    def host_timed(fn):
        for _ in range(2):
            fn()
        stream.synchronize()
        replicas.barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            fn()
            stream.synchronize()
        t1 = time.perf_counter()
        sampler.window(t0, t1)
        return replicas.max_over_ranks((t1 - t0) * 1e3 / e2e_steps)

    e2e_seq_ms = host_timed(pack_unpack)
    e2e_kern_ms = host_timed(via_host_kernels)
    c_e0 = llx.counters()
    e2e_ms = host_timed(via_host)
    e2e_launches = (llx.counters()["kernel_launches"] - c_e0["kernel_launches"]) // (e2e_steps + 2)
    e2e_val = replicas.sum_over_ranks(2 * n * w.src.block_bytes) / (e2e_ms * 1e-3) / 1e9
    e2e_seq_val = replicas.sum_over_ranks(2 * n * w.src.block_bytes) / (e2e_seq_ms * 1e-3) / 1e9
    e2e_kern_val = replicas.sum_over_ranks(2 * n * w.src.block_bytes) / (e2e_kern_ms * 1e-3) / 1e9
    pin.free()
    link = None
    if world == 1:
        import bench_suite
        link = bench_suite.link_peak(torch)      # the host link's own peak, measured in this run

    # ---- final-stage downtime (S4): host wall clock around the C-ABI call + stream sync ----
    downtime = measure_downtime(torch, llx, w, stream, reps=args.downtime_reps)
    clocks = sampler.stop()

    block_bytes = w.src.block_bytes
    traffic = profiled_traffic()
    suite = None
    configs = None
    overlap_on = w.stage_opts is not None
    if world == 1 and (args.suite or not args.no_configs):
        del w
        import bench_suite
        bench_suite._free(torch)
        if not args.no_configs:
            configs = bench_suite.baseline_configs(torch, llx, stream)      # configs[2..4] + reference points, bounded
        if args.suite:
            suite = run_suite(torch, llx, stream)

    if rank != 0:
        return 0
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "u16", "data": "synthetic",
        "config": {"workload": WORKLOAD, "shape": "L32 H32 D128 S16 fp16, 2 pools x 2000 blocks (15.6 GiB each)",
                   "request": "128 scattered blocks (2048 tokens), stages 112/14/2, 8-token appends between stages; "
                              "consecutive steps migrate two such requests alternately",
                   "streams": ("copies on the migration stream, appends on the source's decode stream (PAPER.md:134, :235); the final "
                               "stage waits for the appends" if dec is not None else "everything on one stream (--serial-appends)"),
                   "stage_order": ("stages 0 and 1 are launched with llx_launch_opts.overlap_prev=1 (independent of every launch back "
                                   "to the previous final stage: disjoint blocks; they may start while it drains, completion order kept); "
                                   "the final stage in plain stream order" if overlap_on
                                   else "plain stream order for every stage"),
                   "bytes_per_step_rd_plus_wr": step_bytes(g), "parallelism": f"replicas x{world} (no collective)",
                   "l2": "inputs larger than L2 (2.1 GB of traffic per step vs 126 MB L2), no flush needed",
                   "copy_kernel": "bulk-async smem ring (llx_copy_bulk)" if llx.get_option(llx.OPT_COPY_KERNEL) in (0, 2) else "vec16"},
        "pct_of_nominal_8TBps": 100.0 * value / world / NOMINAL_HBM_GBS,
        "pct_of_measured_copy_peak": 100.0 * value / world / peak,
        "value_round1_definition": round1_def,
        "downtime_us": downtime,
        "breakdown": breakdown,
        "single_shot_2048": single_shot,
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "traffic": traffic["bytes"], "traffic_source": traffic["source"], "traffic_commit": traffic["commit"],
                     "kernel": "llx_copy_bulk (stage 0: 112 blocks)", "peak_source": peak_src,
                     "algorithmic_bytes_per_launch": stage0_bytes, "avg_launch_ms": stage0_ms,
                     "frac_of_nominal_8TBps": achieved / NOMINAL_HBM_GBS,
                     "whole_step_frac_of_nominal_8TBps": value / world / NOMINAL_HBM_GBS,
                     "downtime_us": {k: downtime[k] for k in ("host_median", "host_p99", "host_wait_call_median", "gpu_median") if k in downtime},
                     "configs": configs if configs is not None else "not run (--no-configs, or N > 1)"},
        "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": n * block_bytes,
                "d2h_bytes_per_step": n * block_bytes, "ms_per_step": e2e_ms, "steps": e2e_steps,
                "gpu_launches_per_step": e2e_launches,
                "link_peak_gbs": link,
                "frac_of_link_duplex": (e2e_val / link["duplex_GBps_both_directions_summed"]) if link else None,
                "kernel_route_frac_of_link_duplex": (e2e_kern_val / link["duplex_GBps_both_directions_summed"]) if link else None,
                "path": "llx_migrate_via_host, default host leg: one pitched copy-engine transfer per block (2L tiles at a constant "
                        "stride) into the pinned buffer and out of it, D2H and H2D at the same time in groups of ~16 MiB; no kernel "
                        "on this route (host wall clock incl. stream sync)",
                "gather_scatter_kernels_through_bounce_buffers": {
                    "value": e2e_kern_val, "ms_per_step": e2e_kern_ms,
                    "path": "LLX_OPT_VIA_HOST_MODE=3: gather kernel -> device bounce buffer -> copy engine D2H | H2D -> bounce "
                            "buffer -> scatter kernel, 64 MiB chunks (round 1's route)"},
                "sequential_pack_then_unpack": {"value": e2e_seq_val, "ms_per_step": e2e_seq_ms,
                                                "path": "llx_pack (gather kernel into a device bounce buffer, copy engine D2H, 64 MiB chunks) "
                                                        "then llx_unpack (copy engine H2D, scatter kernel), one after the other"}},
        "gpu_launches": launches,
        "clocks": clocks,
        "paper_context": "Llumnix reports 20-30 ms downtime on A10 + 64 Gb/s Gloo (PAPER.md:287); no GB/s figure",
    }
    if args.no_cpu_baseline:
        out["cpu_baseline"] = None
    else:
        out["cpu_baseline"] = cpu_baseline()
        out["cpu_baseline_all_cores"] = cpu_baseline_all_cores()
    if suite is not None:
        out["suite_file"] = suite
    print(json.dumps(out))
    return 0


def measure_downtime(torch, llx, w, stream, reps=100):
    """SURVEY.md §8(d) protocol: stages 0..N-2 done and synchronised, last append done ("source stops the
    request"), then t0 -> llx_migrate_stage(final) -> cudaStreamSynchronize -> t1."""
    import ctypes as C
    lib = llx.lib()
    g = w.g
    n_final = SCHEDULE[-1]
    m = sum(SCHEDULE[:-1])
    s_ids = np.ascontiguousarray(w.s_tab[m:m + n_final], dtype=np.int32)
    d_ids = np.ascontiguousarray(w.d_tab[m:m + n_final], dtype=np.int32)
    sp = s_ids.ctypes.data_as(C.POINTER(C.c_int32))
    dp = d_ids.ctypes.data_as(C.POINTER(C.c_int32))
    sh, dh, st = w.src.handle, w.dst.handle, stream.cuda_stream
    tok_bytes = g["layers"] * 2 * g["kv_heads"] * g["head_dim"] * 2
    host_us, gpu_us, wait_us = [], [], []
    ea, eb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

    def earlier_stages():
        tokens, mm = START_TOKENS, 0
        for k, n in enumerate(SCHEDULE[:-1]):
            llx.migrate_stage(w.src, w.s_tab[mm:mm + n], w.dst, w.d_tab[mm:mm + n], stream=stream)
            mm += n
            llx.append_tokens(w.src, w.s_tab, tokens, tokens + APPENDS[k],
                              w.append_dev.data_ptr() + (tokens - START_TOKENS) * tok_bytes, stream=stream)
            tokens += APPENDS[k]
        stream.synchronize()

    for rep in range(reps + 5):      # the library's own blocking call: completion flag in pinned host memory
        earlier_stages()
        t0 = time.perf_counter_ns()
        rc = lib.llx_migrate_stage_wait(sh, sp, dh, dp, n_final, st)
        t1 = time.perf_counter_ns()
        assert rc == 0
        if rep >= 5:
            wait_us.append((t1 - t0) / 1e3)
    wait_us.sort()
    for rep in range(reps + 5):
        tokens, mm = START_TOKENS, 0
        for k, n in enumerate(SCHEDULE[:-1]):
            llx.migrate_stage(w.src, w.s_tab[mm:mm + n], w.dst, w.d_tab[mm:mm + n], stream=stream)
            mm += n
            llx.append_tokens(w.src, w.s_tab, tokens, tokens + APPENDS[k],
                              w.append_dev.data_ptr() + (tokens - START_TOKENS) * tok_bytes, stream=stream)
            tokens += APPENDS[k]
        stream.synchronize()
        ea.record(stream)
        t0 = time.perf_counter_ns()
        rc = lib.llx_migrate_stage(sh, sp, dh, dp, n_final, st)
        stream.synchronize()
        t1 = time.perf_counter_ns()
        assert rc == 0
        # GPU duration measured on a second, untimed-by-host launch so that the events do not sit inside t0..t1
        ea.record(stream)
        lib.llx_migrate_stage(sh, sp, dh, dp, n_final, st)
        eb.record(stream)
        stream.synchronize()
        if rep >= 5:
            host_us.append((t1 - t0) / 1e3)
            gpu_us.append(ea.elapsed_time(eb) * 1e3)
    host_us.sort()
    gpu_us.sort()
    q = lambda v, p: v[min(len(v) - 1, int(p * len(v)))]
    return {"final_stage_blocks": n_final, "final_stage_bytes_rd_plus_wr": 2 * n_final * w.src.block_bytes,
            "host_median": q(host_us, 0.5), "host_p99": q(host_us, 0.99), "host_min": host_us[0],
            "host_wait_call_median": q(wait_us, 0.5), "host_wait_call_p99": q(wait_us, 0.99), "host_wait_call_min": wait_us[0],
            "gpu_median": q(gpu_us, 0.5), "gpu_min": gpu_us[0], "reps": reps,
            "definition": "host_*: host wall clock from entering llx_migrate_stage(final) to return of the stream "
                          "synchronize; host_wait_call_*: the same interval around ONE llx_migrate_stage_wait call "
                          "(the kernel's last CTA writes a pinned host word the caller spins on); gpu_* = CUDA-event "
                          "duration of the same launch repeated (L2-warm)"}


def run_suite(torch, llx, stream):
    import bench_suite
    res = bench_suite.run(torch, llx, stream)
    os.makedirs(os.path.join(ROOT, "gpurun_out"), exist_ok=True)
    path = os.path.join("gpurun_out", "suite.json")
    with open(os.path.join(ROOT, path), "w") as f:
        json.dump(res, f, indent=1)
    for k, v in res.items():
        print(json.dumps({k: v}), file=sys.stderr)
    return path


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=1000)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", choices=["llx", "reference"], default="llx")
    ap.add_argument("--suite", action="store_true", help="also run the length sweep, 30B batch and interference configs")
    ap.add_argument("--downtime-reps", type=int, default=200)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-configs", action="store_true",
                    help="skip the bounded legs over BASELINE.json configs[2..4] and the reference points (about a minute)")
    ap.add_argument("--no-overlap", action="store_true",
                    help="launch every stage in plain stream order (no llx_launch_opts.overlap_prev on stages 0 and 1)")
    ap.add_argument("--serial-appends", action="store_true",
                    help="enqueue the appends on the migration stream between the stages (round-1 behaviour) instead of a decode stream")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3
    if args.impl == "reference":
        return run_reference(args)
    return run_llx(args)


if __name__ == "__main__":
    sys.exit(main())
