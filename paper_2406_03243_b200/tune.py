"""Sweep the copy-kernel launch options on the current GPU and print GB/s (rd+wr) per configuration.

    python -m paper_2406_03243_b200.tune [--blocks 128,112,14,2] [--top 25] [--quick]
    python -m paper_2406_03243_b200.tune --mode tail     # dynamic-tail share x batch, then ring shapes under it
    python -m paper_2406_03243_b200.tune --mode step     # the whole configs[1] step under global option sets

The defaults compiled into libllx.so (llx_api.cu, launch_copy) come from this sweep on a B200; the output
of one run is kept in profiles/r01_copy_sweep.md.  Workload: configs[1] pools (LLaMA-7B shape, 2 x 2000
blocks), one llx_migrate_stage of the given number of scattered blocks, CUDA events on the launching stream,
median of 15; stages of <= 16 blocks are measured L2-cold (a 512 MiB write precedes every launch)."""
from __future__ import annotations

import argparse
import itertools
import statistics
import sys

import numpy as np


def _setup():
    import torch

    import paper_2406_03243_b200 as llx
    import synth
    from paper_2406_03243_b200.suite import Pools
    llx.load()
    g = synth.CONFIGS["llama7b"]
    nb = g["num_blocks"]
    p = Pools(torch, llx, g, nb, nb)
    return torch, llx, synth, g, nb, p, torch.cuda.Stream()


def _back_to_back(torch, st, fn, reps=7, inner=10):
    """us per launch, `inner` launches between one pair of events (launch gaps overlapped as in a real stream)."""
    for _ in range(3):
        fn()
    st.synchronize()
    ts = []
    for _ in range(reps):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(st)
        for _ in range(inner):
            fn()
        b.record(st)
        st.synchronize()
        ts.append(a.elapsed_time(b) / inner)
    return statistics.median(ts) * 1e3


def mode_tail():
    torch, llx, synth, g, nb, p, st = _setup()
    s_tab, d_tab = synth.block_permutation(1, nb), synth.block_permutation(2, nb)
    for n in (112, 128, 256):
        nbytes = 2 * n * p.src.block_bytes
        mig = lambda: llx.migrate_stage(p.src, s_tab[:n], p.dst, d_tab[:n], stream=st)
        print(f"\n== {n} blocks, bulk kernel, back-to-back launches; GB/s = rd+wr")
        print("| us | GB/s | chunk | stages | CTAs | tail % | batch |\n|---|---|---|---|---|---|---|")
        for chunk, stages, cap in ((8192, 4, 296), (32768, 3, 148), (32768, 2, 296), (8192, 3, 444)):
            for pct, batch in [(0, 0)] + [(q, b) for q in (1, 3, 6, 10, 15, 30, 100) for b in ((4,) if q != 6 else (1, 4, 16, 32))]:
                with llx.options(chunk_bytes=chunk, ring_stages=stages, max_ctas=cap, dynamic_tail_pct=pct, dynamic_tail_batch=batch):
                    t = _back_to_back(torch, st, mig)
                print(f"| {t:.1f} | {nbytes / t / 1e3:.0f} | {chunk} | {stages} | {cap} | {pct} | {batch or '-'} |")
    return 0


def mode_step():
    torch, llx, synth, g, nb, p, st = _setup()
    s_tab, d_tab = synth.block_permutation(1, nb)[:128], synth.block_permutation(2, nb)[:128]
    tok_bytes = g["layers"] * 2 * g["kv_heads"] * g["head_dim"] * 2
    vals = torch.zeros(16 * tok_bytes, dtype=torch.uint8, device="cuda")
    schedule, start = (112, 14, 2), 2032

    def step():
        tokens, m = start, 0
        for k, n in enumerate(schedule):
            llx.migrate_stage(p.src, s_tab[m:m + n], p.dst, d_tab[m:m + n], stream=st)
            m += n
            if k < 2:
                llx.append_tokens(p.src, s_tab, tokens, tokens + 8, vals.data_ptr() + (tokens - start) * tok_bytes, stream=st)
                tokens += 8
    nbytes = 2 * 128 * p.src.block_bytes
    cfgs = {"8Kx4 2/SM static (round-1 default until now)": dict(chunk_bytes=8192, ring_stages=4, max_ctas=296, dynamic_tail_pct=0),
            "auto (32Kx3 1/SM tail 6 %; short stages 8Kx4 2/SM)": dict(),
            "8Kx4 2/SM tail 6 %": dict(chunk_bytes=8192, ring_stages=4, max_ctas=296),
            "8Kx3 3/SM tail 6 %": dict(chunk_bytes=8192, ring_stages=3, max_ctas=444),
            "8Kx3 3/SM static": dict(chunk_bytes=8192, ring_stages=3, max_ctas=444, dynamic_tail_pct=0),
            "32Kx3 1/SM tail 6 %": dict(chunk_bytes=32768, ring_stages=3, max_ctas=148),
            "32Kx2 2/SM tail 6 %": dict(chunk_bytes=32768, ring_stages=2, max_ctas=296),
            "16Kx3 2/SM tail 6 %": dict(chunk_bytes=16384, ring_stages=3, max_ctas=296)}
    print("configs[1] step (stages 112/14/2 + two 8-token appends), 600 steps back to back, us per step\n")
    print("| option set (all three stages) | exact residency | PDL | us/step | GB/s |\n|---|---|---|---|---|")
    for name, o in cfgs.items():
        for pad, pdl in ((1, 1), (0, 1), (1, 0)):
            with llx.options(exact_residency=pad, pdl=pdl, **o):
                t = _back_to_back(torch, st, step, reps=3, inner=200)
            print(f"| {name} | {pad} | {pdl} | {t:.2f} | {nbytes / t / 1e3:.0f} |")
    return 0


def mode_refcopy():
    """torch's contiguous copy_ of stage 0's byte count next to llx_migrate_stage of 112 blocks (for an ncu comparison)."""
    torch, llx, synth, g, nb, p, st = _setup()
    s_tab, d_tab = synth.block_permutation(1, nb)[:112], synth.block_permutation(2, nb)[:112]
    a = torch.empty(112 * p.src.block_bytes, dtype=torch.uint8, device="cuda")
    b = torch.empty_like(a)
    with torch.cuda.stream(st):
        for _ in range(5):
            b.copy_(a)
            llx.migrate_stage(p.src, s_tab, p.dst, d_tab, stream=st)
        t1 = _back_to_back(torch, st, lambda: b.copy_(a))
    t2 = _back_to_back(torch, st, lambda: llx.migrate_stage(p.src, s_tab, p.dst, d_tab, stream=st))
    nbytes = 2 * a.numel()
    print(f"torch copy_ {t1:.1f} us {nbytes / t1 / 1e3:.0f} GB/s | llx_migrate_stage {t2:.1f} us {nbytes / t2 / 1e3:.0f} GB/s")
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--mode", choices=["sweep", "tail", "step", "refcopy"], default="sweep")
    ap.add_argument("--blocks", default="128,112,14,2")
    ap.add_argument("--top", type=int, default=25)
    ap.add_argument("--quick", action="store_true")
    args = ap.parse_args()
    if args.mode == "tail":
        return mode_tail()
    if args.mode == "step":
        return mode_step()
    if args.mode == "refcopy":
        return mode_refcopy()
    import torch

    import paper_2406_03243_b200 as llx
    import synth
    from paper_2406_03243_b200.suite import Pools
    llx.load()
    g = synth.CONFIGS["llama7b"]
    nb = g["num_blocks"]
    p = Pools(torch, llx, g, nb, nb)
    st = torch.cuda.Stream()
    flushbuf = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")
    s_tab = synth.block_permutation(1, nb)
    d_tab = synth.block_permutation(2, nb)

    def timeit(fn, reps=15, warm=2, flush=False):
        for _ in range(warm):
            fn()
        st.synchronize()
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(reps)]
        with torch.cuda.stream(st):
            for a, b in evs:
                if flush:
                    flushbuf.fill_(1)
                a.record(st)
                fn()
                b.record(st)
        st.synchronize()
        ts = [a.elapsed_time(b) for a, b in evs]
        return statistics.median(ts), min(ts)

    # reference: a contiguous copy of the same number of bytes (cudaMemcpy D2D through torch)
    a = torch.empty(128 * p.src.block_bytes, dtype=torch.uint8, device="cuda")
    b = torch.empty_like(a)
    with torch.cuda.stream(st):
        med, mn = timeit(lambda: b.copy_(a))
    print(f"torch contiguous copy_ of 1 GiB: median {2 * a.numel() / med / 1e6:.0f} GB/s, best {2 * a.numel() / mn / 1e6:.0f} GB/s")
    del a, b

    for n in [int(x) for x in args.blocks.split(",")]:
        nbytes = 2 * n * p.src.block_bytes
        off = 0 if n >= 112 else 112
        mig = lambda: llx.migrate_stage(p.src, s_tab[off:off + n], p.dst, d_tab[off:off + n], stream=st)
        cold = n <= 16
        res = []
        chunks = [8192, 16384, 32768] if args.quick else [4096, 8192, 16384, 32768, 65536]
        for chunk, stages, cap, hint, order, rings in itertools.product(
                chunks, [2, 3, 4, 6], [148, 296, 444], [0, 3], [0, 1], [1, 2]):
            per_sm = max(1, cap // 148)
            if per_sm * (rings * chunk * stages + 2048) > 227 * 1024:
                continue
            with llx.options(copy_kernel=2, chunk_bytes=chunk, ring_stages=stages, max_ctas=cap, l2_hint=hint,
                             unit_order=order, rings_per_cta=rings):
                med, mn = timeit(mig, flush=cold)
            res.append((nbytes / med / 1e6, nbytes / mn / 1e6, med * 1e3, "bulk", chunk, stages, cap, hint, order, rings,
                        per_sm * rings * chunk * stages // 1024))
        for chunk, cap, order in itertools.product([4096, 8192, 16384, 32768], [296, 592, 1184], [0, 1]):
            with llx.options(copy_kernel=1, chunk_bytes=chunk, max_ctas=cap, unit_order=order):
                med, mn = timeit(mig, flush=cold)
            res.append((nbytes / med / 1e6, nbytes / mn / 1e6, med * 1e3, "vec16", chunk, 0, cap, 0, order, 0, 0))
        with llx.options():
            med, mn = timeit(mig, flush=cold)
        print(f"\n== {n} blocks ({nbytes / 2**20:.0f} MiB rd+wr){' L2-cold' if cold else ''}: library defaults "
              f"{nbytes / med / 1e6:.0f} GB/s median ({med * 1e3:.1f} us)")
        res.sort(reverse=True)
        print("| median GB/s | best GB/s | us | kernel | chunk | stages | CTAs | l2_hint | order | rings | ring KiB/SM |")
        print("|---|---|---|---|---|---|---|---|---|---|---|")
        for r in res[:args.top]:
            print("| %.0f | %.0f | %.1f | %s | %d | %d | %d | %d | %d | %d | %d |" % r)
        print(f"| … {len(res)} configurations; worst: %.0f GB/s (%s chunk=%d stages=%d CTAs=%d order=%d) |" %
              (res[-1][0], res[-1][3], res[-1][4], res[-1][5], res[-1][6], res[-1][8]))
        # marginals over the bulk kernel
        for name, idx in (("order (0 striped, 1 contiguous ranges)", 8), ("l2_hint", 7), ("ring KiB per SM", 10)):
            d = {}
            for r in res:
                if r[3] == "bulk":
                    d.setdefault(r[idx], []).append(r[0])
            print(f"best/median GB/s by {name}: " +
                  ", ".join(f"{k}: {max(v):.0f}/{statistics.median(v):.0f}" for k, v in sorted(d.items())))
    return 0


if __name__ == "__main__":
    sys.exit(main())
