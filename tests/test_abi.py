"""The C-ABI boundary without a GPU: the library builds for sm_100a, loads, exports every symbol
include/llx.h declares, and its host-only entry points behave.  No compute calls here."""
import ctypes
import os
import re
import subprocess

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "llx.h")


@pytest.fixture(scope="module")
def llx():
    from paper_2406_03243_b200 import build
    build.build()
    import paper_2406_03243_b200 as m
    m.load()
    return m


def declared_symbols():
    text = open(HEADER).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(llx_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_all_exported_and_bound(llx):
    names = declared_symbols()
    assert len(names) >= 25 and "llx_migrate_stage" in names and "llx_pack" in names
    raw = ctypes.CDLL(os.path.join(ROOT, "paper_2406_03243_b200", "libllx.so"))
    for n in names:
        assert hasattr(raw, n), f"{n} declared in llx.h but not exported by libllx.so"
    assert sorted(llx.EXPORTS) == names, "binding.EXPORTS and include/llx.h disagree"


def test_library_is_sm100a_and_uses_bulk_async_copy():
    lib = os.path.join(ROOT, "paper_2406_03243_b200", "libllx.so")
    out = subprocess.run(["cuobjdump", "-lelf", lib], capture_output=True, text=True)
    if out.returncode != 0:
        pytest.skip("cuobjdump unavailable")
    assert "sm_100a" in out.stdout
    sass = subprocess.run(["cuobjdump", "-sass", lib], capture_output=True, text=True).stdout
    assert "UBLKCP" in sass and "LDG.E.128" in sass and "STG.E.128" in sass


def test_geometry_arithmetic_matches_paper_example(llx):
    # 16-bit LLaMA-7B: 128 KB per block (K or V, 16 tokens, one layer)
    assert llx.pool_bytes_for(1, 32, 128, 16, llx.F16, 1) == 2 * 131072
    assert llx.pool_bytes_for(32, 32, 128, 16, llx.F16, 2000) == 2000 * 8 * 2**20
    assert llx.pool_bytes_for(60, 52, 128, 16, llx.F16, 3000) == 3000 * 120 * 208 * 1024
    assert llx.pool_bytes_for(2, 4, 64, 16, llx.F16, 256) == 8 * 2**20
    assert llx.pool_bytes_for(2, 4, 64, 16, llx.U8, 256) == 4 * 2**20
    for bad in [(0, 4, 64, 16, 0, 1), (2, 4, 64, 16, 7, 1), (2, 1, 1, 1, 0, 4), (2, 4, 64, 16, 0, 0), (2, 4, 64, -1, 0, 1)]:
        assert llx.pool_bytes_for(*bad) == 0


def test_options_validate_and_roundtrip(llx):
    old = llx.get_option(llx.OPT_CHUNK_BYTES)
    llx.set_option(llx.OPT_CHUNK_BYTES, 8192)
    assert llx.get_option(llx.OPT_CHUNK_BYTES) == 8192
    with pytest.raises(llx.LlxError) as e:
        llx.set_option(llx.OPT_CHUNK_BYTES, 100)          # not a multiple of 16
    assert e.value.name == "LLX_ERR_INVALID_ARG"
    with pytest.raises(llx.LlxError):
        llx.set_option(llx.OPT_COPY_KERNEL, 9)
    with pytest.raises(llx.LlxError):
        llx.set_option(llx.OPT_IDS_BY_VALUE_MAX, 100000)
    llx.set_option(llx.OPT_CHUNK_BYTES, old)
    with llx.options(copy_kernel=1, max_ctas=3):
        assert llx.get_option(llx.OPT_COPY_KERNEL) == 1 and llx.get_option(llx.OPT_MAX_CTAS) == 3
    assert llx.get_option(llx.OPT_COPY_KERNEL) == 0 and llx.get_option(llx.OPT_MAX_CTAS) == 0


def test_status_strings_and_counters(llx):
    l = llx.lib()
    assert l.llx_status_str(0) == b"LLX_OK" and l.llx_status_str(-4) == b"LLX_ERR_DUPLICATE_DST"
    assert l.llx_status_str(-99) == b"LLX_ERR_UNKNOWN"
    llx.reset_counters()
    assert llx.counters() == dict(kernel_launches=0, copy_launches=0, bytes_moved=0, id_uploads=0)
    assert "sm_100a" in llx.version()


def test_no_cpu_fallback_without_a_device(llx):
    """On a box without a GPU every data call must fail loudly (LLX_ERR_CUDA), never compute on the CPU."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present; the no-device behaviour is checked on the CPU box")
    with pytest.raises(llx.LlxError) as e:
        llx.pool_create(2, 4, 64, 16, llx.F16, 256)
    assert e.value.name == "LLX_ERR_CUDA"
    host = np.zeros(1 << 16, dtype=np.uint8)
    with pytest.raises(llx.LlxError):
        llx.pool_wrap(host.ctypes.data, host.nbytes, 1, 1, 8, 1, llx.F16, 4)


def test_null_and_trivial_arguments(llx):
    l = llx.lib()
    assert l.llx_pool_destroy(None) == 0
    assert l.llx_pool_data(None, 0, 0) is None
    assert l.llx_pool_tile_bytes(None) == 0 and l.llx_pool_bytes(None) == 0 and l.llx_pool_num_blocks(None) == 0
    assert l.llx_staging_bytes(None, 4) == 0
    assert l.llx_staging_free_pinned(None) == 0
    rc = l.llx_migrate_stage(None, None, None, None, 0, None)
    assert rc == -1 and b"NULL" in l.llx_last_error()


def test_plan_stage_matches_oracle_on_every_state(llx):
    """S1 is host arithmetic: the library's planner against oracle.plan_stage for every (tokens, migrated)."""
    from oracle import kv_migration as om
    for S, last in ((16, 2), (4, 1), (5, 3)):
        for tokens in range(0, 150):
            for m in range(0, -(-tokens // S) + 1):
                assert llx.plan_stage(tokens, m, S, last) == om.plan_stage(tokens, m, S, last)
    assert llx.plan_stage(2032, 0, 16, 2) == (127, False)
    assert llx.plan_stage(2048, 126, 16, 2) == (2, True)
    for bad in [(16, 2, 16, 2), (-1, 0, 16, 2), (16, 0, 0, 2), (16, 0, 16, 0)]:
        with pytest.raises(llx.LlxError):
            llx.plan_stage(*bad)


def test_predicted_stage_sizes_match_oracle_and_a_time_stepped_simulation(llx):
    """llx_predict_stage_sizes (the planner "driven by measured copy / decode rates")
    against oracle.stage_sizes on seeded rates, and both against a pin that shares nothing with the recurrence: a
    time-stepped simulation in exact rational arithmetic that copies blocks one by one while a decoder appends tokens."""
    from fractions import Fraction

    import numpy as np

    from oracle import kv_migration as om

    def simulate(n0, c, r, S, cap):
        # stage k copies n_k blocks one after the other (1/c s each); tokens decoded in the stage's duration, counted
        # exactly, turn into ceil(tokens / S) new blocks (at least the one open block of the final stage)
        c, r = Fraction(c), Fraction(r)
        sizes, n = [n0], n0
        while n > 1 and len(sizes) < cap:
            duration = sum((1 / c for _ in range(n)), Fraction(0)) if n <= 5000 else n / c
            tokens = r * duration
            blocks = -((-tokens.numerator) // (tokens.denominator * S))     # ceil(tokens / S) on exact rationals
            n = max(1, int(blocks))
            sizes.append(n)
        return sizes

    rng = np.random.default_rng(7)
    for _ in range(300):
        n0 = int(rng.integers(1, 600))
        S = int(rng.choice([4, 16, 32]))
        c = float(rng.integers(1, 4000)) / 4.0                                # quarter-integers: exact in binary and as Fraction
        r = float(rng.integers(0, 4000)) / 4.0
        if rng.random() < 0.8:                                                # mostly the convergent regime: c*S > r
            c = max(c, float(int(2 * r / S) + 1))
        want = om.stage_sizes(n0, c, r, S, max_stages=12)
        if max(want) > 2**31 - 1:                                             # decoding outruns the copy: sizes leave int32
            with pytest.raises(llx.LlxError):
                llx.predict_stage_sizes(n0, c, r, S, cap=12)
        else:
            # (quotients below 2^31 with denominators below 2^17 are at least 7e-6 from an integer unless they are one:
            # double rounding cannot move the ceiling, so the exact simulation and the double recurrence must agree)
            assert want == simulate(n0, c, r, S, 12), (n0, c, r, S)
            assert llx.predict_stage_sizes(n0, c, r, S, cap=12) == want, (n0, c, r, S)
    # the paper's regime: copy much faster than decode -> two stages, whatever the length
    for n0 in (16, 128, 512):
        assert llx.predict_stage_sizes(n0, 950.0, 15.4, 16) == [n0, 1]
    # B200, LLaMA-7B blocks of 8 MiB: 6.5 TB/s rd+wr = 387,000 blocks/s unthrottled; 12 GB/s budget = 715 blocks/s;
    # one request decoding at ~180 tokens/s (5.5 ms per step): two stages in both cases
    assert llx.predict_stage_sizes(128, 387000.0, 180.0, 16) == [128, 1]
    assert llx.predict_stage_sizes(128, 715.0, 180.0, 16) == [128, 3, 1]
    assert llx.predict_stage_sizes(1, 1.0, 1.0, 16) == [1]
    assert llx.predict_stage_sizes(64, 4.0, 16.0, 16) == [64, 16, 4, 1]
    assert llx.predict_stage_sizes(64, 1.0, 64.0, 16, cap=5) == [64, 256, 1024, 4096, 16384]   # decoding outruns the copy
    for bad in [(0, 1.0, 1.0, 16), (4, 0.0, 1.0, 16), (4, 1.0, -1.0, 16), (4, 1.0, 1.0, 0), (4, float("nan"), 1.0, 16),
                (4, float("inf"), 1.0, 16)]:
        with pytest.raises(llx.LlxError):
            llx.predict_stage_sizes(*bad)
    import ctypes as C
    k = C.c_int()
    assert llx.lib().llx_predict_stage_sizes(4, 1.0, 1.0, 16, (C.c_int32 * 1)(), 0, C.byref(k)) == -1     # cap = 0
    assert llx.lib().llx_predict_stage_sizes(4, 1.0, 1.0, 16, None, 4, C.byref(k)) == -1


def test_header_is_plain_c99_and_a_c_client_links_and_runs(llx, tmp_path):
    """The boundary is a C ABI: the header compiles as C99 with -pedantic, and a C program (tests/c/abi_smoke.c)
    drives the host-only entry points — planner, block manager, handshake, Algorithm 1 — through libllx.so."""
    import shutil
    gcc = shutil.which("gcc")
    if not gcc:
        pytest.skip("gcc unavailable")
    r = subprocess.run([gcc, "-fsyntax-only", "-x", "c", "-std=c99", "-Wall", "-Wextra", "-Werror", "-pedantic", HEADER],
                       capture_output=True, text=True)
    assert r.returncode == 0, r.stderr
    libdir = os.path.join(ROOT, "paper_2406_03243_b200")
    exe = str(tmp_path / "abi_smoke")
    r = subprocess.run([gcc, "-std=c99", "-Wall", "-Wextra", "-Werror", "-pedantic", "-I", os.path.join(ROOT, "include"),
                        os.path.join(ROOT, "tests", "c", "abi_smoke.c"), "-o", exe, "-L", libdir, "-lllx",
                        "-Wl,-rpath," + libdir], capture_output=True, text=True)
    assert r.returncode == 0, r.stderr
    r = subprocess.run([exe], capture_output=True, text=True)
    assert r.returncode == 0 and "abi_smoke ok" in r.stdout, r.stdout + r.stderr


def test_host_side_under_asan_and_ubsan(tmp_path):
    """The host side of the library (validation, planner, block manager, handshake, Algorithm 1) built with
    -fsanitize=address,undefined and driven by the C client: no report, exit 0.  (The device side cannot be run under
    compute-sanitizer on this pool of machines.)"""
    import shutil
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    gcc = shutil.which("gcc")
    if not gcc or not os.path.exists(nvcc):
        pytest.skip("toolchain unavailable")
    probe = subprocess.run([gcc, "-fsanitize=address,undefined", "-x", "c", "-", "-o", str(tmp_path / "probe")],
                           input="int main(void){return 0;}", capture_output=True, text=True)
    if probe.returncode != 0:
        pytest.skip("libasan/libubsan unavailable")
    csrc = os.path.join(ROOT, "paper_2406_03243_b200", "csrc")
    lib = str(tmp_path / "libllx.so")
    r = subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O1", "-g", "-std=c++17", "-shared", "-Xcompiler",
                        "-fPIC,-fsanitize=address,-fsanitize=undefined,-fno-omit-frame-pointer", "-diag-suppress", "550",
                        "-o", lib, os.path.join(csrc, "llx_api.cu"), os.path.join(csrc, "llx_coord.cu"), "-lasan", "-lubsan"],
                       capture_output=True, text=True)
    assert r.returncode == 0, r.stderr[-2000:]
    exe = str(tmp_path / "abi_smoke_asan")
    r = subprocess.run([gcc, "-std=c99", "-g", "-fsanitize=address,undefined", "-I", os.path.join(ROOT, "include"),
                        os.path.join(ROOT, "tests", "c", "abi_smoke.c"), "-o", exe, "-L", str(tmp_path), "-lllx",
                        "-Wl,-rpath," + str(tmp_path)], capture_output=True, text=True)
    assert r.returncode == 0, r.stderr
    env = dict(os.environ, ASAN_OPTIONS="detect_leaks=0:protect_shadow_gap=0:halt_on_error=1", UBSAN_OPTIONS="halt_on_error=1")
    r = subprocess.run([exe], capture_output=True, text=True, env=env)
    assert r.returncode == 0 and "abi_smoke ok" in r.stdout and "runtime error" not in r.stderr and "AddressSanitizer" not in r.stderr, \
        r.stdout + r.stderr[-3000:]


def test_launch_opts_are_validated_before_any_device_work(llx):
    """llx_launch_opts: init sets every field to LLX_OPT_DEFAULT; a bad field, an unknown route or a struct_size this
    library does not know is LLX_ERR_INVALID_ARG — reported before the pools are even looked at (so also without a GPU)."""
    import ctypes as C
    o = llx.LaunchOpts()
    assert o.struct_size == C.sizeof(llx.LaunchOpts) == 68
    assert all(getattr(o, f) == llx.OPT_DEFAULT for f, _ in o._fields_ if f != "struct_size")
    l = llx.lib()
    ids = (C.c_int32 * 2)(0, 1)
    for bad in (dict(chunk_bytes=100), dict(copy_kernel=7), dict(bandwidth_gbps=-5), dict(route=9), dict(ring_stages=1),
                dict(overlap_prev=2)):
        rc = l.llx_migrate_stage_ex(None, ids, None, ids, 2, None, C.byref(llx.LaunchOpts(**bad)))
        assert rc == -1 and b"llx_launch_opts." in l.llx_last_error(), (bad, l.llx_last_error())
    o = llx.LaunchOpts()
    o.struct_size = 6
    assert l.llx_migrate_stage_ex(None, ids, None, ids, 2, None, C.byref(o)) == -1 and b"struct_size" in l.llx_last_error()
    o.struct_size = 400
    assert l.llx_migrate_batch_ex(None, None, ids, ids, ids, 1, None, C.byref(o)) == -1 and b"struct_size" in l.llx_last_error()
    with pytest.raises(TypeError):
        llx.LaunchOpts(no_such_field=1)
    # a good policy passes validation and the call then fails on the NULL pools, not on the policy
    rc = l.llx_migrate_stage_ex(None, ids, None, ids, 2, None, C.byref(llx.LaunchOpts(bandwidth_gbps=25, route=llx.ROUTE_PEER)))
    assert rc == -1 and b"pool is NULL" in l.llx_last_error()
    # the process-wide defaults that are not per-call fields
    assert llx.get_option(llx.OPT_COPY_SMEM_CARVEOUT_PCT) == 50 and llx.get_option(llx.OPT_PACED_SLICE_US) == 1000
    with pytest.raises(llx.LlxError):
        llx.set_option(llx.OPT_COPY_SMEM_CARVEOUT_PCT, 101)


def test_ipc_handle_is_checked(llx):
    import ctypes as C
    l = llx.lib()
    assert llx.IPC_HANDLE_BYTES == 96
    with pytest.raises(llx.LlxError) as e:
        llx.pool_ipc_open(b"\0" * llx.IPC_HANDLE_BYTES)                  # no magic: not an llx handle
    assert e.value.name == "LLX_ERR_INVALID_ARG"
    with pytest.raises(llx.LlxError):
        llx.pool_ipc_open(b"short")
    # the right magic ("LLX2") but no valid checksum behind it: refused before any CUDA call is made
    import struct
    forged = b"\x11" * 64 + struct.pack("<I6iI", 0x4C4C5832, 32, 32, 128, 16, 0, 2000, 0)
    assert len(forged) == llx.IPC_HANDLE_BYTES
    with pytest.raises(llx.LlxError) as e:
        llx.pool_ipc_open(forged)
    assert e.value.name == "LLX_ERR_INVALID_ARG" and "checksum" in str(e.value)
    out = C.c_void_p()
    assert l.llx_pool_ipc_open(None, C.byref(out)) == -1 and l.llx_pool_ipc_export(None, None) == -1
    # session policy: a struct size the library cannot read is refused (an older, shorter struct is served), NULL resets
    a, b = llx.BlockManager(8), llx.BlockManager(8)
    mig = llx.Migration(None, a, None, b, 4, 1)
    mig.set_stage_opts(dict(bandwidth_gbps=25))
    mig.set_stage_opts(None)
    bad = llx.LaunchOpts()
    for size in (6, 400):
        bad.struct_size = size
        with pytest.raises(llx.LlxError):
            mig.set_stage_opts(bad)
    older = llx.LaunchOpts(bandwidth_gbps=25, overlap_prev=1)
    older.struct_size = 64                                               # round 2's struct before overlap_prev was added
    mig.set_stage_opts(older)
    with pytest.raises(llx.LlxError) as e:
        mig.stage([3, 3, 4, 5], 14)                                       # a table that names a block twice (A33)
    assert e.value.name == "LLX_ERR_INVALID_ARG" and b.num_free == 8
