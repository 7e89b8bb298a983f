"""ctypes binding with the same names as include/llx.h.  Argument marshalling only.

Block-id arguments are anything convertible to a contiguous int32 NumPy array (host memory, as the
ABI requires); device buffers are passed as integer addresses (`tensor.data_ptr()`); streams as the
integer `torch.cuda.Stream.cuda_stream` (0 / None = legacy default stream).
"""
from __future__ import annotations

import contextlib
import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libllx.so")

F16, BF16, U8 = 0, 1, 2
(OPT_COPY_KERNEL, OPT_MAX_CTAS, OPT_CHUNK_BYTES, OPT_RING_STAGES, OPT_IDS_BY_VALUE_MAX, OPT_ATTN_SPLIT_TOKENS,
 OPT_UNIT_ORDER, OPT_L2_HINT, OPT_RINGS_PER_CTA, OPT_PDL, OPT_BANDWIDTH_GBPS, OPT_VIA_HOST_MODE, OPT_DYNAMIC_TAIL_PCT,
 OPT_DYNAMIC_TAIL_BATCH, OPT_EXACT_RESIDENCY, OPT_COPY_SMEM_CARVEOUT_PCT, OPT_PACED_SLICE_US,
 OPT_OVERLAP_PREV) = range(18)

_vp, _i, _sz, _i32p = C.c_void_p, C.c_int, C.c_size_t, C.POINTER(C.c_int32)


class ReqInfo(C.Structure):
    _fields_ = [("is_queuing", C.c_int32), ("is_head_of_line", C.c_int32), ("is_fake", C.c_int32),
                ("priority", C.c_int32), ("demand", C.c_double), ("physical_usage", C.c_double)]


OPT_DEFAULT = -1
ROUTE_AUTO, ROUTE_PEER, ROUTE_COPY_ENGINE = 0, 1, 2


class LaunchOpts(C.Structure):
    """llx_launch_opts: the launch policy of ONE call.  LaunchOpts(bandwidth_gbps=25) leaves every other field at
    LLX_OPT_DEFAULT (inherit the process default)."""
    _fields_ = [("struct_size", C.c_uint32)] + [(k, C.c_int32) for k in (
        "bandwidth_gbps", "max_ctas", "copy_kernel", "chunk_bytes", "ring_stages", "rings_per_cta", "ids_by_value_max",
        "unit_order", "l2_hint", "pdl", "dynamic_tail_pct", "dynamic_tail_batch", "exact_residency", "via_host_mode",
        "route", "overlap_prev")]

    def __init__(self, **kw):
        super().__init__()
        load().llx_launch_opts_init(C.byref(self))
        for k, v in kw.items():
            if k not in dict(self._fields_) or k == "struct_size":
                raise TypeError(f"llx_launch_opts has no field {k!r}")
            setattr(self, k, int(v))


def _opts(o):
    """None | dict | LaunchOpts -> pointer argument of the *_ex entry points."""
    if o is None:
        return None
    if isinstance(o, dict):
        o = LaunchOpts(**o)
    return C.byref(o)


class _Counters(C.Structure):
    _fields_ = [("kernel_launches", C.c_ulonglong), ("copy_launches", C.c_ulonglong),
                ("bytes_moved", C.c_ulonglong), ("id_uploads", C.c_ulonglong)]


#: every symbol include/llx.h declares: name -> (restype, argtypes)
EXPORTS = {
    "llx_pool_create": (_i, [_i, _i, _i, _i, _i, _i, C.POINTER(_vp)]),
    "llx_pool_wrap": (_i, [_vp, _sz, _i, _i, _i, _i, _i, _i, C.POINTER(_vp)]),
    "llx_pool_destroy": (_i, [_vp]),
    "llx_pool_data": (_vp, [_vp, _i, _i]),
    "llx_pool_tile_bytes": (_sz, [_vp]),
    "llx_pool_block_bytes": (_sz, [_vp]),
    "llx_pool_bytes": (_sz, [_vp]),
    "llx_pool_num_blocks": (_i, [_vp]),
    "llx_pool_bytes_for": (_sz, [_i, _i, _i, _i, _i, _i]),
    "llx_pool_ipc_export": (_i, [_vp, _vp]),
    "llx_pool_ipc_open": (_i, [_vp, C.POINTER(_vp)]),
    "llx_pool_upload": (_i, [_vp, _i, _i, _i, _i, _vp, _vp]),
    "llx_pool_download": (_i, [_vp, _i, _i, _i, _i, _vp, _vp]),
    "llx_pool_fill_u16": (_i, [_vp, C.c_uint16, _vp]),
    "llx_plan_stage": (_i, [_i, _i, _i, _i, C.POINTER(_i), C.POINTER(_i)]),
    "llx_predict_stage_sizes": (_i, [_i, C.c_double, C.c_double, _i, _i32p, _i, C.POINTER(_i)]),
    "llx_launch_opts_init": (None, [C.POINTER(LaunchOpts)]),
    "llx_migrate_stage": (_i, [_vp, _i32p, _vp, _i32p, _i, _vp]),
    "llx_migrate_stage_ex": (_i, [_vp, _i32p, _vp, _i32p, _i, _vp, C.POINTER(LaunchOpts)]),
    "llx_migrate_stage_wait": (_i, [_vp, _i32p, _vp, _i32p, _i, _vp]),
    "llx_migrate_stage_wait_ex": (_i, [_vp, _i32p, _vp, _i32p, _i, _vp, C.POINTER(LaunchOpts)]),
    "llx_migrate_batch": (_i, [_vp, _vp, _i32p, _i32p, _i32p, _i, _vp]),
    "llx_migrate_batch_ex": (_i, [_vp, _vp, _i32p, _i32p, _i32p, _i, _vp, C.POINTER(LaunchOpts)]),
    "llx_staging_bytes": (_sz, [_vp, _i]),
    "llx_staging_alloc_pinned": (_i, [_sz, C.POINTER(_vp), C.POINTER(_vp)]),
    "llx_staging_free_pinned": (_i, [_vp]),
    "llx_pack": (_i, [_vp, _i32p, _i, _vp, _sz, _vp]),
    "llx_pack_ex": (_i, [_vp, _i32p, _i, _vp, _sz, _vp, C.POINTER(LaunchOpts)]),
    "llx_unpack": (_i, [_vp, _sz, _vp, _i32p, _i, _vp]),
    "llx_unpack_ex": (_i, [_vp, _sz, _vp, _i32p, _i, _vp, C.POINTER(LaunchOpts)]),
    "llx_migrate_via_host": (_i, [_vp, _i32p, _vp, _i32p, _i, _vp, _sz, _i, _vp]),
    "llx_migrate_via_host_ex": (_i, [_vp, _i32p, _vp, _i32p, _i, _vp, _sz, _i, _vp, C.POINTER(LaunchOpts)]),
    "llx_blockmgr_create": (_i, [_i, C.POINTER(_vp)]),
    "llx_blockmgr_destroy": (_i, [_vp]),
    "llx_blockmgr_num_free": (_i, [_vp]),
    "llx_blockmgr_num_blocks": (_i, [_vp]),
    "llx_blockmgr_alloc": (_i, [_vp, _i, _i32p]),
    "llx_blockmgr_release": (_i, [_vp, _i32p, _i]),
    "llx_migration_begin": (_i, [_vp, _vp, _vp, _vp, _i, _i, C.POINTER(_vp)]),
    "llx_migration_stage": (_i, [_vp, _i32p, _i, _i, _i, _vp, C.POINTER(_i), C.POINTER(_i), _i32p]),
    "llx_migration_commit": (_i, [_vp, _i32p, _i, _i, _i32p, _i, C.POINTER(_i)]),
    "llx_migration_abort": (_i, [_vp, _i]),
    "llx_migration_set_stage_opts": (_i, [_vp, C.POINTER(LaunchOpts)]),
    "llx_budget_ctl_create": (_i, [C.c_double, _i, _i, _i, _i, C.POINTER(_vp)]),
    "llx_budget_ctl_destroy": (_i, [_vp]),
    "llx_budget_ctl_observe": (_i, [_vp, C.c_double, _i, C.POINTER(_i)]),
    "llx_budget_ctl_gbps": (_i, [_vp]),
    "llx_budget_ctl_last_slowdown_pct": (C.c_double, [_vp]),
    "llx_budget_ctl_adjustments": (_i, [_vp]),
    "llx_migration_state": (_i, [_vp]),
    "llx_migration_abort_reason": (_i, [_vp]),
    "llx_migration_blocks_migrated": (_i, [_vp]),
    "llx_migration_stages": (_i, [_vp]),
    "llx_migration_destroy": (_i, [_vp]),
    "llx_calc_freeness": (_i, [C.POINTER(ReqInfo), _i, C.c_double, C.POINTER(C.c_double), _i, _i,
                               C.POINTER(C.c_double), C.POINTER(C.c_double)]),
    "llx_pair_instances": (_i, [C.POINTER(C.c_double), _i, C.c_double, C.c_double, _i32p, _i32p, _i, C.POINTER(_i)]),
    "llx_migration_order": (_i, [_i32p, _i32p, _i, _i32p]),
    "llx_plan_migration_batch": (_i, [C.POINTER(ReqInfo), _i32p, _i, C.c_double, C.POINTER(C.c_double), _i, _i, C.c_double,
                                      _i32p, _i32p, _vp, _i, _i32p, C.POINTER(_i), _i32p, _i32p, _i32p, _i, C.POINTER(_i)]),
    "llx_append_tokens": (_i, [_vp, _i32p, _i, _i, _i, _vp, _vp]),
    "llx_decode_attention": (_i, [_vp, _i, _vp, _vp, _vp, _vp, _i, _i, C.c_float, _vp]),
    "llx_decode_attention_static_ws": (_i, [_vp, _i, _vp, _vp, _vp, _vp, _i, _i, C.c_float, _vp]),
    "llx_set_option": (_i, [_i, C.c_longlong]),
    "llx_get_option": (C.c_longlong, [_i]),
    "llx_get_counters": (None, [C.POINTER(_Counters)]),
    "llx_reset_counters": (None, []),
    "llx_synchronize": (_i, [_vp]),
    "llx_status_str": (C.c_char_p, [_i]),
    "llx_last_error": (C.c_char_p, []),
    "llx_version": (C.c_char_p, []),
}

_lib = None


class LlxError(RuntimeError):
    def __init__(self, status: int, name: str, detail: str):
        super().__init__(f"{name} ({status}): {detail}")
        self.status, self.name, self.detail = status, name, detail


def load():
    """dlopen libllx.so and declare every prototype.  Fails loudly if the library is not built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2406_03243_b200.build` "
                          "(the llx path has no CPU fallback)")
    lib_ = C.CDLL(LIB_PATH)
    for name, (res, args) in EXPORTS.items():
        fn = getattr(lib_, name)
        fn.restype, fn.argtypes = res, args
    _lib = lib_
    return _lib


def lib():
    return load()


def _check(rc: int):
    if rc != 0:
        l = load()
        raise LlxError(rc, l.llx_status_str(rc).decode(), l.llx_last_error().decode())


def _ids(x):
    a = np.ascontiguousarray(np.asarray(x, dtype=np.int32).reshape(-1))
    return a, a.ctypes.data_as(_i32p)


def _stream(s) -> int:
    if s is None:
        return 0
    return int(getattr(s, "cuda_stream", s))


class Pool:
    """Handle of one serving instance's KV pool (llx_pool*)."""

    def __init__(self, handle: int, keepalive=None):
        self._h = handle
        self._keep = keepalive

    @property
    def handle(self) -> int:
        if not self._h:
            raise LlxError(-1, "LLX_ERR_INVALID_ARG", "pool already destroyed")
        return self._h

    tile_bytes = property(lambda self: load().llx_pool_tile_bytes(self.handle))
    block_bytes = property(lambda self: load().llx_pool_block_bytes(self.handle))
    nbytes = property(lambda self: load().llx_pool_bytes(self.handle))
    num_blocks = property(lambda self: load().llx_pool_num_blocks(self.handle))

    def data(self, layer: int, kv: int) -> int:
        p = load().llx_pool_data(self.handle, layer, kv)
        if not p:
            raise LlxError(-1, "LLX_ERR_INVALID_ARG", f"bad (layer={layer}, kv={kv})")
        return p

    def upload(self, layer, kv, first_block, host: np.ndarray, stream=None):
        host = np.ascontiguousarray(host)
        nb, rem = divmod(host.nbytes, self.tile_bytes)
        assert rem == 0, "host array must hold whole tiles"
        _check(load().llx_pool_upload(self.handle, layer, kv, first_block, nb, host.ctypes.data, _stream(stream)))

    def download(self, layer, kv, first_block, n_blocks, stream=None, dtype=np.uint16) -> np.ndarray:
        out = np.empty((n_blocks, self.tile_bytes // np.dtype(dtype).itemsize), dtype=dtype)
        _check(load().llx_pool_download(self.handle, layer, kv, first_block, n_blocks, out.ctypes.data, _stream(stream)))
        return out

    def fill_u16(self, pattern: int, stream=None):
        _check(load().llx_pool_fill_u16(self.handle, pattern, _stream(stream)))

    def destroy(self):
        if self._h:
            load().llx_pool_destroy(self._h)
            self._h = 0
            self._keep = None

    def __del__(self):
        with contextlib.suppress(Exception):
            self.destroy()


def pool_bytes_for(layers, kv_heads, head_dim, block_size, dtype, num_blocks) -> int:
    return load().llx_pool_bytes_for(layers, kv_heads, head_dim, block_size, dtype, num_blocks)


def pool_create(layers, kv_heads, head_dim, block_size, dtype, num_blocks) -> Pool:
    h = _vp()
    _check(load().llx_pool_create(layers, kv_heads, head_dim, block_size, dtype, num_blocks, C.byref(h)))
    return Pool(h.value)


def pool_wrap(dev_ptr: int, nbytes: int, layers, kv_heads, head_dim, block_size, dtype, num_blocks, keepalive=None) -> Pool:
    h = _vp()
    _check(load().llx_pool_wrap(dev_ptr, nbytes, layers, kv_heads, head_dim, block_size, dtype, num_blocks, C.byref(h)))
    return Pool(h.value, keepalive)


IPC_HANDLE_BYTES = 96


def pool_ipc_export(pool: Pool) -> bytes:
    """Handle of a library-allocated pool for another process (llx_pool_ipc_export): send the bytes, open them there."""
    buf = C.create_string_buffer(IPC_HANDLE_BYTES)
    _check(load().llx_pool_ipc_export(pool.handle, buf))
    return buf.raw


def pool_ipc_open(handle: bytes) -> Pool:
    if len(handle) != IPC_HANDLE_BYTES:
        raise LlxError(-1, "LLX_ERR_INVALID_ARG", "an llx pool handle has %d bytes" % IPC_HANDLE_BYTES)
    h = _vp()
    _check(load().llx_pool_ipc_open(C.c_char_p(handle), C.byref(h)))
    return Pool(h.value)


def plan_stage(num_tokens: int, blocks_migrated: int, block_size: int, last_stage_max_blocks: int):
    """-> (n, is_final): the logical blocks [blocks_migrated, blocks_migrated+n) of the next stage."""
    n, f = _i(), _i()
    _check(load().llx_plan_stage(num_tokens, blocks_migrated, block_size, last_stage_max_blocks, C.byref(n), C.byref(f)))
    return n.value, bool(f.value)


def predict_stage_sizes(n0: int, copy_blocks_per_s: float, decode_tokens_per_s: float, block_size: int, cap: int = 64):
    """-> [n_0, n_1, ...]: the stage sizes a migration takes at these measured rates (llx_predict_stage_sizes)."""
    out, k = (C.c_int32 * cap)(), _i()
    _check(load().llx_predict_stage_sizes(n0, copy_blocks_per_s, decode_tokens_per_s, block_size, out, cap, C.byref(k)))
    return [int(out[i]) for i in range(k.value)]


def migrate_stage(src: Pool, src_block_ids, dst: Pool, dst_block_ids, stream=None, opts=None):
    """opts: None (llx_migrate_stage), or a dict / LaunchOpts = this call's own launch policy (llx_migrate_stage_ex)."""
    s, sp = _ids(src_block_ids)
    d, dp = _ids(dst_block_ids)
    if s.size != d.size:
        raise LlxError(-1, "LLX_ERR_INVALID_ARG", "src/dst id lists differ in length")
    if opts is None:
        _check(load().llx_migrate_stage(src.handle, sp, dst.handle, dp, s.size, _stream(stream)))
    else:
        _check(load().llx_migrate_stage_ex(src.handle, sp, dst.handle, dp, s.size, _stream(stream), _opts(opts)))


def migrate_stage_wait(src: Pool, src_block_ids, dst: Pool, dst_block_ids, stream=None, opts=None):
    """llx_migrate_stage + wait for its completion (the final stage: downtime ends when this returns)."""
    s, sp = _ids(src_block_ids)
    d, dp = _ids(dst_block_ids)
    if s.size != d.size:
        raise LlxError(-1, "LLX_ERR_INVALID_ARG", "src/dst id lists differ in length")
    if opts is None:
        _check(load().llx_migrate_stage_wait(src.handle, sp, dst.handle, dp, s.size, _stream(stream)))
    else:
        _check(load().llx_migrate_stage_wait_ex(src.handle, sp, dst.handle, dp, s.size, _stream(stream), _opts(opts)))


def migrate_batch(src: Pool, dst: Pool, req_offsets, src_block_ids, dst_block_ids, stream=None, opts=None):
    o, op = _ids(req_offsets)
    s, sp = _ids(src_block_ids)
    d, dp = _ids(dst_block_ids)
    if o.size < 1 or s.size != d.size or int(o[-1]) != s.size:
        raise LlxError(-1, "LLX_ERR_INVALID_ARG", "req_offsets[-1] must equal the number of id pairs")
    if opts is None:
        _check(load().llx_migrate_batch(src.handle, dst.handle, op, sp, dp, o.size - 1, _stream(stream)))
    else:
        _check(load().llx_migrate_batch_ex(src.handle, dst.handle, op, sp, dp, o.size - 1, _stream(stream), _opts(opts)))


def staging_bytes(pool: Pool, n: int) -> int:
    return load().llx_staging_bytes(pool.handle, n)


class PinnedStaging:
    """Pinned, mapped host staging buffer (llx_staging_alloc_pinned)."""

    def __init__(self, nbytes: int):
        h, d = _vp(), _vp()
        _check(load().llx_staging_alloc_pinned(nbytes, C.byref(h), C.byref(d)))
        self.host_ptr, self.dev_alias, self.nbytes = h.value, d.value, nbytes

    def as_numpy(self, dtype=np.uint16) -> np.ndarray:
        buf = (C.c_char * self.nbytes).from_address(self.host_ptr)
        return np.frombuffer(buf, dtype=dtype)

    def free(self):
        if self.host_ptr:
            load().llx_staging_free_pinned(self.host_ptr)
            self.host_ptr = 0

    def __del__(self):
        with contextlib.suppress(Exception):
            self.free()


def pack(src: Pool, src_block_ids, staging_ptr: int, staging_nbytes: int, stream=None, opts=None):
    s, sp = _ids(src_block_ids)
    if opts is None:
        _check(load().llx_pack(src.handle, sp, s.size, staging_ptr, staging_nbytes, _stream(stream)))
    else:
        _check(load().llx_pack_ex(src.handle, sp, s.size, staging_ptr, staging_nbytes, _stream(stream), _opts(opts)))


def unpack(staging_ptr: int, staging_nbytes: int, dst: Pool, dst_block_ids, stream=None, opts=None):
    d, dp = _ids(dst_block_ids)
    if opts is None:
        _check(load().llx_unpack(staging_ptr, staging_nbytes, dst.handle, dp, d.size, _stream(stream)))
    else:
        _check(load().llx_unpack_ex(staging_ptr, staging_nbytes, dst.handle, dp, d.size, _stream(stream), _opts(opts)))


def migrate_via_host(src: Pool, src_block_ids, dst: Pool, dst_block_ids, staging_ptr: int, staging_nbytes: int,
                     chunk_blocks: int = 0, stream=None, opts=None):
    s, sp = _ids(src_block_ids)
    d, dp = _ids(dst_block_ids)
    if s.size != d.size:
        raise LlxError(-1, "LLX_ERR_INVALID_ARG", "src/dst id lists differ in length")
    if opts is None:
        _check(load().llx_migrate_via_host(src.handle, sp, dst.handle, dp, s.size, staging_ptr, staging_nbytes,
                                           chunk_blocks, _stream(stream)))
    else:
        _check(load().llx_migrate_via_host_ex(src.handle, sp, dst.handle, dp, s.size, staging_ptr, staging_nbytes,
                                              chunk_blocks, _stream(stream), _opts(opts)))


REQ_RUNNING, REQ_FINISHED, REQ_PREEMPTED, REQ_PEER_FAILED = range(4)
MIG_READY, MIG_COPYING, MIG_FINAL_COPYING, MIG_COMMITTED, MIG_ABORTED = range(5)
ABORT_NONE, ABORT_FINISHED, ABORT_PREEMPTED, ABORT_PEER_FAILED, ABORT_NO_SPACE = range(5)


class BlockManager:
    """One instance's free list of block ids (llx_blockmgr*)."""

    def __init__(self, num_blocks: int):
        h = _vp()
        _check(load().llx_blockmgr_create(num_blocks, C.byref(h)))
        self._h = h.value

    handle = property(lambda self: self._h)
    num_free = property(lambda self: load().llx_blockmgr_num_free(self._h))
    num_blocks = property(lambda self: load().llx_blockmgr_num_blocks(self._h))

    def alloc(self, n: int) -> np.ndarray:
        out = np.empty(max(n, 0), dtype=np.int32)
        _check(load().llx_blockmgr_alloc(self._h, n, out.ctypes.data_as(_i32p)))
        return out

    def release(self, ids):
        a, ap = _ids(ids)
        _check(load().llx_blockmgr_release(self._h, ap, a.size))

    def __del__(self):
        with contextlib.suppress(Exception):
            if self._h:
                load().llx_blockmgr_destroy(self._h)
                self._h = 0


class BudgetController:
    """The bandwidth budget of the non-final stages chosen from the decode steps the engine observes (llx_budget_ctl*)."""

    def __init__(self, target_slowdown_pct: float, min_gbps: int, max_gbps: int, start_gbps: int, window: int = 8):
        h = _vp()
        _check(load().llx_budget_ctl_create(float(target_slowdown_pct), min_gbps, max_gbps, start_gbps, window, C.byref(h)))
        self._h = h.value

    gbps = property(lambda self: load().llx_budget_ctl_gbps(self._h))
    last_slowdown_pct = property(lambda self: load().llx_budget_ctl_last_slowdown_pct(self._h))
    adjustments = property(lambda self: load().llx_budget_ctl_adjustments(self._h))

    def observe(self, step_ms: float, migrating: bool) -> int:
        b = _i()
        _check(load().llx_budget_ctl_observe(self._h, float(step_ms), 1 if migrating else 0, C.byref(b)))
        return b.value

    def __del__(self):
        with contextlib.suppress(Exception):
            if self._h:
                load().llx_budget_ctl_destroy(self._h)
                self._h = 0


class Migration:
    """One request's migration through the handshake of PAPER.md:142 (llx_migration*)."""

    def __init__(self, src, src_mgr: BlockManager, dst, dst_mgr: BlockManager, block_size: int,
                 last_stage_max_blocks: int):
        h = _vp()
        _check(load().llx_migration_begin(src.handle if src is not None else None, src_mgr.handle,
                                          dst.handle if dst is not None else None, dst_mgr.handle,
                                          block_size, last_stage_max_blocks, C.byref(h)))
        self._h, self._keep = h.value, (src, src_mgr, dst, dst_mgr)

    state = property(lambda self: load().llx_migration_state(self._h))
    abort_reason = property(lambda self: load().llx_migration_abort_reason(self._h))
    blocks_migrated = property(lambda self: load().llx_migration_blocks_migrated(self._h))
    stages = property(lambda self: load().llx_migration_stages(self._h))

    def stage(self, src_block_table, num_tokens: int, status: int = REQ_RUNNING, stream=None):
        """-> (n, is_final, dst_ids) of the stage just issued; n == 0 and state MIG_ABORTED after an abort."""
        t, tp = _ids(src_block_table)
        n, f = _i(), _i()
        out = np.empty(max(t.size, 1), dtype=np.int32)
        _check(load().llx_migration_stage(self._h, tp, t.size, num_tokens, status, _stream(stream), C.byref(n),
                                          C.byref(f), out.ctypes.data_as(_i32p)))
        return n.value, bool(f.value), out[:n.value].copy()

    def commit(self, src_block_table, status: int = REQ_RUNNING):
        """-> the request's block table on the destination, or None when the commit turned into an abort."""
        t, tp = _ids(src_block_table)
        out = np.empty(max(t.size, 1), dtype=np.int32)
        n = _i()
        _check(load().llx_migration_commit(self._h, tp, t.size, status, out.ctypes.data_as(_i32p), out.size, C.byref(n)))
        return out[:n.value].copy() if self.state == MIG_COMMITTED else None

    def abort(self, reason: int = ABORT_PEER_FAILED):
        _check(load().llx_migration_abort(self._h, reason))

    def set_stage_opts(self, opts):
        """Launch policy of the non-final stages (dict / LaunchOpts / None); the final stage always runs unthrottled."""
        _check(load().llx_migration_set_stage_opts(self._h, _opts(opts)))

    def __del__(self):
        with contextlib.suppress(Exception):
            if self._h:
                load().llx_migration_destroy(self._h)
                self._h = 0


def calc_freeness(reqs, M: float, headroom_for_priority, is_terminating: bool = False):
    """reqs: iterable of (is_queuing, is_head_of_line, is_fake, priority, demand, physical_usage) -> (F, sum V)"""
    reqs = list(reqs)
    arr = (ReqInfo * max(len(reqs), 1))(*[ReqInfo(int(a), int(b), int(c), int(p), float(d), float(u))
                                          for a, b, c, p, d, u in reqs])
    hr = (C.c_double * len(headroom_for_priority))(*[float(x) for x in headroom_for_priority])
    f, tot = C.c_double(), C.c_double()
    _check(load().llx_calc_freeness(arr, len(reqs), float(M), hr, len(headroom_for_priority), int(is_terminating),
                                    C.byref(f), C.byref(tot)))
    return f.value, tot.value


def pair_instances(freeness, src_below: float, dst_above: float):
    f = np.ascontiguousarray(np.asarray(freeness, dtype=np.float64).reshape(-1))
    s, d = np.empty(max(f.size, 1), np.int32), np.empty(max(f.size, 1), np.int32)
    n = _i()
    _check(load().llx_pair_instances(f.ctypes.data_as(C.POINTER(C.c_double)), f.size, src_below, dst_above,
                                     s.ctypes.data_as(_i32p), d.ctypes.data_as(_i32p), f.size, C.byref(n)))
    return list(zip(s[:n.value].tolist(), d[:n.value].tolist()))


def migration_order(priority, seq_len):
    p, pp = _ids(priority)
    q, qp = _ids(seq_len)
    if p.size != q.size:
        raise LlxError(-1, "LLX_ERR_INVALID_ARG", "priority/seq_len differ in length")
    out = np.empty(max(p.size, 1), np.int32)
    _check(load().llx_migration_order(pp, qp, p.size, out.ctypes.data_as(_i32p)))
    return out[:p.size].tolist()


def plan_migration_batch(reqs, seq_len, M: float, headroom_for_priority, src_below: float, block_tables,
                         dst_mgr: BlockManager, dst_reserve_blocks: int = 0, is_terminating: bool = False):
    """llx_plan_migration_batch.  reqs as in calc_freeness; block_tables: one id list per request (empty for queuing
    requests).  -> (chosen, req_offsets, src_ids, dst_ids): the last three are the arguments of migrate_batch."""
    reqs = list(reqs)
    n = len(reqs)
    arr = (ReqInfo * max(n, 1))(*[ReqInfo(int(a), int(b), int(c), int(p), float(d), float(u)) for a, b, c, p, d, u in reqs])
    hr = (C.c_double * len(headroom_for_priority))(*[float(x) for x in headroom_for_priority])
    sl, slp = _ids(seq_len)
    if sl.size != n or len(block_tables) != n:
        raise LlxError(-1, "LLX_ERR_INVALID_ARG", "reqs / seq_len / block_tables differ in length")
    off = np.zeros(n + 1, dtype=np.int32)
    for r, t in enumerate(block_tables):
        off[r + 1] = off[r] + len(t)
    flat, flatp = _ids(np.concatenate([np.asarray(t, dtype=np.int32).reshape(-1) for t in block_tables])
                       if n else np.zeros(0, np.int32))
    cap = int(off[-1])
    chosen, ro = np.empty(max(n, 1), np.int32), np.empty(n + 1, np.int32)
    s_out, d_out = np.empty(max(cap, 1), np.int32), np.empty(max(cap, 1), np.int32)
    nc, npairs = _i(), _i()
    _check(load().llx_plan_migration_batch(arr, slp, n, float(M), hr, len(headroom_for_priority), int(is_terminating),
                                           float(src_below), off.ctypes.data_as(_i32p), flatp, dst_mgr.handle,
                                           int(dst_reserve_blocks), chosen.ctypes.data_as(_i32p), C.byref(nc),
                                           ro.ctypes.data_as(_i32p), s_out.ctypes.data_as(_i32p), d_out.ctypes.data_as(_i32p),
                                           cap, C.byref(npairs)))
    k, m = nc.value, npairs.value
    return chosen[:k].tolist(), ro[:k + 1].copy(), s_out[:m].copy(), d_out[:m].copy()


def append_tokens(pool: Pool, block_table, t0: int, t1: int, dev_values_ptr: int, stream=None):
    t, tp = _ids(block_table)
    _check(load().llx_append_tokens(pool.handle, tp, t.size, t0, t1, dev_values_ptr, _stream(stream)))


def decode_attention(pool: Pool, layer: int, dev_q: int, dev_out: int, dev_block_tables: int, dev_ctx_lens: int,
                     B: int, max_blocks: int, scale: float, stream=None):
    _check(load().llx_decode_attention(pool.handle, layer, dev_q, dev_out, dev_block_tables, dev_ctx_lens,
                                       B, max_blocks, scale, _stream(stream)))


ATTN_STATIC_WS_BYTES = 16 << 20   # LLX_ATTN_STATIC_WS_BYTES of include/llx.h


def decode_attention_static_ws(pool: Pool, layer: int, dev_q: int, dev_out: int, dev_block_tables: int, dev_ctx_lens: int,
                               B: int, max_blocks: int, scale: float, stream=None):
    """llx_decode_attention for a caller that must not allocate device memory while it runs (an engine that gave all
    free HBM to its KV pool, a decode loop that cannot afford cudaMalloc's device-wide stall): same arguments and
    result, the split-KV partials live in a fixed ATTN_STATIC_WS_BYTES array inside the library instead of a
    cudaMalloc'ed per-pool workspace.  Larger shapes raise LLX_ERR_INVALID_ARG; calls that overlap on the GPU race on
    the shared array; make the first call on a device outside any stream capture (include/llx.h has the details)."""
    _check(load().llx_decode_attention_static_ws(pool.handle, layer, dev_q, dev_out, dev_block_tables, dev_ctx_lens,
                                                 B, max_blocks, scale, _stream(stream)))


def set_option(opt: int, value: int):
    _check(load().llx_set_option(opt, value))


def get_option(opt: int) -> int:
    return load().llx_get_option(opt)


@contextlib.contextmanager
def options(**kw):
    """Temporarily set PROCESS-WIDE default options by lower-case name, e.g. options(copy_kernel=1, max_ctas=16).
    For experiments; the policy of one call belongs in its `opts=` argument (llx_launch_opts)."""
    names = dict(copy_kernel=OPT_COPY_KERNEL, max_ctas=OPT_MAX_CTAS, chunk_bytes=OPT_CHUNK_BYTES,
                 ring_stages=OPT_RING_STAGES, ids_by_value_max=OPT_IDS_BY_VALUE_MAX,
                 attn_split_tokens=OPT_ATTN_SPLIT_TOKENS, unit_order=OPT_UNIT_ORDER, l2_hint=OPT_L2_HINT,
                 rings_per_cta=OPT_RINGS_PER_CTA, pdl=OPT_PDL, bandwidth_gbps=OPT_BANDWIDTH_GBPS,
                 via_host_mode=OPT_VIA_HOST_MODE, dynamic_tail_pct=OPT_DYNAMIC_TAIL_PCT,
                 dynamic_tail_batch=OPT_DYNAMIC_TAIL_BATCH, exact_residency=OPT_EXACT_RESIDENCY,
                 copy_smem_carveout_pct=OPT_COPY_SMEM_CARVEOUT_PCT, paced_slice_us=OPT_PACED_SLICE_US,
                 overlap_prev=OPT_OVERLAP_PREV)
    old = {k: get_option(names[k]) for k in kw}
    try:
        for k, v in kw.items():
            set_option(names[k], v)
        yield
    finally:
        for k, v in old.items():
            set_option(names[k], v)


def synchronize(stream=None):
    _check(load().llx_synchronize(_stream(stream)))


def counters() -> dict:
    c = _Counters()
    load().llx_get_counters(C.byref(c))
    return {f: int(getattr(c, f)) for f, _ in c._fields_}


def reset_counters():
    load().llx_reset_counters()


def version() -> str:
    return load().llx_version().decode()
