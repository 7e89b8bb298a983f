/* llx.h — C ABI of the B200-native live-migration path for a paged KV cache.
 *
 * What this library computes is fixed by Llumnix (arxiv 2406.03243); citations are
 * "PAPER.md:<line>" of the paper text plus the section the line falls in.
 *
 *   - §4.2 "Live Migration of LLM Requests" (Fig. 6): the KV cache is
 *     append-only, so the blocks of completed iterations are copied to the destination
 *     instance in STAGES while decoding continues; a short final stage copies the last
 *     blocks once the source has stopped the request.
 *   - §4.2 handshake (Fig. 7): the destination RESERVES the blocks of a stage
 *     before the stage runs; the caller therefore passes the destination block ids in.
 *   - §5 "Block fusion": the copy unit is the block = K *or* V of block_size
 *     tokens of ONE layer (128 KB for 16-bit LLaMA-7B); the many small blocks of a request
 *     are fused into ONE contiguous buffer for the transport.
 *   - §5 "KV cache transfer": copies run on their own CUDA stream so that
 *     inference is not blocked.
 *
 * Memory model.  A pool is one serving instance's KV cache:
 *
 *     pool[layer][kv][block][slot][head][dim]       kv: 0 = K, 1 = V
 *
 * one dense allocation in that order, i.e. per layer and per K|V a row-major tensor
 * [num_blocks, block_size, kv_heads, head_dim].  A "tile" is pool[layer][kv][block] —
 * tile_bytes = block_size*kv_heads*head_dim*elem_bytes contiguous bytes — the paper's block.
 * A "block id" names the same row index in every (layer, kv) slice; block_bytes =
 * 2*layers*tile_bytes.  tile_bytes must be a multiple of 16 and the base 16-byte aligned.
 *
 * Conventions for every call.
 *   - Pointers named *_ids / req_offsets are HOST int32 arrays owned by the caller; the
 *     library copies them before returning, so they may be reused at once.
 *   - Pointers named dev_* are DEVICE pointers.  `staging` may be a device pointer or a
 *     pinned, mapped host pointer (UVA tells them apart).
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).
 *     Data calls only ENQUEUE work on it and return; completion is observed by the caller
 *     through the stream.  Pools and staging buffers must outlive the enqueued work.
 *   - Errors are return codes; nothing throws or aborts across this boundary.  Argument
 *     errors are found on the host BEFORE anything is launched: a failed call changes no
 *     byte of any pool.  An asynchronous CUDA fault surfaces as LLX_ERR_CUDA from a later
 *     call.  n == 0 (or R == 0) is LLX_OK and launches nothing.
 *   - The library never allocates or frees BLOCKS: reservation is the caller's job
 *     (the paper's PRE-ALLOC).  An aborted migration needs no byte rollback.
 *   - There is no CPU fallback: without a CUDA device every data call returns LLX_ERR_CUDA.
 *   - Threads.  Data calls may be issued from several host threads at once, on distinct streams, between the same
 *     or different pools; work of one stream runs in the order enqueued.  Launch policy is PER CALL
 *     (llx_launch_opts, the *_ex entry points): one thread's bandwidth budget never touches another thread's final
 *     stage.  llx_set_option only changes the process defaults that a call inherits for fields it leaves at
 *     LLX_OPT_DEFAULT.  llx_decode_attention calls on one pool must be ordered on one stream (they share the pool's
 *     workspace); llx_blockmgr / llx_migration objects are not thread-safe per object.
 *   - CUDA graphs.  llx_migrate_stage(_ex), llx_migrate_batch(_ex), llx_pack / llx_unpack with a DEVICE buffer (id lists of
 *     <= 256 pairs: the ids then travel in the kernel parameters), llx_append_tokens (<= 256 tokens) and
 *     llx_decode_attention (workspace already large enough) may be stream-captured and replayed on any stream.
 *     Calls that would have to allocate, synchronise or stage ids through pinned memory while `cuda_stream` is
 *     capturing return LLX_ERR_STATE and enqueue nothing (longer id lists, pinned-host staging,
 *     llx_migrate_via_host, llx_migrate_stage_wait, a first-use allocation).  Captured long stages run without the
 *     dynamic tail (its claim counter belongs to a stream, a graph may replay anywhere).
 */
#ifndef LLX_H_
#define LLX_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct llx_pool llx_pool; /* opaque */

/* Only the element size matters to migration; decode attention requires LLX_F16. */
typedef enum { LLX_F16 = 0, LLX_BF16 = 1, LLX_U8 = 2 } llx_dtype;

typedef enum {
    LLX_OK = 0,
    LLX_ERR_INVALID_ARG = -1,       /* NULL pointer, negative size, unsupported shape */
    LLX_ERR_GEOMETRY_MISMATCH = -2, /* src and dst pools differ in layers / tile_bytes */
    LLX_ERR_BLOCK_OUT_OF_RANGE = -3,
    LLX_ERR_DUPLICATE_DST = -4,     /* a destination block id appears twice in one call */
    LLX_ERR_ALIAS = -5,             /* src and dst are the same pool / overlap */
    LLX_ERR_STAGING_TOO_SMALL = -6,
    LLX_ERR_OOM = -7,
    LLX_ERR_CUDA = -8,
    LLX_ERR_NO_SPACE = -9,          /* the block manager has fewer free blocks than asked for */
    LLX_ERR_STATE = -10             /* call not allowed in the migration's current state */
} llx_status;

/* ---- pools (D1 in SURVEY.md; PagedAttention blocks) ------------------ */

/* Allocates layers*2*num_blocks tiles with cudaMalloc on the current device; contents are
 * undefined.  *out is owned by the caller and released with llx_pool_destroy. */
llx_status llx_pool_create(int layers, int kv_heads, int head_dim, int block_size, llx_dtype dtype,
                           int num_blocks, llx_pool** out);
/* Describes caller-owned device memory (e.g. a torch tensor) of at least llx_pool_bytes;
 * `bytes` is checked.  llx_pool_destroy of a wrapped pool frees only the handle. */
llx_status llx_pool_wrap(void* dev_ptr, size_t bytes, int layers, int kv_heads, int head_dim, int block_size,
                         llx_dtype dtype, int num_blocks, llx_pool** out);
llx_status llx_pool_destroy(llx_pool* pool);

void*  llx_pool_data(const llx_pool* pool, int layer, int kv); /* device address of pool[layer][kv][0]; NULL on bad args */
size_t llx_pool_tile_bytes(const llx_pool* pool);              /* block_size*kv_heads*head_dim*elem_bytes */
size_t llx_pool_block_bytes(const llx_pool* pool);             /* 2*layers*tile_bytes */
size_t llx_pool_bytes(const llx_pool* pool);                   /* num_blocks*block_bytes */
int    llx_pool_num_blocks(const llx_pool* pool);
/* Bytes a pool of this geometry needs (for sizing memory passed to llx_pool_wrap); 0 on bad args. */
size_t llx_pool_bytes_for(int layers, int kv_heads, int head_dim, int block_size, llx_dtype dtype, int num_blocks);

/* The destination instance as ANOTHER PROCESS (instances are separate actors; here one process per
 * GPU / per instance): the owner of a library-allocated pool exports a handle (LLX_IPC_HANDLE_BYTES opaque bytes, sent
 * to the peer by whatever channel the caller has), the peer opens it and gets a pool that names the SAME device memory.
 * llx_migrate_stage / _batch into an opened pool then store straight into the other process's KV cache — on the same GPU
 * (two instances sharing one device) or on another one (the mapping enables peer access; the copy takes the cross-GPU
 * route).  The handle carries the pool's geometry, so the opened pool cannot disagree with the exporter's: its last
 * 4 bytes are a checksum (32-bit FNV-1a of the 92 bytes in front of them) and llx_pool_ipc_open also compares the geometry
 * with the size of the allocation it has just mapped — a truncated, corrupted or stale handle (one that names more
 * blocks or layers than the exporter's allocation holds) is LLX_ERR_INVALID_ARG, not a pool that writes past the mapping.
 * llx_pool_destroy of an opened pool unmaps it; the exporter must keep its pool alive meanwhile.  Only pools from
 * llx_pool_create can be exported (the handle names a whole allocation); LLX_ERR_CUDA when the handle is opened in the
 * process that exported it (the driver refuses that). */
#define LLX_IPC_HANDLE_BYTES 96
llx_status llx_pool_ipc_export(const llx_pool* pool, void* handle_out);
llx_status llx_pool_ipc_open(const void* handle, llx_pool** out);

/* Plain stream-ordered copies between HOST memory and n_blocks consecutive tiles
 * pool[layer][kv][first_block ...]: how the owner of a library-allocated pool fills and
 * inspects it.  `host` holds n_blocks*tile_bytes bytes; pinned memory makes them truly async. */
llx_status llx_pool_upload(llx_pool* pool, int layer, int kv, int first_block, int n_blocks, const void* host,
                           void* cuda_stream);
llx_status llx_pool_download(const llx_pool* pool, int layer, int kv, int first_block, int n_blocks, void* host,
                             void* cuda_stream);
/* Sets every 16-bit word of the whole pool to `pattern` (the tests' sentinel). */
llx_status llx_pool_fill_u16(llx_pool* pool, uint16_t pattern, void* cuda_stream);

/* ---- S1: stage planning (host arithmetic, no device work) -------------------- */

/* Which logical blocks [blocks_migrated, blocks_migrated + *n) of a request the NEXT stage takes.
 * A non-final stage copies "the KV cache blocks of completed iterations" that can no longer
 * change: the full blocks, never the one being appended to.  When at most
 * last_stage_max_blocks blocks remain the stage is final (*is_final = 1): the caller stops the
 * request first, and the stage takes everything left including the partly filled block.
 * LLX_ERR_INVALID_ARG if blocks_migrated exceeds ceil(num_tokens/block_size) or a size is bad. */
llx_status llx_plan_stage(int num_tokens, int blocks_migrated, int block_size, int last_stage_max_blocks, int* n,
                          int* is_final);

/* How many stages a migration will take, from MEASURED rates ("copying is generally much faster than the
 * computation", so "the number of new blocks is typically small"; "the migration only takes two stages").
 * While stage k copies n_k blocks at copy_blocks_per_s, the request decodes decode_tokens_per_s * n_k / copy_blocks_per_s
 * tokens, i.e. the next stage has  n_{k+1} = max(1, ceil(n_k * decode_tokens_per_s / (copy_blocks_per_s * block_size)))
 * blocks; the sequence ends with the first stage of ONE block (the final stage).  Writes n_0 = n0, n_1, ... to sizes_out
 * (HOST int32[cap]) and their count to *n_stages.  A caller picks a bandwidth budget for the non-final stages with it:
 * copy_blocks_per_s = budget / (2 * block_bytes); if the sequence has not reached 1 within cap entries (the last entry
 * is > 1), decoding outruns the copy at that budget.  LLX_ERR_INVALID_ARG: n0 < 1, a rate that is not finite,
 * copy_blocks_per_s <= 0, decode_tokens_per_s < 0, block_size <= 0, cap < 1.  Host arithmetic only. */
llx_status llx_predict_stage_sizes(int n0, double copy_blocks_per_s, double decode_tokens_per_s, int block_size,
                                   int32_t* sizes_out, int cap, int* n_stages);

/* ---- launch policy of ONE call -------------------------------------------------------------------------------
 *
 * The paper's own scenario needs two policies at once: non-final stages must not slow the co-running requests
 * (<= 1 %) while the final stage must be as short as possible because its duration IS the downtime
 * (PAPER.md:134), and a source migrates several requests continuously.  Policy is therefore an
 * argument of the call, not process state.  Every field: LLX_OPT_DEFAULT (-1) = inherit the process default
 * (llx_set_option; shipped defaults are "auto"), otherwise the meaning and range of the llx_option of the same name. */
#define LLX_OPT_DEFAULT (-1)
typedef enum {
    LLX_ROUTE_AUTO = 0, /* peer route exactly when the pools live on different GPUs */
    LLX_ROUTE_PEER = 1, /* take the cross-GPU route (kernel choice, launch shape, addressing of SURVEY NEXT-2) although both
                           pools are on one device: how a single-GPU box executes that branch.  Results are unchanged. */
    LLX_ROUTE_COPY_ENGINE = 2 /* llx_migrate_stage / _batch only: no kernel at all — one pitched copy-engine transfer per block
                           (2L tiles at the pools' slice strides), same or different GPUs.  No SM is used on either GPU, so
                           a migration to another GPU cannot slow a decode step's kernels except through HBM and the link;
                           on ONE GPU it is the slow way (measured there: 1.9 TB/s against the kernels' 6.6).  Unmeasured over NVLink.
                           llx_migrate_stage_wait falls back to the stream synchronize.  The copy engines cannot be paced or
                           capped: with a non-zero bandwidth_gbps or max_ctas (from the call or the process defaults) the
                           call returns LLX_ERR_INVALID_ARG instead of running unthrottled; every other launch-policy field
                           (copy_kernel, chunk_bytes, ring_stages, overlap_prev, ...) has no meaning here and is ignored.
                           Counters: bytes_moved grows, kernel_launches / copy_launches do not (no kernel ran).  The same
                           holds for the copy-engine host legs (LLX_OPT_VIA_HOST_MODE 2, and 0 for llx_migrate_via_host):
                           budget and CTA cap do not apply to them (the link, not HBM, is their bound; they are NOT refused),
                           an explicit copy_kernel selects the kernel + bounce route instead.  A pool whose slice stride
                           num_blocks*tile_bytes exceeds the pitch limit of a pitched transfer (2^31-1 bytes) is served
                           tile by tile (2L transfers per block); llx_migrate_via_host's AUTO then prefers the bounce route */
} llx_route;
typedef struct llx_launch_opts {
    uint32_t struct_size;      /* sizeof(llx_launch_opts) as the caller compiled it; set by llx_launch_opts_init */
    int32_t bandwidth_gbps;    /* LLX_OPT_BANDWIDTH_GBPS: budget of THIS call in GB/s read+written, 0 = unlimited */
    int32_t max_ctas;          /* LLX_OPT_MAX_CTAS */
    int32_t copy_kernel;       /* LLX_OPT_COPY_KERNEL */
    int32_t chunk_bytes;       /* LLX_OPT_CHUNK_BYTES */
    int32_t ring_stages;       /* LLX_OPT_RING_STAGES */
    int32_t rings_per_cta;     /* LLX_OPT_RINGS_PER_CTA */
    int32_t ids_by_value_max;  /* LLX_OPT_IDS_BY_VALUE_MAX */
    int32_t unit_order;        /* LLX_OPT_UNIT_ORDER */
    int32_t l2_hint;           /* LLX_OPT_L2_HINT */
    int32_t pdl;               /* LLX_OPT_PDL */
    int32_t dynamic_tail_pct;  /* LLX_OPT_DYNAMIC_TAIL_PCT */
    int32_t dynamic_tail_batch;/* LLX_OPT_DYNAMIC_TAIL_BATCH */
    int32_t exact_residency;   /* LLX_OPT_EXACT_RESIDENCY */
    int32_t via_host_mode;     /* LLX_OPT_VIA_HOST_MODE */
    int32_t route;             /* llx_route; LLX_OPT_DEFAULT = LLX_ROUTE_AUTO */
    int32_t overlap_prev;      /* LLX_OPT_OVERLAP_PREV: 1 = this copy is independent of every launch back to the last one without the flag */
} llx_launch_opts;
/* Sets struct_size and every field to LLX_OPT_DEFAULT. */
void llx_launch_opts_init(llx_launch_opts* opts);

/* ---- S3/S4: one migration stage (reserved dst blocks PAPER.md:142) -------- */

/* for i<n, l<layers, kv<2:  dst[l][kv][dst_block_ids[i]][:] = src[l][kv][src_block_ids[i]][:]
 * Whole tiles, including unused token slots of a partly filled last block.  One kernel
 * launch on `cuda_stream` (a stage under a bandwidth budget: a chain of launches, LLX_OPT_PACED_SLICE_US).  Checked: same geometry (num_blocks may differ), ids in range,
 * no duplicate destination id (duplicate source ids are legal: prefix-shared blocks),
 * src and dst distinct and non-overlapping.  src is never written.
 * The call runs on the SOURCE pool's device (which must be current; cuda_stream belongs to it).  dst may live on
 * another GPU with peer access: the kernel then stores straight into the peer-mapped pool (the two
 * instances are different machines); LLX_ERR_INVALID_ARG if the devices cannot access each other.
 * Long stages claim their last chunks from a small per-stream counter array the library allocates on first use
 * (that one call synchronises the device). */
llx_status llx_migrate_stage(const llx_pool* src, const int32_t* src_block_ids, llx_pool* dst,
                             const int32_t* dst_block_ids, int n, void* cuda_stream);
/* The same with this call's own launch policy (opts == NULL: process defaults, i.e. llx_migrate_stage).
 * LLX_ERR_INVALID_ARG for a field out of its option's range or a struct_size this library does not know. */
llx_status llx_migrate_stage_ex(const llx_pool* src, const int32_t* src_block_ids, llx_pool* dst,
                                const int32_t* dst_block_ids, int n, void* cuda_stream, const llx_launch_opts* opts);

/* The final stage as ONE blocking call (its duration is the request's downtime): llx_migrate_stage,
 * then the call returns only when the copy — and everything enqueued on cuda_stream before it — is complete.
 * The kernel's last CTA writes a word in pinned host memory that the calling thread spins on (measured on B200: no
 * shorter than a stream synchronize through the driver, 18.2 vs 17.4 us median — the driver's completion path is a spin
 * too; this is the convenient form, not an optimisation); if that is not possible (another copy kernel selected, all
 * flag slots in use) it falls back to the stream synchronize.  Always runs UNTHROTTLED: a bandwidth budget or CTA cap,
 * from the process defaults or from `opts`, is ignored — the downtime is not where bandwidth is saved.
 * Same checks and errors as llx_migrate_stage; LLX_ERR_CUDA also reports an asynchronous fault of the copy itself;
 * LLX_ERR_STATE while cuda_stream is being captured. */
llx_status llx_migrate_stage_wait(const llx_pool* src, const int32_t* src_block_ids, llx_pool* dst,
                                  const int32_t* dst_block_ids, int n, void* cuda_stream);
llx_status llx_migrate_stage_wait_ex(const llx_pool* src, const int32_t* src_block_ids, llx_pool* dst,
                                     const int32_t* dst_block_ids, int n, void* cuda_stream, const llx_launch_opts* opts);

/* ---- S5: many requests in ONE launch (the source migrates its chosen
 * requests one after another; batching them is this build's extension) -------------------- */

/* Request r owns pairs [req_offsets[r], req_offsets[r+1]) of the flat id lists;
 * req_offsets[0] == 0, non-decreasing, R+1 entries.  Result == R successive
 * llx_migrate_stage calls.  Destination ids must be distinct across the whole batch. */
llx_status llx_migrate_batch(const llx_pool* src, llx_pool* dst, const int32_t* req_offsets,
                             const int32_t* src_block_ids, const int32_t* dst_block_ids, int R, void* cuda_stream);
llx_status llx_migrate_batch_ex(const llx_pool* src, llx_pool* dst, const int32_t* req_offsets,
                                const int32_t* src_block_ids, const int32_t* dst_block_ids, int R, void* cuda_stream,
                                const llx_launch_opts* opts);

/* ---- S6: block fusion — gather into / scatter from ONE contiguous buffer -- */

/* Staging layout: staging[i][layer][kv][tile_bytes], i = position in the id list, so the
 * buffers of consecutive stages concatenate.  llx_staging_bytes = n*block_bytes. */
size_t     llx_staging_bytes(const llx_pool* pool, int n);
/* Pinned, mapped host memory for a staging buffer the kernels can address directly.
 * *host_ptr is the CPU address, *dev_alias the address to pass as `staging` (equal under UVA). */
llx_status llx_staging_alloc_pinned(size_t bytes, void** host_ptr, void** dev_alias);
llx_status llx_staging_free_pinned(void* host_ptr);
/* staging[i][l][kv][:] = src[l][kv][src_block_ids[i]][:]
 * With a pinned-host buffer the tiles are gathered into a library-owned device bounce buffer in ~64 MiB chunks and
 * each chunk crosses the host link on the copy engine (all on cuda_stream; first use allocates the bounce buffers and
 * synchronises the device).  LLX_OPT_VIA_HOST_MODE selects the other host legs: 1 (or an explicit LLX_OPT_COPY_KERNEL)
 * makes the kernel write the pinned buffer directly (zero-copy), 2 lets the copy engine gather by itself. */
llx_status llx_pack(const llx_pool* src, const int32_t* src_block_ids, int n, void* staging, size_t staging_bytes,
                    void* cuda_stream);
/* dst[l][kv][dst_block_ids[i]][:] = staging[i][l][kv][:]   (dst ids distinct) */
llx_status llx_unpack(const void* staging, size_t staging_bytes, llx_pool* dst, const int32_t* dst_block_ids, int n,
                      void* cuda_stream);
llx_status llx_pack_ex(const llx_pool* src, const int32_t* src_block_ids, int n, void* staging, size_t staging_bytes,
                       void* cuda_stream, const llx_launch_opts* opts);
llx_status llx_unpack_ex(const void* staging, size_t staging_bytes, llx_pool* dst, const int32_t* dst_block_ids, int n,
                         void* cuda_stream, const llx_launch_opts* opts);

/* The paper's whole transfer route in one call: gather into the contiguous buffer, then scatter
 * from it into the destination's reserved blocks.  Result: dst as after llx_migrate_stage, staging as after llx_pack.
 * The request is cut into chunks of `chunk_blocks` blocks (<= 0: auto, ~64 MiB); chunk k is scattered on an internal
 * stream while chunk k+1 is gathered on `cuda_stream`.  With a pinned-host buffer the chunks cross the host link on the
 * copy engines, device->host and host->device at the same time (the source and destination machines of the paper work
 * concurrently in the same way): by default as one pitched copy per block in groups of ~16 MiB (no kernel at all), with
 * LLX_OPT_VIA_HOST_MODE = 3 or a destination on another GPU through library-owned device bounce buffers (4 x chunk
 * bytes, allocated on first use: that call synchronises the device).  `cuda_stream` is joined with the internal streams before the call returns: work
 * enqueued on it afterwards sees the complete migration.  Checks as llx_migrate_stage + llx_pack; nothing is launched
 * when a check fails.  Calls are serialised per process (they share the internal streams). */
llx_status llx_migrate_via_host(const llx_pool* src, const int32_t* src_block_ids, llx_pool* dst,
                                const int32_t* dst_block_ids, int n, void* staging, size_t staging_bytes,
                                int chunk_blocks, void* cuda_stream);
llx_status llx_migrate_via_host_ex(const llx_pool* src, const int32_t* src_block_ids, llx_pool* dst,
                                   const int32_t* dst_block_ids, int n, void* staging, size_t staging_bytes,
                                   int chunk_blocks, void* cuda_stream, const llx_launch_opts* opts);

/* ---- NEXT-3: block manager + migration handshake (Fig. 7) -- host logic only ------------------
 *
 * llx_blockmgr is one instance's free list of block ids.  Policy (A23): a stack; a fresh manager hands
 * out 0,1,2,...; released ids are pushed in the order given and handed out again last-in-first-out.
 * llx_migration drives ONE request's migration through the handshake of PAPER.md:142:
 *   before each stage  PRE-ALLOC n blocks on the destination (all or nothing, A24) -> proceed | abort
 *   after each stage   the source checks the request: finished / preempted / peer failed -> abort, the destination
 *                      releases everything reserved for this migration (A25); no byte is rolled back
 *   after the final stage  the source releases its blocks, the destination commits: the request resumes there.
 * Not thread-safe per object; distinct objects are independent. */
typedef struct llx_blockmgr llx_blockmgr;
typedef struct llx_migration llx_migration;
typedef enum { LLX_REQ_RUNNING = 0, LLX_REQ_FINISHED = 1, LLX_REQ_PREEMPTED = 2, LLX_REQ_PEER_FAILED = 3 } llx_req_status;
typedef enum {
    LLX_MIG_READY = 0,         /* no stage issued yet */
    LLX_MIG_COPYING = 1,       /* a non-final stage was issued; the request keeps decoding on the source */
    LLX_MIG_FINAL_COPYING = 2, /* the final stage was issued; the request is stopped (downtime) */
    LLX_MIG_COMMITTED = 3,
    LLX_MIG_ABORTED = 4
} llx_mig_state;
typedef enum { LLX_ABORT_NONE = 0, LLX_ABORT_FINISHED = 1, LLX_ABORT_PREEMPTED = 2, LLX_ABORT_PEER_FAILED = 3,
               LLX_ABORT_NO_SPACE = 4 } llx_abort_reason;

llx_status llx_blockmgr_create(int num_blocks, llx_blockmgr** out);
llx_status llx_blockmgr_destroy(llx_blockmgr* mgr);
int        llx_blockmgr_num_free(const llx_blockmgr* mgr);   /* -1 on NULL */
int        llx_blockmgr_num_blocks(const llx_blockmgr* mgr); /* -1 on NULL */
/* n ids into ids_out (HOST int32[n]); LLX_ERR_NO_SPACE when fewer than n are free: nothing is allocated. */
llx_status llx_blockmgr_alloc(llx_blockmgr* mgr, int n, int32_t* ids_out);
/* Returns ids to the free list; LLX_ERR_BLOCK_OUT_OF_RANGE / LLX_ERR_INVALID_ARG (already free, or twice in the
 * list): nothing is released. */
llx_status llx_blockmgr_release(llx_blockmgr* mgr, const int32_t* ids, int n);

/* src / dst may both be NULL: the session then only coordinates (no copy is enqueued) — how the handshake is
 * tested without a device.  The managers are borrowed, not owned. */
llx_status llx_migration_begin(const llx_pool* src, llx_blockmgr* src_mgr, llx_pool* dst, llx_blockmgr* dst_mgr,
                               int block_size, int last_stage_max_blocks, llx_migration** out);
/* One round.  (1) the source's check: status != RUNNING aborts (reserved destination blocks are released).
 * (2) llx_plan_stage(num_tokens, blocks migrated so far).  (3) PRE-ALLOC of *n blocks on the destination manager;
 * LLX_ERR_NO_SPACE aborts likewise.  (4) with pools: llx_migrate_stage of src_block_table[m .. m+*n) into the
 * reserved ids is enqueued on cuda_stream.  src_block_table: HOST int32[table_len], the request's logical->physical
 * table on the source, table_len >= ceil(num_tokens/block_size).  dst_ids_out (may be NULL): the *n reserved ids.
 * Returns LLX_OK also when the round ended in an abort: read llx_migration_state(). */
llx_status llx_migration_stage(llx_migration* mig, const int32_t* src_block_table, int table_len, int num_tokens,
                               llx_req_status status, void* cuda_stream, int* n, int* is_final, int32_t* dst_ids_out);
/* After the final stage's copy has completed (the caller synchronised its stream).  status != RUNNING aborts (A26).
 * Otherwise the source's blocks src_block_table[0 .. blocks migrated) go back to src_mgr and the request's
 * destination table is written to dst_table_out (HOST int32[cap], cap >= blocks migrated); state COMMITTED. */
llx_status llx_migration_commit(llx_migration* mig, const int32_t* src_block_table, int table_len, llx_req_status status,
                                int32_t* dst_table_out, int cap, int* n_out);
/* Either side may abort before the commit ("if the other side fails"). */
llx_status llx_migration_abort(llx_migration* mig, llx_abort_reason reason);
/* Launch policy of the session's NON-FINAL stages (the struct is copied; NULL = back to the process defaults), e.g. a
 * bandwidth budget that keeps the co-running decode steps within 1 %.  The FINAL stage ignores
 * bandwidth_gbps and max_ctas and always runs at full speed: its duration is the request's downtime. */
llx_status llx_migration_set_stage_opts(llx_migration* mig, const llx_launch_opts* opts);
llx_mig_state    llx_migration_state(const llx_migration* mig);
llx_abort_reason llx_migration_abort_reason(const llx_migration* mig);
int              llx_migration_blocks_migrated(const llx_migration* mig);
int              llx_migration_stages(const llx_migration* mig); /* stages issued so far */
llx_status       llx_migration_destroy(llx_migration* mig);     /* an uncommitted session is aborted first */

/* ---- NEXT-4: virtual usage, freeness, pairing (Algorithm 1; §4.4.3) -- host arithmetic
 *
 * The step before the hot path: which instances migrate to which, and which requests go first.  Usages, demands,
 * headrooms and M share one unit (tokens or blocks).  Readings A27-A30 in DESIGN.md. */
typedef struct {
    int32_t is_queuing;      /* not yet running on the instance */
    int32_t is_head_of_line; /* first in the instance's queue (only read when is_queuing) */
    int32_t is_fake;         /* the infinite-usage request of a terminating instance */
    int32_t priority;        /* 0 = normal ... num_priorities-1 = highest */
    double demand;           /* memory the queuing request needs to start */
    double physical_usage;   /* memory the running request occupies */
} llx_req_info;
/* CalcFreeness: *freeness = (M - sum of CalcVirtualUsage) / B, B = running requests (1 if none).  A terminating
 * instance gets the fake request: -inf.  *total_virtual_usage may be NULL. */
llx_status llx_calc_freeness(const llx_req_info* reqs, int n, double M, const double* headroom_for_priority,
                             int num_priorities, int is_terminating, double* freeness, double* total_virtual_usage);
/* Sources: freeness < src_below; destinations: freeness > dst_above (src_below <= dst_above).  Pairs the lowest
 * source with the highest destination repeatedly (ties: lower index first).  *n_pairs = min(#src, #dst); the pairs
 * are written to src_out / dst_out (HOST int32[cap]); LLX_ERR_INVALID_ARG if cap is too small (*n_pairs still set). */
llx_status llx_pair_instances(const double* freeness, int n, double src_below, double dst_above, int32_t* src_out,
                              int32_t* dst_out, int cap, int* n_pairs);
/* The order in which a source offers its requests: lower priority first, then shorter sequence, then lower index. */
llx_status llx_migration_order(const int32_t* priority, const int32_t* seq_len, int n, int32_t* order_out);

/* One migration round of ONE (source, destination) pair as ONE batch: the step between the policy and the hot path
 * ("The llumlet of each source instance then starts to migrate requests to the destination continuously,
 * until it is no longer set in the source state.  The llumlet prefers the requests with lower priorities and shorter
 * sequence lengths").  Reading A31:
 *   1. candidates = the source's RUNNING requests (not queuing, not fake) in llx_migration_order(priority, seq_len);
 *   2. while the source's freeness — llx_calc_freeness over the requests it still has — is below src_below (it is still
 *      "in the source state") and a candidate is left: PRE-ALLOC all blocks of the next candidate on dst_mgr, all or
 *      nothing; the first request the destination cannot hold while keeping dst_reserve_blocks free
 *      ends the round; otherwise the request joins the batch and leaves the source's request set.
 * reqs / seq_len: HOST arrays of n entries.  Request r's block table on the source is
 * src_block_tables[table_offsets[r] .. table_offsets[r+1]) (HOST int32; n+1 offsets; empty for queuing requests).
 * Outputs (HOST): chosen_out int32[n] = the requests taken, in the order taken; *n_chosen; and exactly the arguments of
 * llx_migrate_batch: req_offsets_out int32[n+1] (the first *n_chosen+1 entries are written), src_ids_out / dst_ids_out
 * int32[cap_pairs], *n_pairs.  The destination ids are RESERVED in dst_mgr when the call returns LLX_OK; after the batch
 * has completed the caller releases src_ids_out on the source's manager (the commit of PAPER.md:142) — or releases
 * dst_ids_out on dst_mgr to abort.  LLX_ERR_INVALID_ARG (cap_pairs too small, bad offsets, ...) reserves nothing.
 * Host arithmetic only; nothing is launched. */
llx_status llx_plan_migration_batch(const llx_req_info* reqs, const int32_t* seq_len, int n, double M,
                                    const double* headroom_for_priority, int num_priorities, int is_terminating,
                                    double src_below, const int32_t* table_offsets, const int32_t* src_block_tables,
                                    llx_blockmgr* dst_mgr, int dst_reserve_blocks, int32_t* chosen_out, int* n_chosen,
                                    int32_t* req_offsets_out, int32_t* src_ids_out, int32_t* dst_ids_out, int cap_pairs,
                                    int* n_pairs);

/* ---- NEXT-1: the bandwidth budget of the non-final stages, chosen from what the engine observes ------------------
 *
 * live migration costs the co-running requests "nearly zero (up to 1%)".  On the paper's hardware that
 * holds because the copy is slow; on a B200 the copy can take the whole HBM, so the share has to be CHOSEN
 * (llx_launch_opts.bandwidth_gbps), and the budget that holds a given slowdown depends on the co-running batch, the
 * GPU's power state and what else runs — only the engine sees that.  The engine therefore reports every decode step's
 * duration, saying whether a budgeted stage was in flight, and asks the controller for the budget of the next stage.
 * Rule (A34): every `window` steps observed WITH a migration,
 *     s = median(those steps) / median(the last 2*window steps observed WITHOUT one) - 1
 *     budget <- clamp(budget * f, min_gbps, max_gbps),   f = 2 if s <= target/4, else clamp(target / s, 1/2, 2).
 * Steps with a migration are ignored until a step without one has been reported.  Host arithmetic only; one controller
 * per decode loop; not thread-safe per object.  The final stage is never budgeted. */
typedef struct llx_budget_ctl llx_budget_ctl;
/* target_slowdown_pct > 0; 1 <= min_gbps <= start_gbps <= max_gbps <= 100000; 2 <= window <= 256. */
llx_status llx_budget_ctl_create(double target_slowdown_pct, int min_gbps, int max_gbps, int start_gbps, int window,
                                 llx_budget_ctl** out);
llx_status llx_budget_ctl_destroy(llx_budget_ctl* ctl);
/* One decode step took step_ms (> 0, finite); migrating != 0: a budgeted stage was in flight during it.
 * *budget_gbps (may be NULL) = the budget to give the next non-final stage. */
llx_status llx_budget_ctl_observe(llx_budget_ctl* ctl, double step_ms, int migrating, int* budget_gbps);
int    llx_budget_ctl_gbps(const llx_budget_ctl* ctl);              /* current budget, GB/s read + written; -1 on NULL */
double llx_budget_ctl_last_slowdown_pct(const llx_budget_ctl* ctl); /* s of the last adjustment in %, NaN before the first */
int    llx_budget_ctl_adjustments(const llx_budget_ctl* ctl);       /* adjustments made so far; -1 on NULL */

/* ---- S8: append-only growth while decoding continues --------------- */

/* Writes the K and V vectors of tokens t0..t1-1 of one request into their slots: token t
 * lives in block block_table[t / block_size], slot t % block_size.
 * dev_values: DEVICE buffer [t1-t0][layers][2][kv_heads*head_dim] elements (token-major).
 * block_table: HOST int32[table_len] with table_len > (t1-1)/block_size.  Nothing else is written. */
llx_status llx_append_tokens(llx_pool* pool, const int32_t* block_table, int table_len, int t0, int t1,
                             const void* dev_values, void* cuda_stream);

/* ---- S7: stand-in paged decode attention (measurement only) ------------- */

/* One query token per sequence, MHA (q heads = kv heads), fp16 in, fp32 accumulate, fp16 out:
 *   o[b][h] = sum_t softmax_t(scale * q[b][h].k_t[h]) v_t[h],  t < dev_ctx_lens[b],
 * K/V of token t read from block dev_block_tables[b*max_blocks + t/block_size], slot t%block_size.
 * dev_q, dev_out: DEVICE fp16 [B, kv_heads, head_dim].  Requires LLX_F16, head_dim 64 or 128.
 * ctx_len 0 gives zeros.  Precondition: dev_ctx_lens[b] <= max_blocks*block_size and every table entry a sequence
 * uses is a valid block id; the lengths live on the device, so they are not checked on the host — a longer ctx_len is
 * CLAMPED to max_blocks*block_size in the kernels (never an out-of-row table read).  Uses a per-pool workspace that grows
 * on demand (first call and growth synchronise the device); calls on one pool must be ordered on one stream. */
llx_status llx_decode_attention(const llx_pool* pool, int layer, const void* dev_q, void* dev_out,
                                const int32_t* dev_block_tables, const int32_t* dev_ctx_lens, int B, int max_blocks,
                                float scale, void* cuda_stream);

/* The same attention for callers that are not allowed to allocate device memory.
 *
 * Who that is: a serving engine that has handed all of the GPU's free memory to its KV-cache pool at start-up (so a
 * later cudaMalloc fails or trips its out-of-memory accounting), a decode loop on a latency budget (cudaMalloc and
 * cudaFree may synchronise the whole device and stall every stream, the migration's included), and code that runs
 * where the CUDA allocator must not be entered at all (inside a host callback of a stream, or under a memory-pool
 * policy that forbids growth after initialisation).  llx_decode_attention grows a per-pool workspace with
 * cudaMalloc/cudaFree whenever a larger shape arrives; this entry point never does.
 *
 * Arguments, result and preconditions are exactly those of llx_decode_attention.  The split-KV partials
 * (B * kv_heads * ceil(max_blocks*block_size / split) rows of (head_dim + 4) floats, split = LLX_OPT_ATTN_SPLIT_TOKENS,
 * 256 by default) go into ONE fixed array of LLX_ATTN_STATIC_WS_BYTES that is part of the library image: every GPU
 * that loads libllx.so holds those bytes from the moment the library's code is loaded on it until the process exits,
 * whether or not this function is ever called.  16 MiB covers BASELINE.json configs[4]'s decode batch (32 sequences x
 * 32 heads x up to 4096 tokens of context, head_dim 128: 8.25 MiB) with room for a batch of 62 at that length.
 *
 *   - A shape whose partials need more than LLX_ATTN_STATIC_WS_BYTES is refused with LLX_ERR_INVALID_ARG before anything
 *     is launched (llx_last_error gives the bytes needed and the limit); nothing is allocated instead.  A larger
 *     LLX_OPT_ATTN_SPLIT_TOKENS shrinks the need.
 *   - No cudaMalloc, cudaFree, cudaHostAlloc or other allocating routine is called, on the first call or any later one.
 *   - First call on each device: with that device current (the pool's device — the call checks it) the library looks up
 *     the array's device address once and keeps it.  Make that first call during start-up, before any stream capture.
 *   - The array is shared by every pool, stream and thread of the process on that device and keeps what the last call
 *     left in it.  Nothing in it has to start at zero: a call writes every partial it later reads.  Two calls that are
 *     in flight on the GPU at the same time (different streams, or different threads) race on it and both may return
 *     wrong outputs silently: order all calls of one device on one stream, or with events.  It does not touch the
 *     per-pool workspace, so it may overlap llx_decode_attention calls freely. */
#define LLX_ATTN_STATIC_WS_BYTES (16u << 20)
llx_status llx_decode_attention_static_ws(const llx_pool* pool, int layer, const void* dev_q, void* dev_out,
                                          const int32_t* dev_block_tables, const int32_t* dev_ctx_lens, int B,
                                          int max_blocks, float scale, void* cuda_stream);

/* ---- tuning, counters, errors ----------------------------------------------------------- */

typedef enum {
    LLX_OPT_COPY_KERNEL = 0,    /* 0 auto, 1 = 16-byte LDG/STG kernel, 2 = bulk-async (1-D TMA) smem ring, 3 = the same ring fed by 4-D
                                   tensor-map boxes (cp.async.bulk.tensor: one instruction moves the tiles of one block in several
                                   (layer, K|V) slices) — pool-to-pool copies on one device with tiles of at most 16 KiB only,
                                   LLX_ERR_INVALID_ARG elsewhere; never taken by auto (it ties the 1-D ring, measured) */
    LLX_OPT_MAX_CTAS = 1,       /* cap on the copy grid (0 = auto: fill the GPU); the throttle of SURVEY NEXT-1 */
    LLX_OPT_CHUNK_BYTES = 2,    /* bytes of one tile one CTA moves per step (multiple of 16; 0 = auto) */
    LLX_OPT_RING_STAGES = 3,    /* smem stages per ring of the bulk-async kernel (0 = auto) */
    LLX_OPT_IDS_BY_VALUE_MAX = 4, /* pairs up to which ids travel in the kernel parameters (<= 256) */
    LLX_OPT_ATTN_SPLIT_TOKENS = 5, /* tokens per KV split of decode attention (multiple of 8; 0 = auto) */
    LLX_OPT_UNIT_ORDER = 6,     /* 0: worker w copies chunks w, w+W, w+2W, ... (striped); 1: a contiguous range each */
    LLX_OPT_L2_HINT = 7,        /* bulk kernel: bit0 loads, bit1 stores carry an L2::evict_first policy */
    LLX_OPT_RINGS_PER_CTA = 8,  /* bulk kernel: independent smem rings (warps) per CTA (0 = auto) */
    LLX_OPT_PDL = 9,            /* 1 (default): launch copy/append kernels with programmatic stream serialization so that
                                   a kernel's prologue overlaps the previous kernel's tail; results are unchanged */
    LLX_OPT_BANDWIDTH_GBPS = 10,/* bandwidth budget of device<->device copies in GB/s, read + written (0 = unlimited), so that a
                                   co-running decode step keeps its speed (<= 1 %).  Below 500 GB/s: a paced
                                   register-staged copy, one small CTA per SM, every SM loses the same small share.  From
                                   500 GB/s: budget/60 full-speed bulk CTAs (about 60 GB/s each), which costs the decode
                                   step less per byte than pacing at those rates */
    LLX_OPT_DYNAMIC_TAIL_PCT = 12, /* bulk kernel: share (%) of a long stage's chunks that is not pre-assigned to a ring but
                                   claimed in small batches by whichever ring finishes its range first (default 6; 0 = off) */
    LLX_OPT_DYNAMIC_TAIL_BATCH = 13, /* chunks per claim of the dynamic tail (0 = auto: 4) */
    LLX_OPT_EXACT_RESIDENCY = 14, /* 1 (default): the bulk kernel asks for enough shared memory that no SM can hold more of its
                                   CTAs than intended, early-launched CTAs of the next kernel included */
    LLX_OPT_COPY_SMEM_CARVEOUT_PCT = 15, /* PROCESS-WIDE ONLY (a property of the kernel function, not of a launch): preferred
                                   shared-memory carve-out, in % of the SM's maximum, of the register-staged copy kernel that
                                   serves bandwidth budgets below 500 GB/s and the host zero-copy / peer routes.  That kernel
                                   keeps a small CTA resident on every SM for the whole stage, and an SM cannot change its
                                   L1/shared split while a CTA is resident: a co-running kernel that needs more shared memory
                                   than the split offers waits for the end of the launch (a slice of the stage, see
                                   LLX_OPT_PACED_SLICE_US).  Default 50 (132 KB shared / 124 KB L1): the stand-in decode step
                                   loses nothing (measured; 75 costs it +2..5 %, 100 +11..30 %).  0 = the driver's choice ("all
                                   L1").  100: not even a kernel that needs the whole 227 KB ever waits.  llx's own bulk ring
                                   (164 KB split) does not rely on this: while a register-staged stage is in flight the library
                                   routes its auto-selected copies through the register-staged kernel */
    LLX_OPT_PACED_SLICE_US = 16, /* PROCESS-WIDE ONLY.  A paced stage (bandwidth budget below 500 GB/s) is issued as a chain of launches
                                   of about this many microseconds each (at most 256 per call) instead of ONE kernel resident
                                   for the whole stage, so that a co-running kernel waiting for an SM to change its L1/shared
                                   split waits for the end of a slice, not of the stage (75 ms for 112 blocks at 25 GB/s).
                                   Default 1000; 0 = one launch.  Costs ~3 us of host time per slice inside the call; the rate
                                   and the decode step's slowdown are unchanged (measured).  Counters count every launch */
    LLX_OPT_OVERLAP_PREV = 17,  /* 1: the caller states that this copy is INDEPENDENT of every launch on cuda_stream from the most
                                   recent one made WITHOUT overlap_prev (an llx call that left the flag at 0, or any work that
                                   is not an llx kernel) up to the one enqueued just before it — it reads no byte they write and
                                   writes no byte they read or write.  So in a chain  F, O1, O2  (F plain; O1, O2 with the flag)
                                   O2 must be independent of O1 AND of F: an overlapped kernel lets its successor launch before
                                   it has waited itself, so O2 may run next to F.  Everything enqueued BEFORE F has completed
                                   when O1 or O2 starts: every llx kernel that does not defer its wait lets dependents launch
                                   only after that wait has returned, so a plain launch fences the start of what follows it
                                   (a small or CTA-capped plain launch included).
                                   True for consecutive non-final stages of one request (disjoint blocks on both sides; full
                                   blocks are never written again) and for stages of different requests
                                   (PAPER.md:225).  The copy may then START while those kernels' slowest CTAs are still running
                                   (the wait of the programmatic dependent launch moves from the kernel's prologue to its end),
                                   which hides the ~3 us an SM otherwise idles between two stages.  COMPLETION order is kept:
                                   when this copy has completed, everything enqueued before it on the stream has completed, so
                                   events, synchronises and later kernels see both.  Dependencies that cross streams (an event
                                   wait before the call) are honoured as always.  Only the unthrottled bulk ring with
                                   LLX_OPT_PDL uses it; every other kernel / route ignores it, and so do llx_migrate_stage_wait
                                   and a session's final stage (they read the block the source appended to last) and the routes
                                   whose own kernels depend on one another (llx_migrate_via_host, pinned-host llx_pack /
                                   llx_unpack).  Default 0: plain stream order */
    LLX_OPT_VIA_HOST_MODE = 11  /* the host leg of llx_pack / llx_unpack / llx_migrate_via_host with a pinned-host buffer.
                                   0 (default) auto: llx_migrate_via_host lets the copy engines gather and scatter by themselves
                                   (mode 2; measured 93.8 vs 84.9 GB/s), llx_pack / llx_unpack go through the bounce buffers
                                   (mode 3; equal speed, measured).  1: the kernels address the host buffer directly (zero-copy).
                                   2: one pitched copy-engine transfer per block (2L tiles at a constant stride): no kernel, no
                                   bounce buffer, no SM.  3: a gather / scatter kernel per 64 MiB chunk into / out of device bounce
                                   buffers, the copy engine crosses the link */
} llx_option;
/* Process-wide DEFAULTS: what a later call uses for every policy field it does not set itself (llx_launch_opts).
 * For experiments and process-wide tuning; per-request policy belongs in the call.  LLX_ERR_INVALID_ARG for a bad value. */
llx_status llx_set_option(llx_option opt, long long value);
long long  llx_get_option(llx_option opt);

typedef struct {
    unsigned long long kernel_launches; /* kernels this library launched */
    unsigned long long copy_launches;   /* of which gather/scatter copy kernels */
    unsigned long long bytes_moved;     /* payload bytes those copies wrote */
    unsigned long long id_uploads;      /* stages whose ids went through the pinned ring (not by value) */
} llx_counters;
void llx_get_counters(llx_counters* out);
void llx_reset_counters(void);

/* Waits until everything enqueued on cuda_stream (NULL: the legacy default stream) has completed; LLX_ERR_CUDA reports an
 * asynchronous fault of that work.  For clients that do not link the CUDA runtime themselves. */
llx_status llx_synchronize(void* cuda_stream);

const char* llx_status_str(llx_status s);
const char* llx_last_error(void); /* thread-local detail of this thread's last failed call */
const char* llx_version(void);

#ifdef __cplusplus
}
#endif
#endif /* LLX_H_ */
