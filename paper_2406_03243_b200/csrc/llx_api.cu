// C-ABI of the llx library (include/llx.h): pools, host-side validation, id hand-off and the
// kernel launches.  Every data step runs in the kernels of llx_copy.cuh / llx_attention.cuh;
// this file only checks arguments, stages the block ids and enqueues.  There is no CPU path.
#include "../../include/llx.h"

#include <cuda.h>  // CUtensorMap types only: cuTensorMapEncodeTiled is fetched through cudaGetDriverEntryPoint, libcuda is not linked

#include <atomic>
#include <cmath>
#include <cstdarg>
#include <cstddef>
#include <new>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <unordered_map>
#include <vector>

#include "llx_attention.cuh"
#include "llx_copy.cuh"
#include "llx_internal.h"

using namespace llx;

struct llx_pool {
    unsigned char* data = nullptr;
    int layers = 0, kv_heads = 0, head_dim = 0, block_size = 0, num_blocks = 0;
    llx_dtype dtype = LLX_F16;
    int elem_bytes = 2;
    long long tile_bytes = 0;
    int device = 0;
    bool owned = false;
    bool ipc_mapped = false;  // data comes from cudaIpcOpenMemHandle: destroy unmaps it
    // decode-attention workspace (grows on demand)
    float* attn_ws = nullptr;
    size_t attn_ws_bytes = 0;
    // small tiles (<= 16 KiB): a 4-D tensor map over the pool, dims (row, rows of a tile, block, slice), whose box is the
    // tiles of ONE block in tma_k consecutive (layer, K|V) slices; 0 = no map (large tiles, no driver entry point)
    int tma_k = 0;
    llx::TensorMap tmap;
};

namespace llx {
thread_local char g_err[512] = "";

llx_status fail(llx_status s, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
    return s;
}
}  // namespace llx

namespace {

llx_status cuda_fail(cudaError_t e, const char* what) {
    return fail(LLX_ERR_CUDA, "%s: %s", what, cudaGetErrorString(e));
}
#define LLX_CUDA(call)                                   \
    do {                                                 \
        cudaError_t e_ = (call);                         \
        if (e_ != cudaSuccess) return cuda_fail(e_, #call); \
    } while (0)

int elem_bytes_of(llx_dtype d) {
    switch (d) {
        case LLX_F16:
        case LLX_BF16: return 2;
        case LLX_U8: return 1;
    }
    return 0;
}

// ---- options / counters -------------------------------------------------------------------
std::atomic<long long> g_opt_kernel{0}, g_opt_max_ctas{0}, g_opt_chunk{0}, g_opt_stages{0}, g_opt_byval{kIdsByValueCap},
    g_opt_attn_split{0}, g_opt_order{1}, g_opt_l2hint{0}, g_opt_rings{0}, g_opt_pdl{1}, g_opt_budget{0}, g_opt_via_host{0}, g_opt_dyn_pct{6}, g_opt_dyn_batch{0}, g_opt_smem_pad{1}, g_opt_carveout{50}, g_opt_slice_us{1000}, g_opt_overlap{0};
std::atomic<unsigned long long> g_launches{0}, g_copy_launches{0}, g_bytes{0}, g_id_uploads{0};

// Range of every option: shared by llx_set_option (process defaults) and by the per-call llx_launch_opts.
bool opt_valid(int opt, long long v) {
    switch (opt) {
        case LLX_OPT_COPY_KERNEL: return v >= 0 && v <= 3;
        case LLX_OPT_MAX_CTAS: return v >= 0 && v <= (1 << 20);
        case LLX_OPT_CHUNK_BYTES: return v >= 0 && (v % 16) == 0 && v <= (200 << 10);
        case LLX_OPT_RING_STAGES: return v >= 0 && v != 1 && v <= 14;
        case LLX_OPT_IDS_BY_VALUE_MAX: return v >= 0 && v <= kIdsByValueCap;
        case LLX_OPT_ATTN_SPLIT_TOKENS: return v >= 0 && (v % 8) == 0;
        case LLX_OPT_UNIT_ORDER: return v >= 0 && v <= 1;
        case LLX_OPT_L2_HINT: return v >= 0 && v <= 3;
        case LLX_OPT_RINGS_PER_CTA: return v >= 0 && v <= 8;
        case LLX_OPT_PDL: return v >= 0 && v <= 1;
        case LLX_OPT_BANDWIDTH_GBPS: return v >= 0 && v <= 100000;
        case LLX_OPT_VIA_HOST_MODE: return v >= 0 && v <= 3;
        case LLX_OPT_DYNAMIC_TAIL_PCT: return v >= 0 && v <= 100;
        case LLX_OPT_DYNAMIC_TAIL_BATCH: return v >= 0 && v <= 4096;
        case LLX_OPT_EXACT_RESIDENCY: return v >= 0 && v <= 1;
        case LLX_OPT_COPY_SMEM_CARVEOUT_PCT: return v >= 0 && v <= 100;
        case LLX_OPT_PACED_SLICE_US: return v >= 0 && v <= 1000000;
        case LLX_OPT_OVERLAP_PREV: return v >= 0 && v <= 1;
    }
    return false;
}

// The launch policy of ONE call: the process defaults overridden by whatever the call's llx_launch_opts sets.
// Resolved once at the entry point and passed down by value, so concurrent callers never see each other's policy.
struct Policy {
    long long kernel, max_ctas, chunk, stages, byval, order, l2hint, rings, pdl, budget, via_host, dyn_pct, dyn_batch, smem_pad, overlap;
    int route;
};

llx_status resolve_policy(const llx_launch_opts* o, Policy* p) {
    p->kernel = g_opt_kernel.load();
    p->max_ctas = g_opt_max_ctas.load();
    p->chunk = g_opt_chunk.load();
    p->stages = g_opt_stages.load();
    p->byval = g_opt_byval.load();
    p->order = g_opt_order.load();
    p->l2hint = g_opt_l2hint.load();
    p->rings = g_opt_rings.load();
    p->pdl = g_opt_pdl.load();
    p->budget = g_opt_budget.load();
    p->via_host = g_opt_via_host.load();
    p->dyn_pct = g_opt_dyn_pct.load();
    p->dyn_batch = g_opt_dyn_batch.load();
    p->smem_pad = g_opt_smem_pad.load();
    p->overlap = g_opt_overlap.load();
    p->route = LLX_ROUTE_AUTO;
    if (o) {
        // a caller compiled against an older, shorter struct is served: fields beyond its struct_size keep the defaults
        if (o->struct_size < 2 * sizeof(int32_t) || o->struct_size > sizeof(llx_launch_opts) || (o->struct_size % sizeof(int32_t)) != 0)
            return fail(LLX_ERR_INVALID_ARG, "llx_launch_opts.struct_size = %u (this library: %zu); use llx_launch_opts_init", o->struct_size, sizeof(llx_launch_opts));
#define LLX_FIELD(field, opt, dst)                                                                            \
    if (offsetof(llx_launch_opts, field) + sizeof(int32_t) <= o->struct_size && o->field != LLX_OPT_DEFAULT) { \
        if (!opt_valid(opt, o->field)) return fail(LLX_ERR_INVALID_ARG, "llx_launch_opts." #field " = %d: bad value", (int)o->field); \
        p->dst = o->field;                                                                                    \
    }
        LLX_FIELD(bandwidth_gbps, LLX_OPT_BANDWIDTH_GBPS, budget)
        LLX_FIELD(max_ctas, LLX_OPT_MAX_CTAS, max_ctas)
        LLX_FIELD(copy_kernel, LLX_OPT_COPY_KERNEL, kernel)
        LLX_FIELD(chunk_bytes, LLX_OPT_CHUNK_BYTES, chunk)
        LLX_FIELD(ring_stages, LLX_OPT_RING_STAGES, stages)
        LLX_FIELD(rings_per_cta, LLX_OPT_RINGS_PER_CTA, rings)
        LLX_FIELD(ids_by_value_max, LLX_OPT_IDS_BY_VALUE_MAX, byval)
        LLX_FIELD(unit_order, LLX_OPT_UNIT_ORDER, order)
        LLX_FIELD(l2_hint, LLX_OPT_L2_HINT, l2hint)
        LLX_FIELD(pdl, LLX_OPT_PDL, pdl)
        LLX_FIELD(dynamic_tail_pct, LLX_OPT_DYNAMIC_TAIL_PCT, dyn_pct)
        LLX_FIELD(dynamic_tail_batch, LLX_OPT_DYNAMIC_TAIL_BATCH, dyn_batch)
        LLX_FIELD(exact_residency, LLX_OPT_EXACT_RESIDENCY, smem_pad)
        LLX_FIELD(via_host_mode, LLX_OPT_VIA_HOST_MODE, via_host)
        LLX_FIELD(overlap_prev, LLX_OPT_OVERLAP_PREV, overlap)
#undef LLX_FIELD
        if (offsetof(llx_launch_opts, route) + sizeof(int32_t) <= o->struct_size && o->route != LLX_OPT_DEFAULT) {
            if (o->route != LLX_ROUTE_AUTO && o->route != LLX_ROUTE_PEER && o->route != LLX_ROUTE_COPY_ENGINE)
                return fail(LLX_ERR_INVALID_ARG, "llx_launch_opts.route = %d", (int)o->route);
            p->route = o->route;
        }
    }
    return LLX_OK;
}

// Is work enqueued on `st` being captured into a CUDA graph?  Calls that must allocate, synchronise or stage ids through
// pinned memory refuse (LLX_ERR_STATE) instead of invalidating the capture.
llx_status stream_capturing(cudaStream_t st, bool* capturing) {
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    cudaError_t e = cudaStreamIsCapturing(st, &cs);
    if (e != cudaSuccess) return fail(LLX_ERR_CUDA, "cudaStreamIsCapturing: %s", cudaGetErrorString(e));
    *capturing = cs != cudaStreamCaptureStatusNone;
    return LLX_OK;
}
llx_status refuse_if_capturing(cudaStream_t st, const char* what) {
    bool cap = false;
    llx_status rc = stream_capturing(st, &cap);
    if (rc != LLX_OK) return rc;
    if (cap) return fail(LLX_ERR_STATE, "%s cannot be captured into a CUDA graph (it allocates, synchronises or stages through pinned memory)", what);
    return LLX_OK;
}

// ---- device properties (cached per device) ------------------------------------------------
struct DevInfo {
    int sm_count = 0;
    int max_smem_optin = 0;
    int smem_per_sm = 0;
    int carveout_applied = -1;  // LLX_OPT_COPY_SMEM_CARVEOUT_PCT as last set on the register-staged copy kernel
    bool ready = false;
};
std::mutex g_dev_mu;
DevInfo g_dev[64];

// `dev` must be the CURRENT device (cudaFuncSetAttribute acts on it): every caller passes the device its kernel runs on.
llx_status dev_info(int dev, DevInfo** out, bool capturing = false) {
    if (dev < 0 || dev >= 64) return fail(LLX_ERR_INVALID_ARG, "device %d unsupported", dev);
    std::lock_guard<std::mutex> lk(g_dev_mu);
    DevInfo& d = g_dev[dev];
    if (!d.ready) {
        if (capturing) return fail(LLX_ERR_STATE, "first llx call on device %d inside a stream capture: warm up outside the capture", dev);
        LLX_CUDA(cudaDeviceGetAttribute(&d.sm_count, cudaDevAttrMultiProcessorCount, dev));
        LLX_CUDA(cudaDeviceGetAttribute(&d.max_smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
        LLX_CUDA(cudaDeviceGetAttribute(&d.smem_per_sm, cudaDevAttrMaxSharedMemoryPerMultiprocessor, dev));
        LLX_CUDA(cudaFuncSetAttribute(llx_copy_bulk<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, d.max_smem_optin));
        LLX_CUDA(cudaFuncSetAttribute(llx_copy_bulk<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, d.max_smem_optin));
        LLX_CUDA(cudaFuncSetAttribute(llx_copy_tma<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, d.max_smem_optin));
        LLX_CUDA(cudaFuncSetAttribute(llx_copy_tma<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, d.max_smem_optin));
        d.ready = true;
    }
    // Shared-memory carve-out preference of the register-staged copy kernel (LLX_OPT_COPY_SMEM_CARVEOUT_PCT; see the
    // co-residency note at paced_in_flight below).  0 = the driver's default.
    const int want_carveout = (int)g_opt_carveout.load();
    if (d.carveout_applied != want_carveout && !capturing) {
        const int v = want_carveout > 0 ? want_carveout : cudaSharedmemCarveoutDefault;
        LLX_CUDA(cudaFuncSetAttribute(llx_copy_vec16<true, 4>, cudaFuncAttributePreferredSharedMemoryCarveout, v));
        LLX_CUDA(cudaFuncSetAttribute(llx_copy_vec16<false, 4>, cudaFuncAttributePreferredSharedMemoryCarveout, v));
        d.carveout_applied = want_carveout;
    }
    *out = &d;
    return LLX_OK;
}

// ---- id ring: pinned host slots + device slots, reused in order, guarded by events ---------
struct IdSlot {
    int32_t* host = nullptr;
    int32_t* dev = nullptr;
    size_t cap = 0;  // int32 entries
    cudaEvent_t ev = nullptr;
    bool used = false;
};
constexpr int kIdSlots = 8;
struct IdRing {  // one per device: a slot's device buffer and event belong to the device whose kernels read it
    std::mutex mu;
    IdSlot slots[kIdSlots];
    int next = 0;
};
IdRing g_ring[64];

// Copies `count` ids made of up to two host arrays (a then b) into a slot and enqueues the H2D
// copy; returns the device address.  The caller records the slot's event after its launch.
llx_status ring_stage(IdRing& ring, const int32_t* a, size_t na, const int32_t* b, size_t nb, cudaStream_t st, int32_t** dev_out,
                      IdSlot** slot_out) {
    // the caller holds ring.mu from here until it has recorded the slot's event behind its kernel launch:
    // another thread must not be handed this slot before that event exists
    IdSlot& s = ring.slots[ring.next];
    ring.next = (ring.next + 1) % kIdSlots;
    if (s.used) LLX_CUDA(cudaEventSynchronize(s.ev));
    const size_t need = na + nb;
    if (need > s.cap) {
        size_t cap = 1024;
        while (cap < need) cap *= 2;
        if (s.host) cudaFreeHost(s.host);
        if (s.dev) cudaFree(s.dev);
        s.host = nullptr;
        s.dev = nullptr;
        s.cap = 0;
        if (cudaMallocHost(&s.host, cap * sizeof(int32_t)) != cudaSuccess ||
            cudaMalloc(&s.dev, cap * sizeof(int32_t)) != cudaSuccess) {
            cudaGetLastError();
            return fail(LLX_ERR_OOM, "id ring: cannot allocate %zu ids", cap);
        }
        s.cap = cap;
    }
    if (!s.ev) LLX_CUDA(cudaEventCreateWithFlags(&s.ev, cudaEventDisableTiming));
    if (na) memcpy(s.host, a, na * sizeof(int32_t));
    if (nb) memcpy(s.host + na, b, nb * sizeof(int32_t));
    LLX_CUDA(cudaMemcpyAsync(s.dev, s.host, need * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    s.used = true;
    *dev_out = s.dev;
    *slot_out = &s;
    return LLX_OK;
}

// Records the slot's event behind the launch that reads it.  If the record fails the slot would be reused while its
// copy or kernel is still pending, so the stream is drained instead and the error reported.
llx_status ring_close(IdSlot* slot, cudaStream_t st) {
    if (!slot) return LLX_OK;
    cudaError_t e = cudaEventRecord(slot->ev, st);
    if (e == cudaSuccess) return LLX_OK;
    cudaStreamSynchronize(st);
    slot->used = false;
    return cuda_fail(e, "cudaEventRecord (id ring)");
}

// ---- claim counters of the bulk kernel's dynamic tail: one per (device, stream).  Launches of one stream are
// ordered (with programmatic dependent launch too: the claims come after griddepcontrol.wait), and every launch
// leaves its counter at zero again (its last claim resets it), so a stream's launches can share one counter
// without any event between them — an event record between two kernels would cost the PDL overlap. ----------
constexpr int kDynCounters = 4096;
std::mutex g_dyn_mu;
unsigned int* g_dyn_counters[64] = {};
std::unordered_map<cudaStream_t, int> g_dyn_of_stream[64];

// *counter = nullptr when the device's counters are all taken (the launch then runs without a dynamic tail)
llx_status dyn_counter_get(int dev, cudaStream_t st, unsigned int** counter) {
    std::lock_guard<std::mutex> lk(g_dyn_mu);
    if (!g_dyn_counters[dev]) {
        LLX_CUDA(cudaMalloc(&g_dyn_counters[dev], kDynCounters * sizeof(unsigned int)));
        LLX_CUDA(cudaMemset(g_dyn_counters[dev], 0, kDynCounters * sizeof(unsigned int)));
        LLX_CUDA(cudaDeviceSynchronize());
    }
    auto& m = g_dyn_of_stream[dev];
    auto it = m.find(st);
    if (it == m.end()) {
        if ((int)m.size() >= kDynCounters) {
            *counter = nullptr;
            return LLX_OK;
        }
        it = m.emplace(st, (int)m.size()).first;
    }
    *counter = g_dyn_counters[dev] + it->second;
    return LLX_OK;
}

// ---- co-residency of the register-staged copy kernel -----------------------------------------------------------
// The register-staged kernel (paced copies of NEXT-1, host zero-copy and peer routes) holds no shared memory, but its
// small CTAs stay resident on EVERY SM for a whole stage (75 ms for 112 blocks at 25 GB/s), and an SM cannot change its
// L1/shared-memory split while any CTA is resident.  Whatever split an SM has when such a CTA arrives is pinned until
// the END OF THE STAGE, and a kernel that needs more shared memory than that split offers waits that long.  Measured on
// B200 with the driver's default preference ("all L1" for a kernel without shared memory): a 2-block final stage (bulk
// ring, 2 x 76 KB of shared memory) next to a 25 GB/s stage: median 53 us, p90 75 ms; a 4096^3 bf16 GEMM: up to 75 ms.
// Three measures:
//  (1) the kernel asks for a 50 % carve-out (LLX_OPT_COPY_SMEM_CARVEOUT_PCT): arriving on idle SMs it leaves 132 KB of
//      shared memory configured and 124 KB of L1, which costs the L1-hungry stand-in decode step nothing (measured by
//      preference at a 20 GB/s budget: 0/50/64 %: +0.4..0.5 %, 75 %: +2.1 %, 100 %: +11 %).  That helps kernels of other
//      libraries up to 131 KB; llx's own bulk ring asks for the 164 KB split and still waits at 50 %, hence (2) and (3);
//  (2) the library remembers the register-staged launches that may still be running (one event each) and, while any
//      is, sends its own auto-selected copies through the register-staged kernel too: no shared memory, placed at once
//      (a short stage takes the same time: 23.3 vs 23.6 us; a long one runs at 6.1 instead of 6.5 TB/s next to the
//      budgeted stage);
//  (3) a budgeted stage is a chain of ~1 ms launches (LLX_OPT_PACED_SLICE_US, in launch_copy): whoever waits for an SM
//      to change its split waits for the end of a slice, not of the stage.
struct PacedTracker {
    std::mutex mu;
    static constexpr int kSlots = 16;
    cudaEvent_t ev[kSlots] = {};
    bool live[kSlots] = {};
    int next = 0;
};
PacedTracker g_paced[64];

bool paced_in_flight(int dev) {
    PacedTracker& t = g_paced[dev];
    std::lock_guard<std::mutex> lk(t.mu);
    bool any = false;
    for (int i = 0; i < PacedTracker::kSlots; ++i) {
        if (!t.live[i]) continue;
        const cudaError_t q = cudaEventQuery(t.ev[i]);
        if (q == cudaErrorNotReady) {
            any = true;
        } else {
            if (q != cudaSuccess) cudaGetLastError();
            t.live[i] = false;
        }
    }
    return any;
}
void paced_mark(int dev, cudaStream_t st) {
    PacedTracker& t = g_paced[dev];
    std::lock_guard<std::mutex> lk(t.mu);
    int slot = -1;
    for (int i = 0; i < PacedTracker::kSlots && slot < 0; ++i)
        if (!t.live[i]) slot = i;
    if (slot < 0) {  // all in use: the oldest is given up (it is then no longer tracked)
        slot = t.next;
        t.next = (t.next + 1) % PacedTracker::kSlots;
    }
    if (!t.ev[slot] && cudaEventCreateWithFlags(&t.ev[slot], cudaEventDisableTiming) != cudaSuccess) {
        cudaGetLastError();
        t.ev[slot] = nullptr;
        return;
    }
    t.live[slot] = cudaEventRecord(t.ev[slot], st) == cudaSuccess;
    if (!t.live[slot]) cudaGetLastError();
}

// ---- completion flags of llx_migrate_stage_wait: a word in mapped pinned host memory that the kernel's last
// ring writes, plus the device counter that finds the last ring.  A few slots, one per concurrent waiter. ----
struct DoneSlot {
    volatile unsigned int* host = nullptr;  // mapped pinned word
    unsigned int* dev_alias = nullptr;
    unsigned int* counter = nullptr;  // device
    unsigned int seq = 0;
    bool busy = false;
};
constexpr int kDoneSlots = 16;
std::mutex g_done_mu;
DoneSlot g_done[64][kDoneSlots];

struct DoneReq {  // set by llx_migrate_stage_wait around its launch_copy
    DoneSlot* slot = nullptr;
    bool armed = false;  // launch_copy attached the flag to the kernel it launched
};
thread_local DoneReq* tl_done = nullptr;

llx_status done_slot_get(int dev, DoneSlot** out) {
    std::lock_guard<std::mutex> lk(g_done_mu);
    for (auto& d : g_done[dev]) {
        if (d.busy) continue;
        if (!d.host) {
            void* h = nullptr;
            LLX_CUDA(cudaHostAlloc(&h, 64, cudaHostAllocMapped | cudaHostAllocPortable));
            void* da = nullptr;
            LLX_CUDA(cudaHostGetDevicePointer(&da, h, 0));
            LLX_CUDA(cudaMalloc(&d.counter, sizeof(unsigned int)));
            LLX_CUDA(cudaMemset(d.counter, 0, sizeof(unsigned int)));
            LLX_CUDA(cudaDeviceSynchronize());
            d.host = (volatile unsigned int*)h;
            *d.host = 0;
            d.dev_alias = (unsigned int*)da;
        }
        d.busy = true;
        *out = &d;
        return LLX_OK;
    }
    *out = nullptr;  // all slots taken: the caller falls back to the stream synchronize
    return LLX_OK;
}
void done_slot_put(DoneSlot* d) {
    std::lock_guard<std::mutex> lk(g_done_mu);
    d->busy = false;
}

// ---- validation ------------------------------------------------------------------------------
llx_status check_pool(const llx_pool* p, const char* name) {
    if (!p || !p->data) return fail(LLX_ERR_INVALID_ARG, "%s pool is NULL", name);
    int dev = -1;
    LLX_CUDA(cudaGetDevice(&dev));
    if (dev != p->device) return fail(LLX_ERR_INVALID_ARG, "%s pool lives on device %d, current device is %d", name, p->device, dev);
    return LLX_OK;
}
llx_status check_range(const int32_t* ids, long long n, int num_blocks, const char* name) {
    for (long long i = 0; i < n; ++i)
        if (ids[i] < 0 || ids[i] >= num_blocks)
            return fail(LLX_ERR_BLOCK_OUT_OF_RANGE, "%s_block_ids[%lld] = %d not in [0,%d)", name, i, ids[i], num_blocks);
    return LLX_OK;
}
llx_status check_unique(const int32_t* ids, long long n, int num_blocks) {
    thread_local std::vector<unsigned char> seen;
    seen.assign((size_t)num_blocks, 0);
    for (long long i = 0; i < n; ++i) {
        if (seen[ids[i]]) return fail(LLX_ERR_DUPLICATE_DST, "destination block id %d appears twice (second at %lld)", ids[i], i);
        seen[ids[i]] = 1;
    }
    return LLX_OK;
}
size_t pool_bytes(const llx_pool* p) { return (size_t)p->num_blocks * 2 * p->layers * (size_t)p->tile_bytes; }

// ---- launch helper: programmatic dependent launch (PDL) lets the next kernel of the stream become
// resident and run its prologue while the previous one drains; the kernels order their memory
// accesses themselves with griddepcontrol.wait, so stream semantics are unchanged. ----------------
template <typename... KArgs, typename... Args>
cudaError_t launch_k(bool pdl, void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

// ---- copy launch -----------------------------------------------------------------------------
struct Side {
    const unsigned char* base;
    const int32_t* ids;  // host ids or nullptr (contiguous side)
    long long slice_stride, item_stride;
    bool host_memory;  // staging in mapped host memory
    int device = -1;   // pool side: the device its memory lives on (-1: staging)
    const llx_pool* pool = nullptr;  // pool side: the pool (its tensor map serves the small-tile kernel)
};

// `device` = the device the kernel runs on = the current device (the source pool's for a migration).
llx_status launch_copy(const Policy& pol, const Side& src, const Side& dst, long long n, int layers, long long tile_bytes,
                       int device, cudaStream_t st) {
    bool capturing = false;
    llx_status rc = stream_capturing(st, &capturing);
    if (rc != LLX_OK) return rc;
    DevInfo* di = nullptr;
    if ((rc = dev_info(device, &di, capturing)) != LLX_OK) return rc;

    // kernel choice: the bulk-async ring for device<->device, the LDG/STG kernel when a side is host memory
    long long kern = pol.kernel;
    // a peer-mapped destination (another GPU) is written with plain 16-byte stores: NVLink, not HBM, is the bound.
    // LLX_ROUTE_PEER takes the same route with both pools on one device (how a single-GPU box executes this branch).
    const bool peer = pol.route == LLX_ROUTE_PEER || (src.device >= 0 && dst.device >= 0 && src.device != dst.device);
    if (kern == 0) kern = (src.host_memory || dst.host_memory || peer) ? 1 : 2;
    // Bandwidth budget: paced register-staged copies, no shared memory.  Measured
    // on B200: a co-resident CTA that holds > ~6 KB of shared memory shrinks the L1 of its SM and slows a
    // bandwidth-bound decode kernel by 30 %, and a few full-speed CTAs turn their SMs into stragglers.
    // Above ~500 GB/s pacing on every SM stops paying: measured per GB/s of migration the decode step loses 0.026 % at
    // 400 GB/s paced but 0.045 % at 800 and 0.060 % at 2400, while a FEW full-speed bulk CTAs stay at 0.023-0.030 %
    // (about 60 GB/s per CTA: 7 CTAs 447 GB/s, 14: 864, 29: 1623, 43: 2243).  High budgets are therefore met by the
    // CTA count of the unpaced bulk kernel, low ones by the paced kernel.
    // while a register-staged stage may be resident on every SM, auto-selected copies avoid shared memory (see paced_in_flight)
    const bool beside_paced = pol.kernel == 0 && kern == 2 && !capturing && paced_in_flight(device);
    if (beside_paced) kern = 1;
    const long long budget_asked = pol.budget;
    const bool budget_by_ctas = budget_asked >= 500 && pol.kernel == 0 && kern == 2;
    const long long budget = budget_by_ctas ? 0 : budget_asked;  // from here on: > 0 means "paced"
    if (budget > 0 && pol.kernel != 2) kern = 1;
    // The tensor-map kernel (copy_kernel = 3): pool -> pool on one device, tiles of at most 16 KiB, both pools described
    // by tensor maps with the same box (same geometry => same box).  One unit = one block in tma_k consecutive slices.
    const bool tensor_possible = src.pool && dst.pool && src.ids && dst.ids && !peer && !src.host_memory && !dst.host_memory &&
                                 src.pool->tma_k >= 2 && dst.pool->tma_k == src.pool->tma_k;
    bool tensor = false;
    if (kern == 3) {
        if (!tensor_possible)
            return fail(LLX_ERR_INVALID_ARG, "copy_kernel = 3 (tensor-map kernel) needs a pool-to-pool copy on one device with tiles of at most 16 KiB");
        kern = 2;
        tensor = true;
    }
    const long long total_bytes = n * 2 * layers * tile_bytes;
    // Never taken by itself: once the 1-D ring's depth follows the loads-in-flight rule below, the two tie on every small
    // tile measured (4 KiB: 6.55 / 6.53 TB/s, 8 KiB: 6.48 / 6.48, 16 KiB: 6.53 / 6.51, 12 KiB: 6.41 / 6.38, 3.75 KiB: 6.17 / 6.02);
    // the tensor-map kernel gets there with ONE ring per SM instead of two or four.
    const int tma_k = tensor ? src.pool->tma_k : 1;

    long long chunk = pol.chunk;
    int nstages = (int)pol.stages;
    int threads = 256, grid = 0, long_per_sm = 1;
    size_t smem = 0;
    const int slices = 2 * layers;

    if (kern == 2) {
        // Tuned on B200 (round-1 CUDA-event sweeps, summarised in profiles/r01_ncu_summary.md; re-checked in round 2): ONE CTA
        // per SM with one ring of 3 x 32 KiB,
        // every ring streaming a contiguous range of chunks and the last 6 % of the stage claimed dynamically
        // (6.57 TB/s at 112 blocks, 6.66 TB/s at >= 256).  More bytes in flight per SM lowers DRAM efficiency.
        // A short stage (the final one: 2 blocks) is latency-bound: smaller chunks over twice as many rings.
        const bool short_stage = total_bytes < (64ll << 20) && !budget_by_ctas;
        // Long stages of tiles that are not a multiple of 32 KiB (any head count that is not a multiple of 8: 13 heads of
        // a TP=4 rank of LLaMA-30B = 52 KiB).  "32 KiB, then the rest" leaves a short chunk per tile that occupies a whole
        // ring stage, so fewer bytes are in flight and DRAM idles: 52 KiB tiles ran at 6.13 TB/s, 40 KiB at 5.4, 36 KiB at 5.0.
        // Measured over 13 tile sizes from 20 to 208 KiB (one ring per SM): what matters is (a) chunks of EQUAL size and
        // (b) about 62 KiB of loads in flight per SM — (stages - 1) x chunk; 52 KiB is too little, 78 KiB already too
        // much — with chunks of at least 13 KiB.  So: split the tile into m equal chunks, m from ceil(tile / 32 KiB) up, and
        // take the (m, stages) whose loads in flight are closest to 62 KiB, the larger chunk unless a smaller one is 2 KiB closer.  Multiples of 32 KiB keep
        // 3 x 32 KiB; 52 KiB -> 4 x 13 KiB, 6 stages: 6.48 TB/s; 40 KiB -> 2 x 20 KiB, 4 stages: 6.41; 36 KiB: 6.18; 72 KiB: 6.49;
        // 80 KiB: 6.55; 208 KiB -> 10 x 20.8 KiB, 4 stages: 6.67 (from 6.63).
        bool equal_split = false;
        if (chunk <= 0 && nstages <= 0 && pol.rings <= 0 && !tensor && !short_stage && budget <= 0 && tile_bytes > 16384) {
            const long long target = 62ll << 10, m0 = (tile_bytes + 32767) / 32768;
            long long best = -1;
            for (long long m = m0; m <= m0 + 12; ++m) {
                const long long c = ((tile_bytes + m - 1) / m + 15) & ~15ll;
                if (m > m0 && c < 13312) break;
                for (int sg = 3; sg <= 8 && c * sg <= (160ll << 10); ++sg) {
                    const long long fl = (sg - 1) * c, score = fl > target ? fl - target : target - fl;
                    if (best < 0 || score + 2048 < best) {  // a smaller chunk has to be clearly closer (2 KiB) to replace a larger one
                        best = score;
                        chunk = c;
                        nstages = sg;
                    }
                }
            }
            equal_split = true;
        }
        if (chunk <= 0) chunk = budget > 0 ? 2048 : short_stage ? 8192 : 32768;  // paced: a 4 KiB ring stays below the L1 carve-out step
        if (chunk > tile_bytes) chunk = tile_bytes;
        chunk &= ~15ll;
        if (tensor) chunk = tma_k * tile_bytes;  // one box = one ring stage
        // Small tiles cap the chunk, and one thread cannot issue small bulk copies fast enough to keep its SM's share
        // of HBM busy (measured, long stages: 8 KiB tiles 3.5 TB/s with one ring per SM, 6.0 TB/s with two; 4 KiB
        // tiles 2.0 -> 6.0 TB/s with four): more CTAs per SM, ~64-96 KiB in flight per SM in every case.
        long_per_sm = (chunk >= 16384 || equal_split || tensor) ? 1 : chunk >= 8192 ? 2 : 4;
        if (nstages <= 0 && budget <= 0 && !short_stage) {
            // ring depth from the same measurement as above: ~62 KiB of loads in flight per SM, over all rings of the SM.
            // 32 KiB chunks: 3 stages; 16 KiB: 5 (6.19 -> 6.54 TB/s; 6 stages = 80 KiB in flight is already too much);
            // two rings of 8 KiB or four of 4 KiB: 5 each; a 24 KiB tensor-map box: 4 (6.18 -> 6.38)
            const long long per_stage = (long long)long_per_sm * chunk;
            nstages = 1 + (int)(((62ll << 10) + per_stage / 2) / per_stage);
            if (nstages < 3) nstages = 3;
            if (nstages > 8) nstages = 8;
            if (long_per_sm == 4) nstages = 4;  // four rings of 4 KiB: 48 KiB in flight measured best (6.55 vs 6.45 TB/s with 5 stages)
        }
        if (nstages <= 0) nstages = budget > 0 ? 2 : 4;
        int rings = (int)pol.rings;
        if (rings <= 0) rings = 1;
        threads = 32 * rings;
        smem = (((size_t)rings * nstages * 12 + 127) & ~(size_t)127) + (size_t)rings * nstages * chunk;
        if ((long long)smem > di->max_smem_optin) return fail(LLX_ERR_INVALID_ARG, "ring of %d x %lld bytes exceeds shared memory", nstages, chunk);
    } else {
        if (budget > 0) {  // ~2 GB/s (rd+wr) per warp keeps the loads latency-bound and gentle; spread over all SMs
            long long warps = (budget + 1) / 2;
            int ctas_per_sm = (int)((warps + (long long)di->sm_count * 8 - 1) / ((long long)di->sm_count * 8));
            if (ctas_per_sm < 1) ctas_per_sm = 1;
            if (ctas_per_sm > 8) ctas_per_sm = 8;
            grid = di->sm_count * ctas_per_sm;
            long long wpc = (warps + grid - 1) / grid;
            if (wpc < 1) wpc = 1;
            if (wpc > 8) wpc = 8;
            threads = (int)wpc * 32;
            if (pol.rings > 0) threads = (int)pol.rings * 32;  // experiments: warps per paced CTA
            if (chunk <= 0) chunk = (long long)threads * 16 * 4;
        } else if (chunk <= 0) {
            chunk = 256 * 16 * 4;
        }
        if (chunk > tile_bytes) chunk = tile_bytes;
        chunk &= ~15ll;
    }
    const long long cpt = tensor ? 1 : (tile_bytes + chunk - 1) / chunk;
    const long long units = tensor ? n * (slices / tma_k) : n * slices * cpt;
    if (units >= (1ll << 31)) return fail(LLX_ERR_INVALID_ARG, "stage too large: %lld units", units);

    if (kern == 2) {
        int per_sm = (int)((size_t)di->max_smem_optin / (smem + 1024));  // 1 KiB per-CTA reservation
        if (per_sm > 2) per_sm = 2;
        if (per_sm < 1 || budget > 0) per_sm = 1;
        if (budget <= 0 && (total_bytes >= (64ll << 20) || budget_by_ctas)) per_sm = long_per_sm;
        grid = di->sm_count * per_sm;
        // Exact residency: with programmatic dependent launch the NEXT kernel's CTAs are placed while this kernel
        // still runs, wherever shared memory is free — several on one SM if they fit.  A ring's share of the stage is
        // fixed, so an SM that ends up with more rings than its neighbours becomes the straggler (measured: 3 CTAs/SM
        // of 25 KiB: 351 us per step without PDL, 449-509 us with it).  Asking for just over 1/(per_sm+1) of the
        // SM's shared memory caps every SM at per_sm bulk CTAs, of this launch and of the next one together.
        long long want = per_sm;  // CTAs per SM the launch is meant to have
        const long long capv = pol.max_ctas;
        if (capv > 0) want = (capv % di->sm_count == 0) ? capv / di->sm_count : 0;
        if (pol.smem_pad && budget <= 0 && want >= 1 && want <= 6) {
            const size_t floor_bytes = (size_t)di->smem_per_sm / (size_t)(want + 1) - 1024 + 128;
            if (smem < floor_bytes && floor_bytes <= (size_t)di->max_smem_optin) smem = floor_bytes;
        }
    } else if (budget <= 0) {
        // A side in host memory is bound by the host link (~52 GB/s): one CTA per SM already saturates it
        // (measured: 52.7 GB/s with 74..296 CTAs, 51.5 with 1184) and leaves the SMs to whatever else is running.
        // Device <-> device: FOUR CTAs per SM, i.e. 4 x 256 threads x 4 loads x 16 B = 64 KiB of loads in flight per SM — the
        // same optimum as the bulk ring's (~62 KiB).  Round 1 launched eight (128 KiB in flight): 5.57 TB/s for 128 blocks of
        // LLaMA-7B, 5.80 for 512; four: 6.05 and 6.14-6.22; three or five are slower again.
        grid = (src.host_memory || dst.host_memory) ? di->sm_count : di->sm_count * 4;
    }
    long long cap = pol.max_ctas;
    if (cap <= 0 && budget_by_ctas) cap = (budget_asked + 30) / 60;
    if (cap > 0) grid = (int)cap;  // explicit grid: the throttle (fewer CTAs) or an experiment (more)
    {
        const long long workers_per_cta = (kern == 2) ? threads / 32 : 1;  // rings per CTA
        const long long need = (units + workers_per_cta - 1) / workers_per_cta;
        if (grid > need) grid = (int)need;
    }
    long long pace_ns = 0;
    if (budget > 0) {
        const long long workers = (kern == 2) ? (long long)grid * (threads / 32) : grid;  // rings or CTAs
        pace_ns = workers * 2 * chunk / budget;  // per worker; bytes/ns == GB/s, read + written
        if (pace_ns > 1000000000ll) pace_ns = 1000000000ll;
    }

    CopyArgs a;
    a.src_base = src.base;
    a.dst_base = const_cast<unsigned char*>(dst.base);
    a.src_slice_stride = src.slice_stride;
    a.src_item_stride = src.item_stride;
    a.dst_slice_stride = dst.slice_stride;
    a.dst_item_stride = dst.item_stride;
    a.src_indexed = src.ids != nullptr;
    a.dst_indexed = dst.ids != nullptr;
    a.src_ids = a.dst_ids = nullptr;
    a.tile_bytes = (int)(tensor ? chunk : tile_bytes);
    a.chunk_bytes = (int)chunk;
    a.chunks_per_tile = (int)cpt;
    a.slices = tensor ? slices / tma_k : slices;
    a.tma_k = tma_k;
    a.total_units = (int)units;
    a.unit_begin = 0;
    a.blocked_order = (int)pol.order;
    a.l2_hint = (int)pol.l2hint;
    a.pace_ns = (int)pace_ns;
    // LLX_OPT_OVERLAP_PREV: only the unthrottled bulk ring starts before the previous kernel has finished, and only with
    // programmatic dependent launch (without it the stream serialises the kernels anyway)
    a.defer_wait = (kern == 2 && pol.overlap != 0 && pol.pdl != 0 && budget <= 0) ? 1 : 0;
    a.dyn_units = 0;
    a.dyn_batch = 1;
    a.dyn_claims = 0;
    a.dyn_counter = nullptr;
    a.done_counter = nullptr;
    a.done_flag = nullptr;
    a.done_value = 0;
    a.done_rings = 0;
    if (tl_done && tl_done->slot && kern == 2) {
        DoneSlot* d = tl_done->slot;
        a.done_counter = d->counter;
        a.done_flag = d->dev_alias;
        a.done_value = ++d->seq;
        a.done_rings = (unsigned int)((long long)grid * (threads / 32));
        tl_done->armed = true;
    }
    {
        // Dynamic tail (bulk kernel, blocked order, stages long enough to have a tail worth evening out): SMs do not
        // stream at exactly the same rate, so with fixed ranges the fastest rings idle at the end (ncu: SM active
        // cycles avg 96.4 % vs max 98.9 % of the kernel).  The last dyn_pct % of the units are claimed in batches.
        // Measured (B200, 7B tiles): 112 blocks 295.4 -> 291.3 us, 256 blocks 672 -> 656 us at 4-8 %; 1 % and 15 %
        // give half of that, 100 % (no contiguous ranges at all) is 3 % slower than none.
        // Not under stream capture: the claim counter belongs to the LAUNCHING stream, and a captured launch may be
        // replayed on any stream, concurrently with direct launches of the capture stream that share the counter
        // (a ring that reads an inflated claim index would stop early and chunks would never be copied).
        const long long pct = pol.dyn_pct;
        const long long nrings = (long long)grid * (threads / 32);
        if (kern == 2 && a.blocked_order && pct > 0 && budget <= 0 && units >= nrings * 16 && !capturing) {
            const long long batch = pol.dyn_batch > 0 ? pol.dyn_batch : 4;
            long long dyn = units * pct / 100 / batch * batch;
            if (dyn > 0) {
                if ((rc = dyn_counter_get(device, st, &a.dyn_counter)) != LLX_OK) return rc;
                if (a.dyn_counter) {
                    a.dyn_units = (int)dyn;
                    a.dyn_batch = (int)batch;
                    a.dyn_claims = (unsigned int)(dyn / batch + nrings);
                }
            }
        }
    }

    static thread_local IdPack pack;  // 2 KiB; only the first n entries are meaningful
    const bool byval = n <= pol.byval || (!src.ids && !dst.ids);
    IdRing& ring = g_ring[device];
    std::unique_lock<std::mutex> ring_lk(ring.mu, std::defer_lock);
    IdSlot* slot = nullptr;
    if (byval) {
        if (src.ids) memcpy(pack.src, src.ids, n * sizeof(int32_t));
        if (dst.ids) memcpy(pack.dst, dst.ids, n * sizeof(int32_t));
    } else {
        if (capturing)
            return fail(LLX_ERR_STATE, "a stage of %lld pairs cannot be captured into a CUDA graph: id lists longer than %lld go through a pinned ring "
                        "(host copy + event wait at launch); split the stage into calls of <= %d pairs", n, pol.byval, kIdsByValueCap);
        int32_t* dev_ids = nullptr;
        ring_lk.lock();
        rc = ring_stage(ring, src.ids, src.ids ? n : 0, dst.ids, dst.ids ? n : 0, st, &dev_ids, &slot);
        if (rc != LLX_OK) return rc;
        if (src.ids) a.src_ids = dev_ids;
        if (dst.ids) a.dst_ids = dev_ids + (src.ids ? n : 0);
        g_id_uploads++;
    }

    cudaError_t e = cudaSuccess;
    const bool pdl = pol.pdl != 0;
    int launches = 1;
    if (kern == 2 && tensor) {
        if (byval)
            e = launch_k(pdl, llx_copy_tma<true>, grid, threads, smem, st, a, pack, nstages, src.pool->tmap, dst.pool->tmap);
        else
            e = launch_k(pdl, llx_copy_tma<false>, grid, threads, smem, st, a, pack, nstages, src.pool->tmap, dst.pool->tmap);
    } else if (kern == 2) {
        if (byval)
            e = launch_k(pdl, llx_copy_bulk<true>, grid, threads, smem, st, a, pack, nstages);
        else
            e = launch_k(pdl, llx_copy_bulk<false>, grid, threads, smem, st, a, pack, nstages);
    } else {
        // A paced stage is issued as a chain of short launches (LLX_OPT_PACED_SLICE_US, default 1 ms): its CTAs sit on every
        // SM, and an SM whose L1/shared split is too small for a waiting kernel can only be reconfigured when no CTA is
        // resident (see paced_in_flight).  With slices, such a kernel waits for the end of a slice, not of the stage.
        // Measured next to a 25 GB/s stage of 112 blocks (75 ms): a kernel that needs the 164 KB split: p99 75 ms as one
        // launch, 1.0 ms with 1 ms slices, 0.27 ms with 250 us slices; a 4096^3 GEMM likewise; the stage still runs at
        // 24.9 / 24.6 GB/s and the decode step's slowdown is unchanged (+0.4 % at 25 GB/s, +3.6 % at 100 GB/s).  Price: ~3 us
        // of host time per slice inside the call.  Slices after the first are launched WITHOUT programmatic dependent
        // launch: an early-launched successor would keep the SMs occupied across the boundary.  Every CTA restarts its
        // pacing clock at its slice's start.
        const long long slice_us = g_opt_slice_us.load();
        long long per_slice = units;
        if (budget > 0 && slice_us > 0 && pace_ns > 0 && !capturing) {
            const long long chunks_per_cta = slice_us * 1000 / pace_ns;  // chunks one CTA moves within one slice
            per_slice = (chunks_per_cta < 1 ? 1 : chunks_per_cta) * (long long)grid;
            const long long floor_units = ((units + 255) / 256 + grid - 1) / grid * grid;  // at most 256 launches per call
            if (per_slice < floor_units) per_slice = floor_units;
            if (per_slice * 3 / 2 >= units) per_slice = units;  // not worth cutting
        }
        for (long long u0 = 0; u0 < units && e == cudaSuccess; u0 += per_slice) {
            a.unit_begin = (int)u0;
            a.total_units = (int)(u0 + per_slice < units ? u0 + per_slice : units);
            const bool p = pdl && u0 == 0;
            if (byval)
                e = launch_k(p, llx_copy_vec16<true, 4>, grid, threads, 0, st, a, pack);
            else
                e = launch_k(p, llx_copy_vec16<false, 4>, grid, threads, 0, st, a, pack);
            if (u0 > 0) ++launches;
        }
    }
    if (e == cudaSuccess) e = cudaGetLastError();
    const llx_status rc_ring = ring_close(slot, st);
    if (e != cudaSuccess) return cuda_fail(e, "copy kernel launch");
    if (rc_ring != LLX_OK) return rc_ring;
    // a register-staged stage that will be resident for a while (every paced one; unpaced ones from 8 MiB): remember it
    if (kern == 1 && !capturing && (budget > 0 || total_bytes >= (8ll << 20))) paced_mark(device, st);
    g_launches += (unsigned long long)launches;
    g_copy_launches += (unsigned long long)launches;
    g_bytes += (unsigned long long)total_bytes;
    return LLX_OK;
}

Side pool_side(const llx_pool* p, const int32_t* ids) {
    return Side{p->data, ids, (long long)p->num_blocks * p->tile_bytes, p->tile_bytes, false, p->device, p};
}
llx_status staging_side(const void* staging, int layers, long long tile_bytes, Side* out) {
    cudaPointerAttributes at;
    LLX_CUDA(cudaPointerGetAttributes(&at, staging));
    if (at.type != cudaMemoryTypeDevice && at.type != cudaMemoryTypeHost && at.type != cudaMemoryTypeManaged)
        return fail(LLX_ERR_INVALID_ARG, "staging buffer is neither device nor pinned host memory");
    const void* p = staging;
    if (at.type == cudaMemoryTypeHost) p = at.devicePointer ? at.devicePointer : staging;
    if (((uintptr_t)p & 15) != 0) return fail(LLX_ERR_INVALID_ARG, "staging buffer must be 16-byte aligned");
    *out = Side{(const unsigned char*)p, nullptr, tile_bytes, 2ll * layers * tile_bytes, at.type == cudaMemoryTypeHost};
    return LLX_OK;
}

llx_status check_pair(const llx_pool* src, const llx_pool* dst) {
    llx_status rc = check_pool(src, "src");
    if (rc != LLX_OK) return rc;
    // The destination may live on ANOTHER GPU (the two instances are different
    // machines): the kernel runs on the source's device and stores straight into the peer-mapped pool over NVLink.
    if (dst && dst->data && dst->device != src->device) {
        int can = 0;
        LLX_CUDA(cudaDeviceCanAccessPeer(&can, src->device, dst->device));
        if (!can) return fail(LLX_ERR_INVALID_ARG, "device %d cannot access the dst pool on device %d", src->device, dst->device);
        cudaError_t e = cudaDeviceEnablePeerAccess(dst->device, 0);
        if (e == cudaErrorPeerAccessAlreadyEnabled) cudaGetLastError();
        else if (e != cudaSuccess) return cuda_fail(e, "cudaDeviceEnablePeerAccess");
    } else {
        rc = check_pool(dst, "dst");
        if (rc != LLX_OK) return rc;
    }
    if (src == dst) return fail(LLX_ERR_ALIAS, "src and dst are the same pool");
    const unsigned char *a0 = src->data, *a1 = a0 + pool_bytes(src), *b0 = dst->data, *b1 = b0 + pool_bytes(dst);
    if (a0 < b1 && b0 < a1) return fail(LLX_ERR_ALIAS, "src and dst pools overlap in memory");
    if (src->layers != dst->layers || src->tile_bytes != dst->tile_bytes || src->kv_heads != dst->kv_heads ||
        src->head_dim != dst->head_dim || src->block_size != dst->block_size || src->elem_bytes != dst->elem_bytes)
        return fail(LLX_ERR_GEOMETRY_MISMATCH, "src (L=%d,H=%d,D=%d,S=%d,e=%d) vs dst (L=%d,H=%d,D=%d,S=%d,e=%d)", src->layers,
                    src->kv_heads, src->head_dim, src->block_size, src->elem_bytes, dst->layers, dst->kv_heads,
                    dst->head_dim, dst->block_size, dst->elem_bytes);
    return LLX_OK;
}

// ---- the pipelined host route (llx_migrate_via_host): two internal streams, a ring of events and four
// device bounce buffers per device ------------------------------------------------------------------------
struct Pipe {
    cudaStream_t d2h = nullptr, h2d = nullptr;
    cudaEvent_t ev[64] = {};
    int next = 0;
    unsigned char* bounce[4] = {};  // [0,1] gather side, [2,3] scatter side
    size_t bounce_bytes = 0;        // of each
    cudaEvent_t idle = nullptr;     // recorded when a call's last use of the bounce buffers is enqueued; the next
    bool idle_valid = false;        // call (maybe on another stream) waits for it before touching them
    cudaEvent_t take() {
        cudaEvent_t e = ev[next];
        next = (next + 1) % 64;
        return e;
    }
};
std::mutex g_pipe_mu;
Pipe g_pipe[64];

llx_status pipe_get(int dev, size_t bounce_bytes, Pipe** out) {
    Pipe& p = g_pipe[dev];
    if (!p.d2h) {
        LLX_CUDA(cudaStreamCreateWithFlags(&p.d2h, cudaStreamNonBlocking));
        LLX_CUDA(cudaStreamCreateWithFlags(&p.h2d, cudaStreamNonBlocking));
        for (auto& e : p.ev) LLX_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        LLX_CUDA(cudaEventCreateWithFlags(&p.idle, cudaEventDisableTiming));
    }
    if (bounce_bytes > p.bounce_bytes) {  // first use or growth: synchronises the device
        LLX_CUDA(cudaDeviceSynchronize());
        for (auto& b : p.bounce) {
            if (b) cudaFree(b);
            b = nullptr;
        }
        p.bounce_bytes = 0;
        for (auto& b : p.bounce)
            if (cudaMalloc(&b, bounce_bytes) != cudaSuccess) {
                cudaGetLastError();
                return fail(LLX_ERR_OOM, "bounce buffers of %zu bytes", bounce_bytes);
            }
        p.bounce_bytes = bounce_bytes;
    }
    *out = &p;
    return LLX_OK;
}


// llx_pack / llx_unpack with a pinned-host buffer: the copy engine crosses the host link (57 GB/s device->host,
// 55.6 host->device on this B200) faster than kernels addressing the pinned buffer directly (52.7 / 51.4 GB/s),
// so the tiles are gathered into (scattered from) a device bounce buffer chunk by chunk and the chunk is moved
// with cudaMemcpyAsync, all on the caller's stream (a 64 MiB chunk: 10 us of kernel per 1.1 ms of link).
llx_status staged_through_bounce(const Policy& pol, bool to_host, const llx_pool* pool, const int32_t* ids, int n, const Side& stg, cudaStream_t st) {
    llx_status rc = refuse_if_capturing(st, "llx_pack / llx_unpack through a pinned-host buffer");
    if (rc != LLX_OK) return rc;
    const long long block_bytes = 2ll * pool->layers * pool->tile_bytes;
    int chunk_blocks = (int)((64ll << 20) / block_bytes);
    if (chunk_blocks < 1) chunk_blocks = 1;
    if (chunk_blocks > n) chunk_blocks = n;
    if (chunk_blocks > kIdsByValueCap) chunk_blocks = kIdsByValueCap;
    std::lock_guard<std::mutex> lk(g_pipe_mu);
    Pipe* pipe = nullptr;
    if ((rc = pipe_get(pool->device, (size_t)chunk_blocks * block_bytes, &pipe)) != LLX_OK) return rc;
    if (pipe->idle_valid) LLX_CUDA(cudaStreamWaitEvent(st, pipe->idle, 0));
    unsigned char* bounce = pipe->bounce[to_host ? 0 : 2];
    const Side dev_side = Side{bounce, nullptr, stg.slice_stride, stg.item_stride, false};
    cudaError_t ce = cudaSuccess;
    for (int k = 0; k < n && rc == LLX_OK && ce == cudaSuccess; k += chunk_blocks) {
        const int m = (n - k < chunk_blocks) ? n - k : chunk_blocks;
        unsigned char* host = const_cast<unsigned char*>(stg.base) + (long long)k * block_bytes;
        const size_t bytes = (size_t)m * block_bytes;
        if (to_host) {
            rc = launch_copy(pol, pool_side(pool, ids + k), dev_side, m, pool->layers, pool->tile_bytes, pool->device, st);
            if (rc == LLX_OK) ce = cudaMemcpyAsync(host, bounce, bytes, cudaMemcpyDefault, st);
        } else {
            ce = cudaMemcpyAsync(bounce, host, bytes, cudaMemcpyDefault, st);
            if (ce == cudaSuccess) rc = launch_copy(pol, dev_side, pool_side(pool, ids + k), m, pool->layers, pool->tile_bytes, pool->device, st);
        }
    }
    // also on an error path: whatever was enqueued still uses the bounce buffers, the next call must wait for it
    if (cudaEventRecord(pipe->idle, st) == cudaSuccess) pipe->idle_valid = true;
    if (rc != LLX_OK) return rc;
    if (ce != cudaSuccess) return cuda_fail(ce, "cudaMemcpyAsync (bounce buffer)");
    return LLX_OK;
}

// LLX_OPT_VIA_HOST_MODE = 2: the copy engine gathers / scatters by itself.  One block is 2L tiles at a constant
// stride (num_blocks*tile_bytes) in the pool and 2L consecutive tiles in the staging buffer: ONE pitched copy per block
// (cudaMemcpy2DAsync: width = tile_bytes, height = 2L) crosses the link with no kernel, no bounce buffer and no SM.
// A pitched transfer's pitch is limited (cudaDevAttrMaxPitch, 2^31-1 bytes on B200), and a pool's slice stride
// num_blocks*tile_bytes passes that in big pools (LLaMA-7B tiles: from 16384 blocks = 128 GiB of pool; fewer layers, sooner).
// Such a pool is served tile by tile: 2L plain copies per block instead of one pitched one — still the copy engines, no
// kernel, more calls.  (llx_migrate_via_host's AUTO route prefers the bounce route there, see below.)
bool pitch_ok(const llx_pool* pool) {
    static std::atomic<long long> cache[64];
    const int dev = pool->device;
    long long lim = (dev >= 0 && dev < 64) ? cache[dev].load() : 0;
    if (lim <= 0) {
        int v = 0;
        if (cudaDeviceGetAttribute(&v, cudaDevAttrMaxPitch, dev) != cudaSuccess || v <= 0) {
            cudaGetLastError();
            v = 0x7fffffff;
        }
        lim = v;
        if (dev >= 0 && dev < 64) cache[dev] = lim;
    }
    return (long long)pool->num_blocks * pool->tile_bytes <= lim;
}

llx_status ce_blocks(bool to_host, const llx_pool* pool, const int32_t* ids, int first, int count, const Side& stg, cudaStream_t st) {
    const size_t tile = (size_t)pool->tile_bytes, pool_pitch = (size_t)pool->num_blocks * tile;
    const size_t rows = 2 * (size_t)pool->layers, block_bytes = rows * tile;
    const bool pitched = pitch_ok(pool);
    for (int i = first; i < first + count; ++i) {
        unsigned char* p = pool->data + (size_t)ids[i] * tile;
        unsigned char* h = const_cast<unsigned char*>(stg.base) + (size_t)i * block_bytes;
        if (!pitched) {
            for (size_t r = 0; r < rows; ++r) {
                if (to_host)
                    LLX_CUDA(cudaMemcpyAsync(h + r * tile, p + r * pool_pitch, tile, cudaMemcpyDefault, st));
                else
                    LLX_CUDA(cudaMemcpyAsync(p + r * pool_pitch, h + r * tile, tile, cudaMemcpyDefault, st));
            }
        } else if (to_host) {
            LLX_CUDA(cudaMemcpy2DAsync(h, tile, p, pool_pitch, tile, rows, cudaMemcpyDefault, st));
        } else {
            LLX_CUDA(cudaMemcpy2DAsync(p, pool_pitch, h, tile, tile, rows, cudaMemcpyDefault, st));
        }
    }
    return LLX_OK;
}

// ---- tensor map of a small-tile pool (llx_copy_tma) ---------------------------------------------------------------
// One tile is at most 16 KiB here, so a 1-D bulk copy moves little per instruction and one thread cannot issue them fast
// enough for its SM's share of HBM.  The pool is therefore also described to the TMA unit as a 4-D
// tensor of 8-byte elements — (row of <= 2 KiB, rows of a tile, block, slice) — with a box that spans ONE block in tma_k
// consecutive (layer, K|V) slices: one instruction then moves tma_k tiles (<= 32 KiB), gathered by the TMA unit itself.
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn encode_tiled_fn() {
    static EncodeTiledFn fn = [] {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q = cudaDriverEntryPointSymbolNotFound;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess) {
            cudaGetLastError();
            p = nullptr;
        }
        return (EncodeTiledFn)p;
    }();
    return fn;
}
void build_tensor_map(llx_pool* p) {
    static_assert(sizeof(CUtensorMap) == sizeof(llx::TensorMap), "CUtensorMap is 128 bytes");
    p->tma_k = 0;
    const long long tile = p->tile_bytes, slices = 2ll * p->layers;
    if (tile > (16 << 10)) return;
    int k = 0;
    for (int c = 2; c <= 256 && c <= slices; ++c)
        if (slices % c == 0 && c * tile <= (32 << 10) && (c * tile) % 128 == 0) k = c;
    long long row = 0;
    for (long long d = 16; d <= 2048 && d <= tile; d += 16)
        if (tile % d == 0) row = d;
    if (k < 2 || row == 0 || tile / row > 256) return;
    EncodeTiledFn enc = encode_tiled_fn();
    if (!enc) return;
    const cuuint64_t dims[4] = {(cuuint64_t)(row / 8), (cuuint64_t)(tile / row), (cuuint64_t)p->num_blocks, (cuuint64_t)slices};
    const cuuint64_t strides[3] = {(cuuint64_t)row, (cuuint64_t)tile, (cuuint64_t)p->num_blocks * (cuuint64_t)tile};
    const cuuint32_t box[4] = {(cuuint32_t)(row / 8), (cuuint32_t)(tile / row), 1u, (cuuint32_t)k};
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    if (strides[2] >= (1ull << 40)) return;
    const CUresult r = enc(reinterpret_cast<CUtensorMap*>(&p->tmap), CU_TENSOR_MAP_DATA_TYPE_UINT64, 4, p->data, dims, strides, box, estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r == CUDA_SUCCESS) p->tma_k = k;
}

llx_status make_pool(void* ptr, size_t bytes, bool owned, int layers, int kv_heads, int head_dim, int block_size,
                     llx_dtype dtype, int num_blocks, llx_pool** out) {
    if (!out) return fail(LLX_ERR_INVALID_ARG, "out is NULL");
    *out = nullptr;
    const size_t need = llx_pool_bytes_for(layers, kv_heads, head_dim, block_size, dtype, num_blocks);
    if (need == 0) return fail(LLX_ERR_INVALID_ARG, "bad geometry L=%d H=%d D=%d S=%d dtype=%d blocks=%d (tile must be a positive multiple of 16 bytes)",
                               layers, kv_heads, head_dim, block_size, (int)dtype, num_blocks);
    int dev = 0;
    LLX_CUDA(cudaGetDevice(&dev));
    if (owned) {
        cudaError_t e = cudaMalloc(&ptr, need);
        if (e != cudaSuccess) {
            cudaGetLastError();
            return e == cudaErrorMemoryAllocation ? fail(LLX_ERR_OOM, "cudaMalloc of %zu bytes failed", need)
                                                  : cuda_fail(e, "cudaMalloc");
        }
    } else {
        if (!ptr) return fail(LLX_ERR_INVALID_ARG, "dev_ptr is NULL");
        if (((uintptr_t)ptr & 15) != 0) return fail(LLX_ERR_INVALID_ARG, "dev_ptr must be 16-byte aligned");
        if (bytes < need) return fail(LLX_ERR_INVALID_ARG, "wrapped memory has %zu bytes, pool needs %zu", bytes, need);
        cudaPointerAttributes at;
        LLX_CUDA(cudaPointerGetAttributes(&at, ptr));
        if (at.type != cudaMemoryTypeDevice && at.type != cudaMemoryTypeManaged)
            return fail(LLX_ERR_INVALID_ARG, "dev_ptr is not device memory");
        dev = at.device;
    }
    llx_pool* p = new (std::nothrow) llx_pool();
    if (!p) {
        if (owned) cudaFree(ptr);
        return fail(LLX_ERR_OOM, "host allocation failed");
    }
    p->data = (unsigned char*)ptr;
    p->layers = layers;
    p->kv_heads = kv_heads;
    p->head_dim = head_dim;
    p->block_size = block_size;
    p->num_blocks = num_blocks;
    p->dtype = dtype;
    p->elem_bytes = elem_bytes_of(dtype);
    p->tile_bytes = (long long)block_size * kv_heads * head_dim * p->elem_bytes;
    p->device = dev;
    p->owned = owned;
    build_tensor_map(p);
    *out = p;
    return LLX_OK;
}

}  // namespace

extern "C" {

size_t llx_pool_bytes_for(int layers, int kv_heads, int head_dim, int block_size, llx_dtype dtype, int num_blocks) {
    const int e = elem_bytes_of(dtype);
    if (layers <= 0 || kv_heads <= 0 || head_dim <= 0 || block_size <= 0 || num_blocks <= 0 || e == 0) return 0;
    const unsigned long long tile = (unsigned long long)block_size * kv_heads * head_dim * e;
    if (tile % 16 != 0 || tile > (1ull << 30)) return 0;
    return (size_t)(tile * 2ull * layers * num_blocks);
}

llx_status llx_pool_create(int layers, int kv_heads, int head_dim, int block_size, llx_dtype dtype, int num_blocks,
                           llx_pool** out) {
    return make_pool(nullptr, 0, true, layers, kv_heads, head_dim, block_size, dtype, num_blocks, out);
}
llx_status llx_pool_wrap(void* dev_ptr, size_t bytes, int layers, int kv_heads, int head_dim, int block_size,
                         llx_dtype dtype, int num_blocks, llx_pool** out) {
    return make_pool(dev_ptr, bytes, false, layers, kv_heads, head_dim, block_size, dtype, num_blocks, out);
}
struct IpcHandle {  // LLX_IPC_HANDLE_BYTES: the CUDA handle of the allocation + the pool's geometry
    cudaIpcMemHandle_t mem;
    uint32_t magic;
    int32_t layers, kv_heads, head_dim, block_size, dtype, num_blocks;
    uint32_t checksum;  // FNV-1a over every byte in front of it: a truncated, stale or corrupted handle is refused
};
static_assert(sizeof(IpcHandle) == LLX_IPC_HANDLE_BYTES, "LLX_IPC_HANDLE_BYTES must match IpcHandle");
constexpr uint32_t kIpcMagic = 0x4C4C5832u;  // "LLX2" (round 3: the last word became the checksum)

uint32_t ipc_checksum(const IpcHandle& h) {
    const unsigned char* b = reinterpret_cast<const unsigned char*>(&h);
    uint32_t x = 2166136261u;
    for (size_t i = 0; i < offsetof(IpcHandle, checksum); ++i) x = (x ^ b[i]) * 16777619u;
    return x;
}

// Size of the allocation (or IPC mapping) that contains `ptr`, 0 when the driver cannot say.  cuMemGetAddressRange is
// fetched like cuTensorMapEncodeTiled: libcuda is not linked.
size_t mapped_range_bytes(const void* ptr) {
    typedef CUresult (*RangeFn)(CUdeviceptr*, size_t*, CUdeviceptr);
    static RangeFn fn = [] {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q = cudaDriverEntryPointSymbolNotFound;
        if (cudaGetDriverEntryPoint("cuMemGetAddressRange", &p, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess) {
            cudaGetLastError();
            p = nullptr;
        }
        return (RangeFn)p;
    }();
    if (!fn) return 0;
    CUdeviceptr base = 0;
    size_t size = 0;
    if (fn(&base, &size, (CUdeviceptr)(uintptr_t)ptr) != CUDA_SUCCESS) return 0;
    const size_t skip = (size_t)((uintptr_t)ptr - (uintptr_t)base);
    return size > skip ? size - skip : 0;
}

llx_status llx_pool_ipc_export(const llx_pool* p, void* handle_out) {
    if (!p || !p->data || !handle_out) return fail(LLX_ERR_INVALID_ARG, "NULL argument");
    if (!p->owned) return fail(LLX_ERR_INVALID_ARG, "only a pool allocated by llx_pool_create can be exported (the handle names a whole allocation)");
    IpcHandle h;
    memset(&h, 0, sizeof h);
    LLX_CUDA(cudaIpcGetMemHandle(&h.mem, p->data));
    h.magic = kIpcMagic;
    h.layers = p->layers;
    h.kv_heads = p->kv_heads;
    h.head_dim = p->head_dim;
    h.block_size = p->block_size;
    h.dtype = (int32_t)p->dtype;
    h.num_blocks = p->num_blocks;
    h.checksum = ipc_checksum(h);
    memcpy(handle_out, &h, sizeof h);
    return LLX_OK;
}

llx_status llx_pool_ipc_open(const void* handle, llx_pool** out) {
    if (!out) return fail(LLX_ERR_INVALID_ARG, "out is NULL");
    *out = nullptr;
    if (!handle) return fail(LLX_ERR_INVALID_ARG, "handle is NULL");
    IpcHandle h;
    memcpy(&h, handle, sizeof h);
    if (h.magic != kIpcMagic) return fail(LLX_ERR_INVALID_ARG, "not an llx pool handle");
    if (h.checksum != ipc_checksum(h)) return fail(LLX_ERR_INVALID_ARG, "llx pool handle is corrupted or truncated (checksum mismatch)");
    const size_t need = llx_pool_bytes_for(h.layers, h.kv_heads, h.head_dim, h.block_size, (llx_dtype)h.dtype, h.num_blocks);
    if (need == 0) return fail(LLX_ERR_INVALID_ARG, "handle carries a bad geometry");
    void* ptr = nullptr;
    cudaError_t e = cudaIpcOpenMemHandle(&ptr, h.mem, cudaIpcMemLazyEnablePeerAccess);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return fail(LLX_ERR_CUDA, "cudaIpcOpenMemHandle: %s", cudaGetErrorString(e));
    }
    // The geometry came with the handle; the mapping is what the exporter really allocated.  A handle that names more
    // blocks or layers than that (stale: the exporter re-created its pool; or forged with a matching checksum) would let
    // stages write past the mapping into whatever the other process keeps behind it.
    const size_t mapped = mapped_range_bytes(ptr);
    if (mapped != 0 && mapped < need) {
        cudaIpcCloseMemHandle(ptr);
        return fail(LLX_ERR_INVALID_ARG, "llx pool handle names a pool of %zu bytes but the exporter's allocation has %zu", need, mapped);
    }
    llx_status rc = make_pool(ptr, mapped != 0 ? mapped : need, false, h.layers, h.kv_heads, h.head_dim, h.block_size, (llx_dtype)h.dtype,
                              h.num_blocks, out);
    if (rc != LLX_OK) {
        cudaIpcCloseMemHandle(ptr);
        return rc;
    }
    (*out)->ipc_mapped = true;
    return LLX_OK;
}

llx_status llx_pool_destroy(llx_pool* p) {
    if (!p) return LLX_OK;
    if (p->attn_ws) cudaFree(p->attn_ws);
    if (p->ipc_mapped && p->data) cudaIpcCloseMemHandle(p->data);
    if (p->owned && p->data) cudaFree(p->data);
    delete p;
    return LLX_OK;
}
void* llx_pool_data(const llx_pool* p, int layer, int kv) {
    if (!p || layer < 0 || layer >= p->layers || kv < 0 || kv > 1) return nullptr;
    return p->data + ((long long)layer * 2 + kv) * p->num_blocks * p->tile_bytes;
}
size_t llx_pool_tile_bytes(const llx_pool* p) { return p ? (size_t)p->tile_bytes : 0; }
size_t llx_pool_block_bytes(const llx_pool* p) { return p ? (size_t)p->tile_bytes * 2 * p->layers : 0; }
size_t llx_pool_bytes(const llx_pool* p) { return p ? pool_bytes(p) : 0; }
int llx_pool_num_blocks(const llx_pool* p) { return p ? p->num_blocks : 0; }

static llx_status pool_xfer(const llx_pool* p, int layer, int kv, int first, int nb, void* host, bool up, void* stream) {
    llx_status rc = check_pool(p, "pool");
    if (rc != LLX_OK) return rc;
    if (layer < 0 || layer >= p->layers || kv < 0 || kv > 1) return fail(LLX_ERR_INVALID_ARG, "bad (layer=%d, kv=%d)", layer, kv);
    if (nb < 0 || first < 0 || (long long)first + nb > p->num_blocks)
        return fail(LLX_ERR_BLOCK_OUT_OF_RANGE, "blocks [%d,%d) not in [0,%d)", first, first + nb, p->num_blocks);
    if (nb == 0) return LLX_OK;
    if (!host) return fail(LLX_ERR_INVALID_ARG, "host pointer is NULL");
    unsigned char* d = (unsigned char*)llx_pool_data(p, layer, kv) + (long long)first * p->tile_bytes;
    const size_t bytes = (size_t)nb * p->tile_bytes;
    if (up)
        LLX_CUDA(cudaMemcpyAsync(d, host, bytes, cudaMemcpyHostToDevice, (cudaStream_t)stream));
    else
        LLX_CUDA(cudaMemcpyAsync(host, d, bytes, cudaMemcpyDeviceToHost, (cudaStream_t)stream));
    return LLX_OK;
}
llx_status llx_pool_upload(llx_pool* p, int layer, int kv, int first, int nb, const void* host, void* stream) {
    return pool_xfer(p, layer, kv, first, nb, const_cast<void*>(host), true, stream);
}
llx_status llx_pool_download(const llx_pool* p, int layer, int kv, int first, int nb, void* host, void* stream) {
    return pool_xfer(p, layer, kv, first, nb, host, false, stream);
}
llx_status llx_pool_fill_u16(llx_pool* p, uint16_t pattern, void* stream) {
    llx_status rc = check_pool(p, "pool");
    if (rc != LLX_OK) return rc;
    bool capturing = false;
    if ((rc = stream_capturing((cudaStream_t)stream, &capturing)) != LLX_OK) return rc;
    DevInfo* di = nullptr;
    if ((rc = dev_info(p->device, &di, capturing)) != LLX_OK) return rc;
    const long long nvec = (long long)(pool_bytes(p) / 16);
    const uint32_t w = (uint32_t)pattern | ((uint32_t)pattern << 16);
    llx_fill_u16_kernel<<<di->sm_count * 8, 256, 0, (cudaStream_t)stream>>>((uint4*)p->data, nvec, w);
    LLX_CUDA(cudaGetLastError());
    g_launches++;
    return LLX_OK;
}

llx_status llx_plan_stage(int num_tokens, int blocks_migrated, int block_size, int last_stage_max_blocks, int* n,
                          int* is_final) {
    if (!n || !is_final) return fail(LLX_ERR_INVALID_ARG, "NULL output");
    if (num_tokens < 0 || blocks_migrated < 0 || block_size <= 0 || last_stage_max_blocks < 1)
        return fail(LLX_ERR_INVALID_ARG, "bad arguments (tokens=%d, migrated=%d, S=%d, last=%d)", num_tokens, blocks_migrated, block_size, last_stage_max_blocks);
    const int total = (int)(((long long)num_tokens + block_size - 1) / block_size);
    const int full = num_tokens / block_size;
    if (blocks_migrated > total) return fail(LLX_ERR_INVALID_ARG, "%d blocks migrated, request has %d", blocks_migrated, total);
    const int remaining = total - blocks_migrated;
    if (remaining <= last_stage_max_blocks) {
        *n = remaining;
        *is_final = 1;
    } else {
        *n = full - blocks_migrated;
        *is_final = 0;
    }
    return LLX_OK;
}

llx_status llx_predict_stage_sizes(int n0, double copy_blocks_per_s, double decode_tokens_per_s, int block_size,
                                   int32_t* sizes_out, int cap, int* n_stages) {
    if (!sizes_out || !n_stages) return fail(LLX_ERR_INVALID_ARG, "NULL output");
    *n_stages = 0;
    if (n0 < 1 || block_size <= 0 || cap < 1 || !(copy_blocks_per_s > 0.0) || !(decode_tokens_per_s >= 0.0) ||
        !std::isfinite(copy_blocks_per_s) || !std::isfinite(decode_tokens_per_s))
        return fail(LLX_ERR_INVALID_ARG, "bad arguments (n0=%d, copy=%g blocks/s, decode=%g tokens/s, S=%d, cap=%d)", n0,
                    copy_blocks_per_s, decode_tokens_per_s, block_size, cap);
    int k = 0;
    long long cur = n0;
    sizes_out[k++] = (int32_t)cur;
    while (cur > 1 && k < cap) {
        // stage k lasts cur / c seconds, the request decodes r * cur / c tokens meanwhile = that many / S new blocks
        double nxt = std::ceil((double)cur * decode_tokens_per_s / (copy_blocks_per_s * (double)block_size));
        if (nxt < 1.0) nxt = 1.0;
        if (nxt > 2147483647.0) return fail(LLX_ERR_INVALID_ARG, "stage sizes diverge (decoding outruns the copy)");
        cur = (long long)nxt;
        sizes_out[k++] = (int32_t)cur;
    }
    *n_stages = k;
    return LLX_OK;
}

void llx_launch_opts_init(llx_launch_opts* o) {
    if (!o) return;
    memset(o, 0xFF, sizeof *o);  // every int32 field = -1 = LLX_OPT_DEFAULT
    o->struct_size = (uint32_t)sizeof *o;
}

// LLX_ROUTE_COPY_ENGINE: pool -> pool with one pitched copy-engine transfer per block (2L tiles at the pools' slice
// strides).  No kernel and no SM on either GPU: meant for a destination on another GPU, where the link is the bound.
static llx_status ce_pool_to_pool(const llx_pool* src, const int32_t* src_ids, llx_pool* dst, const int32_t* dst_ids, long long n,
                                  cudaStream_t st) {
    const size_t tile = (size_t)src->tile_bytes, rows = 2 * (size_t)src->layers;
    const size_t sp = (size_t)src->num_blocks * tile, dp = (size_t)dst->num_blocks * tile;
    const bool pitched = pitch_ok(src) && pitch_ok(dst);  // else tile by tile: see pitch_ok
    for (long long i = 0; i < n; ++i) {
        unsigned char* d = dst->data + (size_t)dst_ids[i] * tile;
        const unsigned char* s = src->data + (size_t)src_ids[i] * tile;
        if (pitched) {
            LLX_CUDA(cudaMemcpy2DAsync(d, dp, s, sp, tile, rows, cudaMemcpyDefault, st));
        } else {
            for (size_t r = 0; r < rows; ++r) LLX_CUDA(cudaMemcpyAsync(d + r * dp, s + r * sp, tile, cudaMemcpyDefault, st));
        }
    }
    g_bytes += (unsigned long long)n * rows * tile;
    return LLX_OK;
}

// The copy engines cannot be paced or capped by this library: a budget or CTA cap that silently did nothing would defeat
// its purpose (<= 1 % on the co-running batch), so the combination is refused instead of ignored.
static llx_status ce_route_policy_ok(const Policy& pol) {
    if (pol.budget > 0 || pol.max_ctas > 0)
        return fail(LLX_ERR_INVALID_ARG,
                    "LLX_ROUTE_COPY_ENGINE runs no kernel and cannot honour bandwidth_gbps = %lld / max_ctas = %lld (from this "
                    "call's llx_launch_opts or the process defaults): pace the calls on the host, or use the kernel route",
                    pol.budget, pol.max_ctas);
    return LLX_OK;
}

static llx_status migrate_stage_checked(const Policy& pol, const llx_pool* src, const int32_t* src_ids, llx_pool* dst,
                                        const int32_t* dst_ids, int n, void* stream) {
    llx_status rc = check_pair(src, dst);
    if (rc != LLX_OK) return rc;
    if (n < 0) return fail(LLX_ERR_INVALID_ARG, "n = %d", n);
    if (n == 0) return LLX_OK;
    if (!src_ids || !dst_ids) return fail(LLX_ERR_INVALID_ARG, "block id array is NULL");
    if ((rc = check_range(src_ids, n, src->num_blocks, "src")) != LLX_OK) return rc;
    if ((rc = check_range(dst_ids, n, dst->num_blocks, "dst")) != LLX_OK) return rc;
    if ((rc = check_unique(dst_ids, n, dst->num_blocks)) != LLX_OK) return rc;
    if (pol.route == LLX_ROUTE_COPY_ENGINE) {
        if ((rc = ce_route_policy_ok(pol)) != LLX_OK) return rc;
        return ce_pool_to_pool(src, src_ids, dst, dst_ids, n, (cudaStream_t)stream);
    }
    return launch_copy(pol, pool_side(src, src_ids), pool_side(dst, dst_ids), n, src->layers, src->tile_bytes, src->device,
                       (cudaStream_t)stream);
}

llx_status llx_migrate_stage_ex(const llx_pool* src, const int32_t* src_ids, llx_pool* dst, const int32_t* dst_ids, int n,
                                void* stream, const llx_launch_opts* opts) {
    LLX_TRY
    Policy pol;
    llx_status rc = resolve_policy(opts, &pol);
    if (rc != LLX_OK) return rc;
    return migrate_stage_checked(pol, src, src_ids, dst, dst_ids, n, stream);
    LLX_CATCH
}
llx_status llx_migrate_stage(const llx_pool* src, const int32_t* src_ids, llx_pool* dst, const int32_t* dst_ids, int n,
                             void* stream) {
    return llx_migrate_stage_ex(src, src_ids, dst, dst_ids, n, stream, nullptr);
}

llx_status llx_migrate_stage_wait_ex(const llx_pool* src, const int32_t* src_ids, llx_pool* dst, const int32_t* dst_ids, int n,
                                     void* stream, const llx_launch_opts* opts) {
    LLX_TRY
    Policy pol;
    llx_status rc = resolve_policy(opts, &pol);
    if (rc != LLX_OK) return rc;
    pol.budget = 0;  // the final stage is the downtime: never throttled, whatever the defaults say
    pol.max_ctas = 0;
    pol.overlap = 0;  // and it reads the block the source appended to last: plain stream order
    if (n <= 0 || !src) return migrate_stage_checked(pol, src, src_ids, dst, dst_ids, n, stream);  // nothing to wait for / argument error
    if ((rc = refuse_if_capturing((cudaStream_t)stream, "llx_migrate_stage_wait (a blocking call)")) != LLX_OK) return rc;
    DoneSlot* slot = nullptr;
    if ((rc = done_slot_get(src->device, &slot)) != LLX_OK) return rc;
    DoneReq req;
    req.slot = slot;
    tl_done = &req;
    rc = migrate_stage_checked(pol, src, src_ids, dst, dst_ids, n, stream);
    tl_done = nullptr;
    if (rc != LLX_OK) {
        if (slot) done_slot_put(slot);
        return rc;
    }
    if (!req.armed) {  // no flag on this launch (another kernel was selected, or no free slot)
        if (slot) done_slot_put(slot);
        LLX_CUDA(cudaStreamSynchronize((cudaStream_t)stream));
        return LLX_OK;
    }
    // Spin on the word the kernel's last ring writes.  Every ~1e5 polls the stream is queried: an error there is an
    // asynchronous fault of the copy (the flag will never come); a stream that reports completion has written it.
    const unsigned int want = slot->seq;
    bool seen = false;
    cudaError_t qe = cudaErrorNotReady;
    for (long long i = 0; !seen; ++i) {
        if (*slot->host == want) {
            seen = true;
            break;
        }
        if ((i % 100000) == 99999) {
            qe = cudaStreamQuery((cudaStream_t)stream);
            if (qe != cudaErrorNotReady) break;
        }
#if defined(__x86_64__)
        __builtin_ia32_pause();
#endif
    }
    std::atomic_thread_fence(std::memory_order_acquire);
    if (!seen) {
        // The slot goes back only once the kernel that holds its counter is off the device: released earlier, another
        // waiter's kernel would share the counter and a flag could be written before that copy has landed.
        cudaError_t se = cudaStreamSynchronize((cudaStream_t)stream);
        done_slot_put(slot);
        if (qe != cudaSuccess && qe != cudaErrorNotReady) return cuda_fail(qe, "final-stage copy (asynchronous fault)");
        if (se != cudaSuccess) return cuda_fail(se, "cudaStreamSynchronize");
        return LLX_OK;
    }
    done_slot_put(slot);
    LLX_CUDA(cudaGetLastError());  // a sticky asynchronous fault of this or an earlier launch
    return LLX_OK;
    LLX_CATCH
}
llx_status llx_migrate_stage_wait(const llx_pool* src, const int32_t* src_ids, llx_pool* dst, const int32_t* dst_ids, int n,
                                  void* stream) {
    return llx_migrate_stage_wait_ex(src, src_ids, dst, dst_ids, n, stream, nullptr);
}

llx_status llx_migrate_batch_ex(const llx_pool* src, llx_pool* dst, const int32_t* off, const int32_t* src_ids,
                                const int32_t* dst_ids, int R, void* stream, const llx_launch_opts* opts) {
    LLX_TRY
    Policy pol;
    llx_status rc = resolve_policy(opts, &pol);
    if (rc != LLX_OK) return rc;
    if ((rc = check_pair(src, dst)) != LLX_OK) return rc;
    if (R < 0) return fail(LLX_ERR_INVALID_ARG, "R = %d", R);
    if (R == 0) return LLX_OK;
    if (!off) return fail(LLX_ERR_INVALID_ARG, "req_offsets is NULL");
    if (off[0] != 0) return fail(LLX_ERR_INVALID_ARG, "req_offsets[0] = %d, must be 0", off[0]);
    for (int r = 0; r < R; ++r)
        if (off[r + 1] < off[r]) return fail(LLX_ERR_INVALID_ARG, "req_offsets decreases at request %d", r);
    const long long n = off[R];
    if (n == 0) return LLX_OK;
    if (!src_ids || !dst_ids) return fail(LLX_ERR_INVALID_ARG, "block id array is NULL");
    if ((rc = check_range(src_ids, n, src->num_blocks, "src")) != LLX_OK) return rc;
    if ((rc = check_range(dst_ids, n, dst->num_blocks, "dst")) != LLX_OK) return rc;
    if ((rc = check_unique(dst_ids, n, dst->num_blocks)) != LLX_OK) return rc;
    if (pol.route == LLX_ROUTE_COPY_ENGINE) {
        if ((rc = ce_route_policy_ok(pol)) != LLX_OK) return rc;
        return ce_pool_to_pool(src, src_ids, dst, dst_ids, n, (cudaStream_t)stream);
    }
    // every (block, layer, K|V) tile is independent, so the requests are flattened into one grid
    return launch_copy(pol, pool_side(src, src_ids), pool_side(dst, dst_ids), n, src->layers, src->tile_bytes, src->device,
                       (cudaStream_t)stream);
    LLX_CATCH
}
llx_status llx_migrate_batch(const llx_pool* src, llx_pool* dst, const int32_t* off, const int32_t* src_ids,
                             const int32_t* dst_ids, int R, void* stream) {
    return llx_migrate_batch_ex(src, dst, off, src_ids, dst_ids, R, stream, nullptr);
}

size_t llx_staging_bytes(const llx_pool* p, int n) { return (p && n > 0) ? (size_t)n * llx_pool_block_bytes(p) : 0; }

llx_status llx_staging_alloc_pinned(size_t bytes, void** host_ptr, void** dev_alias) {
    if (!host_ptr || !dev_alias || bytes == 0) return fail(LLX_ERR_INVALID_ARG, "bad arguments");
    void* h = nullptr;
    cudaError_t e = cudaHostAlloc(&h, bytes, cudaHostAllocMapped | cudaHostAllocPortable);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return e == cudaErrorMemoryAllocation ? fail(LLX_ERR_OOM, "cudaHostAlloc of %zu bytes failed", bytes)
                                              : cuda_fail(e, "cudaHostAlloc");
    }
    void* d = nullptr;
    e = cudaHostGetDevicePointer(&d, h, 0);
    if (e != cudaSuccess) {
        cudaFreeHost(h);
        return cuda_fail(e, "cudaHostGetDevicePointer");
    }
    *host_ptr = h;
    *dev_alias = d;
    return LLX_OK;
}
llx_status llx_staging_free_pinned(void* host_ptr) {
    if (!host_ptr) return LLX_OK;
    LLX_CUDA(cudaFreeHost(host_ptr));
    return LLX_OK;
}

llx_status llx_pack_ex(const llx_pool* src, const int32_t* src_ids, int n, void* staging, size_t staging_bytes, void* stream,
                       const llx_launch_opts* opts) {
    LLX_TRY
    Policy pol;
    llx_status rc = resolve_policy(opts, &pol);
    if (rc != LLX_OK) return rc;
    if ((rc = check_pool(src, "src")) != LLX_OK) return rc;
    if (n < 0) return fail(LLX_ERR_INVALID_ARG, "n = %d", n);
    if (n == 0) return LLX_OK;
    if (!src_ids || !staging) return fail(LLX_ERR_INVALID_ARG, "NULL argument");
    if (staging_bytes < llx_staging_bytes(src, n))
        return fail(LLX_ERR_STAGING_TOO_SMALL, "staging has %zu bytes, %d blocks need %zu", staging_bytes, n, llx_staging_bytes(src, n));
    if ((rc = check_range(src_ids, n, src->num_blocks, "src")) != LLX_OK) return rc;
    Side stg;
    if ((rc = staging_side(staging, src->layers, src->tile_bytes, &stg)) != LLX_OK) return rc;
    const unsigned char *a0 = src->data, *a1 = a0 + pool_bytes(src), *b0 = stg.base, *b1 = b0 + llx_staging_bytes(src, n);
    if (a0 < b1 && b0 < a1) return fail(LLX_ERR_ALIAS, "staging buffer overlaps the pool");
    if (stg.host_memory && pol.via_host == 2 && pol.kernel == 0) {
        if ((rc = refuse_if_capturing((cudaStream_t)stream, "llx_pack into pinned host memory")) != LLX_OK) return rc;
        if ((rc = ce_blocks(true, src, src_ids, 0, n, stg, (cudaStream_t)stream)) != LLX_OK) return rc;
        g_bytes += (unsigned long long)llx_staging_bytes(src, n);  // copy-engine transfers count bytes, not launches
        return LLX_OK;
    }
    if (stg.host_memory && (pol.via_host == 0 || pol.via_host == 3) && pol.kernel == 0) {
        pol.overlap = 0;  // a chain of dependent kernels and transfers through one bounce buffer: plain stream order
        return staged_through_bounce(pol, true, src, src_ids, n, stg, (cudaStream_t)stream);
    }
    return launch_copy(pol, pool_side(src, src_ids), stg, n, src->layers, src->tile_bytes, src->device, (cudaStream_t)stream);
    LLX_CATCH
}
llx_status llx_pack(const llx_pool* src, const int32_t* src_ids, int n, void* staging, size_t staging_bytes, void* stream) {
    return llx_pack_ex(src, src_ids, n, staging, staging_bytes, stream, nullptr);
}

llx_status llx_unpack_ex(const void* staging, size_t staging_bytes, llx_pool* dst, const int32_t* dst_ids, int n, void* stream,
                         const llx_launch_opts* opts) {
    LLX_TRY
    Policy pol;
    llx_status rc = resolve_policy(opts, &pol);
    if (rc != LLX_OK) return rc;
    if ((rc = check_pool(dst, "dst")) != LLX_OK) return rc;
    if (n < 0) return fail(LLX_ERR_INVALID_ARG, "n = %d", n);
    if (n == 0) return LLX_OK;
    if (!dst_ids || !staging) return fail(LLX_ERR_INVALID_ARG, "NULL argument");
    if (staging_bytes < llx_staging_bytes(dst, n))
        return fail(LLX_ERR_STAGING_TOO_SMALL, "staging has %zu bytes, %d blocks need %zu", staging_bytes, n, llx_staging_bytes(dst, n));
    if ((rc = check_range(dst_ids, n, dst->num_blocks, "dst")) != LLX_OK) return rc;
    if ((rc = check_unique(dst_ids, n, dst->num_blocks)) != LLX_OK) return rc;
    Side stg;
    if ((rc = staging_side(staging, dst->layers, dst->tile_bytes, &stg)) != LLX_OK) return rc;
    const unsigned char *a0 = dst->data, *a1 = a0 + pool_bytes(dst), *b0 = stg.base, *b1 = b0 + llx_staging_bytes(dst, n);
    if (a0 < b1 && b0 < a1) return fail(LLX_ERR_ALIAS, "staging buffer overlaps the pool");
    if (stg.host_memory && pol.via_host == 2 && pol.kernel == 0) {
        if ((rc = refuse_if_capturing((cudaStream_t)stream, "llx_unpack from pinned host memory")) != LLX_OK) return rc;
        if ((rc = ce_blocks(false, dst, dst_ids, 0, n, stg, (cudaStream_t)stream)) != LLX_OK) return rc;
        g_bytes += (unsigned long long)llx_staging_bytes(dst, n);
        return LLX_OK;
    }
    if (stg.host_memory && (pol.via_host == 0 || pol.via_host == 3) && pol.kernel == 0) {
        pol.overlap = 0;  // see llx_pack_ex
        return staged_through_bounce(pol, false, dst, dst_ids, n, stg, (cudaStream_t)stream);
    }
    return launch_copy(pol, stg, pool_side(dst, dst_ids), n, dst->layers, dst->tile_bytes, dst->device, (cudaStream_t)stream);
    LLX_CATCH
}
llx_status llx_unpack(const void* staging, size_t staging_bytes, llx_pool* dst, const int32_t* dst_ids, int n, void* stream) {
    return llx_unpack_ex(staging, staging_bytes, dst, dst_ids, n, stream, nullptr);
}

llx_status llx_migrate_via_host_ex(const llx_pool* src, const int32_t* src_ids, llx_pool* dst, const int32_t* dst_ids, int n,
                                   void* staging, size_t staging_bytes, int chunk_blocks, void* stream,
                                   const llx_launch_opts* opts) {
    LLX_TRY
    Policy pol;
    llx_status rc = resolve_policy(opts, &pol);
    if (rc != LLX_OK) return rc;
    pol.overlap = 0;  // the scatter of a chunk reads what its gather wrote: the route's own kernels keep plain stream order
    if ((rc = check_pair(src, dst)) != LLX_OK) return rc;
    if (n < 0) return fail(LLX_ERR_INVALID_ARG, "n = %d", n);
    if (n == 0) return LLX_OK;
    if (!src_ids || !dst_ids || !staging) return fail(LLX_ERR_INVALID_ARG, "NULL argument");
    if (staging_bytes < llx_staging_bytes(src, n))
        return fail(LLX_ERR_STAGING_TOO_SMALL, "staging has %zu bytes, %d blocks need %zu", staging_bytes, n, llx_staging_bytes(src, n));
    if ((rc = check_range(src_ids, n, src->num_blocks, "src")) != LLX_OK) return rc;
    if ((rc = check_range(dst_ids, n, dst->num_blocks, "dst")) != LLX_OK) return rc;
    if ((rc = check_unique(dst_ids, n, dst->num_blocks)) != LLX_OK) return rc;
    Side stg;
    if ((rc = staging_side(staging, src->layers, src->tile_bytes, &stg)) != LLX_OK) return rc;
    const unsigned char *b0 = stg.base, *b1 = b0 + llx_staging_bytes(src, n);
    for (const llx_pool* p : {src, (const llx_pool*)dst}) {
        const unsigned char *a0 = p->data, *a1 = a0 + pool_bytes(p);
        if (a0 < b1 && b0 < a1) return fail(LLX_ERR_ALIAS, "staging buffer overlaps a pool");
    }
    cudaStream_t st = (cudaStream_t)stream;
    if ((rc = refuse_if_capturing(st, "llx_migrate_via_host (internal streams, bounce buffers)")) != LLX_OK) return rc;
    const long long block_bytes = 2ll * src->layers * src->tile_bytes;
    // Route.  Pinned-host buffer: gather into a device bounce buffer with the copy kernel, move the chunk over
    // the host link with the copy engines (D2H on one internal stream, H2D on another: the link is full duplex,
    // 2 x 1 GiB in 21.6 ms vs 41 ms one after the other), scatter from a second bounce buffer.  Measured on
    // B200: kernels that address the pinned buffer directly reach 52 GB/s per direction but share ~60 GB/s when
    // both directions run at once, so the zero-copy form (LLX_OPT_VIA_HOST_MODE=1) is kept for comparison only.
    // Device buffer: nothing crosses the link; the two kernels of a chunk simply run on two streams.
    // Pinned-host buffer, both pools on one device: the copy engines gather and scatter by themselves (one pitched copy
    // per block, D2H on one internal stream, H2D on the other) — no kernel, no bounce buffer, and the first H2D starts
    // after 16 MiB instead of 64: 22.9 ms per GiB each way = 93.8 GB/s against 25.3 ms = 84.9 GB/s for the bounce route
    // on the same box (the full-duplex floor of the link is 21.6 ms).  The bounce route stays for a destination on
    // another GPU and as mode 3; zero-copy kernels are mode 1.
    // A pool whose slice stride exceeds the pitch limit (pitch_ok) cannot take pitched transfers: AUTO then keeps the bounce
    // route (85 GB/s; tile-by-tile copy-engine transfers are 2L calls per block); an explicit mode 2 gets tile by tile.
    const bool strided_ce = stg.host_memory && src->device == dst->device &&
                            (pol.via_host == 2 || (pol.via_host == 0 && pol.kernel == 0 && pitch_ok(src) && pitch_ok(dst)));
    const bool bounce = stg.host_memory && !strided_ce && pol.via_host != 1;
    if (strided_ce && chunk_blocks <= 0) {  // small groups: the first host->device copy starts after 16 MiB, not 64
        chunk_blocks = (int)((16ll << 20) / block_bytes);
        if (chunk_blocks < 1) chunk_blocks = 1;
    }
    if (chunk_blocks <= 0) {  // ~64 MiB per chunk (measured best on B200: 24.6 ms per GiB each way; 32 MiB 24.9, 128 MiB 25.5)
        chunk_blocks = (int)((64ll << 20) / block_bytes);
        if (chunk_blocks < 1) chunk_blocks = 1;
    }
    if (chunk_blocks > n) chunk_blocks = n;
    if (chunk_blocks > kIdsByValueCap) chunk_blocks = kIdsByValueCap;

    std::lock_guard<std::mutex> lk(g_pipe_mu);  // the internal streams, events and bounce buffers are shared per device
    Pipe* pipe = nullptr;
    if ((rc = pipe_get(src->device, bounce ? (size_t)chunk_blocks * block_bytes : 0, &pipe)) != LLX_OK) return rc;
    if (pipe->idle_valid) LLX_CUDA(cudaStreamWaitEvent(st, pipe->idle, 0));
    if (strided_ce) {
        // device -> host on one internal stream, host -> device on the other, group by group; `st` only orders the call
        cudaError_t ce2 = cudaSuccess;
        cudaEvent_t start = pipe->take();
        if ((ce2 = cudaEventRecord(start, st)) == cudaSuccess) ce2 = cudaStreamWaitEvent(pipe->d2h, start, 0);
        if (ce2 == cudaSuccess) ce2 = cudaStreamWaitEvent(pipe->h2d, start, 0);
        for (int k = 0; k < n && rc == LLX_OK && ce2 == cudaSuccess; k += chunk_blocks) {
            const int m = (n - k < chunk_blocks) ? n - k : chunk_blocks;
            rc = ce_blocks(true, src, src_ids, k, m, stg, pipe->d2h);
            cudaEvent_t landed = pipe->take();
            if (rc == LLX_OK) ce2 = cudaEventRecord(landed, pipe->d2h);
            if (rc == LLX_OK && ce2 == cudaSuccess) ce2 = cudaStreamWaitEvent(pipe->h2d, landed, 0);
            if (rc == LLX_OK && ce2 == cudaSuccess) rc = ce_blocks(false, dst, dst_ids, k, m, stg, pipe->h2d);
        }
        for (cudaStream_t side : {pipe->d2h, pipe->h2d}) {  // join, also after an error
            cudaEvent_t done = pipe->take();
            if (cudaEventRecord(done, side) == cudaSuccess) cudaStreamWaitEvent(st, done, 0);
        }
        if (cudaEventRecord(pipe->idle, st) == cudaSuccess) pipe->idle_valid = true;
        if (rc != LLX_OK) return rc;
        if (ce2 != cudaSuccess) return cuda_fail(ce2, "llx_migrate_via_host (strided copy-engine route)");
        g_bytes += (unsigned long long)n * (unsigned long long)block_bytes;
        return LLX_OK;
    }
    // Every kernel of this call runs on the source's device (the current one); a destination on a peer GPU is written
    // through its peer mapping.  From here on an error does not return at once: whatever was enqueued on the internal
    // streams is joined into the caller's stream and `idle` is recorded first (the next call reuses the bounce buffers).
    cudaError_t ce = cudaSuccess;
#define LLX_STEP(call) \
    if (rc == LLX_OK && ce == cudaSuccess) ce = (call)
#define LLX_COPY(...) \
    if (rc == LLX_OK && ce == cudaSuccess) rc = launch_copy(__VA_ARGS__)
    cudaEvent_t d2h_done[2] = {nullptr, nullptr};
    int idx = 0;
    for (int k = 0; k < n && rc == LLX_OK && ce == cudaSuccess; k += chunk_blocks, ++idx) {
        const int m = (n - k < chunk_blocks) ? n - k : chunk_blocks;
        const long long off = (long long)k * block_bytes;
        Side part = stg;  // chunk k's slice of the caller's buffer
        part.base = stg.base + off;
        if (!bounce) {
            LLX_COPY(pol, pool_side(src, src_ids + k), part, m, src->layers, src->tile_bytes, src->device, st);
            cudaEvent_t ev = pipe->take();
            LLX_STEP(cudaEventRecord(ev, st));
            LLX_STEP(cudaStreamWaitEvent(pipe->h2d, ev, 0));
            LLX_COPY(pol, part, pool_side(dst, dst_ids + k), m, dst->layers, dst->tile_bytes, src->device, pipe->h2d);
            continue;
        }
        const int slot = idx & 1;
        Side ga = Side{pipe->bounce[slot], nullptr, stg.slice_stride, stg.item_stride, false};
        Side sc = Side{pipe->bounce[2 + slot], nullptr, stg.slice_stride, stg.item_stride, false};
        const size_t bytes = (size_t)m * block_bytes;
        if (d2h_done[slot]) {  // bounce buffer free again
            LLX_STEP(cudaStreamWaitEvent(st, d2h_done[slot], 0));
        }
        LLX_COPY(pol, pool_side(src, src_ids + k), ga, m, src->layers, src->tile_bytes, src->device, st);
        cudaEvent_t packed = pipe->take();
        LLX_STEP(cudaEventRecord(packed, st));
        LLX_STEP(cudaStreamWaitEvent(pipe->d2h, packed, 0));
        LLX_STEP(cudaMemcpyAsync(const_cast<unsigned char*>(part.base), ga.base, bytes, cudaMemcpyDefault, pipe->d2h));
        cudaEvent_t landed = pipe->take();
        LLX_STEP(cudaEventRecord(landed, pipe->d2h));
        d2h_done[slot] = landed;
        LLX_STEP(cudaStreamWaitEvent(pipe->h2d, landed, 0));
        LLX_STEP(cudaMemcpyAsync(const_cast<unsigned char*>(sc.base), part.base, bytes, cudaMemcpyDefault, pipe->h2d));
        LLX_COPY(pol, sc, pool_side(dst, dst_ids + k), m, dst->layers, dst->tile_bytes, src->device, pipe->h2d);
    }
#undef LLX_STEP
#undef LLX_COPY
    // join (also after an error): later work on the caller's stream sees everything this call enqueued
    for (cudaStream_t side : {pipe->d2h, pipe->h2d}) {
        cudaEvent_t done = pipe->take();
        if (cudaEventRecord(done, side) == cudaSuccess) cudaStreamWaitEvent(st, done, 0);
    }
    if (cudaEventRecord(pipe->idle, st) == cudaSuccess) pipe->idle_valid = true;
    if (rc != LLX_OK) return rc;
    if (ce != cudaSuccess) return cuda_fail(ce, "llx_migrate_via_host (stream plumbing)");
    return LLX_OK;
    LLX_CATCH
}
llx_status llx_migrate_via_host(const llx_pool* src, const int32_t* src_ids, llx_pool* dst, const int32_t* dst_ids, int n,
                                void* staging, size_t staging_bytes, int chunk_blocks, void* stream) {
    return llx_migrate_via_host_ex(src, src_ids, dst, dst_ids, n, staging, staging_bytes, chunk_blocks, stream, nullptr);
}

llx_status llx_append_tokens(llx_pool* p, const int32_t* table, int table_len, int t0, int t1, const void* dev_values,
                             void* stream) {
    LLX_TRY
    llx_status rc = check_pool(p, "pool");
    if (rc != LLX_OK) return rc;
    if (t0 < 0 || t1 < t0) return fail(LLX_ERR_INVALID_ARG, "bad token range [%d,%d)", t0, t1);
    if (t1 == t0) return LLX_OK;
    if (!table || !dev_values) return fail(LLX_ERR_INVALID_ARG, "NULL argument");
    if ((t1 - 1) / p->block_size >= table_len) return fail(LLX_ERR_INVALID_ARG, "block table of %d entries too short for token %d", table_len, t1 - 1);
    const int token_bytes = p->kv_heads * p->head_dim * p->elem_bytes;
    if (token_bytes % 16 != 0 || ((uintptr_t)dev_values & 15) != 0) return fail(LLX_ERR_INVALID_ARG, "token vector must be a multiple of 16 bytes and 16-byte aligned");
    const int ntok = t1 - t0;
    std::vector<int32_t> tb((size_t)ntok);
    for (int k = 0; k < ntok; ++k) tb[k] = table[(t0 + k) / p->block_size];
    if ((rc = check_range(tb.data(), ntok, p->num_blocks, "table")) != LLX_OK) return rc;
    AppendArgs a;
    a.pool_base = p->data;
    a.values = (const unsigned char*)dev_values;
    a.tok_block = nullptr;
    a.slice_stride = (long long)p->num_blocks * p->tile_bytes;
    a.tile_bytes = (int)p->tile_bytes;
    a.token_bytes = token_bytes;
    a.block_size = p->block_size;
    a.slices = 2 * p->layers;
    a.t0 = t0;
    a.ntok = ntok;
    static thread_local IdPack pack;
    cudaStream_t st = (cudaStream_t)stream;
    IdSlot* slot = nullptr;
    IdRing& ring = g_ring[p->device];
    std::unique_lock<std::mutex> ring_lk(ring.mu, std::defer_lock);
    const int grid = ntok * a.slices;
    const bool pdl = g_opt_pdl.load() != 0;
    cudaError_t e;
    if (ntok <= kIdsByValueCap) {
        memcpy(pack.src, tb.data(), ntok * sizeof(int32_t));
        e = launch_k(pdl, llx_append_kernel<true>, grid, 128, 0, st, a, pack);
    } else {
        if ((rc = refuse_if_capturing(st, "llx_append_tokens of more than 256 tokens (ids go through a pinned ring)")) != LLX_OK) return rc;
        int32_t* dev_ids = nullptr;
        ring_lk.lock();
        if ((rc = ring_stage(ring, tb.data(), ntok, nullptr, 0, st, &dev_ids, &slot)) != LLX_OK) return rc;
        a.tok_block = dev_ids;
        e = launch_k(pdl, llx_append_kernel<false>, grid, 128, 0, st, a, pack);
    }
    if (e == cudaSuccess) e = cudaGetLastError();
    const llx_status rc_ring = ring_close(slot, st);
    if (e != cudaSuccess) return cuda_fail(e, "append kernel launch");
    if (rc_ring != LLX_OK) return rc_ring;
    g_launches++;
    return LLX_OK;
    LLX_CATCH
}

llx_status llx_decode_attention(const llx_pool* pool, int layer, const void* q, void* out, const int32_t* block_tables,
                                const int32_t* ctx_lens, int B, int max_blocks, float scale, void* stream) {
    llx_status rc = check_pool(pool, "pool");
    if (rc != LLX_OK) return rc;
    if (pool->dtype != LLX_F16) return fail(LLX_ERR_INVALID_ARG, "decode attention needs an fp16 pool");
    if (pool->head_dim != 64 && pool->head_dim != 128) return fail(LLX_ERR_INVALID_ARG, "head_dim %d unsupported (64 or 128)", pool->head_dim);
    if (layer < 0 || layer >= pool->layers) return fail(LLX_ERR_INVALID_ARG, "layer %d not in [0,%d)", layer, pool->layers);
    if (B < 0 || max_blocks < 0) return fail(LLX_ERR_INVALID_ARG, "B = %d, max_blocks = %d", B, max_blocks);
    if (B == 0) return LLX_OK;
    if (!q || !out || !block_tables || !ctx_lens) return fail(LLX_ERR_INVALID_ARG, "NULL argument");
    if ((((uintptr_t)q | (uintptr_t)out) & 15) != 0) return fail(LLX_ERR_INVALID_ARG, "q and out must be 16-byte aligned");
    cudaStream_t st = (cudaStream_t)stream;
    llx_pool* p = const_cast<llx_pool*>(pool);
    {
        bool capturing = false;
        if ((rc = stream_capturing(st, &capturing)) != LLX_OK) return rc;
        DevInfo* di = nullptr;  // first use on this device sets the kernels' attributes (L1 preference)
        if ((rc = dev_info(pool->device, &di, capturing)) != LLX_OK) return rc;
    }

    int split = (int)g_opt_attn_split.load();
    if (split <= 0) split = 256;
    const int D = pool->head_dim, H = pool->kv_heads;
    const long long max_tokens = (long long)max_blocks * pool->block_size;
    int max_splits = (int)((max_tokens + split - 1) / split);
    if (max_splits < 1) max_splits = 1;
    if (max_splits > 65535 || B > 65535) return fail(LLX_ERR_INVALID_ARG, "grid too large");
    const size_t need = (size_t)B * H * max_splits * (D + 4) * sizeof(float);
    if (need > p->attn_ws_bytes) {
        if ((rc = refuse_if_capturing(st, "llx_decode_attention that has to grow its workspace (run the shape once outside the capture)")) != LLX_OK) return rc;
        if (p->attn_ws) {
            LLX_CUDA(cudaDeviceSynchronize());
            cudaFree(p->attn_ws);
            p->attn_ws = nullptr;
            p->attn_ws_bytes = 0;
        }
        cudaError_t e = cudaMalloc(&p->attn_ws, need);
        if (e != cudaSuccess) {
            cudaGetLastError();
            return fail(LLX_ERR_OOM, "attention workspace of %zu bytes", need);
        }
        p->attn_ws_bytes = need;
    }
    AttnArgs a;
    a.k_base = (const unsigned char*)llx_pool_data(pool, layer, 0);
    a.v_base = (const unsigned char*)llx_pool_data(pool, layer, 1);
    a.q = (const __half*)q;
    a.out = (__half*)out;
    a.block_tables = block_tables;
    a.ctx_lens = ctx_lens;
    a.part = p->attn_ws;
    a.tile_bytes = pool->tile_bytes;
    a.H = H;
    a.S = pool->block_size;
    a.max_blocks = max_blocks;
    a.max_splits = max_splits;
    a.split_tokens = split;
    a.scale_log2 = scale * 1.4426950408889634f;
    const int hpw = 32 / (D / 8);
    const int head_groups = (H + kAttnWarps * hpw - 1) / (kAttnWarps * hpw);
    dim3 grid1(max_splits, head_groups, B), grid2(H, B);
    cudaError_t e;
    const bool pdl = g_opt_pdl.load() != 0;
    if (D == 128) {
        e = launch_k(pdl, llx_attn_partial<128>, grid1, kAttnWarps * 32, 0, st, a);
        if (e == cudaSuccess) e = launch_k(pdl, llx_attn_merge<128>, grid2, 128, 0, st, a);
    } else {
        e = launch_k(pdl, llx_attn_partial<64>, grid1, kAttnWarps * 32, 0, st, a);
        if (e == cudaSuccess) e = launch_k(pdl, llx_attn_merge<64>, grid2, 64, 0, st, a);
    }
    if (e != cudaSuccess) return cuda_fail(e, "attention kernel launch");
    LLX_CUDA(cudaGetLastError());
    g_launches += 2;
    return LLX_OK;
}

}  // extern "C"

// ---- llx_decode_attention_static_ws: the split-KV partials in memory that is part of the library image ----------
// For callers that cannot allocate device memory once they are running (llx.h says who and why).  The array below is
// device memory the driver sets aside on every GPU when it loads this library's code there; it stays until the process
// exits.  Nothing in it needs an initial value: llx_attn_partial writes the (acc, m, l) row of every split that has
// tokens and llx_attn_merge reads exactly those rows, so stale rows of an earlier call are never read.
static __device__ __align__(256) unsigned char g_attn_static_ws[LLX_ATTN_STATIC_WS_BYTES];

namespace {
// `g_attn_static_ws` in HOST code is only the handle the runtime registered for the symbol, not an address the GPU can
// use; the device address comes from cudaGetSymbolAddress, per device (every device has its own copy of the array).
std::mutex g_attn_static_mu;
float* g_attn_static_ptr[64] = {};

// `dev` is the current device (check_pool has verified that the pool lives on it).  Allocates nothing.
llx_status attn_static_ws(int dev, float** out) {
    if (dev < 0 || dev >= 64) return fail(LLX_ERR_INVALID_ARG, "device %d unsupported", dev);
    std::lock_guard<std::mutex> lk(g_attn_static_mu);
    if (!g_attn_static_ptr[dev]) {
        void* ptr = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&ptr, g_attn_static_ws);
        if (e != cudaSuccess) return cuda_fail(e, "cudaGetSymbolAddress(static attention workspace)");
        if (!ptr || ((uintptr_t)ptr & 255) != 0) return fail(LLX_ERR_CUDA, "static attention workspace: bad device address %p", ptr);
        g_attn_static_ptr[dev] = (float*)ptr;
    }
    *out = g_attn_static_ptr[dev];
    return LLX_OK;
}
}  // namespace

extern "C" {

llx_status llx_decode_attention_static_ws(const llx_pool* pool, int layer, const void* q, void* out, const int32_t* block_tables,
                                          const int32_t* ctx_lens, int B, int max_blocks, float scale, void* stream) {
    llx_status rc = check_pool(pool, "pool");
    if (rc != LLX_OK) return rc;
    if (pool->dtype != LLX_F16) return fail(LLX_ERR_INVALID_ARG, "decode attention needs an fp16 pool");
    if (pool->head_dim != 64 && pool->head_dim != 128) return fail(LLX_ERR_INVALID_ARG, "head_dim %d unsupported (64 or 128)", pool->head_dim);
    if (layer < 0 || layer >= pool->layers) return fail(LLX_ERR_INVALID_ARG, "layer %d not in [0,%d)", layer, pool->layers);
    if (B < 0 || max_blocks < 0) return fail(LLX_ERR_INVALID_ARG, "B = %d, max_blocks = %d", B, max_blocks);
    if (B == 0) return LLX_OK;
    if (!q || !out || !block_tables || !ctx_lens) return fail(LLX_ERR_INVALID_ARG, "NULL argument");
    if ((((uintptr_t)q | (uintptr_t)out) & 15) != 0) return fail(LLX_ERR_INVALID_ARG, "q and out must be 16-byte aligned");
    cudaStream_t st = (cudaStream_t)stream;

    int split = (int)g_opt_attn_split.load();
    if (split <= 0) split = 256;
    const int D = pool->head_dim, H = pool->kv_heads;
    const long long max_tokens = (long long)max_blocks * pool->block_size;
    long long max_splits = (max_tokens + split - 1) / split;
    if (max_splits < 1) max_splits = 1;
    if (max_splits > 65535 || B > 65535) return fail(LLX_ERR_INVALID_ARG, "grid too large");
    // the size check comes before the address look-up: a shape that does not fit is refused without touching the GPU
    const unsigned long long need = (unsigned long long)B * H * max_splits * (D + 4) * sizeof(float);
    if (need > LLX_ATTN_STATIC_WS_BYTES)
        return fail(LLX_ERR_INVALID_ARG,
                    "llx_decode_attention_static_ws: the partials of B = %d, kv_heads = %d, %lld KV splits of %d tokens need %llu bytes; "
                    "the fixed workspace holds %u (LLX_ATTN_STATIC_WS_BYTES) and this call never allocates: shrink the batch or "
                    "raise LLX_OPT_ATTN_SPLIT_TOKENS, or use llx_decode_attention",
                    B, H, max_splits, split, need, (unsigned)LLX_ATTN_STATIC_WS_BYTES);
    float* ws = nullptr;
    if ((rc = attn_static_ws(pool->device, &ws)) != LLX_OK) return rc;

    AttnArgs a;
    a.k_base = (const unsigned char*)llx_pool_data(pool, layer, 0);
    a.v_base = (const unsigned char*)llx_pool_data(pool, layer, 1);
    a.q = (const __half*)q;
    a.out = (__half*)out;
    a.block_tables = block_tables;
    a.ctx_lens = ctx_lens;
    a.part = ws;
    a.tile_bytes = pool->tile_bytes;
    a.H = H;
    a.S = pool->block_size;
    a.max_blocks = max_blocks;
    a.max_splits = (int)max_splits;
    a.split_tokens = split;
    a.scale_log2 = scale * 1.4426950408889634f;
    const int hpw = 32 / (D / 8);
    const int head_groups = (H + kAttnWarps * hpw - 1) / (kAttnWarps * hpw);
    dim3 grid1((unsigned)max_splits, head_groups, B), grid2(H, B);
    cudaError_t e;
    const bool pdl = g_opt_pdl.load() != 0;
    if (D == 128) {
        e = launch_k(pdl, llx_attn_partial<128>, grid1, kAttnWarps * 32, 0, st, a);
        if (e == cudaSuccess) e = launch_k(pdl, llx_attn_merge<128>, grid2, 128, 0, st, a);
    } else {
        e = launch_k(pdl, llx_attn_partial<64>, grid1, kAttnWarps * 32, 0, st, a);
        if (e == cudaSuccess) e = launch_k(pdl, llx_attn_merge<64>, grid2, 64, 0, st, a);
    }
    if (e != cudaSuccess) return cuda_fail(e, "attention kernel launch");
    LLX_CUDA(cudaGetLastError());
    g_launches += 2;
    return LLX_OK;
}

llx_status llx_set_option(llx_option opt, long long v) {
    if (!opt_valid((int)opt, v)) return fail(LLX_ERR_INVALID_ARG, "option %d: bad value %lld", (int)opt, v);
    switch (opt) {
        case LLX_OPT_COPY_KERNEL: g_opt_kernel = v; break;
        case LLX_OPT_MAX_CTAS: g_opt_max_ctas = v; break;
        case LLX_OPT_CHUNK_BYTES: g_opt_chunk = v; break;
        case LLX_OPT_RING_STAGES: g_opt_stages = v; break;
        case LLX_OPT_IDS_BY_VALUE_MAX: g_opt_byval = v; break;
        case LLX_OPT_ATTN_SPLIT_TOKENS: g_opt_attn_split = v; break;
        case LLX_OPT_UNIT_ORDER: g_opt_order = v; break;
        case LLX_OPT_L2_HINT: g_opt_l2hint = v; break;
        case LLX_OPT_RINGS_PER_CTA: g_opt_rings = v; break;
        case LLX_OPT_PDL: g_opt_pdl = v; break;
        case LLX_OPT_BANDWIDTH_GBPS: g_opt_budget = v; break;
        case LLX_OPT_VIA_HOST_MODE: g_opt_via_host = v; break;
        case LLX_OPT_DYNAMIC_TAIL_PCT: g_opt_dyn_pct = v; break;
        case LLX_OPT_DYNAMIC_TAIL_BATCH: g_opt_dyn_batch = v; break;
        case LLX_OPT_EXACT_RESIDENCY: g_opt_smem_pad = v; break;
        case LLX_OPT_COPY_SMEM_CARVEOUT_PCT: g_opt_carveout = v; break;  // applied to the kernel at the next copy launch
        case LLX_OPT_PACED_SLICE_US: g_opt_slice_us = v; break;
        case LLX_OPT_OVERLAP_PREV: g_opt_overlap = v; break;
    }
    return LLX_OK;
}
long long llx_get_option(llx_option opt) {
    switch (opt) {
        case LLX_OPT_COPY_KERNEL: return g_opt_kernel;
        case LLX_OPT_MAX_CTAS: return g_opt_max_ctas;
        case LLX_OPT_CHUNK_BYTES: return g_opt_chunk;
        case LLX_OPT_RING_STAGES: return g_opt_stages;
        case LLX_OPT_IDS_BY_VALUE_MAX: return g_opt_byval;
        case LLX_OPT_ATTN_SPLIT_TOKENS: return g_opt_attn_split;
        case LLX_OPT_UNIT_ORDER: return g_opt_order;
        case LLX_OPT_L2_HINT: return g_opt_l2hint;
        case LLX_OPT_RINGS_PER_CTA: return g_opt_rings;
        case LLX_OPT_PDL: return g_opt_pdl;
        case LLX_OPT_BANDWIDTH_GBPS: return g_opt_budget;
        case LLX_OPT_VIA_HOST_MODE: return g_opt_via_host;
        case LLX_OPT_DYNAMIC_TAIL_PCT: return g_opt_dyn_pct;
        case LLX_OPT_DYNAMIC_TAIL_BATCH: return g_opt_dyn_batch;
        case LLX_OPT_EXACT_RESIDENCY: return g_opt_smem_pad;
        case LLX_OPT_COPY_SMEM_CARVEOUT_PCT: return g_opt_carveout;
        case LLX_OPT_PACED_SLICE_US: return g_opt_slice_us;
        case LLX_OPT_OVERLAP_PREV: return g_opt_overlap;
    }
    return -1;
}

void llx_get_counters(llx_counters* out) {
    if (!out) return;
    out->kernel_launches = g_launches;
    out->copy_launches = g_copy_launches;
    out->bytes_moved = g_bytes;
    out->id_uploads = g_id_uploads;
}
void llx_reset_counters(void) {
    g_launches = 0;
    g_copy_launches = 0;
    g_bytes = 0;
    g_id_uploads = 0;
}

llx_status llx_synchronize(void* stream) {
    llx_status rc = refuse_if_capturing((cudaStream_t)stream, "llx_synchronize");
    if (rc != LLX_OK) return rc;
    LLX_CUDA(cudaStreamSynchronize((cudaStream_t)stream));
    return LLX_OK;
}

const char* llx_status_str(llx_status s) {
    switch (s) {
        case LLX_OK: return "LLX_OK";
        case LLX_ERR_INVALID_ARG: return "LLX_ERR_INVALID_ARG";
        case LLX_ERR_GEOMETRY_MISMATCH: return "LLX_ERR_GEOMETRY_MISMATCH";
        case LLX_ERR_BLOCK_OUT_OF_RANGE: return "LLX_ERR_BLOCK_OUT_OF_RANGE";
        case LLX_ERR_DUPLICATE_DST: return "LLX_ERR_DUPLICATE_DST";
        case LLX_ERR_ALIAS: return "LLX_ERR_ALIAS";
        case LLX_ERR_STAGING_TOO_SMALL: return "LLX_ERR_STAGING_TOO_SMALL";
        case LLX_ERR_OOM: return "LLX_ERR_OOM";
        case LLX_ERR_CUDA: return "LLX_ERR_CUDA";
        case LLX_ERR_NO_SPACE: return "LLX_ERR_NO_SPACE";
        case LLX_ERR_STATE: return "LLX_ERR_STATE";
    }
    return "LLX_ERR_UNKNOWN";
}
const char* llx_last_error(void) { return g_err; }
const char* llx_version(void) { return "llx 0.2 (sm_100a)"; }

}  // extern "C"
