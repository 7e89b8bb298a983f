// Gather/scatter copy kernels for sm_100a: the data path of one migration stage
// (§4.2; block = K or V of block_size tokens of one layer, §5).
//
// One work UNIT = one chunk (<= chunk_bytes) of one tile (block i, layer l, K|V).  Both sides
// of a copy are addressed with the same affine form
//
//     addr(side, i, slice, c) = base + slice*slice_stride + item(side,i)*item_stride + c*chunk_bytes
//
// where slice = l*2+kv and item = ids[i] for a paged pool (slice_stride = num_blocks*tile_bytes,
// item_stride = tile_bytes) or item = i for the contiguous fusion buffer of PAPER.md:237
// (slice_stride = tile_bytes, item_stride = 2*layers*tile_bytes).  migrate = pool->pool,
// pack = pool->buffer, unpack = buffer->pool: one kernel body serves S3, S4, S5 and S6.
//
// Three implementations, selected by the host (LLX_OPT_COPY_KERNEL):
//   llx_copy_vec16 : 256-thread CTAs, 16-byte LDG/STG, UNROLL independent loads in flight per
//                    thread before the first store; lane 0 fetches the pair's block ids and
//                    broadcasts them with __shfl_sync.
//   llx_copy_bulk  : one elected thread per warp drives a ring of shared-memory stages with the
//                    bulk async-copy engine (cp.async.bulk global->shared completing on an
//                    mbarrier, shared->global in bulk groups): no registers or LSU issue slots
//                    per byte, up to 32 KiB per instruction.
//   llx_copy_tma   : the same ring, fed by 4-D tensor-map boxes (cp.async.bulk.tensor): one instruction moves
//                    the tiles of one block in several (layer, K|V) slices — for pools whose tiles are small.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace llx {

constexpr int kIdsByValueCap = 256;

struct IdPack {  // block ids carried in the kernel parameters (constant bank) for short stages
    int32_t src[kIdsByValueCap];
    int32_t dst[kIdsByValueCap];
};

struct CopyArgs {
    const unsigned char* src_base;
    unsigned char* dst_base;
    long long src_slice_stride, src_item_stride;
    long long dst_slice_stride, dst_item_stride;
    const int32_t* src_ids;  // device; nullptr => item = i (contiguous side) or ids by value
    const int32_t* dst_ids;
    int src_indexed, dst_indexed;  // 1 => item = ids[i], 0 => item = i
    int tile_bytes;
    int chunk_bytes;
    int chunks_per_tile;
    int slices;       // 2*layers
    int total_units;  // n * slices * chunks_per_tile (the register-staged kernel: END of this launch's unit range)
    int unit_begin;   // register-staged kernel: this launch handles units [unit_begin, total_units) — a budgeted stage is
                      // issued as a chain of short launches (see launch_copy); the bulk kernel always gets 0
    int blocked_order;  // 0: worker w takes units w, w+W, ...; 1: worker w takes a contiguous range
    int l2_hint;        // bit0: loads L2::evict_first, bit1: stores L2::evict_first (bulk kernel)
    int pace_ns;        // bulk kernel: minimum time between two chunks of one ring (0 = unthrottled)
    int tma_k;          // tensor-map kernel: (layer, K|V) slices one 4-D box covers; there a unit = (pair, group of tma_k slices),
                        // slices = groups per block, chunks_per_tile = 1, chunk_bytes = tile_bytes = tma_k * the pool's tile
    int defer_wait;     // bulk kernel, LLX_OPT_OVERLAP_PREV: the copy is independent of the previous kernel of its stream, so
                        // griddepcontrol.wait moves from the prologue to just before the first dynamic claim / the exit
    // bulk kernel, blocked order: the last dyn_units units are not pre-assigned; rings that finish their
    // contiguous range early claim them in batches of dyn_batch from *dyn_counter (evens out the tail)
    int dyn_units, dyn_batch;
    unsigned int dyn_claims;    // claims this launch makes in total (batches + one failed claim per ring): the last one resets the counter
    unsigned int* dyn_counter;  // device, zero before the launch
    // completion flag (llx_migrate_stage_wait): the ring that finishes last writes done_value to *done_flag
    // (mapped pinned host memory) so that the host can spin on a word instead of going through the driver
    unsigned int* done_counter;  // device, zero before the launch; nullptr = no flag
    volatile unsigned int* done_flag;
    unsigned int done_value, done_rings;
};

__device__ __forceinline__ uint4 ld_stream16(const void* p) {
    uint4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
                 : "l"(p));
    return r;
}
__device__ __forceinline__ void st_stream16(void* p, const uint4& v) {
    asm volatile("st.global.L1::no_allocate.v4.u32 [%0], {%1,%2,%3,%4};" ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z),
                 "r"(v.w)
                 : "memory");
}

// Programmatic dependent launch: let the next kernel of the stream start its prologue now, and
// wait for the previous kernel's memory before touching global memory.  No-ops without the attribute.
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait_prior_grids() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

__device__ __forceinline__ unsigned long long global_timer_ns() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}

struct UnitAddr {
    const unsigned char* src;
    unsigned char* dst;
    int len;
};

// Decode unit u -> (i, slice, c) and form both addresses.  id_s/id_d are the items of pair i.
__device__ __forceinline__ void unit_coords(const CopyArgs& a, int u, int& i, int& slice, int& c) {
    c = u % a.chunks_per_tile;
    int t = u / a.chunks_per_tile;
    slice = t % a.slices;
    i = t / a.slices;
}
__device__ __forceinline__ UnitAddr unit_addr(const CopyArgs& a, int slice, int c, int item_s, int item_d) {
    UnitAddr r;
    long long off = (long long)c * a.chunk_bytes;
    r.src = a.src_base + slice * a.src_slice_stride + item_s * a.src_item_stride + off;
    r.dst = a.dst_base + slice * a.dst_slice_stride + item_d * a.dst_item_stride + off;
    int rem = a.tile_bytes - c * a.chunk_bytes;
    r.len = rem < a.chunk_bytes ? rem : a.chunk_bytes;
    return r;
}

// ------------------------------------------------------------------------------------------
// 16-byte vector kernel.  Persistent-style grid: CTA b handles units b, b+grid, b+2*grid, ...
// ------------------------------------------------------------------------------------------
template <bool BYVAL, int UNROLL>
__global__ void __launch_bounds__(256, 8) llx_copy_vec16(const CopyArgs a, const __grid_constant__ IdPack ids) {
    const int lane = threadIdx.x & 31;
    const int nt = blockDim.x;
    pdl_wait_prior_grids();   // wait first, then let dependents launch: see ring_copy
    pdl_launch_dependents();
    unsigned long long deadline = a.pace_ns > 0 ? global_timer_ns() : 0ull;
    int u_begin = a.unit_begin + blockIdx.x, u_end = a.total_units, u_step = gridDim.x;
    if (a.blocked_order) {
        const long long span = a.total_units - a.unit_begin;
        u_begin = a.unit_begin + (int)((long long)blockIdx.x * span / gridDim.x);
        u_end = a.unit_begin + (int)((long long)(blockIdx.x + 1) * span / gridDim.x);
        u_step = 1;
    }
    for (int u = u_begin; u < u_end; u += u_step) {
        int i, slice, c;
        unit_coords(a, u, i, slice, c);
        int item_s = i, item_d = i;
        if (BYVAL) {
            if (a.src_indexed) item_s = ids.src[i];
            if (a.dst_indexed) item_d = ids.dst[i];
        } else {
            // warp-level index broadcast: one lane reads the pair's ids, the warp shares them
            int vs = 0, vd = 0;
            if (lane == 0) {
                if (a.src_indexed) vs = __ldg(a.src_ids + i);
                if (a.dst_indexed) vd = __ldg(a.dst_ids + i);
            }
            vs = __shfl_sync(0xffffffffu, vs, 0);
            vd = __shfl_sync(0xffffffffu, vd, 0);
            if (a.src_indexed) item_s = vs;
            if (a.dst_indexed) item_d = vd;
        }
        const UnitAddr ua = unit_addr(a, slice, c, item_s, item_d);
        const int nvec = ua.len >> 4;
        const uint4* __restrict__ s = reinterpret_cast<const uint4*>(ua.src);
        uint4* __restrict__ d = reinterpret_cast<uint4*>(ua.dst);
        for (int v0 = threadIdx.x; v0 < nvec; v0 += nt * UNROLL) {
            uint4 r[UNROLL];
#pragma unroll
            for (int j = 0; j < UNROLL; ++j) {
                int v = v0 + j * nt;
                if (v < nvec) r[j] = ld_stream16(s + v);
            }
#pragma unroll
            for (int j = 0; j < UNROLL; ++j) {
                int v = v0 + j * nt;
                if (v < nvec) st_stream16(d + v, r[j]);
            }
        }
        if (a.pace_ns > 0) {  // bandwidth budget: the CTA starts its next chunk only at its next deadline
            deadline += (unsigned long long)a.pace_ns;
            unsigned long long now = global_timer_ns();
            while (now < deadline) {
                const unsigned long long left = deadline - now;
                __nanosleep(left > 2000 ? 2000u : (unsigned)left);
                now = global_timer_ns();
            }
        }
    }
}

// ------------------------------------------------------------------------------------------
// Bulk async-copy (TMA, non-tensor form) ring kernel.
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "LLX_WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra LLX_DONE_%=;\n"
        "bra LLX_WAIT_%=;\n"
        "LLX_DONE_%=:\n"
        "}\n" ::"r"(bar),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst_smem, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     dst_smem),
                 "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}
__device__ __forceinline__ void bulk_s2g(void* dst, uint32_t src_smem, uint32_t bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(src_smem), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ uint64_t policy_evict_first() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ void bulk_g2s_hint(uint32_t dst_smem, const void* src, uint32_t bytes, uint32_t bar, uint64_t pol) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(
            dst_smem),
        "l"(src), "r"(bytes), "r"(bar), "l"(pol)
        : "memory");
}
__device__ __forceinline__ void bulk_s2g_hint(void* dst, uint32_t src_smem, uint32_t bytes, uint64_t pol) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group.L2::cache_hint [%0], [%1], %2, %3;" ::"l"(dst),
                 "r"(src_smem), "r"(bytes), "l"(pol)
                 : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void bulk_wait_read() {
    asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory");
}
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }

// Shared memory: [rings_per_cta][nstages] mbarriers (8 B each) and [rings_per_cta][nstages] unit numbers (4 B each),
// padded to 128 B, then [rings_per_cta][nstages][chunk_bytes] data.  Lane 0 of each warp is the ring's only
// working thread.  Striped order: ring r handles units r, r+nrings, ...  Blocked order: ring r streams the
// contiguous range [r*Ts/W, (r+1)*Ts/W) of the first Ts = total - dyn_units units, then claims batches of the rest.
//
// The ring is the same for both ways of moving a unit; a Mover supplies them:
//   BulkMover   : one 1-D bulk copy per unit (a chunk of one tile), any tile size that is a multiple of 16 bytes;
//   TensorMover : one 4-D tensor-map box per unit = the tiles of ONE block in tma_k consecutive (layer, K|V) slices
//                 (cp.async.bulk.tensor.4d, SASS UTMALDG / UTMASTG): small tiles travel tma_k at a time.
struct BulkMover {
    uint64_t pol;
    bool hint_ld, hint_st;
    __device__ __forceinline__ void load(const CopyArgs&, const UnitAddr& ua, int, int, uint32_t dst_smem, uint32_t bar) const {
        if (hint_ld)
            bulk_g2s_hint(dst_smem, ua.src, (uint32_t)ua.len, bar, pol);
        else
            bulk_g2s(dst_smem, ua.src, (uint32_t)ua.len, bar);
    }
    __device__ __forceinline__ void store(const CopyArgs&, const UnitAddr& ua, int, int, uint32_t src_smem) const {
        if (hint_st)
            bulk_s2g_hint(ua.dst, src_smem, (uint32_t)ua.len, pol);
        else
            bulk_s2g(ua.dst, src_smem, (uint32_t)ua.len);
    }
};
struct TensorMover {
    const void* src_map;  // CUtensorMap in the kernel parameters (__grid_constant__)
    const void* dst_map;
    __device__ __forceinline__ void load(const CopyArgs& a, const UnitAddr&, int item, int group, uint32_t dst_smem, uint32_t bar) const {
        asm volatile(
            "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];" ::"r"(dst_smem),
            "l"(src_map), "r"(0), "r"(0), "r"(item), "r"(group * a.tma_k), "r"(bar)
            : "memory");
    }
    __device__ __forceinline__ void store(const CopyArgs& a, const UnitAddr&, int item, int group, uint32_t src_smem) const {
        asm volatile("cp.async.bulk.tensor.4d.global.shared::cta.tile.bulk_group [%0, {%1, %2, %3, %4}], [%5];" ::"l"(dst_map), "r"(0),
                     "r"(0), "r"(item), "r"(group * a.tma_k), "r"(src_smem)
                     : "memory");
    }
};

template <bool BYVAL, class Mover>
__device__ __forceinline__ void ring_copy(const CopyArgs& a, const IdPack& ids, int nstages, const Mover mover) {
    extern __shared__ __align__(128) unsigned char smem[];
    const int warp = threadIdx.x >> 5;
    const int rings_per_cta = blockDim.x >> 5;
    if ((threadIdx.x & 31) != 0) return;

    const int bar_bytes = ((rings_per_cta * nstages * 12) + 127) & ~127;
    const uint32_t bar0 = smem_u32(smem) + warp * nstages * 8;
    int* unit_of = reinterpret_cast<int*>(smem + rings_per_cta * nstages * 8) + warp * nstages;
    const uint32_t buf0 = smem_u32(smem) + bar_bytes + warp * nstages * a.chunk_bytes;

    for (int s = 0; s < nstages; ++s) mbar_init(bar0 + s * 8, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    // A copy the caller declared independent of the previous kernel (stages of disjoint blocks) starts
    // streaming as soon as its CTA is resident, i.e. while the previous stage's slowest rings are still draining.  The
    // wait is only deferred, never dropped: (1) a ring executes it before its first claim from the dynamic-tail counter,
    // which the previous launch shares and resets with its last claim; (2) every ring executes it before it exits, so
    // "this kernel has completed" still implies "everything before it on the stream has completed" (completion stays
    // transitive although the start is not ordered).
    // Every llx kernel that does NOT defer lets its dependents launch only AFTER its own wait has returned: when a kernel
    // behind it starts, everything in front of it has completed.  A launch without overlap_prev is thus a fence for the
    // start of whatever follows, and a deferred copy can only ever run next to the launches back to (and including) the
    // last such launch — the set llx.h asks the caller to declare it independent of.
    bool waited = a.defer_wait == 0;
    if (waited) pdl_wait_prior_grids();
    pdl_launch_dependents();

    const int ring = blockIdx.x * rings_per_cta + warp;
    const int nrings = gridDim.x * rings_per_cta;
    // the ring's unit stream: a pre-assigned arithmetic sequence, then (blocked order only) claimed batches
    int s_next, s_end, s_step;
    const int static_units = a.total_units - a.dyn_units;
    if (a.blocked_order) {
        s_next = (int)((long long)ring * static_units / nrings);
        s_end = (int)((long long)(ring + 1) * static_units / nrings);
        s_step = 1;
    } else {
        s_next = ring;
        s_end = a.total_units;
        s_step = nrings;
    }
    int d_next = 0, d_end = 0;
    bool dyn_done = a.dyn_units == 0;
    auto next_unit = [&]() -> int {
        if (s_next < s_end) {
            const int u = s_next;
            s_next += s_step;
            return u;
        }
        if (d_next < d_end) return d_next++;
        if (dyn_done) return -1;
        if (!waited) {
            pdl_wait_prior_grids();
            waited = true;
        }
        const unsigned int b = atomicAdd(a.dyn_counter, 1u);
        if (b == a.dyn_claims - 1) *a.dyn_counter = 0;  // every ring fails exactly once: this was the launch's last claim
        const long long lo = (long long)b * a.dyn_batch;
        if (lo >= a.dyn_units) {
            dyn_done = true;
            return -1;
        }
        d_next = static_units + (int)lo;
        d_end = d_next + a.dyn_batch < a.total_units ? d_next + a.dyn_batch : a.total_units;
        return d_next++;
    };
    unsigned long long deadline = a.pace_ns > 0 ? global_timer_ns() : 0ull;

    // unit u -> both addresses (1-D mover) and (item, slice) on both sides (tensor mover)
    auto addr_of = [&](int u, int& item_s, int& item_d, int& slice) -> UnitAddr {
        int i, c;
        unit_coords(a, u, i, slice, c);
        item_s = item_d = i;
        if (a.src_indexed) item_s = BYVAL ? ids.src[i] : __ldg(a.src_ids + i);
        if (a.dst_indexed) item_d = BYVAL ? ids.dst[i] : __ldg(a.dst_ids + i);
        return unit_addr(a, slice, c, item_s, item_d);
    };
    auto issue_load = [&](int s, int u) {
        unit_of[s] = u;
        int item_s, item_d, slice;
        UnitAddr ua = addr_of(u, item_s, item_d, slice);
        mbar_expect_tx(bar0 + s * 8, (uint32_t)ua.len);
        mover.load(a, ua, item_s, slice, buf0 + s * a.chunk_bytes, bar0 + s * 8);
    };

    int issued = 0;
    for (; issued < nstages; ++issued) {
        const int u = next_unit();
        if (u < 0) break;
        issue_load(issued, u);
    }
    for (int k = 0; k < issued; ++k) {
        const int s = k % nstages;
        mbar_wait(bar0 + s * 8, (uint32_t)((k / nstages) & 1));
        int item_s, item_d, slice;
        UnitAddr ua = addr_of(unit_of[s], item_s, item_d, slice);
        mover.store(a, ua, item_d, slice, buf0 + s * a.chunk_bytes);
        bulk_commit();
        if (a.pace_ns > 0) {  // bandwidth budget: this ring may start its next chunk only at its next deadline
            deadline += (unsigned long long)a.pace_ns;
            unsigned long long now = global_timer_ns();
            while (now < deadline) {
                const unsigned long long left = deadline - now;
                __nanosleep(left > 2000 ? 2000u : (unsigned)left);
                now = global_timer_ns();
            }
        }
        // refill the stage whose store was committed one iteration ago: allowing the newest
        // group to stay pending keeps one store and nstages-1 loads in flight per ring
        if (k >= 1 && issued == k - 1 + nstages) {
            const int u = next_unit();
            if (u >= 0) {
                bulk_wait_read<1>();
                issue_load((k - 1) % nstages, u);
                ++issued;
            }
        }
    }
    bulk_wait_all();  // this ring's stores are complete
    if (!waited) pdl_wait_prior_grids();
    if (a.done_counter) {
        __threadfence();
        if (atomicAdd(a.done_counter, 1u) == a.done_rings - 1) {  // every ring has finished its stores
            *a.done_counter = 0;
            __threadfence_system();
            *a.done_flag = a.done_value;
        }
    }
}

template <bool BYVAL>
__global__ void llx_copy_bulk(const CopyArgs a, const __grid_constant__ IdPack ids, int nstages) {
    BulkMover m;
    m.pol = policy_evict_first();
    m.hint_ld = a.l2_hint & 1;
    m.hint_st = a.l2_hint & 2;
    ring_copy<BYVAL>(a, ids, nstages, m);
}

// 128 opaque bytes with the alignment the TMA unit needs: a CUtensorMap, declared here without the driver header
struct alignas(64) TensorMap {
    unsigned long long opaque[16];
};
template <bool BYVAL>
__global__ void llx_copy_tma(const CopyArgs a, const __grid_constant__ IdPack ids, int nstages,
                             const __grid_constant__ TensorMap src_map, const __grid_constant__ TensorMap dst_map) {
    TensorMover m;
    m.src_map = &src_map;
    m.dst_map = &dst_map;
    ring_copy<BYVAL>(a, ids, nstages, m);
}

// ------------------------------------------------------------------------------------------
// S8 append: values[t][l][kv][token_bytes] -> pool[l][kv][blk(t)][slot(t)]
// One CTA per (token, layer, kv).  tok_block = block id of each token (by value or device).
// ------------------------------------------------------------------------------------------
struct AppendArgs {
    unsigned char* pool_base;
    const unsigned char* values;
    const int32_t* tok_block;  // device, or nullptr when by value
    long long slice_stride;    // num_blocks*tile_bytes
    int tile_bytes, token_bytes, block_size, slices, t0, ntok;
};
template <bool BYVAL>
__global__ void __launch_bounds__(128) llx_append_kernel(const AppendArgs a, const __grid_constant__ IdPack ids) {
    pdl_wait_prior_grids();   // wait first, then let dependents launch: see ring_copy
    pdl_launch_dependents();
    const int u = blockIdx.x;  // (tok, slice)
    const int slice = u % a.slices;
    const int k = u / a.slices;
    const int blk = BYVAL ? ids.src[k] : __ldg(a.tok_block + k);
    const int slot = (a.t0 + k) % a.block_size;
    const uint4* s = reinterpret_cast<const uint4*>(a.values + ((long long)k * a.slices + slice) * a.token_bytes);
    uint4* d = reinterpret_cast<uint4*>(a.pool_base + slice * a.slice_stride + (long long)blk * a.tile_bytes +
                                        (long long)slot * a.token_bytes);
    const int nvec = a.token_bytes >> 4;
    for (int v0 = threadIdx.x; v0 < nvec; v0 += 128 * 4) {  // 4 independent 16-byte loads in flight per thread
        uint4 r[4];
#pragma unroll
        for (int j = 0; j < 4; ++j)
            if (v0 + j * 128 < nvec) r[j] = ld_stream16(s + v0 + j * 128);
#pragma unroll
        for (int j = 0; j < 4; ++j)
            if (v0 + j * 128 < nvec) d[v0 + j * 128] = r[j];
    }
}

__global__ void __launch_bounds__(256) llx_fill_u16_kernel(uint4* p, long long nvec, uint32_t word) {
    const uint4 v = make_uint4(word, word, word, word);
    for (long long i = blockIdx.x * 256ll + threadIdx.x; i < nvec; i += (long long)gridDim.x * 256) p[i] = v;
}

}  // namespace llx
