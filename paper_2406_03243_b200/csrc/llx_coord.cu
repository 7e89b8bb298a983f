// Host-side coordination around the copy path: an instance's block manager and the
// migration handshake of Llumnix §4.2 (Figure 7).  No device code here; the only CUDA
// work a session causes is the llx_migrate_stage it enqueues for each stage.
//
//   PRE-ALLOC before each stage ("issues a pre-allocate request with the number of blocks")
//   proceed | abort from the destination ("try to allocate and reserve the blocks")
//   the source's check after each stage ("has completed or been preempted")
//   abort when the other side fails
//   release on the source + commit on the destination after the final stage
#include <cstring>
#include <new>
#include <vector>

#include "llx_internal.h"

using llx::fail;

// ---- block manager: a stack of free ids (A23) ---------------------------------------------
struct llx_blockmgr {
    int num_blocks = 0;
    std::vector<int32_t> free_stack;     // back() is handed out next
    std::vector<unsigned char> is_free;  // per id
};

struct llx_migration {
    const llx_pool* src = nullptr;
    llx_pool* dst = nullptr;
    llx_blockmgr* src_mgr = nullptr;
    llx_blockmgr* dst_mgr = nullptr;
    int block_size = 0, last_stage_max_blocks = 0;
    llx_mig_state state = LLX_MIG_READY;
    llx_abort_reason reason = LLX_ABORT_NONE;
    int blocks_migrated = 0, stages = 0;
    std::vector<int32_t> dst_table;  // blocks reserved on the destination so far, in logical order
    bool has_opts = false;           // launch policy of the non-final stages (llx_migration_set_stage_opts)
    llx_launch_opts stage_opts;
};

extern "C" {

llx_status llx_blockmgr_create(int num_blocks, llx_blockmgr** out) {
    if (!out) return fail(LLX_ERR_INVALID_ARG, "out is NULL");
    *out = nullptr;
    if (num_blocks <= 0) return fail(LLX_ERR_INVALID_ARG, "num_blocks = %d", num_blocks);
    llx_blockmgr* m = new (std::nothrow) llx_blockmgr();
    if (!m) return fail(LLX_ERR_OOM, "host allocation failed");
    try {
        m->num_blocks = num_blocks;
        m->free_stack.resize((size_t)num_blocks);
        for (int i = 0; i < num_blocks; ++i) m->free_stack[(size_t)i] = num_blocks - 1 - i;  // pops give 0, 1, 2, ...
        m->is_free.assign((size_t)num_blocks, 1);
    } catch (...) {
        delete m;
        return fail(LLX_ERR_OOM, "host allocation failed");
    }
    *out = m;
    return LLX_OK;
}

llx_status llx_blockmgr_destroy(llx_blockmgr* m) {
    delete m;
    return LLX_OK;
}

int llx_blockmgr_num_free(const llx_blockmgr* m) { return m ? (int)m->free_stack.size() : -1; }
int llx_blockmgr_num_blocks(const llx_blockmgr* m) { return m ? m->num_blocks : -1; }

llx_status llx_blockmgr_alloc(llx_blockmgr* m, int n, int32_t* ids_out) {
    if (!m) return fail(LLX_ERR_INVALID_ARG, "block manager is NULL");
    if (n < 0) return fail(LLX_ERR_INVALID_ARG, "n = %d", n);
    if (n == 0) return LLX_OK;
    if (!ids_out) return fail(LLX_ERR_INVALID_ARG, "ids_out is NULL");
    if ((size_t)n > m->free_stack.size())
        return fail(LLX_ERR_NO_SPACE, "%d blocks asked for, %zu free", n, m->free_stack.size());
    for (int i = 0; i < n; ++i) {
        const int32_t b = m->free_stack.back();
        m->free_stack.pop_back();
        m->is_free[(size_t)b] = 0;
        ids_out[i] = b;
    }
    return LLX_OK;
}

llx_status llx_blockmgr_release(llx_blockmgr* m, const int32_t* ids, int n) {
    if (!m) return fail(LLX_ERR_INVALID_ARG, "block manager is NULL");
    if (n < 0) return fail(LLX_ERR_INVALID_ARG, "n = %d", n);
    if (n == 0) return LLX_OK;
    if (!ids) return fail(LLX_ERR_INVALID_ARG, "ids is NULL");
    // validate everything first: a failed release changes nothing
    for (int i = 0; i < n; ++i) {
        if (ids[i] < 0 || ids[i] >= m->num_blocks)
            return fail(LLX_ERR_BLOCK_OUT_OF_RANGE, "ids[%d] = %d not in [0,%d)", i, ids[i], m->num_blocks);
        if (m->is_free[(size_t)ids[i]]) return fail(LLX_ERR_INVALID_ARG, "block %d is already free", ids[i]);
    }
    try {
        m->free_stack.reserve(m->free_stack.size() + (size_t)n);  // the pushes below cannot throw after this
    } catch (...) {
        return fail(LLX_ERR_OOM, "host allocation failed");
    }
    for (int i = 0; i < n; ++i) {  // a duplicate inside the list shows up as "already free" on its second visit
        if (m->is_free[(size_t)ids[i]]) {
            for (int j = 0; j < i; ++j) {  // undo
                m->is_free[(size_t)ids[j]] = 0;
                m->free_stack.pop_back();
            }
            return fail(LLX_ERR_INVALID_ARG, "block %d appears twice in the list", ids[i]);
        }
        m->is_free[(size_t)ids[i]] = 1;
        m->free_stack.push_back(ids[i]);
    }
    return LLX_OK;
}

}  // extern "C"

// ---- migration session: the handshake -----------------------------------------------------------------
namespace {

// destination side of an abort ("abort the migration and clean the states"; A25): every block
// reserved for this migration goes back to the destination's free list; the source is untouched
void do_abort(llx_migration* g, llx_abort_reason why) {
    if (!g->dst_table.empty()) llx_blockmgr_release(g->dst_mgr, g->dst_table.data(), (int)g->dst_table.size());
    g->dst_table.clear();
    g->reason = why;
    g->state = LLX_MIG_ABORTED;
}

llx_abort_reason reason_of(llx_req_status s) {
    switch (s) {
        case LLX_REQ_FINISHED: return LLX_ABORT_FINISHED;
        case LLX_REQ_PREEMPTED: return LLX_ABORT_PREEMPTED;
        case LLX_REQ_PEER_FAILED: return LLX_ABORT_PEER_FAILED;
        default: return LLX_ABORT_NONE;
    }
}

}  // namespace

extern "C" {

llx_status llx_migration_begin(const llx_pool* src, llx_blockmgr* src_mgr, llx_pool* dst, llx_blockmgr* dst_mgr,
                               int block_size, int last_stage_max_blocks, llx_migration** out) {
    if (!out) return fail(LLX_ERR_INVALID_ARG, "out is NULL");
    *out = nullptr;
    if (!src_mgr || !dst_mgr) return fail(LLX_ERR_INVALID_ARG, "block manager is NULL");
    if (src_mgr == dst_mgr) return fail(LLX_ERR_ALIAS, "source and destination share one block manager");
    if ((src == nullptr) != (dst == nullptr)) return fail(LLX_ERR_INVALID_ARG, "pass both pools or neither");
    if (block_size <= 0 || last_stage_max_blocks < 1)
        return fail(LLX_ERR_INVALID_ARG, "block_size = %d, last_stage_max_blocks = %d", block_size, last_stage_max_blocks);
    if (src) {
        if (llx_pool_num_blocks(src) != src_mgr->num_blocks || llx_pool_num_blocks(dst) != dst_mgr->num_blocks)
            return fail(LLX_ERR_GEOMETRY_MISMATCH, "a block manager does not match its pool's num_blocks");
    }
    llx_migration* g = new (std::nothrow) llx_migration();
    if (!g) return fail(LLX_ERR_OOM, "host allocation failed");
    g->src = src;
    g->dst = dst;
    g->src_mgr = src_mgr;
    g->dst_mgr = dst_mgr;
    g->block_size = block_size;
    g->last_stage_max_blocks = last_stage_max_blocks;
    *out = g;
    return LLX_OK;
}

llx_status llx_migration_stage(llx_migration* g, const int32_t* table, int table_len, int num_tokens, llx_req_status status,
                               void* stream, int* n_out, int* is_final_out, int32_t* dst_ids_out) {
    LLX_TRY
    if (!g || !n_out || !is_final_out) return fail(LLX_ERR_INVALID_ARG, "NULL argument");
    *n_out = 0;
    *is_final_out = 0;
    if (g->state != LLX_MIG_READY && g->state != LLX_MIG_COPYING)
        return fail(LLX_ERR_STATE, "llx_migration_stage in state %d", (int)g->state);
    // (1) the source's check (A26: also before the first stage)
    if (status != LLX_REQ_RUNNING) {
        do_abort(g, reason_of(status));
        return LLX_OK;
    }
    // (2) which blocks
    int n = 0, fin = 0;
    llx_status rc = llx_plan_stage(num_tokens, g->blocks_migrated, g->block_size, g->last_stage_max_blocks, &n, &fin);
    if (rc != LLX_OK) return rc;
    const int m = g->blocks_migrated;
    if (n > 0 && (!table || table_len < m + n))
        return fail(LLX_ERR_INVALID_ARG, "source block table of %d entries, stage needs [%d,%d)", table_len, m, m + n);
    // The commit hands src_block_table[0 .. blocks migrated) back to the source's manager, which has no reference
    // counts: a table that names a block twice (llx_migrate_stage itself allows that for prefix-shared blocks) could
    // be copied but never committed.  Refused here, before anything is reserved or copied.
    if (n > 0) {
        std::vector<unsigned char> seen((size_t)g->src_mgr->num_blocks, 0);
        for (int i = 0; i < m + n; ++i) {
            const int32_t b = table[i];
            if (b < 0 || b >= g->src_mgr->num_blocks)
                return fail(LLX_ERR_BLOCK_OUT_OF_RANGE, "src_block_table[%d] = %d not in [0,%d)", i, b, g->src_mgr->num_blocks);
            if (seen[(size_t)b])
                return fail(LLX_ERR_INVALID_ARG, "src_block_table names block %d twice (second at %d): a session cannot migrate prefix-shared "
                            "blocks, the block manager keeps no reference counts", b, i);
            seen[(size_t)b] = 1;
        }
    }
    // (3) PRE-ALLOC on the destination: all or nothing
    std::vector<int32_t> ids((size_t)n);
    g->dst_table.reserve(g->dst_table.size() + (size_t)n);  // nothing below can throw once the blocks are reserved
    rc = llx_blockmgr_alloc(g->dst_mgr, n, ids.data());
    if (rc == LLX_ERR_NO_SPACE) {
        do_abort(g, LLX_ABORT_NO_SPACE);
        return LLX_OK;
    }
    if (rc != LLX_OK) return rc;
    // (4) the stage's copy
    if (g->src && n > 0) {
        // the final stage is the downtime: never throttled; earlier stages follow the session's policy
        llx_launch_opts o;
        if (g->has_opts) o = g->stage_opts; else llx_launch_opts_init(&o);
        // ... and never started early: it reads the block the source was still appending to (stream order against the
        // appends must hold), while a non-final stage only reads full blocks nobody writes any more (A3)
        if (fin) o.bandwidth_gbps = 0, o.max_ctas = 0, o.overlap_prev = 0;
        rc = llx_migrate_stage_ex(g->src, table + m, g->dst, ids.data(), n, stream, (g->has_opts || fin) ? &o : nullptr);
        if (rc != LLX_OK) {  // nothing was launched: give the reservation back, the session stays where it was
            llx_blockmgr_release(g->dst_mgr, ids.data(), n);
            return rc;
        }
    }
    g->dst_table.insert(g->dst_table.end(), ids.begin(), ids.end());
    g->blocks_migrated += n;
    g->stages += 1;
    g->state = fin ? LLX_MIG_FINAL_COPYING : LLX_MIG_COPYING;
    if (dst_ids_out)
        for (int i = 0; i < n; ++i) dst_ids_out[i] = ids[(size_t)i];
    *n_out = n;
    *is_final_out = fin;
    return LLX_OK;
    LLX_CATCH
}

llx_status llx_migration_set_stage_opts(llx_migration* g, const llx_launch_opts* opts) {
    if (!g) return fail(LLX_ERR_INVALID_ARG, "migration is NULL");
    if (!opts) {
        g->has_opts = false;
        return LLX_OK;
    }
    // a caller compiled against an older, shorter struct is served (as in the *_ex calls): later fields keep the defaults
    if (opts->struct_size < 2 * sizeof(int32_t) || opts->struct_size > sizeof(llx_launch_opts) || (opts->struct_size % sizeof(int32_t)) != 0)
        return fail(LLX_ERR_INVALID_ARG, "llx_launch_opts.struct_size = %u (this library: %zu); use llx_launch_opts_init", opts->struct_size, sizeof(llx_launch_opts));
    llx_launch_opts_init(&g->stage_opts);
    memcpy(&g->stage_opts, opts, opts->struct_size);
    g->stage_opts.struct_size = (uint32_t)sizeof(llx_launch_opts);
    g->has_opts = true;
    return LLX_OK;
}

llx_status llx_migration_commit(llx_migration* g, const int32_t* table, int table_len, llx_req_status status,
                                int32_t* dst_table_out, int cap, int* n_out) {
    if (!g) return fail(LLX_ERR_INVALID_ARG, "migration is NULL");
    if (n_out) *n_out = 0;
    if (g->state != LLX_MIG_FINAL_COPYING) return fail(LLX_ERR_STATE, "llx_migration_commit in state %d", (int)g->state);
    if (status != LLX_REQ_RUNNING) {  // A26: a request that ended during the final copy is not committed
        do_abort(g, reason_of(status));
        return LLX_OK;
    }
    const int n = g->blocks_migrated;
    if (n > 0 && (!table || table_len < n)) return fail(LLX_ERR_INVALID_ARG, "source block table of %d entries, %d blocks migrated", table_len, n);
    if (n > 0 && (!dst_table_out || cap < n)) return fail(LLX_ERR_INVALID_ARG, "dst_table_out holds %d entries, %d needed", cap, n);
    // the source releases its local blocks ...
    llx_status rc = llx_blockmgr_release(g->src_mgr, table, n);
    if (rc != LLX_OK) return rc;
    // ... and the destination commits: the reserved blocks now belong to the request there
    for (int i = 0; i < n; ++i) dst_table_out[i] = g->dst_table[(size_t)i];
    if (n_out) *n_out = n;
    g->dst_table.clear();
    g->state = LLX_MIG_COMMITTED;
    return LLX_OK;
}

llx_status llx_migration_abort(llx_migration* g, llx_abort_reason reason) {
    if (!g) return fail(LLX_ERR_INVALID_ARG, "migration is NULL");
    if (g->state == LLX_MIG_COMMITTED || g->state == LLX_MIG_ABORTED)
        return fail(LLX_ERR_STATE, "llx_migration_abort in state %d", (int)g->state);
    if (reason <= LLX_ABORT_NONE || reason > LLX_ABORT_NO_SPACE) return fail(LLX_ERR_INVALID_ARG, "reason = %d", (int)reason);
    do_abort(g, reason);
    return LLX_OK;
}

llx_mig_state llx_migration_state(const llx_migration* g) { return g ? g->state : LLX_MIG_ABORTED; }
llx_abort_reason llx_migration_abort_reason(const llx_migration* g) { return g ? g->reason : LLX_ABORT_NONE; }
int llx_migration_blocks_migrated(const llx_migration* g) { return g ? g->blocks_migrated : -1; }
int llx_migration_stages(const llx_migration* g) { return g ? g->stages : -1; }

llx_status llx_migration_destroy(llx_migration* g) {
    if (!g) return LLX_OK;
    if (g->state != LLX_MIG_COMMITTED && g->state != LLX_MIG_ABORTED) do_abort(g, LLX_ABORT_PEER_FAILED);
    delete g;
    return LLX_OK;
}

}  // extern "C"

// ---- NEXT-4: virtual usage and freeness (Algorithm 1), pairing -------------
#include <algorithm>
#include <limits>

extern "C" {

llx_status llx_calc_freeness(const llx_req_info* reqs, int n, double M, const double* headroom_for_priority,
                             int num_priorities, int is_terminating, double* freeness, double* total_virtual_usage) {
    LLX_TRY
    if (n < 0 || num_priorities < 1 || !headroom_for_priority || !freeness || (n > 0 && !reqs))
        return fail(LLX_ERR_INVALID_ARG, "bad arguments (n=%d, num_priorities=%d)", n, num_priorities);
    // instance.numRequests[p]: the running requests of each priority (they share that priority's headroom)
    std::vector<int> per_prio((size_t)num_priorities, 0);
    int running = 0;
    for (int i = 0; i < n; ++i) {
        const llx_req_info& r = reqs[i];
        if (r.priority < 0 || r.priority >= num_priorities)
            return fail(LLX_ERR_INVALID_ARG, "reqs[%d].priority = %d not in [0,%d)", i, r.priority, num_priorities);
        if (!r.is_queuing && !r.is_fake) {
            ++per_prio[(size_t)r.priority];
            ++running;
        }
    }
    double total = 0.0;
    for (int i = 0; i < n; ++i) {
        const llx_req_info& r = reqs[i];
        double v;
        if (r.is_queuing)
            v = r.is_head_of_line ? r.demand : 0.0;  // lines 2-5
        else if (r.is_fake)
            v = std::numeric_limits<double>::infinity();  // lines 6-7
        else
            v = r.physical_usage + headroom_for_priority[r.priority] / per_prio[(size_t)r.priority];  // lines 8, 10
        total += v;
    }
    if (is_terminating) total += std::numeric_limits<double>::infinity();  // lines 12-13: the fake request
    const double B = running > 0 ? (double)running : 1.0;
    *freeness = (M - total) / B;  // line 17
    if (total_virtual_usage) *total_virtual_usage = total;
    return LLX_OK;
    LLX_CATCH
}

llx_status llx_pair_instances(const double* freeness, int n, double src_below, double dst_above, int32_t* src_out,
                              int32_t* dst_out, int cap, int* n_pairs) {
    if (n < 0 || !n_pairs || (n > 0 && !freeness) || cap < 0 || (cap > 0 && (!src_out || !dst_out)))
        return fail(LLX_ERR_INVALID_ARG, "bad arguments");
    if (src_below > dst_above) return fail(LLX_ERR_INVALID_ARG, "thresholds overlap: src_below %g > dst_above %g", src_below, dst_above);
    LLX_TRY
    std::vector<int32_t> src, dst;
    for (int i = 0; i < n; ++i) {
        if (freeness[i] < src_below) src.push_back(i);
        if (freeness[i] > dst_above) dst.push_back(i);
    }
    std::stable_sort(src.begin(), src.end(), [&](int32_t a, int32_t b) { return freeness[a] < freeness[b]; });
    std::stable_sort(dst.begin(), dst.end(), [&](int32_t a, int32_t b) { return freeness[a] > freeness[b]; });
    const int pairs = (int)std::min(src.size(), dst.size());
    *n_pairs = pairs;
    if (pairs > cap) return fail(LLX_ERR_INVALID_ARG, "%d pairs, output holds %d", pairs, cap);
    for (int k = 0; k < pairs; ++k) {
        src_out[k] = src[(size_t)k];
        dst_out[k] = dst[(size_t)k];
    }
    return LLX_OK;
    LLX_CATCH
}

llx_status llx_migration_order(const int32_t* priority, const int32_t* seq_len, int n, int32_t* order_out) {
    if (n < 0 || (n > 0 && (!priority || !seq_len || !order_out))) return fail(LLX_ERR_INVALID_ARG, "bad arguments");
    for (int i = 0; i < n; ++i) order_out[i] = i;
    std::stable_sort(order_out, order_out + n, [&](int32_t a, int32_t b) {
        return priority[a] != priority[b] ? priority[a] < priority[b] : seq_len[a] < seq_len[b];
    });
    return LLX_OK;
}

// One migration round of one (source, destination) pair as one batch (reading A31): the source offers its
// running requests in migration order while it is still below the source threshold; each request's blocks are
// PRE-ALLOCated on the destination, all or nothing; the first request that does not fit ends the round.
// The output is the argument list of llx_migrate_batch.
llx_status llx_plan_migration_batch(const llx_req_info* reqs, const int32_t* seq_len, int n, double M,
                                    const double* headroom_for_priority, int num_priorities, int is_terminating,
                                    double src_below, const int32_t* table_offsets, const int32_t* src_block_tables,
                                    llx_blockmgr* dst_mgr, int dst_reserve_blocks, int32_t* chosen_out, int* n_chosen,
                                    int32_t* req_offsets_out, int32_t* src_ids_out, int32_t* dst_ids_out, int cap_pairs,
                                    int* n_pairs) {
    LLX_TRY
    if (!n_chosen || !n_pairs) return fail(LLX_ERR_INVALID_ARG, "NULL output");
    *n_chosen = 0;
    *n_pairs = 0;
    if (n < 0 || cap_pairs < 0 || dst_reserve_blocks < 0 || !dst_mgr || !req_offsets_out || !headroom_for_priority || num_priorities < 1)
        return fail(LLX_ERR_INVALID_ARG, "bad arguments (n=%d, cap_pairs=%d, dst_reserve_blocks=%d)", n, cap_pairs, dst_reserve_blocks);
    req_offsets_out[0] = 0;
    if (n == 0) return LLX_OK;
    if (!reqs || !seq_len || !table_offsets || !chosen_out) return fail(LLX_ERR_INVALID_ARG, "NULL argument");
    if (table_offsets[0] != 0) return fail(LLX_ERR_INVALID_ARG, "table_offsets[0] = %d, must be 0", table_offsets[0]);
    for (int r = 0; r < n; ++r)
        if (table_offsets[r + 1] < table_offsets[r]) return fail(LLX_ERR_INVALID_ARG, "table_offsets decreases at request %d", r);
    if (table_offsets[n] > 0 && !src_block_tables) return fail(LLX_ERR_INVALID_ARG, "src_block_tables is NULL");

    // 1. candidates: the running requests, lower priority first, then shorter, then lower index (llx_migration_order)
    std::vector<int32_t> prio((size_t)n), order((size_t)n);
    for (int i = 0; i < n; ++i) prio[(size_t)i] = reqs[i].priority;
    llx_status rc = llx_migration_order(prio.data(), seq_len, n, order.data());
    if (rc != LLX_OK) return rc;
    // 2. take requests while the source is still below its threshold and the destination can hold the next one.
    //    First decided on a copy of the request set (nothing is reserved if an output turns out too small) ...
    std::vector<llx_req_info> left(reqs, reqs + n);
    std::vector<int32_t> left_id((size_t)n);
    for (int i = 0; i < n; ++i) left_id[(size_t)i] = i;
    long long dst_free = (long long)llx_blockmgr_num_free(dst_mgr) - dst_reserve_blocks;
    std::vector<int32_t> chosen;
    long long pairs = 0;
    for (int k = 0; k < n; ++k) {
        const int32_t r = order[(size_t)k];
        if (reqs[r].is_queuing || reqs[r].is_fake) continue;  // nothing to migrate: no KV cache on this instance yet
        double F = 0.0;
        rc = llx_calc_freeness(left.data(), (int)left.size(), M, headroom_for_priority, num_priorities, is_terminating, &F, nullptr);
        if (rc != LLX_OK) return rc;
        if (!(F < src_below)) break;  // no longer in the source state
        const long long nb = (long long)table_offsets[r + 1] - table_offsets[r];
        if (nb > dst_free) break;  // PRE-ALLOC fails: the destination aborts this migration and the round ends
        dst_free -= nb;
        pairs += nb;
        chosen.push_back(r);
        for (size_t j = 0; j < left_id.size(); ++j)
            if (left_id[j] == r) {
                left.erase(left.begin() + (long)j);
                left_id.erase(left_id.begin() + (long)j);
                break;
            }
    }
    if (pairs > cap_pairs) {
        *n_pairs = (int)pairs;
        return fail(LLX_ERR_INVALID_ARG, "%lld id pairs, outputs hold %d", pairs, cap_pairs);
    }
    if (pairs > 0 && (!src_ids_out || !dst_ids_out)) return fail(LLX_ERR_INVALID_ARG, "id output is NULL");
    // ... then the PRE-ALLOC itself, request by request in the order taken (all or nothing each)
    long long at = 0;
    for (size_t c = 0; c < chosen.size(); ++c) {
        const int32_t r = chosen[c];
        const int nb = table_offsets[r + 1] - table_offsets[r];
        rc = llx_blockmgr_alloc(dst_mgr, nb, dst_ids_out + at);
        if (rc != LLX_OK) {  // cannot happen after the count above; give everything back and report
            if (at > 0) llx_blockmgr_release(dst_mgr, dst_ids_out, (int)at);
            return rc;
        }
        for (int i = 0; i < nb; ++i) src_ids_out[at + i] = src_block_tables[table_offsets[r] + i];
        at += nb;
        chosen_out[c] = r;
        req_offsets_out[c + 1] = (int32_t)at;
    }
    *n_chosen = (int)chosen.size();
    *n_pairs = (int)at;
    return LLX_OK;
    LLX_CATCH
}

}  // extern "C"

// ---- NEXT-1: the bandwidth budget chosen from the decode steps the engine observes (A34) ----
#include <cmath>

struct llx_budget_ctl {
    double target = 0.0, lo = 0.0, hi = 0.0, budget = 0.0, last_slowdown_pct = NAN;
    int window = 0, adjustments = 0;
    std::vector<double> base, mig;  // the last 2*window steps without a migration; the steps with one since the last adjustment
};

static double median_of(std::vector<double> v) {  // by value: sorted copy
    std::sort(v.begin(), v.end());
    const size_t n = v.size();
    return (n % 2) ? v[n / 2] : (v[n / 2 - 1] + v[n / 2]) / 2.0;
}
static int rounded_gbps(const llx_budget_ctl* c) { return (int)std::floor(c->budget + 0.5); }

extern "C" {

llx_status llx_budget_ctl_create(double target_slowdown_pct, int min_gbps, int max_gbps, int start_gbps, int window,
                                 llx_budget_ctl** out) {
    LLX_TRY
    if (!out) return fail(LLX_ERR_INVALID_ARG, "out is NULL");
    *out = nullptr;
    if (!(target_slowdown_pct > 0.0) || !std::isfinite(target_slowdown_pct) || min_gbps < 1 || start_gbps < min_gbps ||
        max_gbps < start_gbps || max_gbps > 100000 || window < 2 || window > 256)
        return fail(LLX_ERR_INVALID_ARG, "bad arguments (target=%g %%, budget %d <= %d <= %d GB/s, window=%d)", target_slowdown_pct,
                    min_gbps, start_gbps, max_gbps, window);
    llx_budget_ctl* c = new (std::nothrow) llx_budget_ctl();
    if (!c) return fail(LLX_ERR_OOM, "host allocation failed");
    c->target = target_slowdown_pct / 100.0;
    c->lo = (double)min_gbps;
    c->hi = (double)max_gbps;
    c->budget = (double)start_gbps;
    c->window = window;
    try {
        c->base.reserve((size_t)2 * window + 1);
        c->mig.reserve((size_t)window + 1);
    } catch (...) {
        delete c;
        throw;
    }
    *out = c;
    return LLX_OK;
    LLX_CATCH
}

llx_status llx_budget_ctl_destroy(llx_budget_ctl* c) {
    delete c;
    return LLX_OK;
}

llx_status llx_budget_ctl_observe(llx_budget_ctl* c, double step_ms, int migrating, int* budget_gbps) {
    LLX_TRY
    if (!c) return fail(LLX_ERR_INVALID_ARG, "controller is NULL");
    if (!(step_ms > 0.0) || !std::isfinite(step_ms)) return fail(LLX_ERR_INVALID_ARG, "step_ms = %g", step_ms);
    if (!migrating) {
        c->base.push_back(step_ms);
        if (c->base.size() > (size_t)2 * c->window) c->base.erase(c->base.begin());
    } else if (!c->base.empty()) {  // a step with a migration means nothing before a step without one has been seen
        c->mig.push_back(step_ms);
        if (c->mig.size() >= (size_t)c->window) {
            const double s = median_of(c->mig) / median_of(c->base) - 1.0;
            double f = 2.0;  // cost within noise of zero: probe upwards
            if (!(s <= c->target / 4.0)) f = std::min(2.0, std::max(0.5, c->target / s));
            c->budget = std::min(c->hi, std::max(c->lo, c->budget * f));
            c->last_slowdown_pct = 100.0 * s;
            c->adjustments += 1;
            c->mig.clear();
        }
    }
    if (budget_gbps) *budget_gbps = rounded_gbps(c);
    return LLX_OK;
    LLX_CATCH
}

int llx_budget_ctl_gbps(const llx_budget_ctl* c) { return c ? rounded_gbps(c) : -1; }
double llx_budget_ctl_last_slowdown_pct(const llx_budget_ctl* c) { return c ? c->last_slowdown_pct : NAN; }
int llx_budget_ctl_adjustments(const llx_budget_ctl* c) { return c ? c->adjustments : -1; }

}  // extern "C"
