/* Plain C99 client of the llx C ABI: proves the header is C (not C++) and that the host-only entry points
 * link and behave without a device.  Built and run by tests/test_abi.py. */
#include <stdio.h>
#include <string.h>

#include "llx.h"

#define CHECK(cond)                                                   \
    do {                                                              \
        if (!(cond)) {                                                \
            printf("FAILED line %d: %s (%s)\n", __LINE__, #cond, llx_last_error()); \
            return 1;                                                 \
        }                                                             \
    } while (0)

int main(void) {
    int n = 0, fin = 0, i;
    llx_blockmgr *a = NULL, *b = NULL;
    llx_migration* mig = NULL;
    int32_t table[8], ids[8], dst_table[8];
    double f = 0.0, total = 0.0, headroom[2] = {0.0, 12016.0};
    llx_req_info reqs[2];

    CHECK(strstr(llx_version(), "sm_100a") != NULL);
    CHECK(llx_pool_bytes_for(32, 32, 128, 16, LLX_F16, 1) == 2u * 32u * 131072u); /* 128 KB per block */
    CHECK(llx_plan_stage(2032, 0, 16, 2, &n, &fin) == LLX_OK && n == 127 && fin == 0);
    CHECK(llx_plan_stage(2048, 126, 16, 2, &n, &fin) == LLX_OK && n == 2 && fin == 1);
    CHECK(llx_plan_stage(16, 2, 16, 2, &n, &fin) == LLX_ERR_INVALID_ARG);
    {   /* stage sizes from measured rates: the paper's regime gives two stages */
        int32_t sizes[8];
        int k = 0;
        CHECK(llx_predict_stage_sizes(128, 950.0, 15.4, 16, sizes, 8, &k) == LLX_OK && k == 2 && sizes[0] == 128 && sizes[1] == 1);
        CHECK(llx_predict_stage_sizes(64, 4.0, 16.0, 16, sizes, 8, &k) == LLX_OK && k == 4 && sizes[3] == 1);
        CHECK(llx_predict_stage_sizes(64, 4.0, 16.0, 16, sizes, 0, &k) == LLX_ERR_INVALID_ARG);
    }
    {   /* the budget controller (<= 1 %): 2 % observed at a 1 % target halves the budget, 1 % keeps it */
        llx_budget_ctl* ctl = NULL;
        int i, budget = 0;
        CHECK(llx_budget_ctl_create(0.0, 1, 1000, 100, 4, &ctl) == LLX_ERR_INVALID_ARG && ctl == NULL);
        CHECK(llx_budget_ctl_create(1.0, 1, 1000, 100, 4, &ctl) == LLX_OK && llx_budget_ctl_gbps(ctl) == 100);
        for (i = 0; i < 4; ++i) CHECK(llx_budget_ctl_observe(ctl, 4.08, 1, &budget) == LLX_OK && budget == 100); /* no baseline yet: dropped */
        for (i = 0; i < 8; ++i) CHECK(llx_budget_ctl_observe(ctl, 4.0, 0, &budget) == LLX_OK);
        for (i = 0; i < 4; ++i) CHECK(llx_budget_ctl_observe(ctl, 4.08, 1, &budget) == LLX_OK);
        CHECK(budget == 50 && llx_budget_ctl_adjustments(ctl) == 1 && llx_budget_ctl_last_slowdown_pct(ctl) > 1.99);
        for (i = 0; i < 4; ++i) CHECK(llx_budget_ctl_observe(ctl, 4.04, 1, NULL) == LLX_OK);
        CHECK(llx_budget_ctl_gbps(ctl) == 50 && llx_budget_ctl_adjustments(ctl) == 2);
        CHECK(llx_budget_ctl_observe(ctl, -1.0, 0, NULL) == LLX_ERR_INVALID_ARG && llx_budget_ctl_observe(NULL, 1.0, 0, NULL) == LLX_ERR_INVALID_ARG);
        CHECK(llx_budget_ctl_destroy(ctl) == LLX_OK && llx_budget_ctl_destroy(NULL) == LLX_OK);
    }

    /* the handshake without pools: coordination only */
    CHECK(llx_blockmgr_create(16, &a) == LLX_OK && llx_blockmgr_create(6, &b) == LLX_OK);
    CHECK(llx_blockmgr_alloc(a, 8, table) == LLX_OK && table[0] == 0 && table[7] == 7);
    CHECK(llx_migration_begin(NULL, a, NULL, b, 4, 1, &mig) == LLX_OK);
    CHECK(llx_migration_stage(mig, table, 8, 18, LLX_REQ_RUNNING, NULL, &n, &fin, ids) == LLX_OK && n == 4 && !fin);
    CHECK(llx_migration_state(mig) == LLX_MIG_COPYING && llx_blockmgr_num_free(b) == 2);
    CHECK(llx_migration_stage(mig, table, 8, 19, LLX_REQ_RUNNING, NULL, &n, &fin, ids) == LLX_OK && n == 1 && fin);
    CHECK(llx_migration_commit(mig, table, 5, LLX_REQ_RUNNING, dst_table, 8, &n) == LLX_OK && n == 5);
    for (i = 0; i < 5; ++i) CHECK(dst_table[i] == i);
    CHECK(llx_migration_state(mig) == LLX_MIG_COMMITTED && llx_blockmgr_num_free(a) == 13 && llx_blockmgr_num_free(b) == 1);
    CHECK(llx_migration_destroy(mig) == LLX_OK);
    /* destination out of space: abort, nothing reserved */
    CHECK(llx_migration_begin(NULL, a, NULL, b, 4, 1, &mig) == LLX_OK);
    CHECK(llx_migration_stage(mig, table + 5, 3, 12, LLX_REQ_RUNNING, NULL, &n, &fin, ids) == LLX_OK && n == 0);
    CHECK(llx_migration_state(mig) == LLX_MIG_ABORTED && llx_migration_abort_reason(mig) == LLX_ABORT_NO_SPACE);
    CHECK(llx_blockmgr_num_free(b) == 1);
    llx_migration_destroy(mig);
    llx_blockmgr_destroy(a);
    llx_blockmgr_destroy(b);

    /* Algorithm 1 with the paper's numbers: capacity 13,616 tokens, target load 1,600 tokens for high priority */
    memset(reqs, 0, sizeof reqs);
    reqs[0].priority = 1;
    reqs[0].physical_usage = 1000.0;
    reqs[1].physical_usage = 601.0;
    CHECK(llx_calc_freeness(reqs, 2, 13616.0, headroom, 2, 0, &f, &total) == LLX_OK);
    CHECK(total == 1601.0 + 12016.0 && f < 0.0); /* real load 1601 > 1600: virtually overloaded */
    reqs[1].physical_usage = 600.0;
    CHECK(llx_calc_freeness(reqs, 2, 13616.0, headroom, 2, 0, &f, &total) == LLX_OK && f == 0.0);

    /* block manager error paths leave the manager unchanged; pairing and ordering */
    {
        llx_blockmgr* m = NULL;
        int32_t got[4], bad_twice[2] = {1, 1}, bad_range[1] = {9}, order[5], srcs[4], dsts[4];
        int32_t prio[5] = {1, 0, 0, 1, 0}, len[5] = {5, 9, 3, 2, 3};
        double fr[6] = {5.0, 80.0, -3.0, 70.0, 20.0, 61.0};
        int pairs = 0;
        CHECK(llx_blockmgr_create(4, &m) == LLX_OK && llx_blockmgr_alloc(m, 3, got) == LLX_OK);
        CHECK(llx_blockmgr_alloc(m, 2, got) == LLX_ERR_NO_SPACE && llx_blockmgr_num_free(m) == 1);
        CHECK(llx_blockmgr_release(m, bad_twice, 2) == LLX_ERR_INVALID_ARG && llx_blockmgr_num_free(m) == 1);
        CHECK(llx_blockmgr_release(m, bad_range, 1) == LLX_ERR_BLOCK_OUT_OF_RANGE);
        CHECK(llx_blockmgr_release(m, got, 0) == LLX_OK && llx_blockmgr_destroy(m) == LLX_OK);
        CHECK(llx_pair_instances(fr, 6, 10.0, 60.0, srcs, dsts, 4, &pairs) == LLX_OK && pairs == 2);
        CHECK(srcs[0] == 2 && dsts[0] == 1 && srcs[1] == 0 && dsts[1] == 3);
        CHECK(llx_pair_instances(fr, 6, 10.0, 60.0, srcs, dsts, 1, &pairs) == LLX_ERR_INVALID_ARG && pairs == 2);
        CHECK(llx_migration_order(prio, len, 5, order) == LLX_OK);
        CHECK(order[0] == 2 && order[1] == 4 && order[2] == 1 && order[3] == 3 && order[4] == 0);
        CHECK(llx_set_option(LLX_OPT_CHUNK_BYTES, 100) == LLX_ERR_INVALID_ARG);
        CHECK(llx_set_option(LLX_OPT_DYNAMIC_TAIL_PCT, 8) == LLX_OK && llx_get_option(LLX_OPT_DYNAMIC_TAIL_PCT) == 8);
        CHECK(llx_set_option(LLX_OPT_DYNAMIC_TAIL_PCT, 6) == LLX_OK);
    }

    /* one migration round of a pair as one batch (PAPER.md:225 + :142, reading A31): M = 40 blocks, three running requests
     * of 10 / 6 / 12 blocks and a head-of-line queuing request that needs 20: F = (40 - 48)/3 < 2, so the source gives
     * requests away, shortest first, until F >= 2 or the destination (8 free blocks, 1 kept in reserve) is full */
    {
        llx_blockmgr* dstm = NULL;
        llx_req_info rq[4];
        int32_t seq[4] = {150, 90, 180, 300}, offs[5] = {0, 10, 16, 28, 28}, tabs[28], chosen[4], ro[5], so[28], dd[28], got8[8];
        double hr[1] = {0.0};
        int nc = -1, np = -1;
        llx_launch_opts lo;
        memset(rq, 0, sizeof rq);
        for (i = 0; i < 28; ++i) tabs[i] = 100 + i;
        rq[0].physical_usage = 10.0;
        rq[1].physical_usage = 6.0;
        rq[2].physical_usage = 12.0;
        rq[3].is_queuing = 1;
        rq[3].is_head_of_line = 1;
        rq[3].demand = 20.0;
        CHECK(llx_blockmgr_create(16, &dstm) == LLX_OK && llx_blockmgr_alloc(dstm, 8, got8) == LLX_OK);
        CHECK(llx_plan_migration_batch(rq, seq, 4, 40.0, hr, 1, 0, 2.0, offs, tabs, dstm, 1, chosen, &nc, ro, so, dd, 28, &np) == LLX_OK);
        CHECK(nc == 1 && chosen[0] == 1 && np == 6 && ro[0] == 0 && ro[1] == 6);    /* the 6-block request fits, the 10-block one does not */
        CHECK(so[0] == 110 && so[5] == 115 && dd[0] == 8 && dd[5] == 13 && llx_blockmgr_num_free(dstm) == 2);
        CHECK(llx_plan_migration_batch(rq, seq, 4, 40.0, hr, 1, 0, 2.0, offs, tabs, dstm, 0, chosen, &nc, ro, so, dd, 2, &np) == LLX_OK && nc == 0);
        CHECK(llx_plan_migration_batch(rq, seq, 4, 400.0, hr, 1, 0, 2.0, offs, tabs, dstm, 0, chosen, &nc, ro, so, dd, 28, &np) == LLX_OK && nc == 0); /* not a source */
        llx_blockmgr_destroy(dstm);
        llx_launch_opts_init(&lo);
        CHECK(lo.struct_size == sizeof lo && lo.bandwidth_gbps == LLX_OPT_DEFAULT && lo.route == LLX_OPT_DEFAULT);
        lo.chunk_bytes = 100; /* not a multiple of 16: refused before anything else is looked at */
        CHECK(llx_migrate_stage_ex(NULL, NULL, NULL, NULL, 1, NULL, &lo) == LLX_ERR_INVALID_ARG);
    }

    /* no device here or bad arguments: data calls fail loudly, never compute on the CPU */
    CHECK(llx_migrate_stage(NULL, NULL, NULL, NULL, 1, NULL) == LLX_ERR_INVALID_ARG);
    CHECK(strcmp(llx_status_str(LLX_ERR_NO_SPACE), "LLX_ERR_NO_SPACE") == 0);
    printf("abi_smoke ok\n");
    return 0;
}
