/* bench_downtime.c — the final-stage downtime measured by a plain C99 client of the llx ABI:
 * what the LIBRARY costs, without the Python binding that bench.py times through.  Built and run by
 * `python bench_suite.py --only floor` (gcc bench_downtime.c -Iinclude -Lpaper_2406_03243_b200 -lllx).
 *
 *     bench_downtime [reps]
 *
 * Two LLaMA-7B-shaped pools of 300 blocks (llx_pool_create), ids = a fixed stride permutation.  Per repetition: an
 * earlier stage of 14 blocks is enqueued and synchronised (the source has stopped the request), then
 *   t0; llx_migrate_stage(final 2 blocks); llx_synchronize; t1          -> host_us
 *   t0; llx_migrate_stage_wait(final 2 blocks); t1                       -> wait_call_us
 * and the same for a stage that moves nothing worth timing (ONE Tiny-sized block of a second, small pool pair): the
 * floor of one launch + one synchronize through this entry point.  Prints one JSON object. */
#define _POSIX_C_SOURCE 200112L
#include <stdio.h>
#include <stdlib.h>
#include <time.h>

#include "llx.h"

#define CHECK(cond)                                                                 \
    do {                                                                            \
        if (!(cond)) {                                                              \
            printf("{\"error\": \"line %d: %s (%s)\"}\n", __LINE__, #cond, llx_last_error()); \
            return 1;                                                               \
        }                                                                           \
    } while (0)

static double now_us(void) {
    struct timespec ts;
    clock_gettime(CLOCK_MONOTONIC, &ts);
    return (double)ts.tv_sec * 1e6 + (double)ts.tv_nsec * 1e-3;
}
static int cmp(const void* a, const void* b) {
    double x = *(const double*)a, y = *(const double*)b;
    return (x > y) - (x < y);
}
static void stats(double* v, int n, const char* name, int last) {
    qsort(v, (size_t)n, sizeof *v, cmp);
    printf(" \"%s\": {\"median\": %.3f, \"p99\": %.3f, \"min\": %.3f}%s\n", name, v[n / 2], v[(int)(0.99 * (n - 1))], v[0], last ? "" : ",");
}

int main(int argc, char** argv) {
    enum { NB = 300, N_EARLY = 14 };
    int reps = argc > 1 ? atoi(argv[1]) : 300, i, r;
    int32_t s_ids[16], d_ids[16], one_s[1] = {3}, one_d[1] = {5};
    llx_pool *src = NULL, *dst = NULL, *tsrc = NULL, *tdst = NULL;
    double *a, *b, *c, *d;
    if (reps < 10) reps = 10;
    a = (double*)malloc(sizeof(double) * (size_t)reps * 4);
    CHECK(a != NULL);
    b = a + reps; c = b + reps; d = c + reps;
    for (i = 0; i < 16; ++i) {               /* scattered, distinct ids */
        s_ids[i] = (i * 37 + 11) % NB;
        d_ids[i] = (i * 53 + 7) % NB;
    }
    CHECK(llx_pool_create(32, 32, 128, 16, LLX_F16, NB, &src) == LLX_OK);
    CHECK(llx_pool_create(32, 32, 128, 16, LLX_F16, NB, &dst) == LLX_OK);
    CHECK(llx_pool_create(2, 4, 64, 16, LLX_F16, 16, &tsrc) == LLX_OK);
    CHECK(llx_pool_create(2, 4, 64, 16, LLX_F16, 16, &tdst) == LLX_OK);
    CHECK(llx_pool_fill_u16(src, 0x3C00, NULL) == LLX_OK && llx_pool_fill_u16(dst, 0x7BAD, NULL) == LLX_OK);
    CHECK(llx_pool_fill_u16(tsrc, 0x3C00, NULL) == LLX_OK && llx_pool_fill_u16(tdst, 0x7BAD, NULL) == LLX_OK);
    CHECK(llx_synchronize(NULL) == LLX_OK);
    for (r = -20; r < reps; ++r) {           /* 20 warm-up repetitions */
        double t0, t1;
        CHECK(llx_migrate_stage(src, s_ids, dst, d_ids, N_EARLY, NULL) == LLX_OK);
        CHECK(llx_synchronize(NULL) == LLX_OK);
        t0 = now_us();
        CHECK(llx_migrate_stage(src, s_ids + N_EARLY, dst, d_ids + N_EARLY, 2, NULL) == LLX_OK);
        CHECK(llx_synchronize(NULL) == LLX_OK);
        t1 = now_us();
        if (r >= 0) a[r] = t1 - t0;
        CHECK(llx_migrate_stage(src, s_ids, dst, d_ids, N_EARLY, NULL) == LLX_OK);
        CHECK(llx_synchronize(NULL) == LLX_OK);
        t0 = now_us();
        CHECK(llx_migrate_stage_wait(src, s_ids + N_EARLY, dst, d_ids + N_EARLY, 2, NULL) == LLX_OK);
        t1 = now_us();
        if (r >= 0) b[r] = t1 - t0;
        t0 = now_us();
        CHECK(llx_migrate_stage(tsrc, one_s, tdst, one_d, 1, NULL) == LLX_OK);
        t1 = now_us();
        CHECK(llx_synchronize(NULL) == LLX_OK);
        if (r >= 0) {
            d[r] = t1 - t0;
            c[r] = now_us() - t0;
        }
    }
    printf("{\n \"reps\": %d,\n \"final_stage_blocks\": 2,\n \"final_stage_bytes_rd_plus_wr\": %lu,\n", reps,
           (unsigned long)(4 * llx_pool_block_bytes(src)));
    stats(a, reps, "host_us_stage_plus_synchronize", 0);
    stats(b, reps, "host_us_stage_wait_call", 0);
    stats(c, reps, "floor_host_us_one_32KiB_block_plus_synchronize", 0);
    stats(d, reps, "floor_enqueue_us_one_32KiB_block", 1);
    printf("}\n");
    llx_pool_destroy(src); llx_pool_destroy(dst); llx_pool_destroy(tsrc); llx_pool_destroy(tdst);
    free(a);
    return 0;
}
