/* A plain C99 client that MOVES DATA through the llx C ABI: no Python, no CUDA headers, nothing but llx.h.
 *
 *     abi_gpu CASEDIR        CASEDIR written by tests/golden/make_abi_gpu_case.py (synth inputs, oracle expected values)
 *
 * BASELINE configs[0] "Tiny": two library-owned pools (llx_pool_create), the source uploaded from src.bin
 * (llx_pool_upload), the destination filled with the sentinel (llx_pool_fill_u16); the request migrates in two stages
 * (llx_migrate_stage of 5 blocks, then the blocking final stage llx_migrate_stage_wait of 2); the same
 * request is then fused into ONE pinned host buffer (llx_pack), compared with staging.bin, and scattered
 * into a second set of reserved blocks (llx_unpack); the destination comes back with llx_pool_download and must equal
 * dst.bin byte for byte.  Built and run by tests/test_gpu_c_client.py. */
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "llx.h"

#define CHECK(cond)                                                                  \
    do {                                                                             \
        if (!(cond)) {                                                               \
            printf("FAILED line %d: %s (%s)\n", __LINE__, #cond, llx_last_error());  \
            return 1;                                                                \
        }                                                                            \
    } while (0)

enum { L = 2, HEADS = 4, HEAD_DIM = 64, BLOCK = 16, NB = 256, SENTINEL = 0x7BAD };

static void* read_file(const char* dir, const char* name, size_t* bytes) {
    char path[1024];
    FILE* f;
    long sz;
    void* p;
    snprintf(path, sizeof path, "%s/%s", dir, name);
    f = fopen(path, "rb");
    if (!f) return NULL;
    fseek(f, 0, SEEK_END);
    sz = ftell(f);
    fseek(f, 0, SEEK_SET);
    p = malloc((size_t)sz);
    if (p && fread(p, 1, (size_t)sz, f) != (size_t)sz) {
        free(p);
        p = NULL;
    }
    fclose(f);
    *bytes = (size_t)sz;
    return p;
}

int main(int argc, char** argv) {
    size_t ids_bytes = 0, src_bytes = 0, stg_bytes = 0, dst_bytes = 0, tile, pool_bytes, need;
    int32_t *ids, *s_ids, *d_ids, *d2_ids;
    unsigned char *src_img, *stg_img, *dst_img, *got;
    llx_pool *src = NULL, *dst = NULL;
    void *pin_host = NULL, *pin_dev = NULL;
    llx_launch_opts opts;
    llx_counters c0, c1;
    int n, l, kv;

    if (argc != 2) {
        printf("usage: abi_gpu CASEDIR\n");
        return 2;
    }
    ids = (int32_t*)read_file(argv[1], "ids.bin", &ids_bytes);
    src_img = (unsigned char*)read_file(argv[1], "src.bin", &src_bytes);
    stg_img = (unsigned char*)read_file(argv[1], "staging.bin", &stg_bytes);
    dst_img = (unsigned char*)read_file(argv[1], "dst.bin", &dst_bytes);
    CHECK(ids && src_img && stg_img && dst_img);
    n = ids[0];
    CHECK(n > 2 && ids_bytes == (size_t)(1 + 3 * n) * sizeof(int32_t));
    s_ids = ids + 1;
    d_ids = s_ids + n;
    d2_ids = d_ids + n;

    CHECK(llx_pool_create(L, HEADS, HEAD_DIM, BLOCK, LLX_F16, NB, &src) == LLX_OK);
    CHECK(llx_pool_create(L, HEADS, HEAD_DIM, BLOCK, LLX_F16, NB, &dst) == LLX_OK);
    tile = llx_pool_tile_bytes(src);
    pool_bytes = llx_pool_bytes(src);
    CHECK(tile == (size_t)BLOCK * HEADS * HEAD_DIM * 2 && pool_bytes == src_bytes && pool_bytes == dst_bytes);
    for (l = 0; l < L; ++l)
        for (kv = 0; kv < 2; ++kv)
            CHECK(llx_pool_upload(src, l, kv, 0, NB, src_img + ((size_t)l * 2 + (size_t)kv) * NB * tile, NULL) == LLX_OK);
    CHECK(llx_pool_fill_u16(dst, SENTINEL, NULL) == LLX_OK);
    CHECK(llx_synchronize(NULL) == LLX_OK);

    /* stage 0 with this call's own launch policy (a struct, not process state), then the blocking final stage */
    llx_get_counters(&c0);
    llx_launch_opts_init(&opts);
    opts.bandwidth_gbps = 200;
    CHECK(llx_migrate_stage_ex(src, s_ids, dst, d_ids, n - 2, NULL, &opts) == LLX_OK);
    CHECK(llx_migrate_stage_wait(src, s_ids + (n - 2), dst, d_ids + (n - 2), 2, NULL) == LLX_OK);
    llx_get_counters(&c1);
    CHECK(c1.copy_launches == c0.copy_launches + 2);
    CHECK(c1.bytes_moved - c0.bytes_moved == (unsigned long long)n * llx_pool_block_bytes(src));

    /* block fusion through ONE pinned host buffer */
    need = llx_staging_bytes(src, n);
    CHECK(need == stg_bytes);
    CHECK(llx_staging_alloc_pinned(need, &pin_host, &pin_dev) == LLX_OK);
    memset(pin_host, 0x11, need);
    CHECK(llx_pack(src, s_ids, n, pin_dev, need - 16, NULL) == LLX_ERR_STAGING_TOO_SMALL);
    CHECK(llx_pack(src, s_ids, n, pin_dev, need, NULL) == LLX_OK);
    CHECK(llx_synchronize(NULL) == LLX_OK);
    CHECK(memcmp(pin_host, stg_img, need) == 0);
    CHECK(llx_unpack(pin_dev, need, dst, d_ids, n, NULL) == LLX_OK); /* same blocks again: same bytes */
    CHECK(llx_unpack(pin_dev, need, dst, d2_ids, n, NULL) == LLX_OK);

    /* an argument error changes no byte: a duplicate destination id */
    {
        int32_t dup[2];
        dup[0] = dup[1] = d_ids[0];
        CHECK(llx_migrate_stage(src, s_ids, dst, dup, 2, NULL) == LLX_ERR_DUPLICATE_DST);
    }

    got = (unsigned char*)malloc(pool_bytes);
    CHECK(got != NULL);
    for (l = 0; l < L; ++l)
        for (kv = 0; kv < 2; ++kv)
            CHECK(llx_pool_download(dst, l, kv, 0, NB, got + ((size_t)l * 2 + (size_t)kv) * NB * tile, NULL) == LLX_OK);
    CHECK(llx_synchronize(NULL) == LLX_OK);
    if (memcmp(got, dst_img, pool_bytes) != 0) {
        size_t i = 0;
        while (got[i] == dst_img[i]) ++i;
        printf("FAILED: destination pool differs from the oracle at byte %lu (expected 0x%02x, got 0x%02x)\n", (unsigned long)i,
               dst_img[i], got[i]);
        return 1;
    }
    /* the source is never written */
    for (l = 0; l < L; ++l)
        for (kv = 0; kv < 2; ++kv)
            CHECK(llx_pool_download(src, l, kv, 0, NB, got + ((size_t)l * 2 + (size_t)kv) * NB * tile, NULL) == LLX_OK);
    CHECK(llx_synchronize(NULL) == LLX_OK);
    CHECK(memcmp(got, src_img, pool_bytes) == 0);

    CHECK(llx_staging_free_pinned(pin_host) == LLX_OK);
    CHECK(llx_pool_destroy(src) == LLX_OK && llx_pool_destroy(dst) == LLX_OK);
    free(got);
    free(ids);
    free(src_img);
    free(stg_img);
    free(dst_img);
    printf("abi_gpu ok: %d blocks migrated, fused and scattered; destination and staging buffer equal the oracle's\n", n);
    return 0;
}
