/* The C ABI used from plain C99 (no C++, no Python, no CUDA headers): the header must compile
 * as C, every host-side entry point must link and behave.  Built and run by
 * tests/test_c_abi.py with gcc -std=c99 -pedantic -Wall -Wextra -Werror. */
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "lumen_kv.h"

#define CHECK(cond)                                                        \
    do {                                                                   \
        if (!(cond)) {                                                     \
            fprintf(stderr, "FAILED line %d: %s\n", __LINE__, #cond);      \
            return 1;                                                      \
        }                                                                  \
    } while (0)

int main(void) {
    lumen_kv_geom g;
    lumen_kv_req reqs[2];
    lumen_kv_plan* plan = NULL;
    lumen_kv_run_info run;
    lumen_kv_chunk_info chunks[64];
    int32_t pt0[3] = {7, 3, 9}, pt1[1] = {5};
    int64_t n;

    memset(&g, 0, sizeof g);
    g.num_layers = 2; g.kv_heads = 2; g.head_dim = 64; g.page_size = 16; g.elem_bytes = 2;
    g.num_pages = 64;                                   /* BASELINE.json configs[0] geometry */
    reqs[0].page_table = pt0; reqs[0].page_table_len = 3; reqs[0].t_begin = 5; reqs[0].t_end = 37;
    reqs[1].page_table = pt1; reqs[1].page_table_len = 1; reqs[1].t_begin = 0; reqs[1].t_end = 5;

    CHECK(lumen_kv_version() == LUMEN_KV_VERSION);
    CHECK(lumen_kv_plan_build(&g, reqs, 2, LUMEN_KV_HOST_ONLY | LUMEN_KV_VALIDATE_UNIQUE_DST, NULL,
                              &plan) == LUMEN_KV_OK);
    CHECK(lumen_kv_plan_bytes(plan) == (32 + 5) * 1024);          /* 1 KiB per token          */
    CHECK(lumen_kv_plan_req_offset(plan, 1) == 32 * 1024);
    CHECK(lumen_kv_plan_num_runs(plan) == 4);                      /* 11 + 16 + 5 tokens, + 5  */
    CHECK(lumen_kv_plan_get_run(plan, 0, &run) == LUMEN_KV_OK);
    CHECK(run.src_slot == 7 * 16 + 5 && run.dst_token == 0 && run.count == 11 && run.req == 0);
    n = lumen_kv_plan_get_chunks(plan, 4096, chunks, 64);
    CHECK(n > 4 && chunks[0].byte_begin == 0 && chunks[n - 1].byte_end == 37 * 1024);
    CHECK(lumen_kv_plan_num_chunks(plan, 16) == LUMEN_KV_ESIZE);  /* a run must fit a slot    */
    /* a host-only plan cannot be executed, and nothing here touched a GPU */
    CHECK(lumen_kv_checkpoint_pack(plan, NULL, NULL, NULL, 1 << 20, LUMEN_KV_MEM_DEVICE, NULL) ==
          LUMEN_KV_EINVAL);
    lumen_kv_plan_free(plan);
    reqs[1].page_table = pt0;                                      /* same slot of page 7 twice */
    reqs[1].t_begin = 5; reqs[1].t_end = 6;
    CHECK(lumen_kv_plan_build(&g, reqs, 2, LUMEN_KV_HOST_ONLY | LUMEN_KV_VALIDATE_UNIQUE_DST, NULL,
                              &plan) == LUMEN_KV_EOVERLAP);
    CHECK(plan == NULL && strlen(lumen_kv_strerror(LUMEN_KV_EOVERLAP)) > 0);

    {   /* tags + store + controller, host side */
        lumen_kv_tag a[3], b[2];
        lumen_kv_store* st = NULL;
        lumen_kv_segment seg[4];
        static uint16_t arena[64 * 512] __attribute__((aligned(16)));   /* 64 tokens x 1 KiB */
        static uint16_t delta[20 * 512];
        int64_t tok_off[2] = {0, 40};
        double q[3] = {0.0, 1.0, 1.0};
        int64_t held[2] = {10, 10}, avail[3] = {50, 50, 50}, load[3] = {9, 2, 2}, fin[3], sz[2] = {7, 3};
        int32_t hb[4] = {0, 0, 1, 2}, holder = -9, who[2] = {1, 1}, assign[2];
        uint8_t alive[3] = {0, 1, 1}, reuse[2];

        CHECK(lumen_kv_tags_num_pages(tok_off, 1, 16) == 3);
        a[0].hash = 1; a[0].end_pos = 16; a[1].hash = 2; a[1].end_pos = 32; a[2].hash = 3; a[2].end_pos = 40;
        b[0] = a[1]; b[1] = a[0];
        CHECK(lumen_kv_longest_prefix(a, 3, b, 2) == 32);
        CHECK(lumen_kv_store_create(arena, sizeof arena, 1024, 16, 2, &st) == LUMEN_KV_OK);
        CHECK(lumen_kv_store_reserve(st, 42, 40) == LUMEN_KV_OK);
        CHECK(lumen_kv_store_reserve(st, 43, 30) == LUMEN_KV_ENOMEM);   /* 24 tokens left       */
        CHECK(lumen_kv_store_available(st) == 24 * 1024);
        memset(delta, 0x5a, sizeof delta);
        CHECK(lumen_kv_store_append(st, 42, 0, 20, delta, 20 * 1024, a, 1) == LUMEN_KV_OK);
        CHECK(lumen_kv_store_append(st, 42, 20, 40, delta, 20 * 1024, a + 1, 2) == LUMEN_KV_OK);
        CHECK(lumen_kv_store_tokens(st, 42) == 40 && lumen_kv_store_lookup(st, 42, a, 3) == 40);
        CHECK(lumen_kv_store_segments(st, 42, 32, seg, 4) == 2);
        CHECK(seg[1].t_begin == 20 && seg[1].t_end == 32 && seg[1].plane_stride_tokens == 20 &&
              seg[1].buf_offset == 20 * 1024);
        CHECK(lumen_kv_store_release(st, 42) == LUMEN_KV_OK && lumen_kv_store_reserved(st) == 0);
        lumen_kv_store_destroy(st);

        CHECK(lumen_kv_choose_holder(q, held, hb, avail, 3, 0, 10, 1.0, 26.0, &holder) == LUMEN_KV_OK);
        CHECK(holder == 1);                                         /* tie: lowest id          */
        CHECK(lumen_kv_recover(load, alive, 3, who, sz, 2, assign, reuse, fin) == LUMEN_KV_OK);
        /* w1 = 2 + 2 = 4 > average 3: it sheds its smallest checkpoint (size 3) to w2 -> 3, 3 */
        CHECK(assign[0] == 1 && assign[1] == 2 && reuse[0] && !reuse[1] && fin[1] == 3 && fin[2] == 3);
    }
    puts("c abi ok");
    return 0;
}
