/* The C ABI driven end to end from plain C99 on a GPU: no Python, no torch, no C++ -- only
 * include/lumen_kv.h and the CUDA runtime's C API for memory and streams.  Built and run by
 * tests/test_gpu_c_abi.py (gcc -std=c99 -pedantic -Wall -Wextra -Werror).
 *
 * The check needs no oracle (the idea of pin P6, tests/test_oracle_pins.py): every pool word
 * encodes its own (plane, token slot, element), so each word of the packed buffer can be
 * recomputed from the page table alone with the index map the header states:
 *     B[off_r + (plane*n_r + j)*row + b] <-> planes[plane][(PT_r[(tb+j)/S]*S + (tb+j)%S)*row + b]
 * and after the restore every pool word is either such a value at its new place or the fill of
 * the destination pool. */
#include <cuda_runtime_api.h>
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

enum { L = 3, H = 2, D = 64, S = 16, N = 200, R = 5, PLANES = 2 * L, E = H * D };

static uint16_t word(int plane, int64_t slot, int e) {
    return (uint16_t)((slot * 131 + e * 7 + plane * 977 + 12345) & 0xFFFF);
}

/* a permutation of 0..N-1: i -> (a*i + c) mod N with gcd(a, N) = 1 */
static int32_t perm(int64_t i, int64_t a, int64_t c) { return (int32_t)((a * i + c) % N); }

int main(void) {
    static const int64_t len[R] = {37, 100, 5, 64, 333};
    static const int64_t tb[R] = {5, 0, 4, 16, 129};
    const int64_t row = (int64_t)E * 2, words = (int64_t)N * S * E;
    lumen_kv_geom g;
    lumen_kv_req reqs[R], rreqs[R];
    int32_t *pt[R], *rpt[R];
    void *ka[L], *va[L], *kb[L], *vb[L];
    const void *cka[L], *cva[L];
    uint16_t *hplane, *hbuf, *hostbuf = NULL, *stagedbuf = NULL;
    void *dbuf = NULL, *ring = NULL;
    lumen_kv_plan *plan = NULL, *rplan = NULL;
    lumen_kv_stager* stager = NULL;
    cudaStream_t stream;
    int64_t nbytes, used = 0, rused = 0;
    int r, l, p;

    if (cudaSetDevice(0) != cudaSuccess) {
        fprintf(stderr, "no CUDA device\n");
        return 2;
    }
    CHECK(cudaStreamCreate(&stream) == cudaSuccess);
    CHECK(lumen_kv_init() == LUMEN_KV_OK);
    memset(&g, 0, sizeof g);
    g.num_layers = L; g.kv_heads = H; g.head_dim = D; g.page_size = S; g.elem_bytes = 2;
    g.num_pages = N;

    /* page tables: consecutive chunks of two different permutations (source / fresh pages) */
    for (r = 0; r < R; ++r) {
        const int64_t pages = (len[r] + S - 1) / S;
        int64_t i;
        pt[r] = (int32_t*)malloc((size_t)pages * sizeof(int32_t));
        rpt[r] = (int32_t*)malloc((size_t)pages * sizeof(int32_t));
        CHECK(pt[r] && rpt[r]);
        for (i = 0; i < pages; ++i) {
            pt[r][i] = perm(used + i, 7, 3);
            rpt[r][i] = perm(rused + i, 11, 50);
        }
        used += pages; rused += pages;
        reqs[r].page_table = pt[r]; reqs[r].page_table_len = pages;
        reqs[r].t_begin = tb[r]; reqs[r].t_end = len[r];
        rreqs[r] = reqs[r]; rreqs[r].page_table = rpt[r];
    }
    CHECK(used <= N);

    /* pools: 2L separate allocations each; A is address-coded, B is filled with 0xEEEE */
    hplane = (uint16_t*)malloc((size_t)words * 2);
    CHECK(hplane);
    for (l = 0; l < L; ++l) {
        void** dst[4];
        int k;
        dst[0] = &ka[l]; dst[1] = &va[l]; dst[2] = &kb[l]; dst[3] = &vb[l];
        for (k = 0; k < 4; ++k) CHECK(cudaMalloc(dst[k], (size_t)words * 2) == cudaSuccess);
        for (k = 0; k < 2; ++k) {
            int64_t slot;
            int e;
            for (slot = 0; slot < (int64_t)N * S; ++slot)
                for (e = 0; e < E; ++e) hplane[slot * E + e] = word(2 * l + k, slot, e);
            CHECK(cudaMemcpy(k ? va[l] : ka[l], hplane, (size_t)words * 2, cudaMemcpyHostToDevice) ==
                  cudaSuccess);
        }
        CHECK(cudaMemset(kb[l], 0xEE, (size_t)words * 2) == cudaSuccess);
        CHECK(cudaMemset(vb[l], 0xEE, (size_t)words * 2) == cudaSuccess);
        cka[l] = ka[l]; cva[l] = va[l];
    }

    /* a2 + a3: plan, pack to an HBM buffer */
    CHECK(lumen_kv_plan_build(&g, reqs, R, 0, stream, &plan) == LUMEN_KV_OK);
    nbytes = lumen_kv_plan_bytes(plan);
    {
        int64_t tokens = 0;
        for (r = 0; r < R; ++r) tokens += len[r] - tb[r];
        CHECK(nbytes == tokens * PLANES * row);
    }
    CHECK(cudaMalloc(&dbuf, (size_t)nbytes) == cudaSuccess);
    CHECK(cudaMemset(dbuf, 0, (size_t)nbytes) == cudaSuccess);
    CHECK(lumen_kv_checkpoint_pack(plan, cka, cva, dbuf, nbytes - 16, LUMEN_KV_MEM_DEVICE, stream) ==
          LUMEN_KV_ESIZE);
    CHECK(lumen_kv_checkpoint_pack(plan, cka, cva, dbuf, nbytes, LUMEN_KV_MEM_DEVICE, stream) ==
          LUMEN_KV_OK);
    hbuf = (uint16_t*)malloc((size_t)nbytes);
    CHECK(hbuf);
    CHECK(cudaMemcpyAsync(hbuf, dbuf, (size_t)nbytes, cudaMemcpyDeviceToHost, stream) == cudaSuccess);
    CHECK(cudaStreamSynchronize(stream) == cudaSuccess);
    for (r = 0; r < R; ++r) {
        const int64_t n = len[r] - tb[r], off = lumen_kv_plan_req_offset(plan, r) / 2;
        int64_t j;
        int e;
        for (p = 0; p < PLANES; ++p)
            for (j = 0; j < n; ++j) {
                const int64_t t = tb[r] + j, slot = (int64_t)pt[r][t / S] * S + t % S;
                for (e = 0; e < E; ++e)
                    if (hbuf[off + (p * n + j) * E + e] != word(p, slot, e)) {
                        fprintf(stderr, "pack mismatch r=%d plane=%d j=%ld e=%d\n", r, p, (long)j, e);
                        return 1;
                    }
            }
    }

    /* a4: the same bytes in pinned host memory, zero-copy and through the staging ring */
    CHECK(cudaHostAlloc((void**)&hostbuf, (size_t)nbytes, cudaHostAllocMapped) == cudaSuccess);
    CHECK(cudaHostAlloc((void**)&stagedbuf, (size_t)nbytes, cudaHostAllocMapped) == cudaSuccess);
    memset(hostbuf, 0, (size_t)nbytes);
    memset(stagedbuf, 0, (size_t)nbytes);
    CHECK(lumen_kv_checkpoint_pack(plan, cka, cva, hostbuf, nbytes, LUMEN_KV_MEM_HOST_MAPPED, stream) ==
          LUMEN_KV_OK);
    CHECK(cudaMalloc(&ring, 3 * 65536) == cudaSuccess);
    CHECK(lumen_kv_stager_create(ring, 65536, 3, &stager) == LUMEN_KV_OK);
    CHECK(lumen_kv_checkpoint_pack_staged(plan, cka, cva, stagedbuf, nbytes, stager, stream) ==
          LUMEN_KV_OK);
    CHECK(cudaStreamSynchronize(stream) == cudaSuccess);
    CHECK(memcmp(hostbuf, hbuf, (size_t)nbytes) == 0);
    CHECK(memcmp(stagedbuf, hbuf, (size_t)nbytes) == 0);

    /* a6 + a7: restore into pool B under fresh page tables, from the staged host buffer */
    CHECK(lumen_kv_plan_build(&g, rreqs, R, LUMEN_KV_VALIDATE_UNIQUE_DST, stream, &rplan) == LUMEN_KV_OK);
    CHECK(lumen_kv_plan_bytes(rplan) == nbytes);
    CHECK(lumen_kv_restore_unpack_staged(rplan, kb, vb, stagedbuf, nbytes, stager, stream) == LUMEN_KV_OK);
    CHECK(cudaStreamSynchronize(stream) == cudaSuccess);
    for (p = 0; p < PLANES; ++p) {
        int64_t slot, hits = 0, expect = 0;
        CHECK(cudaMemcpy(hplane, (p & 1) ? vb[p / 2] : kb[p / 2], (size_t)words * 2,
                         cudaMemcpyDeviceToHost) == cudaSuccess);
        for (r = 0; r < R; ++r) {            /* every restored token sits at its new slot */
            int64_t t;
            int e;
            for (t = tb[r]; t < len[r]; ++t) {
                const int64_t src = (int64_t)pt[r][t / S] * S + t % S;
                const int64_t dst = (int64_t)rpt[r][t / S] * S + t % S;
                for (e = 0; e < E; ++e) CHECK(hplane[dst * E + e] == word(p, src, e));
                ++expect;
            }
        }
        for (slot = 0; slot < (int64_t)N * S; ++slot) {   /* and nothing else was written */
            int e, untouched = 1;
            for (e = 0; e < E; ++e) untouched &= hplane[slot * E + e] == 0xEEEE;
            hits += !untouched;
        }
        CHECK(hits == expect);   /* a token's 128 words differ from each other: never all 0xEEEE */
    }

    lumen_kv_plan_free(plan);
    lumen_kv_plan_free(rplan);
    lumen_kv_stager_destroy(stager);
    lumen_kv_trim();
    for (l = 0; l < L; ++l) {
        cudaFree(ka[l]); cudaFree(va[l]); cudaFree(kb[l]); cudaFree(vb[l]);
    }
    for (r = 0; r < R; ++r) {
        free(pt[r]); free(rpt[r]);
    }
    cudaFree(dbuf); cudaFree(ring); cudaFreeHost(hostbuf); cudaFreeHost(stagedbuf);
    free(hplane); free(hbuf);
    cudaStreamDestroy(stream);
    printf("c abi gpu ok\n");
    return 0;
}
