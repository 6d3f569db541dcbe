/*
 * lumen_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU statement of what LUMEN's KV checkpoint
 * pack and restore unpack compute.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may load this file.  It
 * shares no code, header, table or helper with paper_2606_17787_b200/ or
 * include/: it declares its own argument structs below.
 *
 * What it follows:
 *   - KV page = "a fixed-size block of cached keys and values for contiguous
 *     token positions" (section 2.1).
 *   - Pack  = step (3) of the incremental checkpoint pipeline: "workers track
 *     checkpoint progress and transmit only newly generated KV pages after
 *     each prefill or decode batch. A background thread copies these pages
 *     from GPU memory to the local pinned buffer" (section 4.2).
 *   - Unpack = KV-reuse recovery: "loading the matching KV pages into GPU
 *     memory" (section 4.3).
 *   - Buffer layout [req][layer][K|V][token][head][dim] is the build
 *     contract's (BASELINE.json configs[0]); SURVEY.md section 8(c) C1/C2
 *     writes the index map out, and this file is that map as five nested
 *     loops with a 2-byte scalar move innermost.  No blocking, no memcpy of
 *     runs, no SIMD, no reordering.
 *
 * The result is exact (a permutation of 16-bit words); parity with the CUDA
 * path is bit-for-bit.  Pins: tests/test_oracle_pins.py (P1-P10 of SURVEY.md
 * section 8(c) C7) and tests/test_golden_pack.py (P11: the hand-worked example
 * tests/golden/pack_tiny.txt).  No function here is "parity unpinned".
 *
 * lumen_oracle_pack_omp / lumen_oracle_unpack_omp are the same loop nest with
 * an OpenMP pragma over (request, layer) and a row memcpy innermost.  They
 * exist only to be *timed* as a multi-core CPU baseline and are asserted
 * equal to the plain functions in the tests before being used.
 */
#include <stdint.h>
#include <stddef.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* geometry of a paged pool: L layers, each with a K plane and a V plane of
 * shape [N pages][S tokens][H heads][D dims] of 16-bit words              */
typedef struct {
    int32_t L, H, D, S;
    int64_t N;
} oracle_geom;

/* one request: its page table (logical page -> physical page) and the token
 * range [tb, te) being checkpointed / restored                             */
typedef struct {
    const int32_t *PT;
    int64_t        PT_len;
    int64_t        tb, te;
} oracle_req;

enum {
    ORACLE_OK       =  0,
    ORACLE_EARG     = -1,   /* bad geometry / null pointer / bad range      */
    ORACLE_EPAGE    = -2,   /* page index outside [0, N) or table too short */
    ORACLE_ESIZE    = -3,   /* buffer too small                             */
    ORACLE_EOVERLAP = -4    /* unpack: two tokens map to one pool slot      */
};

/* ---- sizes (C1: off_0 = 0, off_{r+1} = off_r + n_r * 2L * E) ------------ */

int64_t lumen_oracle_total_elems(const oracle_geom *g, const oracle_req *reqs,
                                 int32_t R)
{
    int64_t E = (int64_t)g->H * g->D, off = 0;
    for (int32_t r = 0; r < R; ++r)
        off += (reqs[r].te - reqs[r].tb) * 2 * g->L * E;
    return off;
}

int64_t lumen_oracle_req_offset_elems(const oracle_geom *g,
                                      const oracle_req *reqs, int32_t r)
{
    int64_t E = (int64_t)g->H * g->D, off = 0;
    for (int32_t q = 0; q < r; ++q)
        off += (reqs[q].te - reqs[q].tb) * 2 * g->L * E;
    return off;
}

static int check_inputs(const oracle_geom *g, const oracle_req *reqs, int32_t R)
{
    if (!g || g->L <= 0 || g->H <= 0 || g->D <= 0 || g->S <= 0 || g->N <= 0)
        return ORACLE_EARG;
    if (R < 0 || (R > 0 && !reqs))
        return ORACLE_EARG;
    for (int32_t r = 0; r < R; ++r) {
        const oracle_req *q = &reqs[r];
        if (q->tb < 0 || q->te < q->tb)
            return ORACLE_EARG;
        for (int64_t t = q->tb; t < q->te; ++t) {
            int64_t lp = t / g->S;
            if (lp >= q->PT_len || !q->PT)
                return ORACLE_EPAGE;
            if (q->PT[lp] < 0 || (int64_t)q->PT[lp] >= g->N)
                return ORACLE_EPAGE;
        }
    }
    return ORACLE_OK;
}

/* ---- C1: pack ------------------------------------------------------------
 * for r, for l, for c in (K=0,V=1), for j in 0..n_r-1, for e in 0..E-1:
 *     t = tb_r + j ; p = PT_r[t div S] ; s = t mod S
 *     B[off_r + ((l*2 + c)*n_r + j)*E + e] = (c==0 ? Kp : Vp)[l][p][s][e]
 */
int lumen_oracle_pack(const oracle_geom *g,
                      const uint16_t *const *Kp, const uint16_t *const *Vp,
                      const oracle_req *reqs, int32_t R,
                      uint16_t *B, int64_t B_elems)
{
    int rc = check_inputs(g, reqs, R);
    if (rc) return rc;
    if (lumen_oracle_total_elems(g, reqs, R) > B_elems) return ORACLE_ESIZE;

    const int64_t E = (int64_t)g->H * g->D;
    const int64_t S = g->S;
    int64_t off = 0;
    for (int32_t r = 0; r < R; ++r) {
        const int64_t n = reqs[r].te - reqs[r].tb;
        for (int32_t l = 0; l < g->L; ++l) {
            for (int32_t c = 0; c < 2; ++c) {
                const uint16_t *plane = (c == 0) ? Kp[l] : Vp[l];
                for (int64_t j = 0; j < n; ++j) {
                    const int64_t t = reqs[r].tb + j;
                    const int64_t p = reqs[r].PT[t / S];
                    const int64_t s = t % S;
                    for (int64_t e = 0; e < E; ++e)
                        B[off + (((int64_t)l * 2 + c) * n + j) * E + e] =
                            plane[((p * S) + s) * E + e];
                }
            }
        }
        off += n * 2 * g->L * E;
    }
    return ORACLE_OK;
}

/* ---- C2: unpack (restore) --------------------------------------------------
 * Same index map with the assignment reversed.  Every pool word not addressed
 * by some (r, l, c, t in [tb_r, te_r)) is left as it was.  Destinations must
 * be disjoint: checked here token-slot by
 * token-slot with a brute-force O(tokens^2) scan when check_overlap != 0
 * (small cases only).
 */
int lumen_oracle_unpack(const oracle_geom *g,
                        uint16_t *const *Kp, uint16_t *const *Vp,
                        const oracle_req *reqs, int32_t R,
                        const uint16_t *B, int64_t B_elems, int check_overlap)
{
    int rc = check_inputs(g, reqs, R);
    if (rc) return rc;
    if (lumen_oracle_total_elems(g, reqs, R) > B_elems) return ORACLE_ESIZE;

    const int64_t E = (int64_t)g->H * g->D;
    const int64_t S = g->S;

    if (check_overlap) {
        for (int32_t r = 0; r < R; ++r)
            for (int64_t t = reqs[r].tb; t < reqs[r].te; ++t) {
                int64_t a = (int64_t)reqs[r].PT[t / S] * S + t % S;
                for (int32_t q = 0; q <= r; ++q)
                    for (int64_t u = reqs[q].tb; u < reqs[q].te; ++u) {
                        if (q == r && u >= t) break;
                        int64_t b = (int64_t)reqs[q].PT[u / S] * S + u % S;
                        if (a == b) return ORACLE_EOVERLAP;
                    }
            }
    }

    int64_t off = 0;
    for (int32_t r = 0; r < R; ++r) {
        const int64_t n = reqs[r].te - reqs[r].tb;
        for (int32_t l = 0; l < g->L; ++l) {
            for (int32_t c = 0; c < 2; ++c) {
                uint16_t *plane = (c == 0) ? Kp[l] : Vp[l];
                for (int64_t j = 0; j < n; ++j) {
                    const int64_t t = reqs[r].tb + j;
                    const int64_t p = reqs[r].PT[t / S];
                    const int64_t s = t % S;
                    for (int64_t e = 0; e < E; ++e)
                        plane[((p * S) + s) * E + e] =
                            B[off + (((int64_t)l * 2 + c) * n + j) * E + e];
                }
            }
        }
        off += n * 2 * g->L * E;
    }
    return ORACLE_OK;
}

/* ---- one output at a time (full-size sampled parity) -----------------------
 * Where does buffer word (r, l, c, j, e) live in B, and which pool word is it?
 * Written straight from C1 so a test can check single words of a 32 GiB
 * buffer without materialising it.
 */
int64_t lumen_oracle_buffer_index(const oracle_geom *g, const oracle_req *reqs,
                                  int32_t r, int32_t l, int32_t c,
                                  int64_t j, int64_t e)
{
    const int64_t E = (int64_t)g->H * g->D;
    const int64_t n = reqs[r].te - reqs[r].tb;
    return lumen_oracle_req_offset_elems(g, reqs, r) +
           (((int64_t)l * 2 + c) * n + j) * E + e;
}

/* index of the pool word, inside plane (l, c), that buffer word (r,*,*,j,e)
 * is copied from (pack) / to (unpack); -1 if the page table does not cover it */
int64_t lumen_oracle_pool_index(const oracle_geom *g, const oracle_req *reqs,
                                int32_t r, int64_t j, int64_t e)
{
    const int64_t E = (int64_t)g->H * g->D;
    const int64_t t = reqs[r].tb + j;
    const int64_t lp = t / g->S;
    if (lp >= reqs[r].PT_len) return -1;
    const int64_t p = reqs[r].PT[lp];
    const int64_t s = t % g->S;
    return (p * g->S + s) * E + e;
}

/* ---- timed multi-core variants (baseline only; see header) ---------------- */

int lumen_oracle_pack_omp(const oracle_geom *g,
                          const uint16_t *const *Kp, const uint16_t *const *Vp,
                          const oracle_req *reqs, int32_t R,
                          uint16_t *B, int64_t B_elems)
{
    int rc = check_inputs(g, reqs, R);
    if (rc) return rc;
    if (lumen_oracle_total_elems(g, reqs, R) > B_elems) return ORACLE_ESIZE;
    const int64_t E = (int64_t)g->H * g->D, S = g->S;
    const int32_t L = g->L;
#pragma omp parallel for collapse(2) schedule(dynamic, 1)
    for (int32_t r = 0; r < R; ++r) {
        for (int32_t l = 0; l < L; ++l) {
            const int64_t n = reqs[r].te - reqs[r].tb;
            const int64_t off = lumen_oracle_req_offset_elems(g, reqs, r);
            for (int32_t c = 0; c < 2; ++c) {
                const uint16_t *plane = (c == 0) ? Kp[l] : Vp[l];
                for (int64_t j = 0; j < n; ++j) {
                    const int64_t t = reqs[r].tb + j;
                    const int64_t p = reqs[r].PT[t / S], s = t % S;
                    memcpy(&B[off + (((int64_t)l * 2 + c) * n + j) * E],
                           &plane[(p * S + s) * E], (size_t)E * 2);
                }
            }
        }
    }
    return ORACLE_OK;
}

int lumen_oracle_unpack_omp(const oracle_geom *g,
                            uint16_t *const *Kp, uint16_t *const *Vp,
                            const oracle_req *reqs, int32_t R,
                            const uint16_t *B, int64_t B_elems)
{
    int rc = check_inputs(g, reqs, R);
    if (rc) return rc;
    if (lumen_oracle_total_elems(g, reqs, R) > B_elems) return ORACLE_ESIZE;
    const int64_t E = (int64_t)g->H * g->D, S = g->S;
    const int32_t L = g->L;
#pragma omp parallel for collapse(2) schedule(dynamic, 1)
    for (int32_t r = 0; r < R; ++r) {
        for (int32_t l = 0; l < L; ++l) {
            const int64_t n = reqs[r].te - reqs[r].tb;
            const int64_t off = lumen_oracle_req_offset_elems(g, reqs, r);
            for (int32_t c = 0; c < 2; ++c) {
                uint16_t *plane = (c == 0) ? Kp[l] : Vp[l];
                for (int64_t j = 0; j < n; ++j) {
                    const int64_t t = reqs[r].tb + j;
                    const int64_t p = reqs[r].PT[t / S], s = t % S;
                    memcpy(&plane[(p * S + s) * E],
                           &B[off + (((int64_t)l * 2 + c) * n + j) * E],
                           (size_t)E * 2);
                }
            }
        }
    }
    return ORACLE_OK;
}

int lumen_oracle_omp_threads(void)
{
    int n = 1;
#ifdef _OPENMP
#pragma omp parallel
    {
#pragma omp single
        n = omp_get_num_threads();
    }
#endif
    return n;
}

/* ---- explicit buffer layout (checkpoint store) ---------------
 * A checkpoint store keeps what it received: a request's checkpoint is the sequence of its
 * delta buffers ("transmit only newly generated KV pages"; one checkpoint per
 * request), and a recovery restores the longest checkpointed prefix
 * (PAPER.md:157), which may end inside the last delta.  So pack / unpack are also defined
 * for a buffer in which request r's block sits at an explicit element offset off_r with an
 * explicit plane stride st_r >= n_r (in tokens):
 *     B[off_r + ((l*2 + c)*st_r + j)*E + e]  <->  plane(l,c)[PT_r[t div S]][t mod S][e]
 * The dense layout of C1 is the special case off_r = prefix sum, st_r = n_r.  Words of B
 * that no (r, l, c, j, e) addresses are never read or written.
 */
typedef struct {
    int64_t off_elems;      /* element offset of the request's block in B */
    int64_t stride_tokens;  /* tokens between consecutive planes, >= n_r  */
} oracle_layout;

static int check_layout(const oracle_geom *g, const oracle_req *reqs, const oracle_layout *lay,
                        int32_t R, int64_t B_elems)
{
    const int64_t E = (int64_t)g->H * g->D;
    if (R > 0 && !lay) return ORACLE_EARG;
    for (int32_t r = 0; r < R; ++r) {
        const int64_t n = reqs[r].te - reqs[r].tb;
        if (lay[r].off_elems < 0 || lay[r].stride_tokens < n) return ORACLE_EARG;
        if (n > 0 &&
            lay[r].off_elems + (((int64_t)2 * g->L - 1) * lay[r].stride_tokens + n) * E > B_elems)
            return ORACLE_ESIZE;
    }
    return ORACLE_OK;
}

int lumen_oracle_pack_layout(const oracle_geom *g,
                             const uint16_t *const *Kp, const uint16_t *const *Vp,
                             const oracle_req *reqs, const oracle_layout *lay, int32_t R,
                             uint16_t *B, int64_t B_elems)
{
    int rc = check_inputs(g, reqs, R);
    if (rc) return rc;
    rc = check_layout(g, reqs, lay, R, B_elems);
    if (rc) return rc;
    const int64_t E = (int64_t)g->H * g->D;
    const int64_t S = g->S;
    for (int32_t r = 0; r < R; ++r) {
        const int64_t n = reqs[r].te - reqs[r].tb;
        for (int32_t l = 0; l < g->L; ++l)
            for (int32_t c = 0; c < 2; ++c) {
                const uint16_t *plane = (c == 0) ? Kp[l] : Vp[l];
                for (int64_t j = 0; j < n; ++j) {
                    const int64_t t = reqs[r].tb + j;
                    const int64_t p = reqs[r].PT[t / S];
                    const int64_t s = t % S;
                    for (int64_t e = 0; e < E; ++e)
                        B[lay[r].off_elems + (((int64_t)l * 2 + c) * lay[r].stride_tokens + j) * E + e] =
                            plane[((p * S) + s) * E + e];
                }
            }
    }
    return ORACLE_OK;
}

int lumen_oracle_unpack_layout(const oracle_geom *g,
                               uint16_t *const *Kp, uint16_t *const *Vp,
                               const oracle_req *reqs, const oracle_layout *lay, int32_t R,
                               const uint16_t *B, int64_t B_elems)
{
    int rc = check_inputs(g, reqs, R);
    if (rc) return rc;
    rc = check_layout(g, reqs, lay, R, B_elems);
    if (rc) return rc;
    const int64_t E = (int64_t)g->H * g->D;
    const int64_t S = g->S;
    for (int32_t r = 0; r < R; ++r) {
        const int64_t n = reqs[r].te - reqs[r].tb;
        for (int32_t l = 0; l < g->L; ++l)
            for (int32_t c = 0; c < 2; ++c) {
                uint16_t *plane = (c == 0) ? Kp[l] : Vp[l];
                for (int64_t j = 0; j < n; ++j) {
                    const int64_t t = reqs[r].tb + j;
                    const int64_t p = reqs[r].PT[t / S];
                    const int64_t s = t % S;
                    for (int64_t e = 0; e < E; ++e)
                        plane[((p * S) + s) * E + e] =
                            B[lay[r].off_elems + (((int64_t)l * 2 + c) * lay[r].stride_tokens + j) * E + e];
                }
            }
    }
    return ORACLE_OK;
}
