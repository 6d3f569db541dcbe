/*
 * tags_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain CPU statement of LUMEN's page tags and of the longest-contiguous-prefix lookup
 * (SURVEY.md section 8(f) row f1).  Shares nothing with paper_2606_17787_b200/ or
 * include/.  What it follows:
 *
 *   "each transferred page carries a page tag: a hash value of the token IDs stored in
 *    page i, paired with the page's end position in the request token sequence (i.e., the
 *    cumulative token length after page i). Since this tag derives purely from the
 *    request's token sequence, any worker can independently reconstruct it using the token
 *    history ... if a failure interrupts a transfer, the lookup simply halts at the last
 *    valid tag" (section 4.2), and "the holder deterministically regenerates
 *    page tags to locate the longest contiguous checkpointed prefix within its local
 *    store" (section 4.3).
 *
 * The paper does not name the hash function nor say whether the tag of page i depends on
 * earlier pages.  Reading A12: the text is taken literally --
 * the hash covers "the token IDs stored in page i" only -- and the hash is 64-bit FNV-1a
 * over the little-endian bytes of the page's int32 token IDs.  THE CHOICE OF HASH IS
 * PARITY UNPINNED (nothing in the paper fixes it); the implementation of the chosen hash is
 * pinned to the published FNV-1a test vectors, and the lookup to brute force
 * (tests/test_tags.py).
 *
 * Page i of a request with `len` tokens and page size S holds tokens
 * [i*S, min((i+1)*S, len)); its end position is min((i+1)*S, len).  A last page that is
 * not full is hashed over the tokens it holds.
 */
#include <stdint.h>
#include <stddef.h>

typedef struct {
    uint64_t hash;      /* FNV-1a 64 of the page's token IDs                      */
    int64_t  end_pos;   /* cumulative token length after this page                */
} oracle_tag;

/* 64-bit FNV-1a, byte by byte: offset basis 0xcbf29ce484222325, prime 0x100000001b3 */
uint64_t tags_oracle_fnv1a64(const uint8_t *bytes, int64_t n) {
    uint64_t h = 0xcbf29ce484222325ULL;
    for (int64_t i = 0; i < n; ++i) {
        h ^= (uint64_t)bytes[i];
        h *= 0x100000001b3ULL;
    }
    return h;
}

/* number of pages of a request of `len` tokens */
int64_t tags_oracle_num_pages(int64_t len, int64_t S) {
    if (len < 0 || S < 1) return -1;
    return (len + S - 1) / S;
}

/* tags of all pages of one request.  out has tags_oracle_num_pages(len, S) entries. */
int tags_oracle_page_tags(const int32_t *token_ids, int64_t len, int64_t S, oracle_tag *out) {
    if (len < 0 || S < 1 || (len > 0 && (!token_ids || !out))) return -1;
    int64_t pages = (len + S - 1) / S;
    for (int64_t i = 0; i < pages; ++i) {
        int64_t first = i * S;
        int64_t end = (i + 1) * S < len ? (i + 1) * S : len;
        uint8_t le[4];
        uint64_t h = 0xcbf29ce484222325ULL;
        for (int64_t t = first; t < end; ++t) {
            uint32_t v = (uint32_t)token_ids[t];
            le[0] = (uint8_t)(v & 0xff);          /* little-endian bytes of the token ID */
            le[1] = (uint8_t)((v >> 8) & 0xff);
            le[2] = (uint8_t)((v >> 16) & 0xff);
            le[3] = (uint8_t)((v >> 24) & 0xff);
            for (int b = 0; b < 4; ++b) {
                h ^= (uint64_t)le[b];
                h *= 0x100000001b3ULL;
            }
        }
        out[i].hash = h;
        out[i].end_pos = end;
    }
    return 0;
}

/*
 * Longest contiguous checkpointed prefix, in tokens: walk the regenerated tags in page order
 * and halt at the first one that is not among the `stored` tags of this request
 * (membership by linear scan: the store is whatever arrived, in any order).
 */
int64_t tags_oracle_longest_prefix(const oracle_tag *regen, int64_t n_regen,
                                   const oracle_tag *stored, int64_t n_stored) {
    int64_t prefix = 0;
    for (int64_t i = 0; i < n_regen; ++i) {
        int found = 0;
        for (int64_t j = 0; j < n_stored; ++j)
            if (stored[j].hash == regen[i].hash && stored[j].end_pos == regen[i].end_pos) {
                found = 1;
                break;
            }
        if (!found) break;
        prefix = regen[i].end_pos;
    }
    return prefix;
}
