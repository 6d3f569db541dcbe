// Host plan builder: step a2 of the hot path.
// Splits each request's token range [t_begin, t_end) -- the KV produced since the
// last checkpoint, PAPER.md:145 -- at page boundaries into token-runs, computes the
// per-request buffer offsets (exclusive prefix sum of n_r * 2L * row), optionally
// merges runs over physically adjacent pages, and validates everything so that the
// kernels never need a bounds check.  Pure C++: no CUDA types or calls in here.
#include "plan.hpp"

#include <algorithm>
#include <limits>

namespace lumen {
namespace {

struct Extent {           // a pool-contiguous, buffer-contiguous stretch of tokens
    int64_t src_off = 0;  // byte offset inside a plane
    int64_t dst_tok = 0;  // request-relative first token
    int64_t count = 0;    // tokens
};

inline void emit(HostPlan* hp, const Extent& x, int32_t req, int64_t chunk_tokens) {
    int64_t done = 0;
    while (done < x.count) {
        const int64_t c = std::min(chunk_tokens, x.count - done);
        const uint64_t off16 = static_cast<uint64_t>(x.src_off + done * hp->row_bytes) >> 4;
        RunDesc d;
        d.src_lo = static_cast<uint32_t>(off16 & 0xFFFFFFFFu);
        d.src_hi = static_cast<uint16_t>(off16 >> 32);
        d.dst_tok = static_cast<uint32_t>(x.dst_tok + done);
        d.req = static_cast<uint32_t>(req);
        d.count = static_cast<uint16_t>(c);
        hp->runs.push_back(d);
        hp->max_count = std::max<int32_t>(hp->max_count, static_cast<int32_t>(c));
        done += c;
    }
}

}  // namespace

int build_host_plan(const lumen_kv_geom* g, const lumen_kv_req* reqs,
                    const lumen_kv_req_layout* layouts, int32_t num_reqs, uint32_t flags,
                    HostPlan* hp) {
    if (!g || !hp) return LUMEN_KV_EINVAL;
    if (num_reqs < 0 || (num_reqs > 0 && !reqs)) return LUMEN_KV_EINVAL;
    const uint32_t known = LUMEN_KV_VALIDATE_UNIQUE_DST | LUMEN_KV_MERGE_ADJACENT |
                           LUMEN_KV_HOST_ONLY | LUMEN_KV_NO_INLINE | LUMEN_KV_KERNEL_MASK;
    if (flags & ~known) return LUMEN_KV_EINVAL;
    if (g->num_layers < 1 || g->kv_heads < 1 || g->head_dim < 1 || g->page_size < 1 ||
        g->elem_bytes < 1 || g->reserved != 0)
        return LUMEN_KV_EINVAL;
    if (g->num_pages < 1 || g->num_pages >= (int64_t{1} << 31)) return LUMEN_KV_EINVAL;
    if (g->num_layers > 32767) return LUMEN_KV_EINVAL;

    const int64_t S = g->page_size;
    const int64_t row = int64_t{g->kv_heads} * g->head_dim * g->elem_bytes;
    if (row % 16 != 0 || row > (int64_t{1} << 30)) return LUMEN_KV_EINVAL;
    if (S > (int64_t{1} << 20)) return LUMEN_KV_EINVAL;
    const int64_t dense = S * row;
    int64_t stride = g->page_stride_bytes;
    if (stride == 0) stride = dense;
    if (stride < dense || stride % 16 != 0) return LUMEN_KV_EINVAL;
    // pool byte offsets must fit 48 bits of 16-byte units
    if (static_cast<long double>(stride) * static_cast<long double>(g->num_pages) >=
        static_cast<long double>(int64_t{1} << 52))
        return LUMEN_KV_EINVAL;

    hp->geom = *g;
    hp->row_bytes = row;
    hp->page_stride = stride;
    hp->runs.clear();
    hp->reqs.assign(static_cast<size_t>(num_reqs), ReqDesc{0, 0});
    hp->req_offset.assign(static_cast<size_t>(num_reqs) + 1, 0);
    hp->req_tokens.assign(static_cast<size_t>(num_reqs), 0);
    hp->req_stride.assign(static_cast<size_t>(num_reqs), 0);
    hp->max_count = 0;

    const bool merge = (flags & LUMEN_KV_MERGE_ADJACENT) && stride == dense;
    const bool unique = (flags & LUMEN_KV_VALIDATE_UNIQUE_DST) != 0;
    const int64_t chunk_tokens =
        std::min<int64_t>(65535, std::max<int64_t>(1, kChunkBytes / row));
    const int64_t planes = 2 * int64_t{g->num_layers};

    // pass 1: validate ranges, sizes and page indices; count touched pages
    int64_t tokens = 0, touched = 0, extent = 0;
    for (int32_t r = 0; r < num_reqs; ++r) {
        const lumen_kv_req& q = reqs[r];
        if (q.t_begin < 0 || q.t_end < q.t_begin || q.page_table_len < 0) return LUMEN_KV_EINVAL;
        const int64_t n = q.t_end - q.t_begin;
        if (n >= (int64_t{1} << 32)) return LUMEN_KV_EINVAL;
        hp->req_tokens[r] = n;
        if (layouts) {
            const lumen_kv_req_layout& ly = layouts[r];
            if (ly.buf_offset < 0 || ly.buf_offset % row != 0 || ly.plane_stride_tokens < n ||
                ly.plane_stride_tokens >= (int64_t{1} << 40) ||
                ly.buf_offset > (std::numeric_limits<int64_t>::max() / 4))
                return LUMEN_KV_EINVAL;
            hp->reqs[r].row_base = ly.buf_offset / row;
            hp->reqs[r].n = ly.plane_stride_tokens;
            hp->req_offset[r] = ly.buf_offset;
            hp->req_stride[r] = ly.plane_stride_tokens;
            if (n > 0) {
                // largest byte addressed + 1 = buf_offset + ((planes-1)*stride + n)*row, every
                // step checked: stride < 2^40, row <= 2^30 and planes <= 65534 alone do not
                // keep the product inside 63 bits
                int64_t rows = 0, ext = 0;
                if (__builtin_mul_overflow(planes - 1, ly.plane_stride_tokens, &rows) ||
                    __builtin_add_overflow(rows, n, &rows) ||
                    __builtin_mul_overflow(rows, row, &ext) ||
                    __builtin_add_overflow(ext, ly.buf_offset, &ext) ||
                    ext > (std::numeric_limits<int64_t>::max() / 4))
                    return LUMEN_KV_EINVAL;
                extent = std::max(extent, ext);
            }
        } else {
            hp->reqs[r].row_base = tokens * planes;
            hp->reqs[r].n = n;
            hp->req_offset[r] = tokens * planes * row;
            hp->req_stride[r] = n;
        }
        if (n == 0) continue;
        const int64_t lp0 = q.t_begin / S, lp1 = (q.t_end - 1) / S;
        if (!q.page_table || lp1 >= q.page_table_len) return LUMEN_KV_ERANGE;
        for (int64_t lp = lp0; lp <= lp1; ++lp) {
            const int32_t p = q.page_table[lp];
            if (p < 0 || int64_t{p} >= g->num_pages) return LUMEN_KV_ERANGE;
        }
        touched += lp1 - lp0 + 1;
        tokens += n;
        if (tokens > (std::numeric_limits<int64_t>::max() / 4) / (planes * row))
            return LUMEN_KV_EINVAL;
    }
    hp->total_tokens = tokens;
    hp->total_bytes = layouts ? extent : tokens * planes * row;
    hp->req_offset[num_reqs] = hp->total_bytes;

    // optional: every pool token slot addressed at most once across the whole plan (A5).
    // Pages are checked first (bitmap or sort); only pages that appear twice -- e.g. two
    // consecutive deltas of one request meeting inside a page -- get the exact slot-interval test.
    if (unique && touched > 0) {
        const int64_t N = g->num_pages;
        std::vector<int32_t> dup;
        if (N <= 64 * touched || N <= (int64_t{1} << 23)) {
            std::vector<uint64_t> bits(static_cast<size_t>((N + 63) / 64), 0);
            for (int32_t r = 0; r < num_reqs; ++r) {
                const lumen_kv_req& q = reqs[r];
                if (q.t_end == q.t_begin) continue;
                for (int64_t lp = q.t_begin / S; lp <= (q.t_end - 1) / S; ++lp) {
                    const uint32_t p = static_cast<uint32_t>(q.page_table[lp]);
                    uint64_t& w = bits[p >> 6];
                    const uint64_t m = uint64_t{1} << (p & 63);
                    if (w & m) dup.push_back(static_cast<int32_t>(p));
                    w |= m;
                }
            }
        } else {
            std::vector<int32_t> all;
            all.reserve(static_cast<size_t>(touched));
            for (int32_t r = 0; r < num_reqs; ++r) {
                const lumen_kv_req& q = reqs[r];
                if (q.t_end == q.t_begin) continue;
                for (int64_t lp = q.t_begin / S; lp <= (q.t_end - 1) / S; ++lp)
                    all.push_back(q.page_table[lp]);
            }
            std::sort(all.begin(), all.end());
            for (size_t i = 1; i < all.size(); ++i)
                if (all[i] == all[i - 1]) dup.push_back(all[i]);
        }
        if (!dup.empty()) {
            std::sort(dup.begin(), dup.end());
            dup.erase(std::unique(dup.begin(), dup.end()), dup.end());
            struct Span { int32_t page; int32_t lo, hi; };
            std::vector<Span> spans;
            for (int32_t r = 0; r < num_reqs; ++r) {
                const lumen_kv_req& q = reqs[r];
                if (q.t_end == q.t_begin) continue;
                for (int64_t lp = q.t_begin / S; lp <= (q.t_end - 1) / S; ++lp) {
                    const int32_t p = q.page_table[lp];
                    if (!std::binary_search(dup.begin(), dup.end(), p)) continue;
                    const int64_t lo = std::max(q.t_begin, lp * S) - lp * S;
                    const int64_t hi = std::min(q.t_end, (lp + 1) * S) - lp * S;
                    spans.push_back(Span{p, static_cast<int32_t>(lo), static_cast<int32_t>(hi)});
                }
            }
            std::sort(spans.begin(), spans.end(), [](const Span& a, const Span& b) {
                return a.page != b.page ? a.page < b.page : a.lo < b.lo;
            });
            for (size_t i = 1; i < spans.size(); ++i)
                if (spans[i].page == spans[i - 1].page && spans[i].lo < spans[i - 1].hi)
                    return LUMEN_KV_EOVERLAP;
            // (sorted by lo, so comparing with the predecessor's hi suffices once overlaps are
            //  rejected: non-overlapping predecessors have increasing hi)
        }
    }

    // pass 2: flatten into runs
    // a page span of k tokens yields ceil(k / chunk_tokens) <= k / chunk_tokens + 1 runs
    hp->runs.reserve(static_cast<size_t>(tokens / chunk_tokens + touched));
    hp->req_run_begin.assign(static_cast<size_t>(num_reqs) + 1, 0);
    for (int32_t r = 0; r < num_reqs; ++r) {
        const lumen_kv_req& q = reqs[r];
        hp->req_run_begin[r] = static_cast<int64_t>(hp->runs.size());
        if (q.t_end == q.t_begin) continue;
        Extent cur;
        int64_t t = q.t_begin;
        while (t < q.t_end) {
            const int64_t lp = t / S, slot = t % S;
            const int64_t cnt = std::min(S - slot, q.t_end - t);
            const int64_t off = int64_t{q.page_table[lp]} * stride + slot * row;
            if (cur.count > 0 && merge && cur.src_off + cur.count * row == off) {
                cur.count += cnt;           // physically adjacent: extend
            } else {
                if (cur.count > 0) emit(hp, cur, r, chunk_tokens);
                cur.src_off = off;
                cur.dst_tok = t - q.t_begin;
                cur.count = cnt;
            }
            t += cnt;
        }
        if (cur.count > 0) emit(hp, cur, r, chunk_tokens);
    }
    hp->req_run_begin[num_reqs] = static_cast<int64_t>(hp->runs.size());
    return LUMEN_KV_OK;
}

int build_chunks(const HostPlan& hp, const RunDesc* runs, int64_t slot_bytes,
                 std::vector<Chunk>* out) {
    out->clear();
    if (slot_bytes < 16 || slot_bytes % 16 != 0) return LUMEN_KV_EINVAL;
    const int64_t row = hp.row_bytes;
    const int32_t planes = 2 * hp.geom.num_layers;
    if (int64_t{hp.max_count} * row > slot_bytes) return LUMEN_KV_ESIZE;
    const int64_t R = static_cast<int64_t>(hp.req_tokens.size());
    Chunk group{0, 0, 0, planes, 0, 0};          // whole, buffer-adjacent requests accumulated so far
    auto flush = [&]() {
        if (group.b1 > group.b0) out->push_back(group);
        group.b0 = group.b1 = 0;
    };
    for (int64_t r = 0; r < R; ++r) {
        const int64_t n = hp.req_tokens[r];
        if (n == 0) continue;
        const int64_t off = hp.req_offset[r];
        const int64_t pitch = hp.req_stride[r] * row;   // bytes between consecutive planes
        const int64_t pb = n * row;                      // bytes of one plane of this request
        const bool dense = (hp.req_stride[r] == n);
        const int64_t bytes = pb * planes;
        const int64_t ra = hp.req_run_begin[r], rb = hp.req_run_begin[r + 1];
        if (dense && bytes <= slot_bytes) {
            const bool open = group.b1 > group.b0;
            if (open && (off != group.b1 || group.b1 - group.b0 + bytes > slot_bytes)) flush();
            if (group.b1 == group.b0) { group.ra = ra; group.b0 = off; }
            group.rb = rb;
            group.b1 = off + bytes;
            continue;
        }
        flush();
        if (pb <= slot_bytes) {
            // dense blocks: as many whole planes as fit; strided blocks: one plane per chunk
            const int32_t k = dense ? static_cast<int32_t>(std::min<int64_t>(planes, slot_bytes / pb)) : 1;
            for (int32_t p0 = 0; p0 < planes; p0 += k) {
                const int32_t p1 = std::min(planes, p0 + k);
                out->push_back(Chunk{ra, rb, p0, p1, off + p0 * pitch, off + (p1 - 1) * pitch + pb});
            }
            continue;
        }
        for (int32_t p = 0; p < planes; ++p) {   // split the token axis at run boundaries
            int64_t a = ra;
            while (a < rb) {
                int64_t b = a, sz = 0;
                while (b < rb && sz + int64_t{runs[b].count} * row <= slot_bytes) {
                    sz += int64_t{runs[b].count} * row;
                    ++b;
                }
                const int64_t b0 = off + p * pitch + int64_t{runs[a].dst_tok} * row;
                out->push_back(Chunk{a, b, p, p + 1, b0, b0 + sz});
                a = b;
            }
        }
    }
    flush();
    return LUMEN_KV_OK;
}

}  // namespace lumen
