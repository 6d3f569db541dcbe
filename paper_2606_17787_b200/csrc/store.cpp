// Checkpoint store (include/lumen_kv.h): reserved footprints in a
// caller-provided host arena, append-only deltas with their page tags, lookups that only see
// completely received deltas.  Pure host C++: no CUDA in here.
#include <algorithm>
#include <condition_variable>
#include <cstring>
#include <map>
#include <mutex>
#include <new>
#include <thread>
#include <unordered_map>
#include <vector>

#include "lumen_kv.h"

namespace {

struct Delta {
    int64_t t_begin, t_end;   // token range
    int64_t offset;           // byte offset in the arena
};

struct Entry {
    int64_t region_off = 0;     // reserved region [region_off, region_off + region_bytes)
    int64_t region_bytes = 0;
    int64_t max_tokens = 0;
    int64_t tokens = 0;         // tokens completely received
    int64_t receiving = 0;      // tokens of appends in progress / claimed (not yet visible)
    int claims = 0;             // outstanding lumen_kv_store_acquire claims (filled in place, in order)
    std::vector<Delta> deltas;
    std::vector<lumen_kv_tag> tags;
};

constexpr int64_t kParallelCopyMin = 1 << 20;   // below this one memcpy beats waking the pool

// Persistent copy threads: an append is cut into slices that the pool's threads and the caller
// copy together.  Waking sleeping threads costs microseconds, starting new ones per append
// (the first version) cost tens -- too much for the 2.5 MiB deltas of a decode step.
class CopyPool {
public:
    explicit CopyPool(int threads) {
        for (int i = 1; i < threads; ++i) workers_.emplace_back([this] { loop(); });
    }
    ~CopyPool() {
        {
            std::lock_guard<std::mutex> g(mu_);
            stop_ = true;
        }
        cv_.notify_all();
        for (auto& t : workers_) t.join();
    }
    // One copy at a time (appends of different requests queue up here: the memory bus is shared).
    void copy(char* dst, const char* src, int64_t bytes) {
        const int64_t parts = static_cast<int64_t>(workers_.size()) + 1;
        if (parts == 1 || bytes < kParallelCopyMin) {
            std::memcpy(dst, src, static_cast<size_t>(bytes));
            return;
        }
        std::lock_guard<std::mutex> one(job_mu_);
        const int64_t slice = ((bytes / parts) + 4095) & ~int64_t{4095};
        {
            std::lock_guard<std::mutex> g(mu_);
            dst_ = dst;
            src_ = src;
            bytes_ = bytes;
            slice_ = slice;
            next_ = slice;          // slice 0 is the caller's
            pending_ = 0;
            for (int64_t at = slice; at < bytes; at += slice) ++pending_;
            ++generation_;
        }
        cv_.notify_all();
        std::memcpy(dst, src, static_cast<size_t>(std::min(slice, bytes)));
        std::unique_lock<std::mutex> lk(mu_);
        done_cv_.wait(lk, [&] { return pending_ == 0; });
    }

private:
    void loop() {
        uint64_t seen = 0;
        std::unique_lock<std::mutex> lk(mu_);
        for (;;) {
            cv_.wait(lk, [&] { return stop_ || (generation_ != seen && next_ < bytes_); });
            if (stop_) return;
            while (next_ < bytes_) {
                const int64_t at = next_;
                next_ += slice_;
                const int64_t n = std::min(slice_, bytes_ - at);
                char* d = dst_ + at;
                const char* s = src_ + at;
                lk.unlock();
                std::memcpy(d, s, static_cast<size_t>(n));
                lk.lock();
                if (--pending_ == 0) done_cv_.notify_all();
            }
            seen = generation_;
        }
    }
    std::vector<std::thread> workers_;
    std::mutex mu_, job_mu_;
    std::condition_variable cv_, done_cv_;
    char* dst_ = nullptr;
    const char* src_ = nullptr;
    int64_t bytes_ = 0, slice_ = 0, next_ = 0, pending_ = 0;
    uint64_t generation_ = 0;
    bool stop_ = false;
};

}  // namespace

struct lumen_kv_store {
    char* arena = nullptr;
    int64_t arena_bytes = 0;
    int64_t token_bytes = 0;
    int32_t page_size = 0;
    int32_t copy_threads = 1;
    mutable std::mutex mu;
    std::map<int64_t, int64_t> free_;                    // offset -> bytes, coalesced
    std::unordered_map<uint64_t, Entry> reqs;
    int64_t reserved = 0;
    int64_t sink_errors = 0;
    CopyPool* pool = nullptr;
    ~lumen_kv_store() { delete pool; }
};

extern "C" {

int lumen_kv_store_create(void* arena, int64_t arena_bytes, int64_t token_bytes,
                          int32_t page_size, int32_t copy_threads, lumen_kv_store** out) {
    if (!out) return LUMEN_KV_EINVAL;
    *out = nullptr;
    if (!arena || (reinterpret_cast<uintptr_t>(arena) & 15) || arena_bytes < 0 ||
        token_bytes < 16 || token_bytes % 16 != 0 || page_size < 1 || copy_threads < 1 ||
        copy_threads > 256)
        return LUMEN_KV_EINVAL;
    lumen_kv_store* s = new (std::nothrow) lumen_kv_store();
    if (!s) return LUMEN_KV_ENOMEM;
    s->arena = static_cast<char*>(arena);
    s->arena_bytes = arena_bytes;
    s->token_bytes = token_bytes;
    s->page_size = page_size;
    s->copy_threads = copy_threads;
    s->pool = new (std::nothrow) CopyPool(copy_threads);
    if (!s->pool) {
        delete s;
        return LUMEN_KV_ENOMEM;
    }
    if (arena_bytes > 0) s->free_[0] = arena_bytes;
    *out = s;
    return LUMEN_KV_OK;
}

void lumen_kv_store_destroy(lumen_kv_store* s) { delete s; }

int64_t lumen_kv_store_available(const lumen_kv_store* s) {
    if (!s) return LUMEN_KV_EINVAL;
    std::lock_guard<std::mutex> g(s->mu);
    return s->arena_bytes - s->reserved;
}

int64_t lumen_kv_store_reserved(const lumen_kv_store* s) {
    if (!s) return LUMEN_KV_EINVAL;
    std::lock_guard<std::mutex> g(s->mu);
    return s->reserved;
}

int lumen_kv_store_reserve(lumen_kv_store* s, uint64_t id, int64_t max_tokens) {
    if (!s || max_tokens < 1 || max_tokens > (int64_t{1} << 40) / s->token_bytes)
        return LUMEN_KV_EINVAL;
    const int64_t need = max_tokens * s->token_bytes;
    std::lock_guard<std::mutex> g(s->mu);
    if (s->reqs.count(id)) return LUMEN_KV_EINVAL;
    for (auto it = s->free_.begin(); it != s->free_.end(); ++it) {   // first fit, lowest offset
        if (it->second < need) continue;
        Entry e;
        e.region_off = it->first;
        e.region_bytes = need;
        e.max_tokens = max_tokens;
        const int64_t rest = it->second - need;
        s->free_.erase(it);
        if (rest > 0) s->free_[e.region_off + need] = rest;
        s->reserved += need;
        s->reqs.emplace(id, std::move(e));
        return LUMEN_KV_OK;
    }
    return LUMEN_KV_ENOMEM;
}

int lumen_kv_store_release(lumen_kv_store* s, uint64_t id) {
    if (!s) return LUMEN_KV_EINVAL;
    std::lock_guard<std::mutex> g(s->mu);
    auto it = s->reqs.find(id);
    if (it == s->reqs.end() || it->second.receiving) return LUMEN_KV_EINVAL;
    int64_t off = it->second.region_off, bytes = it->second.region_bytes;
    s->reserved -= bytes;
    s->reqs.erase(it);
    auto next = s->free_.lower_bound(off);                 // coalesce with the neighbours
    if (next != s->free_.end() && off + bytes == next->first) {
        bytes += next->second;
        next = s->free_.erase(next);
    }
    if (next != s->free_.begin()) {
        auto prev = std::prev(next);
        if (prev->first + prev->second == off) {
            prev->second += bytes;
            return LUMEN_KV_OK;
        }
    }
    s->free_[off] = bytes;
    return LUMEN_KV_OK;
}

int lumen_kv_store_append(lumen_kv_store* s, uint64_t id, int64_t t_begin, int64_t t_end,
                          const void* delta, int64_t delta_bytes, const lumen_kv_tag* tags,
                          int32_t n_tags) {
    if (!s || t_begin < 0 || t_end < t_begin || n_tags < 0 || (n_tags > 0 && !tags))
        return LUMEN_KV_EINVAL;
    const int64_t n = t_end - t_begin;
    if (delta_bytes != n * s->token_bytes) return LUMEN_KV_ESIZE;
    if (n > 0 && !delta) return LUMEN_KV_EINVAL;
    for (int32_t i = 0; i < n_tags; ++i)
        if (tags[i].end_pos <= t_begin || tags[i].end_pos > t_end) return LUMEN_KV_EINVAL;
    char* dst;
    bool in_place = false;
    {
        std::lock_guard<std::mutex> g(s->mu);
        auto it = s->reqs.find(id);
        if (it == s->reqs.end()) return LUMEN_KV_EINVAL;
        Entry& e = it->second;
        if (t_begin != e.tokens || t_end > e.max_tokens) return LUMEN_KV_EINVAL;
        dst = s->arena + e.region_off + e.tokens * s->token_bytes;
        if (e.claims > 0) {
            // commit of the oldest claim (lumen_kv_store_acquire): the bytes are already in place
            if (n == 0 || delta != dst || n > e.receiving) return LUMEN_KV_EINVAL;
            in_place = true;
        } else {
            if (e.receiving) return LUMEN_KV_EINVAL;
            if (n == 0) return LUMEN_KV_OK;
            e.receiving = n;                               // claims the region's tail
        }
    }
    if (!in_place) s->pool->copy(dst, static_cast<const char*>(delta), delta_bytes);
    {
        // publication: the delta and its tags become visible together, after the last byte
        std::lock_guard<std::mutex> g(s->mu);
        auto it = s->reqs.find(id);
        if (it == s->reqs.end()) return LUMEN_KV_EINVAL;
        Entry& e = it->second;
        if (in_place && (e.claims == 0 || t_begin != e.tokens)) return LUMEN_KV_EINVAL;   // aborted meanwhile
        e.deltas.push_back(Delta{t_begin, t_end, static_cast<int64_t>(dst - s->arena)});
        e.tags.insert(e.tags.end(), tags, tags + n_tags);
        e.tokens = t_end;
        e.receiving -= n;
        if (in_place) --e.claims;
    }
    return LUMEN_KV_OK;
}

void* lumen_kv_store_acquire(void* store, uint64_t id, int64_t t_begin, int64_t t_end,
                             int64_t delta_bytes) {
    lumen_kv_store* s = static_cast<lumen_kv_store*>(store);
    if (!s || t_begin < 0 || t_end <= t_begin) return nullptr;
    const int64_t n = t_end - t_begin;
    if (delta_bytes != n * s->token_bytes) return nullptr;
    std::lock_guard<std::mutex> g(s->mu);
    auto it = s->reqs.find(id);
    if (it == s->reqs.end()) return nullptr;
    Entry& e = it->second;
    if (e.receiving != 0 && e.claims == 0) return nullptr;      // a copying append is in progress
    if (t_begin != e.tokens + e.receiving || t_end > e.max_tokens) return nullptr;
    e.receiving += n;
    ++e.claims;
    return s->arena + e.region_off + t_begin * s->token_bytes;
}

void lumen_kv_store_abort(void* store, uint64_t id) {
    lumen_kv_store* s = static_cast<lumen_kv_store*>(store);
    if (!s) return;
    std::lock_guard<std::mutex> g(s->mu);
    auto it = s->reqs.find(id);
    if (it == s->reqs.end() || it->second.claims == 0) return;
    it->second.receiving = 0;                                   // every outstanding claim is void
    it->second.claims = 0;
}

void* lumen_kv_store_arena(const lumen_kv_store* s, int64_t* bytes) {
    if (bytes) *bytes = s ? s->arena_bytes : 0;
    return s ? s->arena : nullptr;
}

int64_t lumen_kv_store_tokens(const lumen_kv_store* s, uint64_t id) {
    if (!s) return LUMEN_KV_EINVAL;
    std::lock_guard<std::mutex> g(s->mu);
    auto it = s->reqs.find(id);
    return it == s->reqs.end() ? int64_t{LUMEN_KV_EINVAL} : it->second.tokens;
}

int64_t lumen_kv_store_lookup(const lumen_kv_store* s, uint64_t id, const lumen_kv_tag* regen,
                              int64_t n_regen) {
    if (!s) return LUMEN_KV_EINVAL;
    std::vector<lumen_kv_tag> stored;
    {
        std::lock_guard<std::mutex> g(s->mu);
        auto it = s->reqs.find(id);
        if (it == s->reqs.end()) return LUMEN_KV_EINVAL;
        stored = it->second.tags;
    }
    return lumen_kv_longest_prefix(regen, n_regen, stored.data(),
                                   static_cast<int64_t>(stored.size()));
}

int lumen_kv_store_sink(void* store, uint64_t id, int64_t t_begin, int64_t t_end,
                        const void* delta, int64_t delta_bytes, const lumen_kv_tag* tags,
                        int32_t n_tags) {
    lumen_kv_store* s = static_cast<lumen_kv_store*>(store);
    if (!s) return LUMEN_KV_EINVAL;
    const int rc = lumen_kv_store_append(s, id, t_begin, t_end, delta, delta_bytes, tags, n_tags);
    if (rc != LUMEN_KV_OK) {
        std::lock_guard<std::mutex> g(s->mu);
        ++s->sink_errors;
    }
    return rc;
}

// internal (recover.cu): the arena the segments' offsets refer to; not exported
const void* lumen_kv_store_arena_(const lumen_kv_store* s, int64_t* bytes) {
    if (bytes) *bytes = s ? s->arena_bytes : 0;
    return s ? s->arena : nullptr;
}

int64_t lumen_kv_store_sink_errors(const lumen_kv_store* s) {
    if (!s) return LUMEN_KV_EINVAL;
    std::lock_guard<std::mutex> g(s->mu);
    return s->sink_errors;
}

int64_t lumen_kv_store_segments(const lumen_kv_store* s, uint64_t id, int64_t prefix_tokens,
                                lumen_kv_segment* out, int64_t cap) {
    if (!s || prefix_tokens < 0 || cap < 0 || (cap > 0 && !out)) return LUMEN_KV_EINVAL;
    std::lock_guard<std::mutex> g(s->mu);
    auto it = s->reqs.find(id);
    if (it == s->reqs.end() || prefix_tokens > it->second.tokens) return LUMEN_KV_EINVAL;
    int64_t n = 0;
    for (const Delta& d : it->second.deltas) {
        if (d.t_begin >= prefix_tokens) break;
        if (n < cap)
            out[n] = lumen_kv_segment{d.t_begin, std::min(d.t_end, prefix_tokens), d.offset,
                                      d.t_end - d.t_begin};
        ++n;
    }
    return n;
}

}  // extern "C"
