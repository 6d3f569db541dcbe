// Background checkpointer (include/lumen_kv.h): one thread per worker that
// tracks checkpoint progress, packs every batch's new KV through the two-stage path into the
// caller's pinned buffer and hands each request's delta to a sink as its chunks commit.
// Built on the public C ABI only (plan_build, pack_staged_commit, get_chunks).
#include <cuda_runtime.h>

#include <atomic>
#include <chrono>
#include <condition_variable>
#include <map>
#include <mutex>
#include <new>
#include <thread>
#include <vector>

#include "lumen_kv.h"

namespace {

struct Pending {
    std::vector<int32_t> pt;   // page table as of the notification
    int64_t t_cur = 0;         // = marks.back().first
    // (t, event): tokens [.., t) exist once the event has fired; ascending in t.  A later
    // notification does not replace an earlier one's event: what is ready now is packed now.
    std::vector<std::pair<int64_t, cudaEvent_t>> marks;
    std::vector<int32_t> toks; // token IDs [tok_base, t_cur), empty if the caller gave none
    int64_t tok_base = 0;      // multiple of the page size, <= the page of the delta's first token
};

struct Tracked {
    int64_t t_prev = 0;        // tokens delivered to the sink
    int64_t t_sent = 0;        // tokens handed to a pack that has been enqueued (>= t_prev)
    bool has_pending = false;
    int in_flight = 0;         // batches enqueued but not yet delivered that contain this request
    bool zombie = false;       // untracked while in flight: erased after delivery
    uint64_t gen = 0;          // bumped when a delivery fails: jobs taken before that are void
    Pending p;
};

struct Job {
    uint64_t id;
    std::vector<int32_t> pt;
    int64_t tb, te;
    cudaEvent_t ev;
    std::vector<lumen_kv_tag> tags;   // tags of the pages [tb, te) touches
    uint64_t gen = 0;                 // the request's generation when the job was taken
};

// tags of a job, from the token IDs the notification carried
std::vector<lumen_kv_tag> tags_of(const Pending& p, int64_t tb, int64_t te, int32_t S) {
    std::vector<lumen_kv_tag> out;
    if (p.toks.empty() || te <= tb) return out;
    out.resize(static_cast<size_t>((te - 1) / S - tb / S + 1));
    if (lumen_kv_page_tags_host(p.toks.data(), p.tok_base, tb, te, S, out.data(),
                                static_cast<int64_t>(out.size())) < 0)
        out.clear();
    return out;
}

// One enqueued pack: it owns one half of the pinned buffer until it has been delivered.
struct Batch {
    std::vector<Job> jobs;
    lumen_kv_plan* plan = nullptr;
    std::vector<lumen_kv_chunk_info> chunks;
    uint64_t epoch = 0;
    int half = 0;
    int rc = LUMEN_KV_OK;
    // direct batches: the copy engine writes every job's delta to dst[i], a position the sink's
    // owner handed out (lumen_kv_ckpt_set_direct); off[i] = dst[i] - region base
    bool direct = false;
    std::vector<char*> dst;
    std::vector<int64_t> off;
    std::vector<char> open_claim;   // acquired and neither committed (sink) nor aborted yet
};

}  // namespace

struct lumen_kv_ckpt {
    lumen_kv_geom geom{};
    std::vector<const void*> k, v;
    int64_t token_bytes = 0, slot_bytes = 0, pinned_bytes = 0;
    char* pinned = nullptr;
    lumen_kv_sink_fn sink = nullptr;
    void* user = nullptr;
    int device = 0;
    lumen_kv_stager* stager = nullptr;
    cudaStream_t stream = nullptr;
    // reserve-then-commit delivery (lumen_kv_ckpt_set_direct); read by the thread under mu
    char* direct_base = nullptr;
    int64_t direct_bytes = 0, direct_min = 0;
    lumen_kv_acquire_fn acquire = nullptr;
    lumen_kv_abort_fn abort_claim = nullptr;
    uint64_t* flags[2] = {nullptr, nullptr};   // pinned, one word per chunk, per buffer half
    int64_t flags_cap[2] = {0, 0};
    uint64_t epoch = 0;

    std::mutex mu;
    std::condition_variable work_cv, idle_cv;
    std::map<uint64_t, Tracked> reqs;
    bool stop = false, busy = false;
    int first_error = 0;
    std::thread thread;
};

namespace {

bool any_pending(const lumen_kv_ckpt* c) {
    for (const auto& kv : c->reqs)
        if (kv.second.has_pending) return true;
    return false;
}

// Waits until flags[idx] == epoch; false if the stream died or finished without the flag.
bool wait_flag(lumen_kv_ckpt* c, const Batch& b, int64_t idx) {
    volatile uint64_t* f = c->flags[b.half] + idx;
    int spins = 0;
    for (;;) {
        if (*f == b.epoch) {
            std::atomic_thread_fence(std::memory_order_acquire);
            return true;
        }
        if (++spins % 64 == 0) {
            const cudaError_t e = cudaStreamQuery(c->stream);
            if (e == cudaSuccess) {                 // everything ran: the flag must be there now
                std::atomic_thread_fence(std::memory_order_acquire);
                return *f == b.epoch;
            }
            if (e != cudaErrorNotReady) {
                (void)cudaGetLastError();
                return false;
            }
            std::this_thread::sleep_for(std::chrono::microseconds(20));
        }
    }
}

// Gives back every claim of the batch that has not been committed.
void release_claims(lumen_kv_ckpt* c, Batch& b) {
    for (size_t i = 0; i < b.open_claim.size(); ++i)
        if (b.open_claim[i]) {
            c->abort_claim(c->user, b.jobs[i].id);
            b.open_claim[i] = 0;
        }
}

// Reserve-then-commit: if the sink's owner hands out a final position for every delta of the
// batch, the batch is packed straight to those positions (an explicit-layout plan whose buffer
// is the owner's region) and the sink call that follows is the commit -- PAPER.md:147's "visible
// only upon complete reception" is then the commit, not the copy.  Small deltas keep the classic
// path (one chunk and one copy per batch instead of one per request).
void try_direct(lumen_kv_ckpt* c, Batch& b, const std::vector<lumen_kv_req>& reqs) {
    b.direct = false;
    lumen_kv_acquire_fn acquire;
    int64_t min_avg;
    {
        std::lock_guard<std::mutex> g(c->mu);
        acquire = c->acquire;
        min_avg = c->direct_min;
    }
    const size_t n = b.jobs.size();
    if (!acquire || n == 0) return;
    int64_t total = 0;
    for (const lumen_kv_req& q : reqs) total += (q.t_end - q.t_begin) * c->token_bytes;
    if (total < min_avg * static_cast<int64_t>(n)) return;
    for (const lumen_kv_req& q : reqs)
        if (q.t_end == q.t_begin) return;
    b.dst.assign(n, nullptr);
    b.off.assign(n, 0);
    b.open_claim.assign(n, 0);
    const int64_t row = c->token_bytes / (2 * c->geom.num_layers);
    for (size_t i = 0; i < n; ++i) {
        const Job& j = b.jobs[i];
        const int64_t bytes = (j.te - j.tb) * c->token_bytes;
        char* p = static_cast<char*>(acquire(c->user, j.id, j.tb, j.te, bytes));
        const int64_t off = p ? p - c->direct_base : -1;
        if (!p || off < 0 || off % row != 0 || off + bytes > c->direct_bytes) {
            if (p) c->abort_claim(c->user, j.id);
            release_claims(c, b);                   // all or nothing: the batch goes the classic way
            return;
        }
        b.dst[i] = p;
        b.off[i] = off;
        b.open_claim[i] = 1;
    }
    b.direct = true;
}

// Stage 1: build the plan of the batch and enqueue its pack into one half of the pinned buffer.
void submit(lumen_kv_ckpt* c, Batch& b) {
    const int32_t n = static_cast<int32_t>(b.jobs.size());
    const int64_t half_bytes = c->pinned_bytes / 2;
    std::vector<lumen_kv_req> reqs(static_cast<size_t>(n));
    for (int32_t i = 0; i < n; ++i) {
        reqs[i].page_table = b.jobs[i].pt.data();
        reqs[i].page_table_len = static_cast<int64_t>(b.jobs[i].pt.size());
        reqs[i].t_begin = b.jobs[i].tb;
        reqs[i].t_end = b.jobs[i].te;
    }
    try_direct(c, b, reqs);
    if (b.direct) {
        std::vector<lumen_kv_req_layout> lays(static_cast<size_t>(n));
        for (int32_t i = 0; i < n; ++i) {
            lays[i].buf_offset = b.off[i];
            lays[i].plane_stride_tokens = b.jobs[i].te - b.jobs[i].tb;
        }
        b.rc = lumen_kv_plan_build_layout(&c->geom, reqs.data(), lays.data(), n, 0, c->stream, &b.plan);
    } else {
        b.rc = lumen_kv_plan_build(&c->geom, reqs.data(), n, 0, c->stream, &b.plan);
    }
    if (b.rc != LUMEN_KV_OK) return;
    const int64_t n_chunks = lumen_kv_plan_num_chunks(b.plan, c->slot_bytes);
    if (n_chunks < 0) {
        b.rc = static_cast<int>(n_chunks);
        return;
    }
    if (n_chunks > c->flags_cap[b.half]) {          // control memory, grown rarely
        if (c->flags[b.half]) cudaFreeHost(c->flags[b.half]);
        c->flags[b.half] = nullptr;
        c->flags_cap[b.half] = 0;
        int64_t cap = 256;
        while (cap < n_chunks) cap <<= 1;
        if (cudaHostAlloc(reinterpret_cast<void**>(&c->flags[b.half]), static_cast<size_t>(cap) * 8,
                          cudaHostAllocDefault) != cudaSuccess) {
            (void)cudaGetLastError();
            b.rc = LUMEN_KV_ENOMEM;
            return;
        }
        for (int64_t i = 0; i < cap; ++i) c->flags[b.half][i] = 0;
        c->flags_cap[b.half] = cap;
    }
    b.chunks.resize(static_cast<size_t>(n_chunks));
    lumen_kv_plan_get_chunks(b.plan, c->slot_bytes, b.chunks.data(), n_chunks);
    cudaEvent_t last = nullptr;
    for (const Job& j : b.jobs)                     // A10: stream order behind the producing batch
        if (j.ev && j.ev != last) {
            if (cudaStreamWaitEvent(c->stream, j.ev, 0) != cudaSuccess) {
                (void)cudaGetLastError();
                b.rc = LUMEN_KV_ECUDA;
                return;
            }
            last = j.ev;
        }
    b.epoch = ++c->epoch;
    if (b.direct)   // the checkpoint buffer IS the sink owner's region: no pinned half in between
        b.rc = lumen_kv_checkpoint_pack_staged_commit(b.plan, c->k.data(), c->v.data(), c->direct_base,
                                                      c->direct_bytes, c->stager, c->stream,
                                                      c->flags[b.half], b.epoch);
    else
        b.rc = lumen_kv_checkpoint_pack_staged_commit(b.plan, c->k.data(), c->v.data(),
                                                      c->pinned + b.half * half_bytes, half_bytes,
                                                      c->stager, c->stream, c->flags[b.half], b.epoch);
}

// Stage 2: hand every request's delta to the sink as soon as the chunks that hold it have
// committed (later chunks, and the next batch's pack into the other half, are still in flight).
// Under the lock: request `t` lost a delta (sink rejection or batch failure).  Its progress stays
// at t_prev, nothing of it remains pending, and jobs of it that are already in the next batch are
// void (their generation is stale): they would reach the sink with a gap in front of them.
void fail_request(Tracked& t) {
    ++t.gen;
    t.has_pending = false;
    t.p.marks.clear();
    t.p.toks.clear();
    t.t_sent = t.t_prev;
}

void deliver(lumen_kv_ckpt* c, Batch& b) {
    const int32_t n = static_cast<int32_t>(b.jobs.size());
    const char* base = c->pinned + b.half * (c->pinned_bytes / 2);
    const int64_t n_chunks = static_cast<int64_t>(b.chunks.size());
    int64_t ci = 0;
    int sink_rc = LUMEN_KV_OK;
    for (int32_t i = 0; i < n && b.rc == LUMEN_KV_OK; ++i) {
        const Job& j = b.jobs[i];
        const int64_t off = lumen_kv_plan_req_offset(b.plan, i);
        const int64_t end = lumen_kv_plan_req_offset(b.plan, i + 1);
        {
            std::lock_guard<std::mutex> g(c->mu);
            auto it = c->reqs.find(j.id);
            if (it == c->reqs.end() || it->second.gen != j.gen) continue;   // void: see fail_request
        }
        bool taken = true;
        if (b.direct) {
            // the block of request i is [off_i, off_i + bytes); chunks commit in index order, so
            // the last chunk that intersects the block completes it
            const int64_t lo = b.off[i], hi = lo + (j.te - j.tb) * c->token_bytes;
            int64_t last = -1;
            for (int64_t k = 0; k < n_chunks; ++k)
                if (b.chunks[static_cast<size_t>(k)].byte_begin < hi &&
                    b.chunks[static_cast<size_t>(k)].byte_end > lo)
                    last = k;
            if (last < 0 || !wait_flag(c, b, last)) {
                b.rc = LUMEN_KV_ECUDA;
                break;
            }
            taken = c->sink(c->user, j.id, j.tb, j.te, b.dst[i], hi - lo, j.tags.data(),
                            static_cast<int32_t>(j.tags.size())) == 0;
            if (taken) b.open_claim[i] = 0;                 // committed
        } else if (end > off) {
            while (ci < n_chunks && b.chunks[static_cast<size_t>(ci)].byte_end < end) ++ci;
            if (ci >= n_chunks || !wait_flag(c, b, ci)) {   // the chunk that completes request i
                b.rc = LUMEN_KV_ECUDA;
                break;
            }
            taken = c->sink(c->user, j.id, j.tb, j.te, base + off, end - off, j.tags.data(),
                            static_cast<int32_t>(j.tags.size())) == 0;
        }
        std::lock_guard<std::mutex> g(c->mu);
        auto it = c->reqs.find(j.id);
        if (it == c->reqs.end()) continue;
        if (taken) {
            it->second.t_prev = j.te;                       // progress (a1)
        } else {
            fail_request(it->second);
            sink_rc = LUMEN_KV_ESINK;
        }
    }
    if (b.rc != LUMEN_KV_OK || b.direct) {
        // a direct batch may hold claims that were not committed (void jobs, a rejection, a
        // failure): the copy engine must have left their bytes before the owner gets them back
        bool open = b.rc != LUMEN_KV_OK;
        for (char oc : b.open_claim) open = open || oc;
        if (open) cudaStreamSynchronize(c->stream);
    }
    if (b.direct) release_claims(c, b);
    if (b.plan) lumen_kv_plan_free(b.plan);
    b.plan = nullptr;
    std::lock_guard<std::mutex> g(c->mu);
    if (c->first_error == 0) c->first_error = b.rc != LUMEN_KV_OK ? b.rc : sink_rc;
    for (const Job& j : b.jobs) {
        auto it = c->reqs.find(j.id);
        if (it == c->reqs.end()) continue;
        Tracked& t = it->second;
        --t.in_flight;
        if (b.rc != LUMEN_KV_OK && t.gen == j.gen && t.t_prev < j.te)   // do not retry for ever
            fail_request(t);
        if (t.zombie && t.in_flight == 0) c->reqs.erase(it);
    }
}

// The newest mark whose event has fired (readiness is monotonic in t); the oldest one if none has.
size_t ready_mark(const Pending& p) {
    size_t k = 0;
    for (size_t i = 0; i < p.marks.size(); ++i) {
        const cudaEvent_t ev = p.marks[i].second;
        if (ev != nullptr && cudaEventQuery(ev) == cudaErrorNotReady) {
            (void)cudaGetLastError();
            break;
        }
        (void)cudaGetLastError();
        k = i;
    }
    return k;
}

// Under the lock: move pending deltas into a batch, at most `room` bytes (one buffer half).
void take_jobs(lumen_kv_ckpt* c, Batch& b, int64_t room) {
    for (auto& kv : c->reqs) {
        Tracked& t = kv.second;
        if (!t.has_pending) continue;
        while (!t.p.marks.empty() && t.p.marks.front().first <= t.t_sent)
            t.p.marks.erase(t.p.marks.begin());     // already on its way
        if (t.p.marks.empty()) {
            t.has_pending = false;
            continue;
        }
        const size_t k = ready_mark(t.p);
        const int64_t te = t.p.marks[k].first;
        const cudaEvent_t ev = t.p.marks[k].second;
        const int64_t want = (te - t.t_sent) * c->token_bytes;
        if (want <= room) {
            const bool last = (k + 1 == t.p.marks.size());
            b.jobs.push_back(Job{kv.first, last ? std::move(t.p.pt) : t.p.pt, t.t_sent, te, ev,
                                 tags_of(t.p, t.t_sent, te, c->geom.page_size), t.gen});
            t.p.marks.erase(t.p.marks.begin(), t.p.marks.begin() + static_cast<long>(k) + 1);
            t.has_pending = !last;
            t.t_sent = te;
            room -= want;
        } else if (b.jobs.empty()) {                // larger than a whole half: take a prefix
            const int64_t fit = room / c->token_bytes;
            if (fit < 1) {
                if (c->first_error == 0) c->first_error = LUMEN_KV_ESIZE;
                t.has_pending = false;
                t.p.marks.clear();
                continue;
            }
            b.jobs.push_back(Job{kv.first, t.p.pt, t.t_sent, t.t_sent + fit, ev,
                                 tags_of(t.p, t.t_sent, t.t_sent + fit, c->geom.page_size), t.gen});
            t.t_sent += fit;                        // the rest stays pending
            room = 0;
        } else {
            break;                                  // next batch
        }
        ++t.in_flight;
        if (room == 0) break;
    }
}

// The thread: a two-deep software pipeline over the two halves of the pinned buffer.  The pack
// of batch k+1 is enqueued before batch k is delivered, so the copy engine fills one half while
// the sink drains the other.
void run(lumen_kv_ckpt* c) {
    cudaSetDevice(c->device);
    const int64_t half_bytes = c->pinned_bytes / 2;
    Batch cur;
    bool have_cur = false;
    int half = 0;
    for (;;) {
        Batch nxt;
        {
            std::unique_lock<std::mutex> lk(c->mu);
            if (!have_cur) {
                c->busy = false;
                c->idle_cv.notify_all();
                c->work_cv.wait(lk, [&] { return c->stop || any_pending(c); });
                if (!any_pending(c)) break;         // stop requested and nothing left
                c->busy = true;
            }
            nxt.half = half;
            take_jobs(c, nxt, half_bytes);
        }
        const bool have_nxt = !nxt.jobs.empty();
        if (have_nxt) {
            half ^= 1;
            submit(c, nxt);
        }
        if (have_cur) deliver(c, cur);
        have_cur = have_nxt;
        if (have_nxt) cur = std::move(nxt);
    }
    std::lock_guard<std::mutex> g(c->mu);
    c->busy = false;
    c->idle_cv.notify_all();
}

}  // namespace

extern "C" {

int lumen_kv_ckpt_create(const lumen_kv_geom* geom, const void* const* k_planes,
                         const void* const* v_planes, void* staging, int64_t slot_bytes,
                         int32_t n_slots, void* pinned, int64_t pinned_bytes,
                         lumen_kv_sink_fn sink, void* user, lumen_kv_ckpt** out) {
    if (!out) return LUMEN_KV_EINVAL;
    *out = nullptr;
    if (!geom || !k_planes || !v_planes || !pinned || !sink || pinned_bytes < 64 ||
        pinned_bytes % 32 != 0 ||
        (reinterpret_cast<uintptr_t>(pinned) & 15) || geom->num_layers < 1)
        return LUMEN_KV_EINVAL;
    lumen_kv_plan* probe = nullptr;                 // validates the geometry, host only
    int rc = lumen_kv_plan_build(geom, nullptr, 0, LUMEN_KV_HOST_ONLY, nullptr, &probe);
    if (rc != LUMEN_KV_OK) return rc;
    lumen_kv_plan_free(probe);
    lumen_kv_ckpt* c = new (std::nothrow) lumen_kv_ckpt();
    if (!c) return LUMEN_KV_ENOMEM;
    c->geom = *geom;
    c->k.assign(k_planes, k_planes + geom->num_layers);
    c->v.assign(v_planes, v_planes + geom->num_layers);
    c->token_bytes = int64_t{2} * geom->num_layers * geom->kv_heads * geom->head_dim * geom->elem_bytes;
    c->slot_bytes = slot_bytes;
    c->pinned = static_cast<char*>(pinned);
    c->pinned_bytes = pinned_bytes;
    c->sink = sink;
    c->user = user;
    rc = lumen_kv_stager_create(staging, slot_bytes, n_slots, &c->stager);
    if (rc == LUMEN_KV_OK && (cudaGetDevice(&c->device) != cudaSuccess ||
                              cudaStreamCreateWithFlags(&c->stream, cudaStreamNonBlocking) != cudaSuccess)) {
        (void)cudaGetLastError();
        rc = LUMEN_KV_ECUDA;
    }
    if (rc != LUMEN_KV_OK) {
        if (c->stager) lumen_kv_stager_destroy(c->stager);
        delete c;
        return rc;
    }
    c->busy = true;
    c->thread = std::thread(run, c);
    *out = c;
    return LUMEN_KV_OK;
}

int lumen_kv_ckpt_set_direct(lumen_kv_ckpt* c, void* region, int64_t region_bytes,
                             lumen_kv_acquire_fn acquire, lumen_kv_abort_fn abort_fn,
                             int64_t min_avg_delta_bytes) {
    if (!c) return LUMEN_KV_EINVAL;
    if (!acquire) {                                 // switch it off
        std::lock_guard<std::mutex> g(c->mu);
        c->acquire = nullptr;
        return LUMEN_KV_OK;
    }
    if (!abort_fn || !region || region_bytes < 16 || min_avg_delta_bytes < 0 ||
        (reinterpret_cast<uintptr_t>(region) & 15))
        return LUMEN_KV_EINVAL;
    void* alias = nullptr;                          // the copy engine writes there: must be pinned
    if (cudaHostGetDevicePointer(&alias, region, 0) != cudaSuccess) {
        (void)cudaGetLastError();
        return LUMEN_KV_EINVAL;
    }
    std::lock_guard<std::mutex> g(c->mu);
    c->direct_base = static_cast<char*>(region);
    c->direct_bytes = region_bytes;
    c->direct_min = min_avg_delta_bytes;
    c->abort_claim = abort_fn;
    c->acquire = acquire;
    return LUMEN_KV_OK;
}

void lumen_kv_ckpt_destroy(lumen_kv_ckpt* c) {
    if (!c) return;
    {
        std::lock_guard<std::mutex> g(c->mu);
        c->stop = true;
    }
    c->work_cv.notify_all();
    if (c->thread.joinable()) c->thread.join();
    cudaStreamSynchronize(c->stream);
    lumen_kv_stager_destroy(c->stager);
    cudaStreamDestroy(c->stream);
    for (int h = 0; h < 2; ++h)
        if (c->flags[h]) cudaFreeHost(c->flags[h]);
    (void)cudaGetLastError();
    delete c;
}

int lumen_kv_ckpt_track(lumen_kv_ckpt* c, uint64_t id, int64_t t_prev) {
    if (!c || t_prev < 0) return LUMEN_KV_EINVAL;
    std::lock_guard<std::mutex> g(c->mu);
    if (c->reqs.count(id)) return LUMEN_KV_EINVAL;
    c->reqs[id].t_prev = c->reqs[id].t_sent = t_prev;
    return LUMEN_KV_OK;
}

int lumen_kv_ckpt_untrack(lumen_kv_ckpt* c, uint64_t id) {
    if (!c) return LUMEN_KV_EINVAL;
    std::lock_guard<std::mutex> g(c->mu);
    auto it = c->reqs.find(id);
    if (it == c->reqs.end() || it->second.zombie) return LUMEN_KV_EINVAL;
    it->second.has_pending = false;
    it->second.p.marks.clear();
    if (it->second.in_flight)
        it->second.zombie = true;
    else
        c->reqs.erase(it);
    return LUMEN_KV_OK;
}

int lumen_kv_ckpt_notify(lumen_kv_ckpt* c, const uint64_t* ids, const lumen_kv_req* reqs,
                         const int32_t* const* token_ids, int32_t n, void* ready_event) {
    if (!c || n < 0 || (n > 0 && (!ids || !reqs))) return LUMEN_KV_EINVAL;
    {
        std::lock_guard<std::mutex> g(c->mu);
        const int64_t S = c->geom.page_size;
        for (int32_t i = 0; i < n; ++i) {           // validate everything before changing anything
            auto it = c->reqs.find(ids[i]);
            if (it == c->reqs.end() || it->second.zombie) return LUMEN_KV_EINVAL;
            const Tracked& t = it->second;
            const int64_t floor_ = t.has_pending ? t.p.t_cur : t.t_sent;
            if (reqs[i].t_end < floor_ || reqs[i].page_table_len < 0 ||
                (reqs[i].t_end > 0 && (!reqs[i].page_table ||
                                       (reqs[i].t_end + S - 1) / S > reqs[i].page_table_len)))
                return LUMEN_KV_EINVAL;
            // the pending delta carries token IDs: a notification without them would lose the
            // tags of pages that are still to be sent
            if (t.has_pending && !t.p.toks.empty() && !(token_ids && token_ids[i]))
                return LUMEN_KV_EINVAL;
        }
        for (int32_t i = 0; i < n; ++i) {
            Tracked& t = c->reqs[ids[i]];
            if (reqs[i].t_end == t.t_sent && !t.has_pending) continue;   // nothing new
            t.p.pt.assign(reqs[i].page_table, reqs[i].page_table + reqs[i].page_table_len);
            t.p.t_cur = reqs[i].t_end;
            if (!t.has_pending) t.p.marks.clear();
            const cudaEvent_t ev = static_cast<cudaEvent_t>(ready_event);
            if (!t.p.marks.empty() && t.p.marks.back().second == ev)
                t.p.marks.back().first = reqs[i].t_end;
            else
                t.p.marks.emplace_back(reqs[i].t_end, ev);
            if (t.p.marks.size() > 256) t.p.marks.erase(t.p.marks.begin());   // covered by its successor
            t.p.toks.clear();
            if (token_ids && token_ids[i]) {        // the tokens of the pages the delta touches
                t.p.tok_base = (t.t_sent / S) * S;
                t.p.toks.assign(token_ids[i] + t.p.tok_base, token_ids[i] + reqs[i].t_end);
            }
            t.has_pending = true;
        }
    }
    c->work_cv.notify_all();
    return LUMEN_KV_OK;
}

int lumen_kv_ckpt_flush(lumen_kv_ckpt* c) {
    if (!c) return LUMEN_KV_EINVAL;
    std::unique_lock<std::mutex> lk(c->mu);
    c->work_cv.notify_all();
    c->idle_cv.wait(lk, [&] { return !c->busy && !any_pending(c); });
    return c->first_error;
}

int64_t lumen_kv_ckpt_progress(lumen_kv_ckpt* c, uint64_t id) {
    if (!c) return LUMEN_KV_EINVAL;
    std::lock_guard<std::mutex> g(c->mu);
    auto it = c->reqs.find(id);
    return it == c->reqs.end() ? int64_t{LUMEN_KV_EINVAL} : it->second.t_prev;
}

}  // extern "C"
