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
    int64_t t_cur = 0;
    cudaEvent_t ev = nullptr;  // fires when tokens [.., t_cur) exist
};

struct Tracked {
    int64_t t_prev = 0;        // tokens delivered to the sink
    bool has_pending = false;
    bool in_flight = false;
    bool zombie = false;       // untracked while in flight: erased after delivery
    Pending p;
};

struct Job {
    uint64_t id;
    std::vector<int32_t> pt;
    int64_t tb, te;
    cudaEvent_t ev;
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
    uint64_t* flags = nullptr;   // pinned, one word per chunk of the plan in flight
    int64_t flags_cap = 0;
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

void set_error(lumen_kv_ckpt* c, int rc) {
    std::lock_guard<std::mutex> g(c->mu);
    if (c->first_error == 0) c->first_error = rc;
}

// Waits until flags[idx] == epoch; false if the stream died or finished without the flag.
bool wait_flag(lumen_kv_ckpt* c, int64_t idx) {
    volatile uint64_t* f = c->flags + idx;
    int spins = 0;
    for (;;) {
        if (*f == c->epoch) {
            std::atomic_thread_fence(std::memory_order_acquire);
            return true;
        }
        if (++spins % 64 == 0) {
            const cudaError_t e = cudaStreamQuery(c->stream);
            if (e == cudaSuccess) {                 // everything ran: the flag must be there now
                std::atomic_thread_fence(std::memory_order_acquire);
                return *f == c->epoch;
            }
            if (e != cudaErrorNotReady) {
                (void)cudaGetLastError();
                return false;
            }
            std::this_thread::sleep_for(std::chrono::microseconds(20));
        }
    }
}

int process(lumen_kv_ckpt* c, std::vector<Job>& jobs) {
    const int32_t n = static_cast<int32_t>(jobs.size());
    std::vector<lumen_kv_req> reqs(static_cast<size_t>(n));
    for (int32_t i = 0; i < n; ++i) {
        reqs[i].page_table = jobs[i].pt.data();
        reqs[i].page_table_len = static_cast<int64_t>(jobs[i].pt.size());
        reqs[i].t_begin = jobs[i].tb;
        reqs[i].t_end = jobs[i].te;
    }
    lumen_kv_plan* plan = nullptr;
    int rc = lumen_kv_plan_build(&c->geom, reqs.data(), n, 0, c->stream, &plan);
    if (rc != LUMEN_KV_OK) return rc;
    const int64_t n_chunks = lumen_kv_plan_num_chunks(plan, c->slot_bytes);
    if (n_chunks < 0) {
        lumen_kv_plan_free(plan);
        return static_cast<int>(n_chunks);
    }
    if (n_chunks > c->flags_cap) {                  // control memory, grown rarely
        if (c->flags) cudaFreeHost(c->flags);
        c->flags = nullptr;
        c->flags_cap = 0;
        int64_t cap = 256;
        while (cap < n_chunks) cap <<= 1;
        if (cudaHostAlloc(reinterpret_cast<void**>(&c->flags), static_cast<size_t>(cap) * 8,
                          cudaHostAllocDefault) != cudaSuccess) {
            (void)cudaGetLastError();
            lumen_kv_plan_free(plan);
            return LUMEN_KV_ENOMEM;
        }
        for (int64_t i = 0; i < cap; ++i) c->flags[i] = 0;
        c->flags_cap = cap;
    }
    std::vector<lumen_kv_chunk_info> chunks(static_cast<size_t>(n_chunks));
    lumen_kv_plan_get_chunks(plan, c->slot_bytes, chunks.data(), n_chunks);
    cudaEvent_t last = nullptr;
    for (const Job& j : jobs)                       // A10: stream order behind the producing batch
        if (j.ev && j.ev != last) {
            if (cudaStreamWaitEvent(c->stream, j.ev, 0) != cudaSuccess) {
                (void)cudaGetLastError();
                lumen_kv_plan_free(plan);
                return LUMEN_KV_ECUDA;
            }
            last = j.ev;
        }
    ++c->epoch;
    rc = lumen_kv_checkpoint_pack_staged_commit(plan, c->k.data(), c->v.data(), c->pinned,
                                                c->pinned_bytes, c->stager, c->stream, c->flags,
                                                c->epoch);
    if (rc == LUMEN_KV_OK) {
        int64_t ci = 0;
        for (int32_t i = 0; i < n && rc == LUMEN_KV_OK; ++i) {
            const int64_t off = lumen_kv_plan_req_offset(plan, i);
            const int64_t end = lumen_kv_plan_req_offset(plan, i + 1);
            if (end > off) {
                while (ci < n_chunks && chunks[static_cast<size_t>(ci)].byte_end < end) ++ci;
                if (ci >= n_chunks || !wait_flag(c, ci)) {   // the chunk that completes request i
                    rc = LUMEN_KV_ECUDA;
                    break;
                }
                c->sink(c->user, jobs[i].id, jobs[i].tb, jobs[i].te, c->pinned + off, end - off);
            }
            std::lock_guard<std::mutex> g(c->mu);
            auto it = c->reqs.find(jobs[i].id);
            if (it != c->reqs.end()) it->second.t_prev = jobs[i].te;   // progress (a1)
        }
    }
    if (rc != LUMEN_KV_OK) cudaStreamSynchronize(c->stream);
    lumen_kv_plan_free(plan);
    return rc;
}

void run(lumen_kv_ckpt* c) {
    cudaSetDevice(c->device);
    for (;;) {
        std::vector<Job> jobs;
        {
            std::unique_lock<std::mutex> lk(c->mu);
            c->busy = false;
            c->idle_cv.notify_all();
            c->work_cv.wait(lk, [&] { return c->stop || any_pending(c); });
            if (!any_pending(c)) break;             // stop requested and nothing left
            c->busy = true;
            int64_t room = c->pinned_bytes;
            for (auto& kv : c->reqs) {
                Tracked& t = kv.second;
                if (!t.has_pending) continue;
                if (t.p.t_cur <= t.t_prev) {        // already delivered by the job that was in flight
                    t.has_pending = false;
                    continue;
                }
                const int64_t want = (t.p.t_cur - t.t_prev) * c->token_bytes;
                if (want <= room) {
                    jobs.push_back(Job{kv.first, std::move(t.p.pt), t.t_prev, t.p.t_cur, t.p.ev});
                    t.has_pending = false;
                    room -= want;
                } else if (jobs.empty()) {          // larger than the whole buffer: take a prefix
                    const int64_t fit = room / c->token_bytes;
                    if (fit < 1) {
                        if (c->first_error == 0) c->first_error = LUMEN_KV_ESIZE;
                        t.has_pending = false;
                        continue;
                    }
                    jobs.push_back(Job{kv.first, t.p.pt, t.t_prev, t.t_prev + fit, t.p.ev});
                    room = 0;                       // the rest stays pending
                } else {
                    break;                          // next round
                }
                t.in_flight = true;
                if (room == 0) break;
            }
        }
        if (!jobs.empty()) {
            const int rc = process(c, jobs);
            if (rc != LUMEN_KV_OK) set_error(c, rc);
            std::lock_guard<std::mutex> g(c->mu);
            for (const Job& j : jobs) {
                auto it = c->reqs.find(j.id);
                if (it == c->reqs.end()) continue;
                it->second.in_flight = false;
                if (rc != LUMEN_KV_OK) it->second.has_pending = false;   // do not retry for ever
                if (it->second.zombie) c->reqs.erase(it);
            }
        }
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
    if (!geom || !k_planes || !v_planes || !pinned || !sink || pinned_bytes < 16 ||
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
    if (c->flags) cudaFreeHost(c->flags);
    (void)cudaGetLastError();
    delete c;
}

int lumen_kv_ckpt_track(lumen_kv_ckpt* c, uint64_t id, int64_t t_prev) {
    if (!c || t_prev < 0) return LUMEN_KV_EINVAL;
    std::lock_guard<std::mutex> g(c->mu);
    if (c->reqs.count(id)) return LUMEN_KV_EINVAL;
    c->reqs[id].t_prev = t_prev;
    return LUMEN_KV_OK;
}

int lumen_kv_ckpt_untrack(lumen_kv_ckpt* c, uint64_t id) {
    if (!c) return LUMEN_KV_EINVAL;
    std::lock_guard<std::mutex> g(c->mu);
    auto it = c->reqs.find(id);
    if (it == c->reqs.end() || it->second.zombie) return LUMEN_KV_EINVAL;
    it->second.has_pending = false;
    if (it->second.in_flight)
        it->second.zombie = true;
    else
        c->reqs.erase(it);
    return LUMEN_KV_OK;
}

int lumen_kv_ckpt_notify(lumen_kv_ckpt* c, const uint64_t* ids, const lumen_kv_req* reqs, int32_t n,
                         void* ready_event) {
    if (!c || n < 0 || (n > 0 && (!ids || !reqs))) return LUMEN_KV_EINVAL;
    {
        std::lock_guard<std::mutex> g(c->mu);
        const int64_t S = c->geom.page_size;
        for (int32_t i = 0; i < n; ++i) {           // validate everything before changing anything
            auto it = c->reqs.find(ids[i]);
            if (it == c->reqs.end() || it->second.zombie) return LUMEN_KV_EINVAL;
            const Tracked& t = it->second;
            const int64_t floor_ = t.has_pending ? t.p.t_cur : t.t_prev;
            if (reqs[i].t_end < floor_ || reqs[i].page_table_len < 0 ||
                (reqs[i].t_end > 0 && (!reqs[i].page_table ||
                                       (reqs[i].t_end + S - 1) / S > reqs[i].page_table_len)))
                return LUMEN_KV_EINVAL;
        }
        for (int32_t i = 0; i < n; ++i) {
            Tracked& t = c->reqs[ids[i]];
            if (reqs[i].t_end == t.t_prev && !t.in_flight && !t.has_pending) continue;   // nothing new
            t.p.pt.assign(reqs[i].page_table, reqs[i].page_table + reqs[i].page_table_len);
            t.p.t_cur = reqs[i].t_end;
            t.p.ev = static_cast<cudaEvent_t>(ready_event);
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
