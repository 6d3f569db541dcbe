// Two-stage host path (include/lumen_kv.h): device staging ring + copy-engine transfers,
// per-chunk commit / ready flags, and the asynchronous form in which a stager-owned thread
// issues the per-chunk stream operations.
#include <cuda_runtime.h>

#include <condition_variable>
#include <deque>
#include <memory>
#include <mutex>
#include <new>
#include <thread>
#include <vector>

#include "internal.hpp"
#include "lumen_kv.h"
#include "plan.hpp"

namespace lumen {
extern thread_local int t_last_cuda_error;   // lib.cu: what lumen_kv_last_cuda_error() returns
// lumen_kv_set_option("fail_after_chunks", n): every staged call fails with ECUDA in front of
// its chunk n (0: before anything is enqueued); -1 (default): off.  For tests of the error paths.
std::atomic<int> g_fail_after_chunks{-1};
}

namespace {

// One asynchronous call waiting for (or being issued by) the stager's thread.
struct Job {
    uint64_t ticket = 0;
    const lumen_kv_plan* plan = nullptr;                        // holds a reference
    std::shared_ptr<const std::vector<lumen::Chunk>> chunks;
    std::vector<const void*> planes;                            // K0,V0,K1,V1,..
    char* host = nullptr;
    unsigned long long flags_dev = 0;
    uint64_t epoch = 0;
    bool pack = true;
    cudaEvent_t begin = nullptr;   // recorded on the caller's stream at the call
};

struct TicketRec {
    uint64_t id = 0;
    cudaEvent_t done = nullptr;    // recorded behind the call's last operation once issued
    int status = LUMEN_KV_OK;
    int cuda_error = 0;            // the cudaError_t behind a failed status (seen on the worker's thread)
    int waiters = 0;               // stager_wait / stager_sync calls holding `done`: not pruned meanwhile
    bool issued = false;
};

}  // namespace

struct lumen_kv_stager {
    char* base = nullptr;          // caller's device staging memory
    int64_t slot_bytes = 0;
    int32_t n_slots = 0;
    int device = 0;                // the device its streams and events belong to
    int64_t next = 0;              // chunks issued so far: chunk i uses slot i % n_slots
    cudaStream_t copy = nullptr;   // the stager's copy stream (non-blocking)
    cudaStream_t work = nullptr;   // kernels of asynchronous calls (non-blocking)
    cudaEvent_t full[16];          // slot holds a complete chunk (producer done)
    cudaEvent_t free_[16];         // slot may be overwritten (consumer done)
    cudaEvent_t join = nullptr;
    std::mutex issue_mu;           // one call is issued at a time (calling threads and the worker)

    std::mutex mu;                 // everything below
    std::condition_variable cv;
    std::deque<Job> queue;
    std::deque<TicketRec> tickets; // ascending id; the front is pruned once complete
    uint64_t next_ticket = 1;
    bool worker_started = false, stop = false;
    std::thread worker;
};

namespace lumen {
namespace {

#define LUMEN_CUDA(x)                                  \
    do {                                               \
        cudaError_t e_ = (x);                          \
        if (e_ != cudaSuccess) return cuda_fail(e_);   \
    } while (0)

// 64-bit stream memory operations (driver API), fetched at run time so that the library has
// no link-time dependency on libcuda: (stream, device address, value, flags)
typedef int (*StreamMemOp64)(cudaStream_t, unsigned long long, unsigned long long, unsigned int);
StreamMemOp64 g_write64 = nullptr, g_wait64 = nullptr;

int load_stream_memops() {
    static std::once_flag once;
    static cudaError_t err = cudaSuccess;
    std::call_once(once, [] {
        void* w = nullptr;
        void* q = nullptr;
        cudaDriverEntryPointQueryResult r1, r2;
        err = cudaGetDriverEntryPoint("cuStreamWriteValue64", &w, cudaEnableDefault, &r1);
        if (err == cudaSuccess)
            err = cudaGetDriverEntryPoint("cuStreamWaitValue64", &q, cudaEnableDefault, &r2);
        if (err == cudaSuccess && (r1 != cudaDriverEntryPointSuccess ||
                                   r2 != cudaDriverEntryPointSuccess || !w || !q))
            err = cudaErrorNotSupported;
        if (err == cudaSuccess) {
            g_write64 = reinterpret_cast<StreamMemOp64>(w);
            g_wait64 = reinterpret_cast<StreamMemOp64>(q);
        }
    });
    return err == cudaSuccess ? LUMEN_KV_OK : cuda_fail(err);
}

// Everything a staged call checks before anything is enqueued; fills the job.
int prepare(const lumen_kv_plan* plan, const void* const* k_planes, const void* const* v_planes,
            void* host, int64_t host_bytes, lumen_kv_stager* st, bool pack, const uint64_t* flags,
            uint64_t epoch, Job* job, bool* empty) {
    *empty = false;
    if (!plan || !st) return LUMEN_KV_EINVAL;
    if (plan->flags & LUMEN_KV_HOST_ONLY) return LUMEN_KV_EINVAL;
    if (host_bytes < plan->hp.total_bytes) return LUMEN_KV_ESIZE;
    if (plan->hp.total_bytes == 0) {
        *empty = true;
        return LUMEN_KV_OK;
    }
    if (!host || (reinterpret_cast<uintptr_t>(host) & 15)) return LUMEN_KV_EINVAL;
    int rc = gather_planes(plan, k_planes, v_planes, &job->planes);
    if (rc != LUMEN_KV_OK) return rc;
    void* alias = nullptr;         // only to reject pageable memory: the copies must be asynchronous
    if (cudaHostGetDevicePointer(&alias, host, 0) != cudaSuccess) {
        (void)cudaGetLastError();
        return LUMEN_KV_EINVAL;
    }
    rc = plan_chunks(plan, st->slot_bytes, &job->chunks);   // cached on the plan
    if (rc != LUMEN_KV_OK) return rc;
    job->flags_dev = 0;            // device alias of the caller's pinned flag array
    if (flags) {
        if (reinterpret_cast<uintptr_t>(flags) & 7) return LUMEN_KV_EINVAL;
        void* fa = nullptr;
        if (cudaHostGetDevicePointer(&fa, const_cast<uint64_t*>(flags), 0) != cudaSuccess) {
            (void)cudaGetLastError();
            return LUMEN_KV_EINVAL;
        }
        job->flags_dev = reinterpret_cast<unsigned long long>(fa);
        rc = load_stream_memops();
        if (rc != LUMEN_KV_OK) return rc;
    }
    job->plan = plan;
    job->host = static_cast<char*>(host);
    job->epoch = epoch;
    job->pack = pack;
    return LUMEN_KV_OK;
}

// The per-chunk pipeline of one call, kernels on `stream`, transfers on the stager's copy
// stream.  Called with st->issue_mu held.
int issue_chunks(lumen_kv_stager* st, const Job& j, cudaStream_t stream) {
    const lumen_kv_plan* plan = j.plan;
    const bool pack = j.pack;
    int64_t ci = 0;                     // chunk index = entry of lumen_kv_plan_get_chunks
    char* h = j.host;
    if (!pack) {   // the host buffer may have been produced by earlier work on `stream`
        LUMEN_CUDA(cudaEventRecord(st->join, stream));
        LUMEN_CUDA(cudaStreamWaitEvent(st->copy, st->join, 0));
    }
    const int fail_at = g_fail_after_chunks.load(std::memory_order_relaxed);
    for (const Chunk& c : *j.chunks) {
        if (fail_at >= 0 && ci >= fail_at) return cuda_fail(cudaErrorUnknown);   // test hook
        const int slot = static_cast<int>(st->next++ % st->n_slots);
        char* sbase = st->base + int64_t{slot} * st->slot_bytes;
        // the address byte 0 of the checkpoint buffer would have if the chunk sat in this slot
        const uintptr_t shifted = reinterpret_cast<uintptr_t>(sbase) - static_cast<uintptr_t>(c.b0);
        const size_t bytes = static_cast<size_t>(c.b1 - c.b0);
        int rc;
        if (pack) {
            LUMEN_CUDA(cudaStreamWaitEvent(stream, st->free_[slot], 0));
            rc = launch_part(plan, j.planes, shifted, false, stream, true, c.ra, c.rb, c.p0, c.p1);
            if (rc != LUMEN_KV_OK) return rc;
            LUMEN_CUDA(cudaEventRecord(st->full[slot], stream));
            LUMEN_CUDA(cudaStreamWaitEvent(st->copy, st->full[slot], 0));
            LUMEN_CUDA(cudaMemcpyAsync(h + c.b0, sbase, bytes, cudaMemcpyDeviceToHost, st->copy));
            LUMEN_CUDA(cudaEventRecord(st->free_[slot], st->copy));
            if (j.flags_dev && g_write64(st->copy, j.flags_dev + 8ull * ci, j.epoch, 0) != 0)
                return cuda_fail(cudaErrorUnknown);
        } else {
            LUMEN_CUDA(cudaStreamWaitEvent(st->copy, st->free_[slot], 0));
            if (j.flags_dev && g_wait64(st->copy, j.flags_dev + 8ull * ci, j.epoch, 0 /* >= */) != 0)
                return cuda_fail(cudaErrorUnknown);
            LUMEN_CUDA(cudaMemcpyAsync(sbase, h + c.b0, bytes, cudaMemcpyHostToDevice, st->copy));
            LUMEN_CUDA(cudaEventRecord(st->full[slot], st->copy));
            LUMEN_CUDA(cudaStreamWaitEvent(stream, st->full[slot], 0));
            rc = launch_part(plan, j.planes, shifted, false, stream, false, c.ra, c.rb, c.p0, c.p1);
            if (rc != LUMEN_KV_OK) return rc;
            LUMEN_CUDA(cudaEventRecord(st->free_[slot], stream));
        }
        ++ci;
    }
    if (pack) {    // work enqueued on `stream` after this call sees the complete host buffer
        LUMEN_CUDA(cudaEventRecord(st->join, st->copy));
        LUMEN_CUDA(cudaStreamWaitEvent(stream, st->join, 0));
    }
    return LUMEN_KV_OK;
}

// A call that fails half-way leaves slot events half-recorded: a kernel may have been launched
// into a slot whose copy was never enqueued, and a later call -- possibly on another stream --
// would find that slot "free" while the kernel still writes it.  So a failed call drains what it
// did enqueue before it reports: once `stream` and the copy stream are idle every recorded slot
// event is complete and any slot may be reused; the stager stays usable.  (A restore with ready
// flags still needs the flags of the chunks it did issue.  Under stream capture nothing can be
// drained; the capture is invalid after an error anyway.)  The error seen first is the one kept
// for lumen_kv_last_cuda_error().
int issue(lumen_kv_stager* st, const Job& j, cudaStream_t stream) {
    const int rc = issue_chunks(st, j, stream);
    if (rc == LUMEN_KV_OK) return rc;
    const int first = t_last_cuda_error;
    cudaStreamSynchronize(stream);
    cudaStreamSynchronize(st->copy);
    (void)cudaGetLastError();
    t_last_cuda_error = first;
    return rc;
}

int run_staged(const lumen_kv_plan* plan, const void* const* k_planes, const void* const* v_planes,
               void* host, int64_t host_bytes, lumen_kv_stager* st, void* stream_, bool pack,
               const uint64_t* flags = nullptr, uint64_t epoch = 0) {
    static thread_local Job job;   // its vectors are reused: no allocation in steady state
    bool empty = false;
    const int rc = prepare(plan, k_planes, v_planes, host, host_bytes, st, pack, flags, epoch, &job,
                           &empty);
    if (rc != LUMEN_KV_OK || empty) return rc;
    std::lock_guard<std::mutex> g(st->issue_mu);
    const int out = issue(st, job, static_cast<cudaStream_t>(stream_));
    job.chunks.reset();
    return out;
}

// The stager's thread: issues queued asynchronous calls in order.
void worker_main(lumen_kv_stager* st) {
    cudaSetDevice(st->device);
    for (;;) {
        Job job;
        {
            std::unique_lock<std::mutex> lk(st->mu);
            st->cv.wait(lk, [&] { return st->stop || !st->queue.empty(); });
            if (st->queue.empty()) return;          // stop requested and nothing left
            job = std::move(st->queue.front());
            st->queue.pop_front();
        }
        int rc = LUMEN_KV_OK;
        cudaEvent_t done = nullptr;
        {
            std::lock_guard<std::mutex> g(st->issue_mu);
            cudaError_t e = cudaStreamWaitEvent(st->work, job.begin, 0);
            if (e != cudaSuccess) rc = cuda_fail(e);
            if (rc == LUMEN_KV_OK) rc = issue(st, job, st->work);
            if (rc == LUMEN_KV_OK) {
                e = cudaEventCreateWithFlags(&done, cudaEventDisableTiming);
                if (e == cudaSuccess) e = cudaEventRecord(done, st->work);
                if (e != cudaSuccess) rc = cuda_fail(e);
            }
        }
        cudaEventDestroy(job.begin);
        plan_release(job.plan);
        {
            std::lock_guard<std::mutex> g(st->mu);
            for (TicketRec& t : st->tickets)
                if (t.id == job.ticket) {
                    t.done = done;
                    t.status = rc;
                    t.cuda_error = rc == LUMEN_KV_OK ? 0 : t_last_cuda_error;
                    t.issued = true;
                }
        }
        st->cv.notify_all();
    }
}

int run_staged_async(const lumen_kv_plan* plan, const void* const* k_planes,
                     const void* const* v_planes, void* host, int64_t host_bytes,
                     lumen_kv_stager* st, void* stream_, bool pack, const uint64_t* flags,
                     uint64_t epoch, uint64_t* ticket) {
    if (!ticket) return LUMEN_KV_EINVAL;
    *ticket = 0;
    Job job;
    bool empty = false;
    int rc = prepare(plan, k_planes, v_planes, host, host_bytes, st, pack, flags, epoch, &job, &empty);
    if (rc != LUMEN_KV_OK) return rc;
    if (!empty) {
        LUMEN_CUDA(cudaEventCreateWithFlags(&job.begin, cudaEventDisableTiming));
        const cudaError_t e = cudaEventRecord(job.begin, static_cast<cudaStream_t>(stream_));
        if (e != cudaSuccess) {
            cudaEventDestroy(job.begin);
            return cuda_fail(e);
        }
        plan_retain(plan);
    }
    try {
        std::lock_guard<std::mutex> g(st->mu);
        // completed tickets leave at the front (calls complete in submission order), unless a
        // stager_wait / stager_sync on another thread still holds their event
        while (st->tickets.size() > 64 && st->tickets.front().issued &&
               st->tickets.front().waiters == 0 &&
               (!st->tickets.front().done ||
                cudaEventQuery(st->tickets.front().done) == cudaSuccess)) {
            if (st->tickets.front().done) cudaEventDestroy(st->tickets.front().done);
            st->tickets.pop_front();
        }
        (void)cudaGetLastError();
        if (!empty && !st->worker_started) {
            st->worker = std::thread(worker_main, st);   // may throw: nothing is queued yet
            st->worker_started = true;
        }
        TicketRec t;
        t.id = st->next_ticket;
        t.issued = empty;          // an empty plan has nothing to issue: complete at once
        st->tickets.push_back(t);
        if (!empty) {
            job.ticket = t.id;
            try {
                st->queue.push_back(std::move(job));
            } catch (...) {
                st->tickets.pop_back();
                throw;
            }
        }
        *ticket = st->next_ticket++;
    } catch (...) {                // bad_alloc, system_error: nothing may cross the C boundary
        if (!empty) {
            cudaEventDestroy(job.begin);
            plan_release(plan);
        }
        return LUMEN_KV_ENOMEM;
    }
    if (!empty) st->cv.notify_all();
    return LUMEN_KV_OK;
}

// Blocks until the ticket has been issued; *done receives its completion event (nullptr: nothing
// to wait for) and the ticket is pinned against pruning until unpin() -- another thread's _async
// call would otherwise be free to destroy the event once it has completed.  Returns the call's
// status; a failed call's cudaError_t is handed to the calling thread (lumen_kv_last_cuda_error).
int wait_issued(lumen_kv_stager* st, uint64_t ticket, cudaEvent_t* done) {
    *done = nullptr;
    std::unique_lock<std::mutex> lk(st->mu);
    if (ticket == 0 || ticket >= st->next_ticket) return LUMEN_KV_EINVAL;
    for (;;) {
        TicketRec* rec = nullptr;
        for (TicketRec& t : st->tickets)
            if (t.id == ticket) rec = &t;
        if (!rec) return LUMEN_KV_OK;              // pruned: complete long ago
        if (rec->issued) {
            if (rec->status != LUMEN_KV_OK) {
                t_last_cuda_error = rec->cuda_error;
                return rec->status;
            }
            if (rec->done) {
                *done = rec->done;
                ++rec->waiters;
            }
            return LUMEN_KV_OK;
        }
        st->cv.wait(lk);
    }
}

void unpin(lumen_kv_stager* st, uint64_t ticket) {
    std::lock_guard<std::mutex> g(st->mu);
    for (TicketRec& t : st->tickets)
        if (t.id == ticket) --t.waiters;
}

}  // namespace
}  // namespace lumen

extern "C" {

int lumen_kv_stager_create(void* staging, int64_t slot_bytes, int32_t n_slots,
                           lumen_kv_stager** out) {
    using namespace lumen;
    if (!out) return LUMEN_KV_EINVAL;
    *out = nullptr;
    if (!staging || (reinterpret_cast<uintptr_t>(staging) & 15) || slot_bytes < 16 ||
        slot_bytes % 16 != 0 || n_slots < 2 || n_slots > 16)
        return LUMEN_KV_EINVAL;
    lumen_kv_stager* st = new (std::nothrow) lumen_kv_stager();
    if (!st) return LUMEN_KV_ENOMEM;
    st->base = static_cast<char*>(staging);
    st->slot_bytes = slot_bytes;
    st->n_slots = n_slots;
    for (int i = 0; i < 16; ++i) st->full[i] = st->free_[i] = nullptr;
    cudaError_t e = cudaGetDevice(&st->device);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&st->copy, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&st->work, cudaStreamNonBlocking);
    for (int i = 0; i < n_slots && e == cudaSuccess; ++i) {
        e = cudaEventCreateWithFlags(&st->full[i], cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&st->free_[i], cudaEventDisableTiming);
    }
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&st->join, cudaEventDisableTiming);
    if (e != cudaSuccess) {
        lumen_kv_stager_destroy(st);
        return cuda_fail(e);
    }
    *out = st;
    return LUMEN_KV_OK;
}

void lumen_kv_stager_destroy(lumen_kv_stager* st) {
    if (!st) return;
    if (st->worker_started) {          // queued calls are issued before the thread leaves
        {
            std::lock_guard<std::mutex> g(st->mu);
            st->stop = true;
        }
        st->cv.notify_all();
        st->worker.join();
    }
    if (st->work) {
        cudaStreamSynchronize(st->work);
        cudaStreamDestroy(st->work);
    }
    if (st->copy) {
        cudaStreamSynchronize(st->copy);
        cudaStreamDestroy(st->copy);
    }
    for (int i = 0; i < 16; ++i) {
        if (st->full[i]) cudaEventDestroy(st->full[i]);
        if (st->free_[i]) cudaEventDestroy(st->free_[i]);
    }
    for (auto& t : st->tickets)
        if (t.done) cudaEventDestroy(t.done);
    if (st->join) cudaEventDestroy(st->join);
    (void)cudaGetLastError();
    delete st;
}

int lumen_kv_checkpoint_pack_staged(const lumen_kv_plan* plan, const void* const* k_planes,
                                    const void* const* v_planes, void* dst_host,
                                    int64_t dst_bytes, lumen_kv_stager* stager, void* stream) {
    return lumen::run_staged(plan, k_planes, v_planes, dst_host, dst_bytes, stager, stream, true);
}

int lumen_kv_restore_unpack_staged(const lumen_kv_plan* plan, void* const* k_planes,
                                   void* const* v_planes, const void* src_host,
                                   int64_t src_bytes, lumen_kv_stager* stager, void* stream) {
    return lumen::run_staged(plan, const_cast<const void* const*>(k_planes),
                             const_cast<const void* const*>(v_planes),
                             const_cast<void*>(src_host), src_bytes, stager, stream, false);
}

int lumen_kv_checkpoint_pack_staged_commit(const lumen_kv_plan* plan, const void* const* k_planes,
                                           const void* const* v_planes, void* dst_host,
                                           int64_t dst_bytes, lumen_kv_stager* stager, void* stream,
                                           uint64_t* flags, uint64_t epoch) {
    return lumen::run_staged(plan, k_planes, v_planes, dst_host, dst_bytes, stager, stream, true,
                             flags, epoch);
}

int lumen_kv_restore_unpack_staged_ready(const lumen_kv_plan* plan, void* const* k_planes,
                                         void* const* v_planes, const void* src_host,
                                         int64_t src_bytes, lumen_kv_stager* stager, void* stream,
                                         const uint64_t* flags, uint64_t epoch) {
    return lumen::run_staged(plan, const_cast<const void* const*>(k_planes),
                             const_cast<const void* const*>(v_planes),
                             const_cast<void*>(src_host), src_bytes, stager, stream, false, flags,
                             epoch);
}

int lumen_kv_checkpoint_pack_staged_async(const lumen_kv_plan* plan, const void* const* k_planes,
                                          const void* const* v_planes, void* dst_host,
                                          int64_t dst_bytes, lumen_kv_stager* stager, void* stream,
                                          uint64_t* flags, uint64_t epoch, uint64_t* ticket) {
    return lumen::run_staged_async(plan, k_planes, v_planes, dst_host, dst_bytes, stager, stream,
                                   true, flags, epoch, ticket);
}

int lumen_kv_restore_unpack_staged_async(const lumen_kv_plan* plan, void* const* k_planes,
                                         void* const* v_planes, const void* src_host,
                                         int64_t src_bytes, lumen_kv_stager* stager, void* stream,
                                         const uint64_t* flags, uint64_t epoch, uint64_t* ticket) {
    return lumen::run_staged_async(plan, const_cast<const void* const*>(k_planes),
                                   const_cast<const void* const*>(v_planes),
                                   const_cast<void*>(src_host), src_bytes, stager, stream, false,
                                   flags, epoch, ticket);
}

int lumen_kv_stager_query(lumen_kv_stager* st, uint64_t ticket) {
    if (!st) return LUMEN_KV_EINVAL;
    std::lock_guard<std::mutex> g(st->mu);
    if (ticket == 0 || ticket >= st->next_ticket) return LUMEN_KV_EINVAL;
    for (const TicketRec& t : st->tickets)
        if (t.id == ticket) {
            if (!t.issued) return 0;
            if (t.status != LUMEN_KV_OK) {
                lumen::t_last_cuda_error = t.cuda_error;
                return t.status;
            }
            if (!t.done) return 1;
            const cudaError_t e = cudaEventQuery(t.done);
            if (e == cudaSuccess) return 1;
            (void)cudaGetLastError();
            return e == cudaErrorNotReady ? 0 : lumen::cuda_fail(e);
        }
    return 1;                                       // pruned: complete long ago
}

int lumen_kv_stager_wait(lumen_kv_stager* st, uint64_t ticket, void* stream) {
    if (!st) return LUMEN_KV_EINVAL;
    cudaEvent_t done = nullptr;
    const int rc = lumen::wait_issued(st, ticket, &done);
    if (rc != LUMEN_KV_OK || !done) return rc;
    const cudaError_t e = cudaStreamWaitEvent(static_cast<cudaStream_t>(stream), done, 0);
    lumen::unpin(st, ticket);
    return e == cudaSuccess ? LUMEN_KV_OK : lumen::cuda_fail(e);
}

int lumen_kv_stager_sync(lumen_kv_stager* st, uint64_t ticket) {
    if (!st) return LUMEN_KV_EINVAL;
    cudaEvent_t done = nullptr;
    const int rc = lumen::wait_issued(st, ticket, &done);
    if (rc != LUMEN_KV_OK || !done) return rc;
    const cudaError_t e = cudaEventSynchronize(done);
    lumen::unpin(st, ticket);
    return e == cudaSuccess ? LUMEN_KV_OK : lumen::cuda_fail(e);
}

int64_t lumen_kv_plan_get_chunks(const lumen_kv_plan* plan, int64_t slot_bytes,
                                 lumen_kv_chunk_info* out, int64_t cap) {
    if (!plan || cap < 0 || (cap > 0 && !out)) return LUMEN_KV_EINVAL;
    std::shared_ptr<const std::vector<lumen::Chunk>> chunks;
    const int rc = lumen::plan_chunks(plan, slot_bytes, &chunks);
    if (rc != LUMEN_KV_OK) return rc;
    const int64_t n = static_cast<int64_t>(chunks->size());
    for (int64_t i = 0; i < n && i < cap; ++i) {
        const lumen::Chunk& c = (*chunks)[static_cast<size_t>(i)];
        out[i] = lumen_kv_chunk_info{c.ra, c.rb, c.p0, c.p1, c.b0, c.b1};
    }
    return n;
}

int64_t lumen_kv_plan_num_chunks(const lumen_kv_plan* plan, int64_t slot_bytes) {
    return lumen_kv_plan_get_chunks(plan, slot_bytes, nullptr, 0);
}

}  // extern "C"
