// Two-stage host path (include/lumen_kv.h): device staging ring + copy-engine transfers,
// per-chunk commit / ready flags.
#include <cuda_runtime.h>

#include <mutex>
#include <new>
#include <vector>

#include "internal.hpp"
#include "lumen_kv.h"
#include "plan.hpp"

struct lumen_kv_stager {
    char* base = nullptr;          // caller's device staging memory
    int64_t slot_bytes = 0;
    int32_t n_slots = 0;
    int64_t next = 0;              // chunks issued so far: chunk i uses slot i % n_slots
    cudaStream_t copy = nullptr;   // the stager's copy stream (non-blocking)
    cudaEvent_t full[16];          // slot holds a complete chunk (producer done)
    cudaEvent_t free_[16];         // slot may be overwritten (consumer done)
    cudaEvent_t join = nullptr;
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

int run_staged(const lumen_kv_plan* plan, const void* const* k_planes, const void* const* v_planes,
               void* host, int64_t host_bytes, lumen_kv_stager* st, void* stream_, bool pack,
               const uint64_t* flags = nullptr, uint64_t epoch = 0) {
    if (!plan || !st) return LUMEN_KV_EINVAL;
    if (plan->flags & LUMEN_KV_HOST_ONLY) return LUMEN_KV_EINVAL;
    if (host_bytes < plan->hp.total_bytes) return LUMEN_KV_ESIZE;
    if (plan->hp.total_bytes == 0) return LUMEN_KV_OK;
    if (!host || (reinterpret_cast<uintptr_t>(host) & 15)) return LUMEN_KV_EINVAL;
    std::vector<const void*> planes;
    int rc = gather_planes(plan, k_planes, v_planes, &planes);
    if (rc != LUMEN_KV_OK) return rc;
    void* alias = nullptr;         // only to reject pageable memory: the copies must be asynchronous
    if (cudaHostGetDevicePointer(&alias, host, 0) != cudaSuccess) {
        (void)cudaGetLastError();
        return LUMEN_KV_EINVAL;
    }
    std::vector<Chunk> chunks;
    rc = build_chunks(plan->hp, plan->h_runs, st->slot_bytes, &chunks);
    if (rc != LUMEN_KV_OK) return rc;
    unsigned long long flags_dev = 0;   // device alias of the caller's pinned flag array
    if (flags) {
        if (reinterpret_cast<uintptr_t>(flags) & 7) return LUMEN_KV_EINVAL;
        void* fa = nullptr;
        if (cudaHostGetDevicePointer(&fa, const_cast<uint64_t*>(flags), 0) != cudaSuccess) {
            (void)cudaGetLastError();
            return LUMEN_KV_EINVAL;
        }
        flags_dev = reinterpret_cast<unsigned long long>(fa);
        rc = load_stream_memops();
        if (rc != LUMEN_KV_OK) return rc;
    }

    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    int64_t ci = 0;                     // chunk index = entry of lumen_kv_plan_get_chunks
    char* h = static_cast<char*>(host);
    if (!pack) {   // the host buffer may have been produced by earlier work on `stream`
        LUMEN_CUDA(cudaEventRecord(st->join, stream));
        LUMEN_CUDA(cudaStreamWaitEvent(st->copy, st->join, 0));
    }
    for (const Chunk& c : chunks) {
        const int slot = static_cast<int>(st->next++ % st->n_slots);
        char* sbase = st->base + int64_t{slot} * st->slot_bytes;
        // the address byte 0 of the checkpoint buffer would have if the chunk sat in this slot
        const uintptr_t shifted = reinterpret_cast<uintptr_t>(sbase) - static_cast<uintptr_t>(c.b0);
        const size_t bytes = static_cast<size_t>(c.b1 - c.b0);
        if (pack) {
            LUMEN_CUDA(cudaStreamWaitEvent(stream, st->free_[slot], 0));
            rc = launch_part(plan, planes, shifted, false, stream, true, c.ra, c.rb, c.p0, c.p1);
            if (rc != LUMEN_KV_OK) return rc;
            LUMEN_CUDA(cudaEventRecord(st->full[slot], stream));
            LUMEN_CUDA(cudaStreamWaitEvent(st->copy, st->full[slot], 0));
            LUMEN_CUDA(cudaMemcpyAsync(h + c.b0, sbase, bytes, cudaMemcpyDeviceToHost, st->copy));
            LUMEN_CUDA(cudaEventRecord(st->free_[slot], st->copy));
            if (flags && g_write64(st->copy, flags_dev + 8ull * ci, epoch, 0) != 0)
                return cuda_fail(cudaErrorUnknown);
        } else {
            LUMEN_CUDA(cudaStreamWaitEvent(st->copy, st->free_[slot], 0));
            if (flags && g_wait64(st->copy, flags_dev + 8ull * ci, epoch, 0 /* >= */) != 0)
                return cuda_fail(cudaErrorUnknown);
            LUMEN_CUDA(cudaMemcpyAsync(sbase, h + c.b0, bytes, cudaMemcpyHostToDevice, st->copy));
            LUMEN_CUDA(cudaEventRecord(st->full[slot], st->copy));
            LUMEN_CUDA(cudaStreamWaitEvent(stream, st->full[slot], 0));
            rc = launch_part(plan, planes, shifted, false, stream, false, c.ra, c.rb, c.p0, c.p1);
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
    cudaError_t e = cudaStreamCreateWithFlags(&st->copy, cudaStreamNonBlocking);
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
    if (st->copy) {
        cudaStreamSynchronize(st->copy);
        cudaStreamDestroy(st->copy);
    }
    for (int i = 0; i < 16; ++i) {
        if (st->full[i]) cudaEventDestroy(st->full[i]);
        if (st->free_[i]) cudaEventDestroy(st->free_[i]);
    }
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

int64_t lumen_kv_plan_get_chunks(const lumen_kv_plan* plan, int64_t slot_bytes,
                                 lumen_kv_chunk_info* out, int64_t cap) {
    if (!plan || cap < 0 || (cap > 0 && !out)) return LUMEN_KV_EINVAL;
    std::vector<lumen::Chunk> chunks;
    const int rc = lumen::build_chunks(plan->hp, plan->h_runs, slot_bytes, &chunks);
    if (rc != LUMEN_KV_OK) return rc;
    const int64_t n = static_cast<int64_t>(chunks.size());
    for (int64_t i = 0; i < n && i < cap; ++i) {
        const lumen::Chunk& c = chunks[static_cast<size_t>(i)];
        out[i] = lumen_kv_chunk_info{c.ra, c.rb, c.p0, c.p1, c.b0, c.b1};
    }
    return n;
}

int64_t lumen_kv_plan_num_chunks(const lumen_kv_plan* plan, int64_t slot_bytes) {
    return lumen_kv_plan_get_chunks(plan, slot_bytes, nullptr, 0);
}

}  // extern "C"
