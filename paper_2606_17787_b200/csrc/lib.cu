// C entry points of include/lumen_kv.h: plan objects, the descriptor arena and the
// marshalling into launch_kv_copy.  All CUDA runtime use outside the kernels is here.
#include <cuda_runtime.h>

#include <cstdlib>
#include <cstring>
#include <map>
#include <memory>
#include <mutex>
#include <new>
#include <stdexcept>
#include <vector>

#include "internal.hpp"
#include "kernels.hpp"
#include "lumen_kv.h"
#include "plan.hpp"

namespace lumen {

thread_local int t_last_cuda_error = 0;

int g_inline_max_runs = -1;   // -1: unset (LUMEN_KV_INLINE_MAX_RUNS, else kInlineRunsL)
int inline_max_runs() {
    if (g_inline_max_runs < 0) {
        const char* e = std::getenv("LUMEN_KV_INLINE_MAX_RUNS");
        const int v = e ? std::atoi(e) : kInlineRunsL;
        g_inline_max_runs = v < 0 ? 0 : (v > kInlineRunsL ? kInlineRunsL : v);
    }
    return g_inline_max_runs;
}

int cuda_fail(cudaError_t e) {
    t_last_cuda_error = static_cast<int>(e);
    (void)cudaGetLastError();  // clear the sticky-free error state
    return LUMEN_KV_ECUDA;
}

// A descriptor blob: pinned host staging + device copy + the events that say when
// the device copy is no longer read by enqueued work.
struct Blob {
    void* host = nullptr;   // cudaHostAlloc (or malloc for HOST_ONLY)
    void* dev = nullptr;    // cudaMalloc, on `device`
    size_t cap = 0;
    int device = -1;        // the device `dev` and the events belong to
    bool host_only = false;
    bool captured = false;  // used under stream capture: a graph may replay it at any time
    cudaEvent_t uploaded = nullptr;   // recorded behind the descriptor copy on the upload stream
    bool upload_seen = false;         // that event has been seen complete: no wait is needed any more
    std::vector<std::pair<cudaStream_t, cudaEvent_t>> uses;  // last use per stream
    // guards upload_seen, uses and captured: a plan handed to an _async staged call is launched
    // from the stager's thread at a time the caller cannot observe, possibly while the caller
    // uses the same plan in another call
    std::mutex mu;
};

namespace {

// Recycles blobs so that a build -> pack -> free loop per decode iteration performs
// no cudaMalloc / cudaHostAlloc in steady state (SURVEY.md section 7.3 hard part 2).
// Free lists are kept per (device, size class): a blob is only ever reused on the device that
// owns its memory and events, and acquire() looks at blobs of the wanted size only.
// Nothing is ever freed here -- cudaFree synchronises the device, and release() runs on the
// decode loop's thread; lumen_kv_trim() is the one place that gives memory back.
class Arena {
public:
    int acquire(size_t bytes, Blob** out) {
        size_t cap = 4096;
        while (cap < bytes) cap <<= 1;
        int dev = 0;
        cudaError_t e = cudaGetDevice(&dev);
        if (e != cudaSuccess) return cuda_fail(e);
        {
            std::lock_guard<std::mutex> g(mu_);
            std::vector<Blob*>& fl = free_[std::make_pair(dev, cap)];
            for (size_t i = 0; i < fl.size(); ++i) {
                Blob* b = fl[i];
                if (!idle(b)) continue;
                fl.erase(fl.begin() + static_cast<long>(i));
                *out = b;
                return LUMEN_KV_OK;
            }
        }
        Blob* b = new (std::nothrow) Blob();
        if (!b) return LUMEN_KV_ENOMEM;
        b->cap = cap;
        b->device = dev;
        e = cudaHostAlloc(&b->host, cap, cudaHostAllocDefault);
        if (e == cudaSuccess) e = cudaMalloc(&b->dev, cap);
        if (e != cudaSuccess) {
            if (b->host) cudaFreeHost(b->host);
            delete b;
            if (e == cudaErrorMemoryAllocation) {
                (void)cudaGetLastError();
                return LUMEN_KV_ENOMEM;
            }
            return cuda_fail(e);
        }
        *out = b;
        return LUMEN_KV_OK;
    }

    void release(Blob* b) {
        if (b->host_only) {
            std::free(b->host);
            delete b;
            return;
        }
        std::lock_guard<std::mutex> g(mu_);
        if (b->captured)
            retired_.push_back(b);   // an instantiated graph may still read it: kept until trim()
        else
            free_[std::make_pair(b->device, b->cap)].push_back(b);
    }

    // Every device that owns cached blobs is synchronised before its blobs are destroyed (a blob
    // of another device than the current one may still have an upload or a kernel in flight).
    void trim() {
        int cur = 0;
        const bool have_cur = cudaGetDevice(&cur) == cudaSuccess;
        std::lock_guard<std::mutex> g(mu_);
        std::map<int, std::vector<Blob*>> by_dev;
        for (auto& kv : free_)
            for (Blob* b : kv.second) by_dev[b->device].push_back(b);
        free_.clear();
        for (Blob* b : retired_) by_dev[b->device].push_back(b);
        retired_.clear();
        for (auto& kv : by_dev) {
            if (cudaSetDevice(kv.first) == cudaSuccess) cudaDeviceSynchronize();
            for (Blob* b : kv.second) destroy(b);
        }
        if (have_cur) cudaSetDevice(cur);
        (void)cudaGetLastError();
    }

private:
    static bool idle(Blob* b) {
        // the descriptor upload reads the pinned staging: a plan built and freed unused must
        // not have it rewritten under the copy
        if (b->uploaded && cudaEventQuery(b->uploaded) != cudaSuccess) {
            (void)cudaGetLastError();
            return false;
        }
        for (auto& u : b->uses)
            if (cudaEventQuery(u.second) != cudaSuccess) {
                (void)cudaGetLastError();
                return false;
            }
        return true;
    }
    static void destroy(Blob* b) {
        for (auto& u : b->uses) cudaEventDestroy(u.second);
        if (b->uploaded) cudaEventDestroy(b->uploaded);
        if (b->host) cudaFreeHost(b->host);
        if (b->dev) cudaFree(b->dev);
        (void)cudaGetLastError();
        delete b;
    }
    std::mutex mu_;
    std::map<std::pair<int, size_t>, std::vector<Blob*>> free_;
    std::vector<Blob*> retired_;
};

Arena& arena() {
    static Arena* a = new Arena();  // leaked on purpose: no CUDA calls at process exit
    return *a;
}

// Descriptor uploads run on a stream of the library's own (one per device), not on the caller's:
// a copy-engine operation between two kernels of one stream costs ~10 us (it cannot start before
// the first kernel has drained, and the second kernel starts cold behind it); on its own stream
// the copy runs while the caller's stream is busy, and the kernel only waits for its event.
constexpr int kMaxDev = 64;
std::mutex g_upload_mu;
cudaStream_t g_upload_stream[kMaxDev] = {};

cudaError_t upload_stream(cudaStream_t* out) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDev) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> g(g_upload_mu);
    if (!g_upload_stream[dev]) {
        e = cudaStreamCreateWithFlags(&g_upload_stream[dev], cudaStreamNonBlocking);
        if (e != cudaSuccess) return e;
    }
    *out = g_upload_stream[dev];
    return cudaSuccess;
}

}  // namespace
}  // namespace lumen

namespace lumen {
namespace {

// Orders `stream` behind the plan's descriptor upload (a no-op once the copy has been seen
// complete, so that no event wait sits between two kernels of a decode loop).
int await_upload(lumen_kv_plan* p, cudaStream_t stream) {
    Blob* b = p->blob;
    if (!b) return LUMEN_KV_OK;
    std::lock_guard<std::mutex> g(b->mu);
    if (b->upload_seen || !b->uploaded) return LUMEN_KV_OK;
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(stream, &cs) != cudaSuccess) (void)cudaGetLastError();
    if (cs != cudaStreamCaptureStatusNone) {
        // An event of a stream outside the capture cannot become a graph dependency, and event
        // queries are illegal under a global-mode capture: the few microseconds of the copy are
        // waited for on the host, once, at capture time, with this thread in relaxed mode.
        cudaStreamCaptureMode mode = cudaStreamCaptureModeRelaxed;
        cudaError_t e = cudaThreadExchangeStreamCaptureMode(&mode);
        if (e != cudaSuccess) return cuda_fail(e);
        e = cudaEventSynchronize(b->uploaded);
        (void)cudaThreadExchangeStreamCaptureMode(&mode);
        if (e != cudaSuccess) return cuda_fail(e);
        b->upload_seen = true;
        return LUMEN_KV_OK;
    }
    cudaError_t e = cudaEventQuery(b->uploaded);
    if (e == cudaSuccess) {
        b->upload_seen = true;
        return LUMEN_KV_OK;
    }
    (void)cudaGetLastError();
    if (e != cudaErrorNotReady) return cuda_fail(e);
    e = cudaStreamWaitEvent(stream, b->uploaded, 0);
    return e == cudaSuccess ? LUMEN_KV_OK : cuda_fail(e);
}

// record "plan still in use on `stream`" so the arena does not recycle the blob early
int note_use(lumen_kv_plan* p, cudaStream_t stream) {
    Blob* b = p->blob;
    // Under stream capture an event record would become a graph node and could never be
    // queried; the plan must outlive the graph anyway (lumen_kv.h), so the blob is simply
    // never recycled.
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(stream, &cs) != cudaSuccess) (void)cudaGetLastError();
    std::lock_guard<std::mutex> g(b->mu);
    if (cs != cudaStreamCaptureStatusNone) {
        b->captured = true;
        return LUMEN_KV_OK;
    }
    for (auto& u : b->uses)
        if (u.first == stream) {
            cudaError_t e = cudaEventRecord(u.second, stream);
            return e == cudaSuccess ? LUMEN_KV_OK : cuda_fail(e);
        }
    cudaEvent_t ev;
    cudaError_t e = cudaEventCreateWithFlags(&ev, cudaEventDisableTiming);
    if (e != cudaSuccess) return cuda_fail(e);
    e = cudaEventRecord(ev, stream);
    if (e != cudaSuccess) {
        cudaEventDestroy(ev);
        return cuda_fail(e);
    }
    b->uses.emplace_back(stream, ev);
    return LUMEN_KV_OK;
}

}  // namespace

int gather_planes(const lumen_kv_plan* plan, const void* const* k_planes,
                  const void* const* v_planes, std::vector<const void*>* planes) {
    if (!k_planes || !v_planes) return LUMEN_KV_EINVAL;
    const int32_t L = plan->hp.geom.num_layers;
    planes->resize(static_cast<size_t>(2 * L));
    for (int32_t l = 0; l < L; ++l) {
        const void* k = k_planes[l];
        const void* v = v_planes[l];
        if (!k || !v) return LUMEN_KV_EINVAL;
        if ((reinterpret_cast<uintptr_t>(k) | reinterpret_cast<uintptr_t>(v)) & 15)
            return LUMEN_KV_EINVAL;
        (*planes)[2 * l] = k;
        (*planes)[2 * l + 1] = v;
    }
    return LUMEN_KV_OK;
}

int launch_part(const lumen_kv_plan* plan, const std::vector<const void*>& planes, uintptr_t buf,
                bool buf_is_host, cudaStream_t stream, bool pack, int64_t ra, int64_t rb,
                int32_t p0, int32_t p1, bool buf_is_peer) {
    if (rb <= ra || p1 <= p0) return LUMEN_KV_OK;
    CopyArgs a;
    a.inline_desc = plan->inline_desc;
    a.runs = (plan->inline_desc ? plan->h_runs : plan->d_runs) + ra;
    a.reqs = plan->inline_desc ? plan->h_reqs : plan->d_reqs;
    a.n_runs = rb - ra;
    a.n_reqs = plan->n_reqs;
    a.row_bytes = plan->hp.row_bytes;
    a.max_count = plan->hp.max_count;
    a.pool_align32 = plan->hp.row_bytes % 32 == 0 && plan->hp.page_stride % 32 == 0;
    a.planes = planes.data() + p0;
    a.n_planes = p1 - p0;
    a.plane_base = p0;
    a.buf = reinterpret_cast<void*>(buf);
    a.buf_is_host = buf_is_host;
    a.buf_is_peer = buf_is_peer;
    a.pack = pack;
    a.kernel = static_cast<int>((plan->flags & LUMEN_KV_KERNEL_MASK) >> LUMEN_KV_KERNEL_SHIFT);
    a.stream = stream;
    if (!plan->inline_desc) {
        const int rc = await_upload(const_cast<lumen_kv_plan*>(plan), stream);
        if (rc != LUMEN_KV_OK) return rc;
    }
    cudaError_t e = launch_kv_copy(a);
    if (e != cudaSuccess) return cuda_fail(e);
    if (plan->inline_desc) return LUMEN_KV_OK;   // nothing on the device to keep alive
    return note_use(const_cast<lumen_kv_plan*>(plan), stream);
}

void plan_retain(const lumen_kv_plan* plan) {
    const_cast<lumen_kv_plan*>(plan)->refs.fetch_add(1, std::memory_order_relaxed);
}

void plan_release(const lumen_kv_plan* plan_) {
    lumen_kv_plan* plan = const_cast<lumen_kv_plan*>(plan_);
    if (plan->refs.fetch_sub(1, std::memory_order_acq_rel) != 1) return;
    if (plan->blob) arena().release(plan->blob);
    delete plan;
}

int plan_chunks(const lumen_kv_plan* plan_, int64_t slot_bytes,
                std::shared_ptr<const std::vector<Chunk>>* out) {
    lumen_kv_plan* plan = const_cast<lumen_kv_plan*>(plan_);
    std::lock_guard<std::mutex> g(plan->chunk_mu);
    if (!plan->chunk_list || plan->chunk_slot_bytes != slot_bytes) {
        auto v = std::make_shared<std::vector<Chunk>>();
        const int rc = build_chunks(plan->hp, plan->h_runs, slot_bytes, v.get());
        if (rc != LUMEN_KV_OK) return rc;
        plan->chunk_list = std::move(v);
        plan->chunk_slot_bytes = slot_bytes;
    }
    *out = plan->chunk_list;
    return LUMEN_KV_OK;
}

namespace {

// LUMEN_KV_MEM_DEVICE promises memory of the current device (its L2 may be asked for the bytes
// early).  A caller that passes a peer GPU's buffer under that kind -- legal before the kinds were
// told apart -- must not get stale data for it: the owner is looked up when a thread sees a
// buffer for the first time (one pointer comparison per call afterwards), and a buffer of
// another device is handled as LUMEN_KV_MEM_DEVICE_PEER.  A lookup that fails decides nothing.
bool buffer_is_local(const void* buf) {
    static thread_local const void* seen_buf = nullptr;
    static thread_local int seen_dev = -1;
    static thread_local bool seen_local = true;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) {
        (void)cudaGetLastError();
        return true;
    }
    if (buf == seen_buf && dev == seen_dev) return seen_local;
    cudaPointerAttributes at;
    bool local = true;
    if (cudaPointerGetAttributes(&at, buf) == cudaSuccess)
        local = !(at.type == cudaMemoryTypeDevice && at.device != dev);
    else
        (void)cudaGetLastError();
    seen_buf = buf;
    seen_dev = dev;
    seen_local = local;
    return local;
}

int run_copy(const lumen_kv_plan* plan, const void* const* k_planes, const void* const* v_planes,
             void* buf, int64_t buf_bytes, int kind, void* stream, bool pack) {
    if (!plan) return LUMEN_KV_EINVAL;
    if (plan->flags & LUMEN_KV_HOST_ONLY) return LUMEN_KV_EINVAL;
    if (kind != LUMEN_KV_MEM_DEVICE && kind != LUMEN_KV_MEM_HOST_MAPPED &&
        kind != LUMEN_KV_MEM_DEVICE_PEER)
        return LUMEN_KV_EINVAL;
    if (buf_bytes < plan->hp.total_bytes) return LUMEN_KV_ESIZE;
    if (plan->hp.total_bytes == 0) return LUMEN_KV_OK;  // A4: empty plan launches nothing
    if (!buf) return LUMEN_KV_EINVAL;
    // reused across calls: after a thread's first call this allocates nothing
    static thread_local std::vector<const void*> planes;
    int rc = gather_planes(plan, k_planes, v_planes, &planes);
    if (rc != LUMEN_KV_OK) return rc;
    void* dev_buf = buf;
    if (kind == LUMEN_KV_MEM_HOST_MAPPED) {
        cudaError_t e = cudaHostGetDevicePointer(&dev_buf, buf, 0);
        if (e != cudaSuccess) {
            t_last_cuda_error = static_cast<int>(e);
            (void)cudaGetLastError();
            return LUMEN_KV_EINVAL;  // not pinned / not mapped
        }
    }
    if (reinterpret_cast<uintptr_t>(dev_buf) & 15) return LUMEN_KV_EINVAL;
    if (kind == LUMEN_KV_MEM_DEVICE && !buffer_is_local(dev_buf)) kind = LUMEN_KV_MEM_DEVICE_PEER;
    return launch_part(plan, planes, reinterpret_cast<uintptr_t>(dev_buf),
                       kind == LUMEN_KV_MEM_HOST_MAPPED, static_cast<cudaStream_t>(stream), pack, 0,
                       plan->n_runs, 0, 2 * plan->hp.geom.num_layers,
                       kind == LUMEN_KV_MEM_DEVICE_PEER);
}

}  // namespace
}  // namespace lumen

extern "C" {

int lumen_kv_plan_build(const lumen_kv_geom* geom, const lumen_kv_req* reqs, int32_t num_reqs,
                        uint32_t flags, void* stream, lumen_kv_plan** out) {
    return lumen_kv_plan_build_layout(geom, reqs, nullptr, num_reqs, flags, stream, out);
}

int lumen_kv_plan_build_layout(const lumen_kv_geom* geom, const lumen_kv_req* reqs,
                               const lumen_kv_req_layout* layouts, int32_t num_reqs,
                               uint32_t flags, void* stream, lumen_kv_plan** out) {
    using namespace lumen;
    if (!out) return LUMEN_KV_EINVAL;
    *out = nullptr;
    const uint32_t ksel = flags & LUMEN_KV_KERNEL_MASK;
    if (ksel != LUMEN_KV_KERNEL_AUTO && ksel != LUMEN_KV_KERNEL_WARP && ksel != LUMEN_KV_KERNEL_BULK)
        return LUMEN_KV_EINVAL;
    lumen_kv_plan* p = new (std::nothrow) lumen_kv_plan();
    if (!p) return LUMEN_KV_ENOMEM;
    int rc;
    try {
        rc = build_host_plan(geom, reqs, layouts, num_reqs, flags, &p->hp);
    } catch (const std::bad_alloc&) {
        rc = LUMEN_KV_ENOMEM;
    } catch (const std::exception&) {   // e.g. length_error: nothing may cross the C boundary
        rc = LUMEN_KV_ENOMEM;
    }
    if (rc != LUMEN_KV_OK) {
        delete p;
        return rc;
    }
    p->flags = flags;
    p->n_runs = static_cast<int64_t>(p->hp.runs.size());
    p->n_reqs = num_reqs;

    const size_t run_bytes = p->hp.runs.size() * sizeof(RunDesc);
    const size_t req_bytes = p->hp.reqs.size() * sizeof(ReqDesc);
    const size_t total = run_bytes + req_bytes;

    // Small plans (a decode step's deltas) need no device copy at all: the kernel receives
    // the descriptors in its parameters.
    if (!(flags & (LUMEN_KV_HOST_ONLY | LUMEN_KV_NO_INLINE)) && p->n_runs <= inline_max_runs() && num_reqs <= kInlineReqsL) {
        p->inline_desc = true;
        p->h_runs = p->hp.runs.data();
        p->h_reqs = p->hp.reqs.data();
        *out = p;
        return LUMEN_KV_OK;
    }

    if (flags & LUMEN_KV_HOST_ONLY) {
        Blob* b = new (std::nothrow) Blob();
        if (!b) { delete p; return LUMEN_KV_ENOMEM; }
        b->host_only = true;
        b->cap = total ? total : 16;
        b->host = std::malloc(b->cap);
        if (!b->host) { delete b; delete p; return LUMEN_KV_ENOMEM; }
        p->blob = b;
    } else if (total > 0) {
        rc = arena().acquire(total, &p->blob);
        if (rc != LUMEN_KV_OK) { delete p; return rc; }
    }
    if (p->blob) {
        char* h = static_cast<char*>(p->blob->host);
        if (run_bytes) std::memcpy(h, p->hp.runs.data(), run_bytes);
        if (req_bytes) std::memcpy(h + run_bytes, p->hp.reqs.data(), req_bytes);
        p->h_runs = reinterpret_cast<const RunDesc*>(h);
        p->h_reqs = reinterpret_cast<const ReqDesc*>(h + run_bytes);
        if (!(flags & LUMEN_KV_HOST_ONLY)) {
            char* d = static_cast<char*>(p->blob->dev);
            p->d_runs = reinterpret_cast<const RunDesc*>(d);
            p->d_reqs = reinterpret_cast<const ReqDesc*>(d + run_bytes);
            (void)stream;   // kept in the signature; the upload has a stream of its own (see above)
            cudaStream_t s = nullptr;
            cudaError_t e = upload_stream(&s);
            Blob* b = p->blob;
            if (e == cudaSuccess && !b->uploaded)
                e = cudaEventCreateWithFlags(&b->uploaded, cudaEventDisableTiming);
            // a recycled blob is idle (Arena::acquire): nothing enqueued still reads its device copy
            if (e == cudaSuccess) e = cudaMemcpyAsync(d, h, total, cudaMemcpyHostToDevice, s);
            if (e == cudaSuccess) e = cudaEventRecord(b->uploaded, s);
            b->upload_seen = false;
            if (e != cudaSuccess) {
                arena().release(p->blob);
                delete p;
                return cuda_fail(e);
            }
        }
    }
    // the vectors are no longer needed: descriptors live in the blob
    std::vector<RunDesc>().swap(p->hp.runs);
    std::vector<ReqDesc>().swap(p->hp.reqs);
    *out = p;
    return LUMEN_KV_OK;
}

int64_t lumen_kv_plan_bytes(const lumen_kv_plan* plan) {
    return plan ? plan->hp.total_bytes : int64_t{LUMEN_KV_EINVAL};
}

int64_t lumen_kv_plan_req_offset(const lumen_kv_plan* plan, int32_t r) {
    if (!plan || r < 0 || r > plan->n_reqs) return LUMEN_KV_EINVAL;
    return plan->hp.req_offset[static_cast<size_t>(r)];
}

int64_t lumen_kv_plan_num_runs(const lumen_kv_plan* plan) {
    return plan ? plan->n_runs : int64_t{LUMEN_KV_EINVAL};
}

int lumen_kv_plan_get_run(const lumen_kv_plan* plan, int64_t i, lumen_kv_run_info* out) {
    if (!plan || !out || i < 0 || i >= plan->n_runs) return LUMEN_KV_EINVAL;
    const lumen::RunDesc& d = plan->h_runs[i];
    const int64_t off = ((static_cast<int64_t>(d.src_hi) << 32) | d.src_lo) << 4;
    const int64_t page = off / plan->hp.page_stride;
    const int64_t slot = (off % plan->hp.page_stride) / plan->hp.row_bytes;
    out->src_slot = page * plan->hp.geom.page_size + slot;
    out->dst_token = d.dst_tok;
    out->req = static_cast<int32_t>(d.req);
    out->count = d.count;
    return LUMEN_KV_OK;
}

int lumen_kv_checkpoint_pack(const lumen_kv_plan* plan, const void* const* k_planes,
                             const void* const* v_planes, void* dst, int64_t dst_bytes,
                             int dst_kind, void* stream) {
    return lumen::run_copy(plan, k_planes, v_planes, dst, dst_bytes, dst_kind, stream, true);
}

int lumen_kv_restore_unpack(const lumen_kv_plan* plan, void* const* k_planes,
                            void* const* v_planes, const void* src, int64_t src_bytes,
                            int src_kind, void* stream) {
    return lumen::run_copy(plan, const_cast<const void* const*>(k_planes),
                           const_cast<const void* const*>(v_planes), const_cast<void*>(src),
                           src_bytes, src_kind, stream, false);
}

void lumen_kv_plan_free(lumen_kv_plan* plan) {
    if (plan) lumen::plan_release(plan);
}

void lumen_kv_trim(void) { lumen::arena().trim(); }

int lumen_kv_set_option(const char* name, int value) {
    if (name && !std::strcmp(name, "inline_max_runs")) {   // A/B: which plans ride in the parameters
        lumen::g_inline_max_runs = value < 0 ? 0 : (value > lumen::kInlineRunsL ? lumen::kInlineRunsL : value);
        return LUMEN_KV_OK;
    }
    if (name && !std::strcmp(name, "fail_after_chunks")) {   // error-path tests of the staged calls
        lumen::g_fail_after_chunks.store(value < 0 ? -1 : value);
        return LUMEN_KV_OK;
    }
    return lumen::set_option(name, value) == 0 ? LUMEN_KV_OK : LUMEN_KV_EINVAL;
}

int lumen_kv_init(void) {
    const cudaError_t e = lumen::init_current_device();
    return e == cudaSuccess ? LUMEN_KV_OK : lumen::cuda_fail(e);
}

const char* lumen_kv_strerror(int status) {
    switch (status) {
        case LUMEN_KV_OK: return "ok";
        case LUMEN_KV_EINVAL: return "invalid argument (null, misaligned, bad geometry, kind or flag)";
        case LUMEN_KV_ERANGE: return "page index or token range outside the page table / pool";
        case LUMEN_KV_EOVERLAP: return "a pool token slot is addressed more than once";
        case LUMEN_KV_ESIZE: return "buffer smaller than the plan's bytes";
        case LUMEN_KV_ENOMEM: return "out of memory (descriptors), or no room for the reservation in the store arena";
        case LUMEN_KV_ECUDA: return "CUDA runtime error (see lumen_kv_last_cuda_error)";
        case LUMEN_KV_ESINK: return "the checkpointer's sink rejected a delta";
        case LUMEN_KV_ECAPACITY:
            return "plan too large for lumen_kv_copy_noalloc (more than 65,536 runs or 4,096 requests)";
        default: return "unknown status";
    }
}

int lumen_kv_last_cuda_error(void) { return lumen::t_last_cuda_error; }
int lumen_kv_version(void) { return LUMEN_KV_VERSION; }

}  // extern "C"
