// Internals shared by the C entry points (lib.cu) and the two-stage host path (stager.cu).
// Not part of the public ABI.
#pragma once
#include <cuda_runtime.h>

#include <atomic>
#include <cstdint>
#include <memory>
#include <mutex>
#include <vector>

#include "lumen_kv.h"
#include "plan.hpp"

namespace lumen {
struct Blob;   // descriptor blob of the arena (lib.cu)

// records the CUDA error for lumen_kv_last_cuda_error() and returns LUMEN_KV_ECUDA
int cuda_fail(cudaError_t e);
// failure injection for the staged paths (stager.cu)
extern std::atomic<int> g_fail_after_chunks;
}  // namespace lumen

struct lumen_kv_plan {
    lumen::HostPlan hp;        // runs/reqs vectors are released after upload unless host-only
    lumen::Blob* blob = nullptr;
    const lumen::RunDesc* h_runs = nullptr;   // inside blob->host
    const lumen::ReqDesc* h_reqs = nullptr;
    const lumen::RunDesc* d_runs = nullptr;   // inside blob->dev
    const lumen::ReqDesc* d_reqs = nullptr;
    int64_t n_runs = 0;
    int32_t n_reqs = 0;
    uint32_t flags = 0;
    bool inline_desc = false;  // small plan: descriptors stay in hp and travel as kernel parameters
    // lumen_kv_plan_free drops the caller's reference; an asynchronous staged call holds one of
    // its own until the stager's thread has issued it
    std::atomic<int> refs{1};
    // the chunk list of the two-stage path, built once per slot size and shared with whoever
    // is still issuing from it
    std::mutex chunk_mu;
    int64_t chunk_slot_bytes = 0;
    std::shared_ptr<const std::vector<lumen::Chunk>> chunk_list;
};

namespace lumen {

void plan_retain(const lumen_kv_plan* plan);
void plan_release(const lumen_kv_plan* plan);   // frees the plan with the last reference

// The plan's chunks for this slot size (build_chunks, cached on the plan); a lumen_kv_status.
int plan_chunks(const lumen_kv_plan* plan, int64_t slot_bytes,
                std::shared_ptr<const std::vector<Chunk>>* out);

// validation shared by the one-shot and the staged calls: interleaves the plane pointers
// (K0,V0,K1,V1,..) into `planes`
int gather_planes(const lumen_kv_plan* plan, const void* const* k_planes,
                  const void* const* v_planes, std::vector<const void*>* planes);

// Enqueue runs [ra, rb) x planes [p0, p1) of the plan.  `buf` is the address that byte 0 of
// the plan's checkpoint buffer would have (for a staging slot: slot base - chunk offset, so
// it may lie outside any allocation; only bytes of the chunk are ever addressed).
int launch_part(const lumen_kv_plan* plan, const std::vector<const void*>& planes, uintptr_t buf,
                bool buf_is_host, cudaStream_t stream, bool pack, int64_t ra, int64_t rb,
                int32_t p0, int32_t p1, bool buf_is_peer = false);

}  // namespace lumen
