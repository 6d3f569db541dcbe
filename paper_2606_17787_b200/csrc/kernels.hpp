// Launcher interface between the C entry points (lib.cu) and the kernels (kernels.cu).
#pragma once
#include <cuda_runtime.h>

#include <cstdint>

#include "plan.hpp"

namespace lumen {

constexpr int kMaxPlanesPerLaunch = 256;  // plane pointers travel as kernel parameters

// Small plans (one decode step: 64 requests x 1-2 runs) travel entirely in the kernel
// parameters: no descriptor upload, no device blob, and a CTA starts its payload loads
// without first waiting on two dependent descriptor loads from global memory.
// Two size classes, so that the common decode step pays for 6 KiB of parameters and a batch of a
// few hundred requests (whose upload would cost ~10 us per launch: a copy-engine hop between two
// kernels) for 24 KiB; the parameter space of a kernel is 32,764 bytes.
constexpr int kInlineRuns = 256;
constexpr int kInlineReqs = 128;
constexpr int kInlineRunsL = 1024;
constexpr int kInlineReqsL = 512;

enum KernelKind : int { kKernelAuto = 0, kKernelWarp = 1, kKernelBulk = 2 };

struct CopyArgs {
    const RunDesc* runs = nullptr;   // device (or host when inline_desc)
    const ReqDesc* reqs = nullptr;   // device (or host when inline_desc)
    int32_t n_reqs = 0;
    bool inline_desc = false;        // descriptors are HOST pointers, passed as kernel parameters
    int64_t n_runs = 0;
    int64_t row_bytes = 0;
    int32_t max_count = 0;           // longest run in tokens
    bool pool_align32 = false;       // row and page stride are multiples of 32 bytes
    const void* const* planes = nullptr;  // HOST array of n_planes device pointers (K0,V0,K1,V1,..)
    int32_t n_planes = 0;
    int32_t plane_base = 0;          // absolute index of planes[0] (a launch over a plane sub-range)
    void* buf = nullptr;             // device-accessible checkpoint buffer
    bool buf_is_host = false;        // mapped pinned host memory
    bool buf_is_peer = false;        // another GPU's memory (peer mapped): never prefetched early
    bool pack = true;                // true: planes -> buf, false: buf -> planes
    int kernel = kKernelAuto;
    cudaStream_t stream = nullptr;
};

// Enqueues the copy.  No synchronisation, no allocation.
cudaError_t launch_kv_copy(const CopyArgs& a);

// One-time initialisation of the CURRENT device (SM count, load of every kernel variant and its
// shared-memory limit); launch_kv_copy does it by itself at the first launch on a device.
cudaError_t init_current_device();

// Tuning knobs (the LUMEN_KV_* environment variables, settable at run time): 0 or -1 (unknown name).
int set_option(const char* name, int value);

// Which kernel AUTO resolves to for these arguments (exposed for tests / bench notes).
int resolve_kernel(const CopyArgs& a);

}  // namespace lumen
