// lumen_kv_copy_noalloc: pack / restore for callers that must not allocate GPU memory.
//
// Who that is.  A serving worker normally gives every free byte of HBM to its KV pool at
// start-up, and the moment it most needs a restore -- a recovery burst, when it takes over a
// failed peer's requests -- is the moment that pool is fullest: a cudaMalloc
// for a plan's descriptors can then fail, and even when it succeeds cudaMalloc / cudaFree
// synchronise the whole device, which a decode loop cannot afford.  Other callers simply run
// under a policy that every device byte comes from their own pool.  The regular calls cover
// plans of up to 1,024 runs without device memory (descriptors ride in the kernel parameters);
// beyond that they upload the descriptors into memory the library allocates.  This file is the
// alternative for the larger plans: the descriptors go into a fixed array that is part of the
// library's image, so nothing is allocated by anyone, at any time.
//
// How.  g_desc below is a file-scope device array (1,088 KiB: 65,536 run descriptors and 4,096
// request descriptors of 16 bytes; every GPU that loads the library carries it until the process
// exits).  A call first writes the plan's descriptors into it with stage_desc -- a tiny kernel
// that receives up to 1,024 descriptors in its parameters and names g_desc directly, so the
// bytes leave the host at launch time and no host buffer has to outlive the call -- and then
// launches kv_copy_static, the warp-per-task gather / scatter of kernels.cu reading its
// descriptors from g_desc.  Host code cannot use the name g_desc as an address (on the host it
// is only a handle for the runtime's symbol table); the kernel is given the pointer that
// cudaGetSymbolAddress returned for the current device, looked up once per device.
#include <cuda_runtime.h>

#include <cstdint>
#include <mutex>

#include "internal.hpp"
#include "lumen_kv.h"
#include "plan.hpp"

namespace lumen {
namespace {

constexpr int64_t kMaxRuns = LUMEN_KV_NOALLOC_MAX_RUNS;
constexpr int64_t kMaxReqs = LUMEN_KV_NOALLOC_MAX_REQS;
static_assert(sizeof(RunDesc) == sizeof(uint4) && sizeof(ReqDesc) == sizeof(uint4), "16-byte descriptors");

// [0, kMaxRuns): run descriptors; [kMaxRuns, kMaxRuns + kMaxReqs): request descriptors.
// Never cleared: a call overwrites entries [0, n_runs) and [kMaxRuns, kMaxRuns + n_reqs) and
// its kernel indexes nothing else, so whatever an earlier call left behind is never read.
static __device__ __align__(256) uint4 g_desc[kMaxRuns + kMaxReqs];

constexpr int kSlice = 1024;          // descriptors per stage_desc launch (16 KiB of parameters)
struct DescSlice {
    uint4 e[kSlice];
};

__global__ void __launch_bounds__(256)
stage_desc(const __grid_constant__ DescSlice s, uint32_t first, uint32_t count) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < count) g_desc[first + i] = s.e[i];      // device code may name the array
}

constexpr int kPlanesPerLaunch = 256;
struct PlaneTable {
    void* p[kPlanesPerLaunch];
};

constexpr int kWarps = 8;
constexpr int kUnroll = 4;

template <int VB>
struct Vec;
template <>
struct Vec<16> {
    uint4 v;
    __device__ __forceinline__ void load(const void* p) {
        asm volatile("ld.global.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                     : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p) : "memory");
    }
    __device__ __forceinline__ void store(void* p) const {
        asm volatile("st.global.L1::no_allocate.v4.u32 [%0], {%1,%2,%3,%4};" ::"l"(p), "r"(v.x),
                     "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
    }
};
template <>
struct Vec<32> {
    uint32_t a[8];
    __device__ __forceinline__ void load(const void* p) {
        asm volatile("ld.global.L1::no_allocate.v8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                     : "=r"(a[0]), "=r"(a[1]), "=r"(a[2]), "=r"(a[3]), "=r"(a[4]), "=r"(a[5]),
                       "=r"(a[6]), "=r"(a[7]) : "l"(p) : "memory");
    }
    __device__ __forceinline__ void store(void* p) const {
        asm volatile("st.global.L1::no_allocate.v8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"l"(p),
                     "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(a[4]), "r"(a[5]), "r"(a[6]),
                     "r"(a[7]) : "memory");
    }
};

// One warp per (run, plane, sub-chunk of kUnroll*32*VB bytes); the index map is the one of
// include/lumen_kv.h (PAPER.md:145 for pack, PAPER.md:157-163 for restore).  `desc` is the
// device address of g_desc.
template <int VB>
__global__ void __launch_bounds__(kWarps * 32)
kv_copy_static(const __grid_constant__ PlaneTable planes, const uint4* __restrict__ desc,
               int64_t n_runs, char* buf, uint32_t row_bytes, int32_t plane0, int sub_shift,
               int pack) {
    constexpr uint32_t kTask = kUnroll * 32 * VB;
    const int lane = threadIdx.x & 31;
    const int64_t task = static_cast<int64_t>(blockIdx.x) * kWarps + (threadIdx.x >> 5);
    const int64_t run = task >> sub_shift;
    if (run >= n_runs) return;
    const uint32_t sub = static_cast<uint32_t>(task & ((int64_t{1} << sub_shift) - 1));
    const uint4 d = __ldg(desc + run);                   // RunDesc: src_lo, dst_tok, req, count | src_hi << 16
    const uint32_t bytes = (d.w & 0xFFFFu) * row_bytes;
    if (sub * kTask >= bytes) return;                    // this run is shorter than the longest one
    const uint64_t off16 = (static_cast<uint64_t>(d.w >> 16) << 32) | d.x;
    const uint4 qw = __ldg(desc + kMaxRuns + d.z);       // ReqDesc: row_base, n (two int64)
    const int64_t row_base = static_cast<int64_t>((static_cast<uint64_t>(qw.y) << 32) | qw.x);
    const int64_t n = static_cast<int64_t>((static_cast<uint64_t>(qw.w) << 32) | qw.z);
    const int64_t row = row_base + static_cast<int64_t>(plane0 + blockIdx.y) * n + d.y;
    char* pool = static_cast<char*>(planes.p[blockIdx.y]) + (off16 << 4);
    char* b = buf + row * static_cast<int64_t>(row_bytes);
    const uint32_t nvec = bytes / VB;
    const uint32_t i = sub * (kUnroll * 32) + lane;
    const char* src = (pack ? pool : b) + static_cast<size_t>(i) * VB;
    char* dst = (pack ? b : pool) + static_cast<size_t>(i) * VB;
    Vec<VB> v[kUnroll];
#pragma unroll
    for (int u = 0; u < kUnroll; ++u)
        if (i + u * 32 < nvec) v[u].load(src + u * (32 * VB));
#pragma unroll
    for (int u = 0; u < kUnroll; ++u)
        if (i + u * 32 < nvec) v[u].store(dst + u * (32 * VB));
}

// Set-up, once per device and with that device current: the device address of g_desc, and the
// load of the three kernels (CUDA loads a kernel lazily at its first launch).
struct DeviceSetup {
    std::once_flag once;
    cudaError_t err = cudaSuccess;
    uint4* desc = nullptr;
};
constexpr int kMaxDev = 64;
DeviceSetup g_setup[kMaxDev];
std::mutex g_enqueue_mu;   // one call's launches are enqueued as a block

cudaError_t setup_current_device(DeviceSetup** out) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDev) return cudaErrorInvalidDevice;
    DeviceSetup& s = g_setup[dev];
    std::call_once(s.once, [&s] {
        void* p = nullptr;
        s.err = cudaGetSymbolAddress(&p, g_desc);
        if (s.err != cudaSuccess) return;
        s.desc = static_cast<uint4*>(p);
        cudaFuncAttributes fa;
        s.err = cudaFuncGetAttributes(&fa, stage_desc);
        if (s.err == cudaSuccess) s.err = cudaFuncGetAttributes(&fa, kv_copy_static<16>);
        if (s.err == cudaSuccess) s.err = cudaFuncGetAttributes(&fa, kv_copy_static<32>);
    });
    *out = &s;
    return s.err;
}

cudaError_t stage(const void* host, int64_t count, int64_t first, cudaStream_t stream) {
    const uint4* src = static_cast<const uint4*>(host);
    for (int64_t at = 0; at < count; at += kSlice) {
        const int64_t n = count - at < kSlice ? count - at : kSlice;
        DescSlice s;                                   // filled on the stack, copied by the launch
        for (int64_t i = 0; i < n; ++i) s.e[i] = src[at + i];
        stage_desc<<<static_cast<unsigned>((n + 255) / 256), 256, 0, stream>>>(
            s, static_cast<uint32_t>(first + at), static_cast<uint32_t>(n));
        const cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

}  // namespace
}  // namespace lumen

extern "C" int lumen_kv_copy_noalloc(const lumen_kv_plan* plan, int direction,
                                     void* const* k_planes, void* const* v_planes, void* buf,
                                     int64_t buf_bytes, int buf_kind, void* stream_) {
    using namespace lumen;
    if (!plan || !k_planes || !v_planes) return LUMEN_KV_EINVAL;
    if (direction != LUMEN_KV_DIR_PACK && direction != LUMEN_KV_DIR_RESTORE) return LUMEN_KV_EINVAL;
    if (buf_kind != LUMEN_KV_MEM_DEVICE && buf_kind != LUMEN_KV_MEM_HOST_MAPPED &&
        buf_kind != LUMEN_KV_MEM_DEVICE_PEER)
        return LUMEN_KV_EINVAL;
    // the size limit comes before anything that touches CUDA
    if (plan->n_runs > kMaxRuns || plan->n_reqs > kMaxReqs) return LUMEN_KV_ECAPACITY;
    if (buf_bytes < plan->hp.total_bytes) return LUMEN_KV_ESIZE;
    if (plan->hp.total_bytes == 0 || plan->n_runs == 0) return LUMEN_KV_OK;
    if (!buf || !plan->h_runs || !plan->h_reqs) return LUMEN_KV_EINVAL;
    const int32_t n_planes = 2 * plan->hp.geom.num_layers;
    bool wide = plan->hp.row_bytes % 32 == 0 && plan->hp.page_stride % 32 == 0;
    for (int32_t l = 0; l < plan->hp.geom.num_layers; ++l) {
        const uintptr_t k = reinterpret_cast<uintptr_t>(k_planes[l]);
        const uintptr_t v = reinterpret_cast<uintptr_t>(v_planes[l]);
        if (!k || !v || ((k | v) & 15)) return LUMEN_KV_EINVAL;
        if ((k | v) & 31) wide = false;
    }

    DeviceSetup* dev = nullptr;
    cudaError_t e = setup_current_device(&dev);
    if (e != cudaSuccess) return cuda_fail(e);

    void* dbuf = buf;
    if (buf_kind == LUMEN_KV_MEM_HOST_MAPPED) {
        e = cudaHostGetDevicePointer(&dbuf, buf, 0);     // a table lookup; fails for unpinned memory
        if (e != cudaSuccess) {
            (void)cuda_fail(e);
            return LUMEN_KV_EINVAL;
        }
    }
    if (reinterpret_cast<uintptr_t>(dbuf) & 15) return LUMEN_KV_EINVAL;
    if (reinterpret_cast<uintptr_t>(dbuf) & 31) wide = false;

    const int64_t item_max = static_cast<int64_t>(plan->hp.max_count) * plan->hp.row_bytes;
    const int64_t task_bytes = (wide ? 32 : 16) * 32 * kUnroll;
    int sub_shift = 0;
    while ((task_bytes << sub_shift) < item_max) ++sub_shift;
    const int64_t gx = ((plan->n_runs << sub_shift) + kWarps - 1) / kWarps;
    if (gx > 0x7fffffffLL) return LUMEN_KV_EINVAL;

    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    std::lock_guard<std::mutex> g(g_enqueue_mu);
    e = stage(plan->h_runs, plan->n_runs, 0, stream);
    if (e == cudaSuccess) e = stage(plan->h_reqs, plan->n_reqs, kMaxRuns, stream);
    for (int32_t p0 = 0; e == cudaSuccess && p0 < n_planes; p0 += kPlanesPerLaunch) {
        const int32_t np = n_planes - p0 < kPlanesPerLaunch ? n_planes - p0 : kPlanesPerLaunch;
        PlaneTable pt;
        for (int32_t i = 0; i < kPlanesPerLaunch; ++i) {
            const int32_t p = p0 + i;                    // plane = 2*layer + (0: K, 1: V)
            pt.p[i] = i < np ? ((p & 1) ? v_planes[p >> 1] : k_planes[p >> 1]) : nullptr;
        }
        const dim3 grid(static_cast<unsigned>(gx), static_cast<unsigned>(np), 1);
        const int pack = direction == LUMEN_KV_DIR_PACK ? 1 : 0;
        if (wide)
            kv_copy_static<32><<<grid, kWarps * 32, 0, stream>>>(
                pt, dev->desc, plan->n_runs, static_cast<char*>(dbuf),
                static_cast<uint32_t>(plan->hp.row_bytes), p0, sub_shift, pack);
        else
            kv_copy_static<16><<<grid, kWarps * 32, 0, stream>>>(
                pt, dev->desc, plan->n_runs, static_cast<char*>(dbuf),
                static_cast<uint32_t>(plan->hp.row_bytes), p0, sub_shift, pack);
        e = cudaGetLastError();
    }
    return e == cudaSuccess ? LUMEN_KV_OK : cuda_fail(e);
}
