// sm_100a kernels for the KV checkpoint pack (gather) and restore unpack (scatter).
//
// Both directions are the same byte permutation (PAPER.md:145 step 3 and
// PAPER.md:157-163; index map in include/lumen_kv.h): a work item is one
// (token-run, plane) pair, `count*row` contiguous bytes on the pool side and on the
// buffer side.  Pure data movement: no tensor cores, no arithmetic on the payload,
// the 16-bit words are never interpreted (they include NaN encodings).
//
// Kernels, chosen per launch:
//   kv_copy_warp32 / kv_copy_warp : SIMT, the HBM <-> HBM path.  One warp per (run, plane,
//                  sub-chunk), 32-byte (LDG/STG.E.256) or 16-byte accesses per lane, UNROLL
//                  independent loads in flight per lane before the first store; descriptors
//                  in global memory or in the kernel parameters (two size classes);
//                  programmatic dependent launch, with an L2 prefetch of the source
//                  (cp.async.bulk.prefetch.L2, UBLKPF) ahead of the stream-order wait.
//   kv_copy_bulk : TMA, the zero-copy host path (small grid).  Persistent single-warp CTAs;
//                  one elected lane moves whole items global -> shared ring -> global with
//                  1-D cp.async.bulk (UBLKCP), completion tracked by mbarriers (loads) and
//                  bulk groups (stores).  The other lanes only decode descriptors.
#include "kernels.hpp"

#include <cstdlib>
#include <cstring>
#include <mutex>

namespace lumen {

int g_host_kernel = kKernelBulk;   // LUMEN_KV_HOST_KERNEL=warp|bulk: what AUTO picks for host buffers

namespace {

struct PlaneTable {
    const void* p[kMaxPlanesPerLaunch];
};

// ---------------------------------------------------------------------------------
// small PTX helpers
// ---------------------------------------------------------------------------------
__device__ __forceinline__ uint4 ld_stream16(const void* p) {
    uint4 v;
    asm volatile("ld.global.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w)
                 : "l"(p)
                 : "memory");
    return v;
}
__device__ __forceinline__ void st_stream16(void* p, const uint4& v) {
    asm volatile("st.global.L1::no_allocate.v4.u32 [%0], {%1,%2,%3,%4};" ::"l"(p), "r"(v.x),
                 "r"(v.y), "r"(v.z), "r"(v.w)
                 : "memory");
}

// Programmatic dependent launch (sm_90+): `launch_dependents` lets the next kernel in the
// stream become resident while this grid's last wave drains; `wait` blocks until every
// prerequisite grid has completed and its memory is visible.  A kernel that was not
// launched with the programmatic attribute executes both as no-ops.
__device__ __forceinline__ void pdl_launch_dependents() {
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
}
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// Hint: bring `bytes` (a multiple of 16) at `p` into L2.  L2 is the device's point of coherence,
// so a line fetched early still shows every store that reaches L2 before the later load.
__device__ __forceinline__ void l2_prefetch_bulk(const void* p, uint32_t bytes) {
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
}

// Where the descriptors live: in global memory (uploaded by plan_build) or, for small
// plans, in the kernel parameters themselves (constant bank, no upload, no dependent
// global loads before the first payload load).
struct GlobalDesc {
    const RunDesc* runs;
    const ReqDesc* reqs;
    static constexpr bool kInline = false;
};
template <int R, int Q>
struct InlineDescT {
    RunDesc runs[R];
    ReqDesc reqs[Q];
    static constexpr bool kInline = true;
};
using InlineDesc = InlineDescT<kInlineRuns, kInlineReqs>;      // 6 KiB: one decode step's deltas
using InlineDescL = InlineDescT<kInlineRunsL, kInlineReqsL>;   // 24 KiB: batches of a few hundred requests
static_assert(sizeof(PlaneTable) + sizeof(InlineDescL) + 64 <= 32764, "kernel parameter space");
__device__ __forceinline__ uint4 load_run(const GlobalDesc& d, int64_t run) {
    return __ldg(reinterpret_cast<const uint4*>(d.runs + run));
}
__device__ __forceinline__ longlong2 load_req(const GlobalDesc& d, uint32_t r) {
    return __ldg(reinterpret_cast<const longlong2*>(d.reqs + r));
}
template <int R, int Q>
__device__ __forceinline__ uint4 load_run(const InlineDescT<R, Q>& d, int64_t run) {
    return *reinterpret_cast<const uint4*>(d.runs + run);
}
template <int R, int Q>
__device__ __forceinline__ longlong2 load_req(const InlineDescT<R, Q>& d, uint32_t r) {
    return *reinterpret_cast<const longlong2*>(d.reqs + r);
}

// Decode one item into (pool pointer, buffer pointer, bytes).
struct Item {
    char* pool;
    char* buf;
    uint32_t bytes;
};

template <class Desc>
__device__ __forceinline__ Item decode_item(const Desc& desc, int64_t run,
                                            const void* plane_base, int32_t plane, char* buf,
                                            uint32_t row_bytes) {
    const uint4 d = load_run(desc, run);
    // d.x = src_lo, d.y = dst_tok, d.z = req, d.w = count | src_hi << 16
    const uint32_t count = d.w & 0xFFFFu;
    const uint64_t off16 = (static_cast<uint64_t>(d.w >> 16) << 32) | d.x;
    const longlong2 q = load_req(desc, d.z);
    // q.x = row_base, q.y = n
    const int64_t row = q.x + static_cast<int64_t>(plane) * q.y + d.y;
    Item it;
    it.pool = const_cast<char*>(static_cast<const char*>(plane_base)) + (off16 << 4);
    it.buf = buf + row * static_cast<int64_t>(row_bytes);
    it.bytes = count * row_bytes;
    return it;
}

// ---------------------------------------------------------------------------------
// SIMT kernels: one warp per (run, plane, sub-chunk)
//
// A task is UNROLL * 32 lanes * VB bytes of one item (VB = bytes per access): every lane
// issues its UNROLL independent loads, then its UNROLL stores, and the warp retires -- no
// loop.  Items are cut into 2^sub_shift sub-chunks so that a 64 x 16-token decode delta
// (about 8,000 items of 32 KiB) becomes tens of thousands of equal tasks: the grid has no
// tail wave, and consecutive warps of a CTA stream consecutive sub-chunks of the same run.
//   kv_copy_warp32 : VB = 32, the default whenever every address is a multiple of 32: sm_100
//                    has 256-bit global loads / stores (LDG.E.256 / STG.E.256); 4 KiB per task,
//                    half the CTAs and half the memory instructions per byte of the 16-byte
//                    form: +1.7 % on cfg 1, +2 % on cfg 4.  An
//                    L2::evict_first priority on both sides was measured too: no gain.
//   kv_copy_warp   : VB = 16 (LDG/STG.E.128), rows / strides / buffers that are only 16-byte
//                    aligned.
// ---------------------------------------------------------------------------------
constexpr int kWarpsPerCta = 8;

template <int VB>
struct Vec;
template <>
struct Vec<16> {
    uint4 v;
    __device__ __forceinline__ void load(const void* p) { v = ld_stream16(p); }
    __device__ __forceinline__ void store(void* p) const { st_stream16(p, v); }
};
template <>
struct Vec<32> {
    uint32_t a[8];
    __device__ __forceinline__ void load(const void* p) {
        asm volatile("ld.global.L1::no_allocate.v8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                     : "=r"(a[0]), "=r"(a[1]), "=r"(a[2]), "=r"(a[3]), "=r"(a[4]), "=r"(a[5]),
                       "=r"(a[6]), "=r"(a[7])
                     : "l"(p)
                     : "memory");
    }
    __device__ __forceinline__ void store(void* p) const {
        asm volatile("st.global.L1::no_allocate.v8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"l"(p),
                     "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(a[4]), "r"(a[5]), "r"(a[6]),
                     "r"(a[7])
                     : "memory");
    }
};

template <int VB, int UNROLL, class Desc>
__device__ __forceinline__ void warp_task(const PlaneTable& planes, const Desc& desc, int64_t n_runs,
                                          char* buf, uint32_t row_bytes, int32_t plane0,
                                          int sub_shift, int pack, int32_t pf_dist) {
    constexpr uint32_t kTask = UNROLL * 32 * VB;          // bytes per warp
    pdl_launch_dependents();
    const int lane = threadIdx.x & 31;
    const int64_t task = static_cast<int64_t>(blockIdx.x) * kWarpsPerCta + (threadIdx.x >> 5);
    const int64_t run = task >> sub_shift;
    if (run >= n_runs) return;
    const uint32_t sub = static_cast<uint32_t>(task & ((int64_t{1} << sub_shift) - 1));
    // descriptors in global memory were written by an earlier copy in the stream; to stay
    // independent of how that copy was ordered, only parameter-resident ones are decoded
    // before the wait
    if (!Desc::kInline) pdl_wait();
    const Item it = decode_item(desc, run, planes.p[blockIdx.y], plane0 + blockIdx.y, buf,
                                row_bytes);
    // L2 prefetch (pf_dist >= 0): one lane asks L2 for the source of the task that the warp
    // pf_dist CTAs further on will copy (0: its own).  L2 is the device's point of coherence, so
    // a line fetched early still shows every store that reaches L2 before the later load; that
    // makes it legal in front of the wait, where the CTAs of the first wave -- resident while the
    // previous grid's last wave drains -- would otherwise sit with nothing in flight.
    const bool live = sub * kTask < it.bytes;              // else: this run is shorter than the longest
    const char* const src0 = (pack ? it.pool : it.buf) + static_cast<size_t>(sub) * kTask;
    auto prefetch_own = [&] {
        const uint32_t left = it.bytes - sub * kTask;
        if (live) l2_prefetch_bulk(src0, left < kTask ? left : kTask);
    };
    auto prefetch_ahead = [&] {
        const uint64_t lin = static_cast<uint64_t>(blockIdx.y) * gridDim.x + blockIdx.x + pf_dist;
        const uint32_t by = static_cast<uint32_t>(lin / gridDim.x);
        const uint32_t bx = static_cast<uint32_t>(lin - static_cast<uint64_t>(by) * gridDim.x);
        const int64_t task2 = static_cast<int64_t>(bx) * kWarpsPerCta + (threadIdx.x >> 5);
        const int64_t run2 = task2 >> sub_shift;
        if (by >= gridDim.y || run2 >= n_runs) return;
        const uint32_t sub2 = static_cast<uint32_t>(task2 & ((int64_t{1} << sub_shift) - 1));
        const Item it2 = decode_item(desc, run2, planes.p[by], plane0 + by, buf, row_bytes);
        if (sub2 * kTask >= it2.bytes) return;
        const uint32_t left = it2.bytes - sub2 * kTask;
        l2_prefetch_bulk((pack ? it2.pool : it2.buf) + static_cast<size_t>(sub2) * kTask,
                         left < kTask ? left : kTask);
    };
    // (one 32 KiB prefetch per CTA instead of 4 KiB per warp was measured as well: no difference)
    const bool leader = pf_dist >= 0 && lane == 0;
    if (Desc::kInline) {
        if (leader) {
            if (pf_dist == 0 || static_cast<uint64_t>(blockIdx.y) * gridDim.x + blockIdx.x <
                                    static_cast<uint32_t>(pf_dist))
                prefetch_own();
            if (pf_dist > 0) prefetch_ahead();
        }
        pdl_wait();
    } else if (leader) {
        // descriptors in global memory: decoding the task ahead would cost two more dependent
        // loads (and, placed behind this warp's own loads, the registers of a fifth CTA per SM:
        // measured, cfg 2 -3 %), so such plans only announce their own task
        prefetch_own();
    }
    if (!live) return;
    const uint32_t nvec = it.bytes / VB;
    const uint32_t i = sub * (UNROLL * 32) + lane;
    const char* src = src0 + static_cast<size_t>(lane) * VB;
    char* dst = (pack ? it.buf : it.pool) + static_cast<size_t>(i) * VB;
    Vec<VB> v[UNROLL];
#pragma unroll
    for (int u = 0; u < UNROLL; ++u)
        if (i + u * 32 < nvec) v[u].load(src + u * (32 * VB));
#pragma unroll
    for (int u = 0; u < UNROLL; ++u)
        if (i + u * 32 < nvec) v[u].store(dst + u * (32 * VB));
}

template <int UNROLL, class Desc>
__global__ void __launch_bounds__(kWarpsPerCta * 32)
kv_copy_warp(const __grid_constant__ PlaneTable planes, const __grid_constant__ Desc desc,
             int64_t n_runs, char* buf, uint32_t row_bytes, int32_t plane0, int sub_shift,
             int pack, int32_t pf_dist) {
    warp_task<16, UNROLL>(planes, desc, n_runs, buf, row_bytes, plane0, sub_shift, pack, pf_dist);
}

template <int UNROLL, class Desc>
__global__ void __launch_bounds__(kWarpsPerCta * 32)
kv_copy_warp32(const __grid_constant__ PlaneTable planes, const __grid_constant__ Desc desc,
               int64_t n_runs, char* buf, uint32_t row_bytes, int32_t plane0, int sub_shift,
               int pack, int32_t pf_dist) {
    warp_task<32, UNROLL>(planes, desc, n_runs, buf, row_bytes, plane0, sub_shift, pack, pf_dist);
}

// ---------------------------------------------------------------------------------
// TMA kernel: persistent single-warp CTAs, 1-D bulk copies through a shared ring
// ---------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(bar),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst_smem, const void* src, uint32_t bytes,
                                         uint32_t bar) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::
            "r"(dst_smem),
        "l"(src), "r"(bytes), "r"(bar)
        : "memory");
}
__device__ __forceinline__ void bulk_s2g(void* dst, uint32_t src_smem, uint32_t bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst),
                 "r"(src_smem), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void bulk_commit() {
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
}
template <int N>
__device__ __forceinline__ void bulk_wait_read() {
    asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory");
}
__device__ __forceinline__ void bulk_wait_all() {
    asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
}

struct StageMeta {
    char* dst;
    uint32_t bytes;
    uint32_t pad;
};

// STAGES ring slots of stage_bytes each; the store of item i is issued LAG
// iterations after its load so that LAG loads are in flight per CTA.
template <int STAGES, class Desc>
__global__ void __launch_bounds__(32)
kv_copy_bulk(const __grid_constant__ PlaneTable planes, const __grid_constant__ Desc desc,
             int64_t n_runs, int32_t n_planes, char* buf, uint32_t row_bytes,
             uint32_t stage_bytes, int32_t plane0, int pack) {
    constexpr int LAG = (STAGES + 1) / 2;
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ __align__(8) uint64_t full_bar[STAGES];
    __shared__ StageMeta meta[STAGES];

    const int lane = threadIdx.x;
    if (lane == 0) {
        for (int s = 0; s < STAGES; ++s) mbar_init(smem_u32(&full_bar[s]), 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncwarp();

    const int64_t total = n_runs * n_planes;     // item = plane * n_runs + run (plane-major)
    const int64_t G = gridDim.x;
    const uint32_t ring = smem_u32(smem);
    int64_t it = 0;                               // items issued by this CTA so far

    for (int64_t base = blockIdx.x; base < total; base += 32 * G) {
        // every lane decodes one of the next 32 items of this CTA
        const int64_t mine = base + static_cast<int64_t>(lane) * G;
        Item my{nullptr, nullptr, 0};
        if (mine < total) {
            const int32_t pl = static_cast<int32_t>(mine / n_runs);
            const int64_t run = mine - static_cast<int64_t>(pl) * n_runs;
            my = decode_item(desc, run, planes.p[pl], plane0 + pl, buf, row_bytes);
        }
        const char* my_src = pack ? my.pool : my.buf;
        char* my_dst = pack ? my.buf : my.pool;
        const int64_t left = (total - base + G - 1) / G;   // items of this CTA from base on
        const int nb = left < 32 ? static_cast<int>(left) : 32;
        for (int k = 0; k < nb; ++k, ++it) {
            const char* src = reinterpret_cast<const char*>(
                __shfl_sync(0xffffffffu, reinterpret_cast<unsigned long long>(my_src), k));
            char* dst = reinterpret_cast<char*>(
                __shfl_sync(0xffffffffu, reinterpret_cast<unsigned long long>(my_dst), k));
            const uint32_t bytes = __shfl_sync(0xffffffffu, my.bytes, k);
            if (lane == 0) {
                const int st = static_cast<int>(it % STAGES);
                // slot st was last read by the store of item it-STAGES: all but the
                // newest STAGES-1-LAG store groups must have finished reading smem
                bulk_wait_read<STAGES - 1 - LAG>();
                const uint32_t bar = smem_u32(&full_bar[st]);
                meta[st].dst = dst;
                meta[st].bytes = bytes;
                mbar_expect_tx(bar, bytes);
                bulk_g2s(ring + st * stage_bytes, src, bytes, bar);
                if (it >= LAG) {
                    const int64_t j = it - LAG;
                    const int sj = static_cast<int>(j % STAGES);
                    mbar_wait(smem_u32(&full_bar[sj]), static_cast<uint32_t>((j / STAGES) & 1));
                    bulk_s2g(meta[sj].dst, ring + sj * stage_bytes, meta[sj].bytes);
                    bulk_commit();
                }
            }
        }
    }
    if (lane == 0) {
        // drain: stores of the last min(it, LAG) items
        for (int64_t j = (it > LAG ? it - LAG : 0); j < it; ++j) {
            const int sj = static_cast<int>(j % STAGES);
            mbar_wait(smem_u32(&full_bar[sj]), static_cast<uint32_t>((j / STAGES) & 1));
            bulk_s2g(meta[sj].dst, ring + sj * stage_bytes, meta[sj].bytes);
            bulk_commit();
        }
        bulk_wait_all();
    }
}

struct BulkCfg {
    int stages;
    uint32_t stage_bytes;
    size_t smem;
    int ctas_per_sm;
    int host_ctas;
};

BulkCfg bulk_config(int64_t item_bytes_max) {
    // round the slot to 128 B; total ring per SM ~192 KiB, more CTAs for small items
    const uint32_t sb = static_cast<uint32_t>((item_bytes_max + 127) & ~int64_t{127});
    BulkCfg c{};
    c.stage_bytes = sb;
    // host_ctas: grid when the buffer is host memory, sized for about 1.5 MB of loads in flight
    // (LAG x slot x CTAs) -- ten times the bandwidth-delay product of the Gen5 x16 link, and
    // little enough that the queued host traffic does not get in the way of HBM traffic
    // (measured: a full grid slows a concurrent HBM copy 1.87x).
    if (sb > 16384)      { c.stages = 3;  c.ctas_per_sm = 2; c.host_ctas = 24; }
    else if (sb > 8192)  { c.stages = 4;  c.ctas_per_sm = 3; c.host_ctas = 48; }
    else if (sb > 4096)  { c.stages = 6;  c.ctas_per_sm = 4; c.host_ctas = 64; }
    else if (sb > 2048)  { c.stages = 8;  c.ctas_per_sm = 6; c.host_ctas = 96; }
    else                 { c.stages = 16; c.ctas_per_sm = 6; c.host_ctas = 96; }
    c.smem = static_cast<size_t>(c.stages) * sb;
    return c;
}

int g_warp_unroll = 4;   // LUMEN_KV_WARP_UNROLL=4|8 (tuning knob, read once; 4 measured best)

int g_host_ctas = 0;   // grid of the bulk kernel when the buffer is host memory (0: default)

template <class D>
void fill_inline(D& d, const CopyArgs& a) {
    std::memcpy(d.runs, a.runs, static_cast<size_t>(a.n_runs) * sizeof(RunDesc));
    std::memcpy(d.reqs, a.reqs, static_cast<size_t>(a.n_reqs) * sizeof(ReqDesc));
}

template <int STAGES, class Desc>
cudaError_t launch_bulk_desc(const PlaneTable& pt, const Desc& d, const CopyArgs& a, int32_t plane0,
                             int32_t np, const BulkCfg& c, int num_sms) {
    auto kern = kv_copy_bulk<STAGES, Desc>;   // dynamic shared memory limit set by preload_all()
    const int64_t total = a.n_runs * np;
    int64_t grid = static_cast<int64_t>(num_sms) * c.ctas_per_sm;
    // A host-memory buffer is bound by the host link (~55 GB/s): a few dozen single-warp
    // CTAs keep it full, and the SMs stay free for whatever else the device is running
    // (checkpointing must stay off the GPU critical path).
    if (a.buf_is_host) grid = g_host_ctas > 0 ? g_host_ctas : c.host_ctas;
    if (grid > total) grid = total;
    kern<<<static_cast<unsigned>(grid), 32, c.smem, a.stream>>>(
        pt, d, a.n_runs, np, static_cast<char*>(a.buf), static_cast<uint32_t>(a.row_bytes),
        c.stage_bytes, a.plane_base + plane0, a.pack ? 1 : 0);
    return cudaGetLastError();
}

template <int STAGES>
cudaError_t launch_bulk(const PlaneTable& pt, const CopyArgs& a, int32_t plane0, int32_t np,
                        const BulkCfg& c, int num_sms) {
    if (a.inline_desc && a.n_runs <= kInlineRuns && a.n_reqs <= kInlineReqs) {
        InlineDesc d;   // unused tail entries are never indexed (run < n_runs)
        fill_inline(d, a);
        return launch_bulk_desc<STAGES>(pt, d, a, plane0, np, c, num_sms);
    }
    if (a.inline_desc) {
        InlineDescL d;
        fill_inline(d, a);
        return launch_bulk_desc<STAGES>(pt, d, a, plane0, np, c, num_sms);
    }
    return launch_bulk_desc<STAGES>(pt, GlobalDesc{a.runs, a.reqs}, a, plane0, np, c, num_sms);
}

struct WarpLaunch {
    dim3 grid;
    cudaStream_t stream;
    int64_t n_runs;
    char* buf;
    uint32_t row_bytes;
    int32_t plane0;
    int sub_shift;
    int pack;
    int32_t pf_dist;   // L2 prefetch distance in CTAs (-1: off, 0: own task)
};

int g_pdl = 1;   // LUMEN_KV_PDL=0 launches without the programmatic attribute (A/B evidence)
int g_wide = 1;   // LUMEN_KV_WIDE=0 keeps the 16-byte kernel even where 32-byte accesses are legal
int g_prefetch = 16;   // LUMEN_KV_PREFETCH=d: L2 prefetch distance in CTAs (-1 off, 0 own task)
constexpr int kWideUnroll = 4;

template <class Desc>
cudaError_t launch_warp32(const PlaneTable& pt, const Desc& d, const WarpLaunch& w) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = w.grid;
    cfg.blockDim = dim3(kWarpsPerCta * 32, 1, 1);
    cfg.stream = w.stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = g_pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kv_copy_warp32<kWideUnroll, Desc>, pt, d, w.n_runs, w.buf,
                              w.row_bytes, w.plane0, w.sub_shift, w.pack, w.pf_dist);
}

template <int UNROLL, class Desc>
cudaError_t launch_warp(const PlaneTable& pt, const Desc& d, const WarpLaunch& w) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = w.grid;
    cfg.blockDim = dim3(kWarpsPerCta * 32, 1, 1);
    cfg.dynamicSmemBytes = 0;
    cfg.stream = w.stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = g_pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kv_copy_warp<UNROLL, Desc>, pt, d, w.n_runs, w.buf,
                              w.row_bytes, w.plane0, w.sub_shift, w.pack, w.pf_dist);
}

// CUDA loads a kernel lazily at its first launch, and that load can wait for kernels that are
// already running -- measured here: the first 1-token delta pack issued while a 70 GiB restore
// was in flight took 1.49 s instead of 0.44 ms.  Touch every variant once, up front.
template <class K>
cudaError_t preload(K kernel, bool big_smem) {
    cudaFuncAttributes fa;
    cudaError_t e = cudaFuncGetAttributes(&fa, kernel);
    if (e == cudaSuccess && big_smem)
        e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    return e;
}

template <int STAGES>
cudaError_t preload_bulk() {
    cudaError_t e = preload(kv_copy_bulk<STAGES, GlobalDesc>, true);
    if (e == cudaSuccess) e = preload(kv_copy_bulk<STAGES, InlineDesc>, true);
    return e != cudaSuccess ? e : preload(kv_copy_bulk<STAGES, InlineDescL>, true);
}

cudaError_t preload_all() {
    cudaError_t e = preload(kv_copy_warp<4, GlobalDesc>, false);
    if (e == cudaSuccess) e = preload(kv_copy_warp<4, InlineDesc>, false);
    if (e == cudaSuccess) e = preload(kv_copy_warp<4, InlineDescL>, false);
    if (e == cudaSuccess) e = preload(kv_copy_warp<8, GlobalDesc>, false);
    if (e == cudaSuccess) e = preload(kv_copy_warp<8, InlineDesc>, false);
    if (e == cudaSuccess) e = preload(kv_copy_warp<8, InlineDescL>, false);
    if (e == cudaSuccess) e = preload(kv_copy_warp32<4, GlobalDesc>, false);
    if (e == cudaSuccess) e = preload(kv_copy_warp32<4, InlineDesc>, false);
    if (e == cudaSuccess) e = preload(kv_copy_warp32<4, InlineDescL>, false);
    if (e == cudaSuccess) e = preload_bulk<3>();
    if (e == cudaSuccess) e = preload_bulk<4>();
    if (e == cudaSuccess) e = preload_bulk<6>();
    if (e == cudaSuccess) e = preload_bulk<8>();
    if (e == cudaSuccess) e = preload_bulk<16>();
    return e;
}

}  // namespace

int resolve_kernel(const CopyArgs& a) {
    int k = a.kernel;
    const int64_t item_max = static_cast<int64_t>(a.max_count) * a.row_bytes;
    if (k == kKernelAuto) k = a.buf_is_host ? g_host_kernel : kKernelWarp;
    if (k == kKernelBulk && item_max > kChunkBytes) k = kKernelWarp;  // one row > ring slot
    return k;
}

// Per-device state: the SM count, and the one-time load of every kernel variant together with
// its dynamic shared memory limit (cudaFuncSetAttribute is per device).  A process that drives
// several GPUs initialises each device at its first launch there.
struct DeviceState {
    std::once_flag once;
    cudaError_t err = cudaSuccess;
    int num_sms = 0;
};
constexpr int kMaxDevices = 64;
DeviceState g_dev[kMaxDevices];

void read_env_once() {
    static std::once_flag once;
    std::call_once(once, [] {
        if (const char* e = getenv("LUMEN_KV_WARP_UNROLL")) g_warp_unroll = (atoi(e) == 8) ? 8 : 4;
        if (const char* e = getenv("LUMEN_KV_PDL")) g_pdl = atoi(e) ? 1 : 0;
        if (const char* e = getenv("LUMEN_KV_WIDE")) g_wide = atoi(e) ? 1 : 0;
        if (const char* e = getenv("LUMEN_KV_PREFETCH")) g_prefetch = atoi(e);
        if (const char* e = getenv("LUMEN_KV_HOST_KERNEL"))
            g_host_kernel = (e[0] == 'w') ? kKernelWarp : kKernelBulk;
        if (const char* e = getenv("LUMEN_KV_HOST_CTAS")) g_host_ctas = atoi(e);
    });
}

int set_option(const char* name, int value) {
    if (!name) return -1;
    read_env_once();                 // so that a later first launch does not overwrite the setting
    if (!strcmp(name, "pdl")) g_pdl = value ? 1 : 0;
    else if (!strcmp(name, "wide")) g_wide = value ? 1 : 0;
    else if (!strcmp(name, "prefetch")) g_prefetch = value;
    else if (!strcmp(name, "warp_unroll")) g_warp_unroll = (value == 8) ? 8 : 4;
    else if (!strcmp(name, "host_kernel")) g_host_kernel = (value == kKernelWarp) ? kKernelWarp : kKernelBulk;
    else if (!strcmp(name, "host_ctas")) g_host_ctas = value > 0 ? value : 0;
    else return -1;
    return 0;
}

cudaError_t device_state(DeviceState** out) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    DeviceState& st = g_dev[dev];
    std::call_once(st.once, [&st, dev] {
        read_env_once();
        st.err = cudaDeviceGetAttribute(&st.num_sms, cudaDevAttrMultiProcessorCount, dev);
        if (st.err == cudaSuccess) st.err = preload_all();
    });
    *out = &st;
    return st.err;
}

cudaError_t init_current_device() {
    DeviceState* st = nullptr;
    return device_state(&st);
}

cudaError_t launch_kv_copy(const CopyArgs& a) {
    if (a.n_runs == 0 || a.n_planes == 0) return cudaSuccess;
    DeviceState* dev = nullptr;
    const cudaError_t init_err = device_state(&dev);   // thread-safe; a table lookup after the first call
    if (init_err != cudaSuccess) return init_err;
    const int kernel = resolve_kernel(a);
    const int64_t item_max = static_cast<int64_t>(a.max_count) * a.row_bytes;

    for (int32_t plane0 = 0; plane0 < a.n_planes; plane0 += kMaxPlanesPerLaunch) {
        const int32_t np = (a.n_planes - plane0 < kMaxPlanesPerLaunch) ? a.n_planes - plane0
                                                                        : kMaxPlanesPerLaunch;
        PlaneTable pt;
        for (int i = 0; i < np; ++i) pt.p[i] = a.planes[plane0 + i];
        for (int i = np; i < kMaxPlanesPerLaunch; ++i) pt.p[i] = nullptr;

        cudaError_t e = cudaSuccess;
        if (kernel == kKernelBulk) {
            const BulkCfg c = bulk_config(item_max);
            switch (c.stages) {
                case 3:  e = launch_bulk<3>(pt, a, plane0, np, c, dev->num_sms); break;
                case 4:  e = launch_bulk<4>(pt, a, plane0, np, c, dev->num_sms); break;
                case 6:  e = launch_bulk<6>(pt, a, plane0, np, c, dev->num_sms); break;
                case 8:  e = launch_bulk<8>(pt, a, plane0, np, c, dev->num_sms); break;
                default: e = launch_bulk<16>(pt, a, plane0, np, c, dev->num_sms); break;
            }
        } else {
            // sub-chunks per item: smallest power of two covering the longest run
            // 32-byte accesses need every address to be a multiple of 32
            bool wide = g_wide != 0 && a.pool_align32 &&
                        (reinterpret_cast<uintptr_t>(a.buf) & 31) == 0;
            for (int i = 0; wide && i < np; ++i)
                wide = (reinterpret_cast<uintptr_t>(pt.p[i]) & 31) == 0;
            const int64_t sub_bytes = wide ? int64_t{1024} * kWideUnroll
                                           : int64_t{512} * g_warp_unroll;
            int sub_shift = 0;
            while ((sub_bytes << sub_shift) < item_max) ++sub_shift;
            const int64_t tasks = a.n_runs << sub_shift;
            const int64_t gx = (tasks + kWarpsPerCta - 1) / kWarpsPerCta;
            if (gx > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
            WarpLaunch w;
            w.grid = dim3(static_cast<unsigned>(gx), static_cast<unsigned>(np), 1);
            w.stream = a.stream;
            w.n_runs = a.n_runs;
            w.buf = static_cast<char*>(a.buf);
            w.row_bytes = static_cast<uint32_t>(a.row_bytes);
            w.plane0 = a.plane_base + plane0;
            w.sub_shift = sub_shift;
            w.pack = a.pack ? 1 : 0;
            // only this device's own memory is cached coherently in its L2: a source in host
            // memory or in a peer GPU's memory is never asked for ahead of the wait
            const bool src_dev = a.pack || !(a.buf_is_host || a.buf_is_peer);
            // the 16-byte kernel (2 KiB tasks, twice the CTAs) loses with it: cfg 1 3,169 -> 3,101 GB/s
            w.pf_dist = (src_dev && wide) ? g_prefetch : -1;
            if (a.inline_desc && a.n_runs <= kInlineRuns && a.n_reqs <= kInlineReqs) {
                InlineDesc d;   // unused tail entries are never indexed (run < n_runs)
                fill_inline(d, a);
                e = wide ? launch_warp32(pt, d, w)
                         : (g_warp_unroll == 4) ? launch_warp<4>(pt, d, w) : launch_warp<8>(pt, d, w);
            } else if (a.inline_desc) {
                InlineDescL d;
                fill_inline(d, a);
                e = wide ? launch_warp32(pt, d, w)
                         : (g_warp_unroll == 4) ? launch_warp<4>(pt, d, w) : launch_warp<8>(pt, d, w);
            } else {
                const GlobalDesc d{a.runs, a.reqs};
                e = wide ? launch_warp32(pt, d, w)
                         : (g_warp_unroll == 4) ? launch_warp<4>(pt, d, w) : launch_warp<8>(pt, d, w);
            }
        }
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

}  // namespace lumen
