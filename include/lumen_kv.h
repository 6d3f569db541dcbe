/*
 * lumen_kv.h -- C ABI of the B200-native KV checkpoint pack / restore unpack.
 *
 * The operation is the data-parallel hot path of LUMEN's load-aware KV
 * checkpointing and recovery:
 *   - pack   = step (3) of the incremental checkpoint pipeline: "workers track
 *     checkpoint progress and transmit only newly generated KV pages after each
 *     prefill or decode batch. A background thread copies these pages from GPU
 *     memory to the local pinned buffer" (section 4.2);
 *   - unpack = KV-reuse recovery: the checkpoint holder locates "the longest
 *     contiguous checkpointed prefix ... subsequently loading the matching KV
 *     pages into GPU memory" (section 4.3).
 *   A "KV page" is "a fixed-size block of cached keys and values for contiguous
 *   token positions" (section 2.1).
 *
 * Data model (BASELINE.json north_star)
 *   Pool: 2L "planes" -- for every layer l one K plane and one V plane, each a
 *   dense device array [num_pages][page_size][kv_heads][head_dim] of opaque
 *   elem_bytes-wide words (bf16 in the paper's models; never interpreted).
 *   row = kv_heads*head_dim*elem_bytes is one token in one plane; it must be a
 *   multiple of 16 bytes and every plane / buffer base must be 16-byte aligned.
 *   A request owns a page table (logical page i -> physical page) shared by all
 *   2L planes, and a token range [t_begin, t_end).
 *   Checkpoint buffer: dense, no padding, laid out
 *       [request][layer][K|V][token][head][dim]
 *   requests in plan order; request r starts at lumen_kv_plan_req_offset(r).
 *   With n_r = t_end - t_begin, plane = 2*layer + (0 for K, 1 for V):
 *       B[off_r + (plane*n_r + j)*row + b]  <->
 *       planes[plane][(PT_r[(t_begin+j)/S]*S + (t_begin+j)%S)*row + b]
 *   pack copies right to left, unpack left to right; unpack leaves every other
 *   pool byte untouched.
 *
 * Conventions
 *   - All functions return LUMEN_KV_OK (0) or a negative lumen_kv_status.
 *   - All validation happens in lumen_kv_plan_build on the host, before any
 *     launch; pack/unpack never read or write out of bounds for a plan that built.
 *   - pack/unpack are asynchronous on the caller's cudaStream_t (passed as
 *     void*): they enqueue one kernel launch per 256 planes and return.  They never
 *     synchronise the device or a stream and never allocate device or pinned memory;
 *     the only CUDA calls besides the launch are cudaGetDevice, for a host buffer one
 *     cudaHostGetDevicePointer (a table lookup), and for a plan with uploaded
 *     descriptors one cudaEventRecord (and, until the upload has been seen complete, one
 *     cudaEventQuery / cudaStreamWaitEvent).  After a thread's first call they do not touch
 *     the heap either.  Results are complete (and, for host destinations,
 *     host-visible) once an event recorded on that stream after the call has fired
 *     (nothing is promised earlier).
 *   - Consecutive launches overlap at their edges (programmatic dependent launch): a
 *     kernel's CTAs become resident while the previous kernel's last wave drains and,
 *     before they wait for it to complete, ask L2 for the source bytes they will copy
 *     (cp.async.bulk.prefetch.L2 -- a hint; the loads themselves come after the wait).
 *     L2 is the point of coherence of a device's OWN memory only, which is why a buffer
 *     in another GPU's memory must be declared LUMEN_KV_MEM_DEVICE_PEER (and pools are
 *     always local): such a source, like a pinned host one, is never asked for early.
 *   - One-time cost: the first launch on a device loads every kernel variant and sets
 *     its shared-memory limit (about twenty cudaFuncGetAttributes / cudaFuncSetAttribute
 *     calls; a lazily loaded kernel can otherwise wait for kernels that are already
 *     running).  Call lumen_kv_init() at start-up to take that outside the first pack.
 *   - Devices: plans, stagers, checkpointers and the library's cached descriptor memory
 *     belong to the device that was current when they were created; every call must be
 *     made with that device current (a stream of another device makes the call fail with
 *     LUMEN_KV_ECUDA).  A process may drive several devices; each is initialised at its
 *     first launch.
 *   - pack/unpack may be captured into a CUDA graph (stream capture); the plan must then
 *     stay alive for as long as the graph can be replayed (its descriptor memory is kept
 *     until lumen_kv_trim()).
 *   - A plan is immutable and direction-agnostic: the same plan drives pack and
 *     unpack.  The caller owns pools, buffers, streams and page tables (page
 *     tables are copied at build time).  Plans may be used concurrently from
 *     different streams and from several host threads (the little state a plan keeps
 *     about its descriptor upload and its last use per stream is locked; a plan handed
 *     to an _async staged call is used by the stager's thread until its ticket is issued).
 *   - There is no CPU fallback: without a CUDA device pack and unpack fail with
 *     LUMEN_KV_ECUDA, and so does every plan_build that has descriptors to upload.
 */
#ifndef LUMEN_KV_H
#define LUMEN_KV_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* 2: lumen_kv_sink_fn returns an int (0 = delta taken; version 1 sinks returned void),
 *    LUMEN_KV_MEM_DEVICE means memory of the CURRENT device, LUMEN_KV_MEM_DEVICE_PEER,
 *    lumen_kv_copy_noalloc, LUMEN_KV_ECAPACITY.  Compare lumen_kv_version() with the header's. */
#define LUMEN_KV_VERSION 2

#if defined(__GNUC__)
#define LUMEN_KV_API __attribute__((visibility("default")))
#else
#define LUMEN_KV_API
#endif

typedef enum {
    LUMEN_KV_OK       =  0,
    LUMEN_KV_EINVAL   = -1,  /* null pointer, bad geometry, misaligned base, bad kind/flag   */
    LUMEN_KV_ERANGE   = -2,  /* page index outside [0, num_pages) or range outside the table */
    LUMEN_KV_EOVERLAP = -3,  /* VALIDATE_UNIQUE_DST: a pool token slot is addressed twice     */
    LUMEN_KV_ESIZE    = -4,  /* buffer smaller than lumen_kv_plan_bytes()                    */
    LUMEN_KV_ENOMEM   = -5,  /* host or device allocation of the descriptors failed          */
    LUMEN_KV_ECUDA    = -6,  /* CUDA runtime error; see lumen_kv_last_cuda_error()           */
    LUMEN_KV_ESINK    = -7,  /* background checkpointer: the sink rejected a delta           */
    LUMEN_KV_ECAPACITY = -8  /* lumen_kv_copy_noalloc: the plan has more runs or requests than
                                the library's built-in descriptor array holds                */
} lumen_kv_status;

/* Geometry of the caller's paged pool (host struct, read during plan_build only). */
typedef struct {
    int32_t num_layers;        /* L >= 1                                              */
    int32_t kv_heads;          /* H >= 1                                              */
    int32_t head_dim;          /* D >= 1                                              */
    int32_t page_size;         /* S >= 1 tokens per page                              */
    int32_t elem_bytes;        /* bytes per element; H*D*elem_bytes must be % 16 == 0 */
    int32_t reserved;          /* must be 0                                           */
    int64_t num_pages;         /* N, 1 <= N < 2^31                                    */
    int64_t page_stride_bytes; /* 0 => dense: S*H*D*elem_bytes; else >= that, % 16    */
} lumen_kv_geom;

/* One request's contribution to a plan (host struct; page_table is a HOST pointer
 * and is copied).  Entries outside [t_begin/S, (t_end-1)/S] are ignored (A6).     */
typedef struct {
    const int32_t* page_table;
    int64_t        page_table_len;
    int64_t        t_begin, t_end;   /* 0 <= t_begin <= t_end <= page_table_len*S  */
} lumen_kv_req;

typedef struct lumen_kv_plan lumen_kv_plan;  /* opaque; library owns its descriptors */

/* plan_build flags */
#define LUMEN_KV_VALIDATE_UNIQUE_DST 0x1u /* reject plans that address a pool token slot twice  */
#define LUMEN_KV_MERGE_ADJACENT      0x2u /* merge runs whose physical pages are adjacent     */
#define LUMEN_KV_HOST_ONLY           0x4u /* build descriptors on the host only (no CUDA call);
                                             such a plan can be inspected, and executed by
                                             lumen_kv_copy_noalloc only                       */
#define LUMEN_KV_NO_INLINE           0x8u /* always upload the descriptors to device memory.
                                             By default a plan of <= 1,024 runs and <= 512
                                             requests (a decode step's deltas, also of a large
                                             batch) is carried in the kernel parameters -- 6 KiB
                                             up to 256 runs / 128 requests, 24 KiB above: no
                                             upload, no device memory, and plan_build makes no
                                             CUDA call for it                                  */
/* kernel selection (default 0 = library heuristic); for benchmarking / evidence   */
#define LUMEN_KV_KERNEL_SHIFT        8
#define LUMEN_KV_KERNEL_MASK         0xF00u
#define LUMEN_KV_KERNEL_AUTO         0x000u
#define LUMEN_KV_KERNEL_WARP         0x100u /* SIMT: warp per (run, plane, sub-chunk), 32 B ld/st */
#define LUMEN_KV_KERNEL_BULK         0x200u /* TMA 1-D bulk copies through a shared-memory ring */

/* where the checkpoint buffer lives */
#define LUMEN_KV_MEM_DEVICE      0  /* device pointer into the CURRENT device's memory (HBM).
                                       A pointer that cudaPointerGetAttributes places on
                                       another device is handled as LUMEN_KV_MEM_DEVICE_PEER
                                       (looked up when a thread first sees the buffer)         */
#define LUMEN_KV_MEM_DEVICE_PEER 2  /* device pointer into ANOTHER GPU's memory (peer access
                                       enabled by the caller): same kernels; the restore does
                                       not ask L2 for its source ahead of the stream-order
                                       wait, because only a device's own memory is cached
                                       coherently in its L2.  Tested on one GPU only (a local
                                       buffer declared as peer): never run against real peer
                                       memory                                                  */
#define LUMEN_KV_MEM_HOST_MAPPED 1  /* pinned host memory (cudaHostAlloc / cudaHostRegister);
                                       pass the HOST pointer, the kernel writes/reads it
                                       directly over the host link (zero-copy).  One launch,
                                       no staging memory; AUTO uses a few dozen single-warp
                                       TMA CTAs so that the SMs stay free.  Every SM-issued
                                       access crosses PCIe as a 128-byte TLP (one L2 line),
                                       the copy engine uses 256-byte TLPs: this path tops out
                                       at 92 % of what cudaMemcpyAsync reaches (measured 52.8
                                       of 57.3 GB/s D2H, 51.5 of 55.6 H2D; counters in
                                       profiles/README.md) whatever kernel, grid or
                                       operation size is used.  The staged calls below move
                                       the same bytes with the copy engine (99 %).            */

/*
 * lumen_kv_plan_build -- step a2: flatten the requests'
 * ranges into token-run descriptors and upload them.
 *   geom, reqs : host pointers, read only during the call.  num_reqs >= 0.
 *   stream     : unused (kept in the signature; pass the stream the plan will run on or
 *                NULL).  Plans that need an upload (more than 1,024 runs or 512 requests,
 *                or LUMEN_KV_NO_INLINE) copy their descriptors on a stream of the
 *                library's own, so that no copy sits between two kernels of the caller's
 *                stream; pack / unpack order themselves behind that copy on whatever
 *                stream they are given (one cudaStreamWaitEvent, none once the copy has
 *                been seen complete; under stream capture the call waits for it on the
 *                host instead).
 *   out        : receives the plan; release with lumen_kv_plan_free.
 * Zero-length ranges and num_reqs == 0 are legal (A4) and yield 0 bytes.
 * Errors: EINVAL, ERANGE, EOVERLAP (with VALIDATE_UNIQUE_DST), ENOMEM, ECUDA.
 */
LUMEN_KV_API int lumen_kv_plan_build(const lumen_kv_geom* geom, const lumen_kv_req* reqs,
                        int32_t num_reqs, uint32_t flags, void* stream,
                        lumen_kv_plan** out);

/*
 * Explicit buffer layout.  A checkpoint store keeps a request's checkpoint as the deltas it
 * received (one checkpoint per request) and a recovery restores
 * the longest checkpointed prefix, which may end inside the last delta.  With
 * a layout, request r's block sits at byte offset buf_offset of the buffer and consecutive
 * planes are plane_stride_tokens rows apart:
 *     B[buf_offset_r + ((plane*plane_stride_tokens_r) + j)*row + b]
 * buf_offset must be a multiple of row, plane_stride_tokens >= n_r.  layouts == NULL is the
 * dense layout of lumen_kv_plan_build.  lumen_kv_plan_bytes() is then the extent (largest
 * byte addressed + 1) and lumen_kv_plan_req_offset(r) returns buf_offset_r (r == num_reqs:
 * the extent).  Blocks of different requests may not overlap for pack; the library does
 * not check that.  Errors as lumen_kv_plan_build.
 */
typedef struct {
    int64_t buf_offset;           /* bytes, multiple of row                       */
    int64_t plane_stride_tokens;  /* >= t_end - t_begin                           */
} lumen_kv_req_layout;
LUMEN_KV_API int lumen_kv_plan_build_layout(const lumen_kv_geom* geom, const lumen_kv_req* reqs,
                        const lumen_kv_req_layout* layouts, int32_t num_reqs, uint32_t flags,
                        void* stream, lumen_kv_plan** out);

/* total checkpoint-buffer bytes = sum_r n_r * 2L * row */
LUMEN_KV_API int64_t lumen_kv_plan_bytes(const lumen_kv_plan* plan);
/* byte offset of request r in the buffer (exclusive prefix sum); r == num_reqs gives the total */
LUMEN_KV_API int64_t lumen_kv_plan_req_offset(const lumen_kv_plan* plan, int32_t r);
/* number of token-run descriptors in the plan */
LUMEN_KV_API int64_t lumen_kv_plan_num_runs(const lumen_kv_plan* plan);

/* One run, for inspection (tests of the plan logic; not needed to use the library). */
typedef struct {
    int64_t src_slot;   /* page*S + first slot, in tokens                    */
    int64_t dst_token;  /* request-relative first token j                    */
    int32_t req;        /* request index                                     */
    int32_t count;      /* tokens in the run                                 */
} lumen_kv_run_info;
LUMEN_KV_API int lumen_kv_plan_get_run(const lumen_kv_plan* plan, int64_t i, lumen_kv_run_info* out);

/*
 * lumen_kv_checkpoint_pack -- steps a3/a4: gather the plan's token ranges from the
 * planes into the contiguous checkpoint buffer dst.
 *   k_planes, v_planes : HOST arrays of num_layers DEVICE pointers (one per layer);
 *                        read during the call, not retained.
 *   dst, dst_bytes     : buffer and its capacity; dst_kind says where it lives.
 * Errors: EINVAL (null / misaligned / host-only plan), ESIZE, ECUDA.
 */
LUMEN_KV_API int lumen_kv_checkpoint_pack(const lumen_kv_plan* plan,
                             const void* const* k_planes, const void* const* v_planes,
                             void* dst, int64_t dst_bytes, int dst_kind, void* stream);

/*
 * lumen_kv_restore_unpack -- step a7: scatter the checkpoint buffer src into the
 * planes under the plan's page tables.  Destinations must be disjoint (use
 * LUMEN_KV_VALIDATE_UNIQUE_DST at build time; otherwise undefined for overlaps).
 */
LUMEN_KV_API int lumen_kv_restore_unpack(const lumen_kv_plan* plan,
                            void* const* k_planes, void* const* v_planes,
                            const void* src, int64_t src_bytes, int src_kind, void* stream);

/*
 * lumen_kv_copy_noalloc -- pack (a3/a4) or restore (a7) for
 * callers that must not allocate GPU memory.
 *
 * Who needs it.  A serving worker usually hands all free HBM to its KV pool at start-up, and
 * that pool is fullest exactly when a restore is most urgent (a recovery burst):
 * a cudaMalloc for a plan's descriptors may then fail, and cudaMalloc / cudaFree synchronise the
 * whole device even when they succeed, which a decode loop cannot absorb.  Other callers run
 * under a rule that all device memory comes from a pool of their own.  The regular calls need no
 * device memory up to 1,024 runs / 512 requests; above that lumen_kv_plan_build allocates (and
 * caches) device and pinned memory for the descriptors.  This call never does: it keeps the
 * descriptors in an array that is part of the library's own image.
 *
 * Use.  Build the plan with LUMEN_KV_HOST_ONLY (host heap only, no CUDA call), then
 *     lumen_kv_copy_noalloc(plan, LUMEN_KV_DIR_PACK or LUMEN_KV_DIR_RESTORE, k_planes, v_planes,
 *                           buf, buf_bytes, buf_kind, stream);
 * Arguments, buffer layout, alignment rules, buffer kinds and stream semantics are those of
 * lumen_kv_checkpoint_pack / lumen_kv_restore_unpack, and so are the bytes that arrive.  Any plan
 * is accepted (not only host-only ones); the plan may be freed as soon as the call returns.
 *
 * Limit.  At most LUMEN_KV_NOALLOC_MAX_RUNS runs and LUMEN_KV_NOALLOC_MAX_REQS requests per call
 * (lumen_kv_plan_num_runs tells; a page-granular 32 GiB prefix restore of 16 requests is 8,192
 * runs).  A larger plan is refused with LUMEN_KV_ECAPACITY before anything is enqueued: split
 * the requests over several plans, or use the regular calls.  The array costs 1,088 KiB of
 * device memory on every GPU that loads the library, held until the process exits.
 *
 * What it does.  It enqueues on `stream` one small kernel per 1,024 descriptors that writes them
 * (they travel in its parameters) into the built-in array, then the copy kernel, one launch per
 * 256 planes.  No cudaMalloc, cudaFree, cudaHostAlloc or other allocating call is made, on any
 * call; nothing is synchronised.  The copy kernel is a plain form of the regular SIMT kernel
 * (no overlap with the neighbouring launches, no L2 prefetch), so expect a few per cent less
 * than the regular call.
 *
 * First call on a device.  It looks up the array's device address (cudaGetSymbolAddress) and
 * loads three kernels; the CUDA runtime may load the library's module at that point.  Make
 * that first call -- an empty plan will not do, it returns before the set-up; any 1-token plan
 * does -- during start-up, with the device current, and before any stream capture is begun.
 *
 * Sharing.  Every call on a device uses the same array, and the array keeps what the last call
 * wrote.  Nothing in it has to start at zero: a call overwrites the entries it will read and
 * reads no others.  But two calls whose GPU work overlaps race on it -- the second call's
 * descriptor writes can land while the first call's copy kernel still reads them, and the first
 * call then moves the wrong bytes, silently.  Issue all calls for a device on ONE stream, or
 * order them with events so that a call's work has completed before the next call's begins.
 * (Calls from several host threads are serialised while they enqueue, so two threads that
 * share a stream are safe; the regular calls never touch the array.)
 *
 * Errors: EINVAL (null, bad direction / kind, misaligned, unpinned host buffer), ECAPACITY,
 * ESIZE (buf_bytes < lumen_kv_plan_bytes), ECUDA.
 */
#define LUMEN_KV_NOALLOC_MAX_RUNS 65536
#define LUMEN_KV_NOALLOC_MAX_REQS 4096
#define LUMEN_KV_DIR_PACK    0   /* planes -> buf */
#define LUMEN_KV_DIR_RESTORE 1   /* buf -> planes */
LUMEN_KV_API int lumen_kv_copy_noalloc(const lumen_kv_plan* plan, int direction,
                             void* const* k_planes, void* const* v_planes,
                             void* buf, int64_t buf_bytes, int buf_kind, void* stream);

/*
 * Two-stage host path (steps a4 / a7 through the copy engines).
 *
 * PAPER.md:145 step 3 copies the new KV "from GPU memory to the local pinned buffer" in
 * the background and PAPER.md:122 requires that this stays off the GPU critical path.
 * lumen_kv_checkpoint_pack with LUMEN_KV_MEM_HOST_MAPPED does it with SM stores over the
 * host link.  The staged form cuts the plan into chunks that are contiguous in the
 * checkpoint buffer, packs chunk c into slot c % n_slots of a caller-provided DEVICE
 * staging ring with the HBM-speed kernel (microseconds of SM time), and moves the slot to
 * dst + chunk offset with cudaMemcpyAsync on the stager's own copy stream while the next
 * chunk is being packed; restore runs the mirror image (H2D copy, then unpack).  The
 * bytes that arrive are identical to the one-shot call's.
 *
 * A stager owns two non-blocking streams (copies; kernels of asynchronous calls), 2*n_slots+1
 * events and, once an _async call has been made, one thread; it holds no payload memory.  staging: device pointer, 16-byte aligned, n_slots*slot_bytes bytes, owned by
 * the caller and not touched by anything else while a staged call is in flight.
 * slot_bytes must be a multiple of 16 and at least as large as the longest run of every
 * plan used with it (32 KiB unless a single row is larger), else ESIZE.  2 <= n_slots <= 16.
 * One stager serves one staged call at a time (calls on it are serialised by its events);
 * use one stager per direction to run pack and restore concurrently.
 *
 * After an error.  A staged call that fails with ECUDA half-way (a launch or copy was refused)
 * first waits for everything it did enqueue -- on `stream` and on the stager's copy stream --
 * and then returns: the staging ring is consistent again and the stager can be used for the next
 * call (a restore with ready flags still needs the flags of the chunks that were issued).  The
 * host buffer (pack) or the plan's pool slots (restore) then hold a mixture of old and new
 * bytes; nothing outside them is touched.  An asynchronous call reports the failure, with its
 * cudaError_t, through lumen_kv_stager_query / _wait / _sync of its ticket; later tickets are
 * still issued.
 *
 * Stream semantics are those of the one-shot calls: the work is ordered after everything
 * enqueued on `stream` before the call, and work enqueued on `stream` after the call sees
 * the complete result (host buffer for pack, pool for restore).  host buffers: pinned
 * host memory (cudaHostAlloc / cudaHostRegister); pass the HOST pointer.
 * Errors: EINVAL, ESIZE, ECUDA.
 */
typedef struct lumen_kv_stager lumen_kv_stager;
LUMEN_KV_API int lumen_kv_stager_create(void* staging, int64_t slot_bytes, int32_t n_slots,
                                        lumen_kv_stager** out);
LUMEN_KV_API void lumen_kv_stager_destroy(lumen_kv_stager* stager);   /* issues what is queued, synchronises its streams */
LUMEN_KV_API int lumen_kv_checkpoint_pack_staged(const lumen_kv_plan* plan,
                             const void* const* k_planes, const void* const* v_planes,
                             void* dst_host, int64_t dst_bytes, lumen_kv_stager* stager,
                             void* stream);
LUMEN_KV_API int lumen_kv_restore_unpack_staged(const lumen_kv_plan* plan,
                             void* const* k_planes, void* const* v_planes,
                             const void* src_host, int64_t src_bytes, lumen_kv_stager* stager,
                             void* stream);
/*
 * Per-chunk commit / ready flags (checkpointed pages "become visible ... only
 * upon complete reception"; the sender of step (4), consumes the pinned buffer
 * while later pages are still being copied).
 *   flags : pinned host array of at least lumen_kv_plan_num_chunks(plan, slot_bytes) 64-bit
 *           words, 8-byte aligned, owned by the caller; NULL = the plain staged call.
 *   pack  : flags[c] = epoch is written in stream order AFTER chunk c's bytes
 *           [byte_begin, byte_end) are complete in dst_host (a release: a host thread that
 *           reads flags[c] == epoch with acquire semantics may read the chunk).
 *   restore: the H2D copy of chunk c waits until flags[c] >= epoch (written by a host
 *           thread after it has filled the chunk, e.g. on reception); chunks are consumed
 *           in order, so a flag that is never raised stalls the call's streams for ever.
 * Chunk c is entry c of lumen_kv_plan_get_chunks.  ECUDA if the driver lacks 64-bit stream
 * memory operations.
 */
LUMEN_KV_API int lumen_kv_checkpoint_pack_staged_commit(const lumen_kv_plan* plan,
                             const void* const* k_planes, const void* const* v_planes,
                             void* dst_host, int64_t dst_bytes, lumen_kv_stager* stager,
                             void* stream, uint64_t* flags, uint64_t epoch);
LUMEN_KV_API int lumen_kv_restore_unpack_staged_ready(const lumen_kv_plan* plan,
                             void* const* k_planes, void* const* v_planes,
                             const void* src_host, int64_t src_bytes, lumen_kv_stager* stager,
                             void* stream, const uint64_t* flags, uint64_t epoch);

/*
 * Asynchronous submission of a staged call.
 *
 * The calls above issue six stream operations per chunk from the calling thread: a decode
 * step's delta (1-6 chunks) costs 10-40 us of host time, but a 32 GiB prefix is 1,024 chunks
 * and a 70 GiB recovery wave 2,300 -- more operations than a CUDA stream queues, so the calling
 * thread is held for most of the transfer.  The _async forms return at once: they validate,
 * record one event on `stream`, and hand the call to a thread owned by the stager, which issues
 * the same per-chunk pipeline on the stager's own streams.
 *   ordering : the transfer starts after everything enqueued on `stream` before the call and
 *              after every earlier call on the same stager.  Nothing enqueued on `stream`
 *              AFTER the call is ordered behind it (CUDA cannot wait for an event that has not
 *              been recorded yet); use lumen_kv_stager_wait for that.
 *   flags, epoch : as in the _commit / _ready forms; NULL = none.
 *   *ticket  : identifies the call (tickets of one stager increase and complete in order).
 *   The plan may be freed and the plane-pointer arrays reused as soon as the call returns; the
 *   host buffer, the pool, the staging ring and (for restore) the flag array must stay valid
 *   until the ticket is complete.  Errors that validation can find (EINVAL, ESIZE) are returned
 *   by the call; errors met while issuing are returned by query / wait / sync.
 * lumen_kv_stager_query : 1 = complete (results visible as after a stream event), 0 = not yet,
 *                         negative = the call failed with that status.  Never blocks.
 * lumen_kv_stager_wait  : makes `stream` wait for the ticket's completion.  Blocks the calling
 *                         thread only until the stager's thread has finished ISSUING the ticket.
 * lumen_kv_stager_sync  : blocks the calling thread until the ticket is complete.
 * Synchronous and asynchronous calls may be mixed on one stager; they are issued one at a time.
 */
LUMEN_KV_API int lumen_kv_checkpoint_pack_staged_async(const lumen_kv_plan* plan,
                             const void* const* k_planes, const void* const* v_planes,
                             void* dst_host, int64_t dst_bytes, lumen_kv_stager* stager,
                             void* stream, uint64_t* flags, uint64_t epoch, uint64_t* ticket);
LUMEN_KV_API int lumen_kv_restore_unpack_staged_async(const lumen_kv_plan* plan,
                             void* const* k_planes, void* const* v_planes,
                             const void* src_host, int64_t src_bytes, lumen_kv_stager* stager,
                             void* stream, const uint64_t* flags, uint64_t epoch,
                             uint64_t* ticket);
LUMEN_KV_API int lumen_kv_stager_query(lumen_kv_stager* stager, uint64_t ticket);
LUMEN_KV_API int lumen_kv_stager_wait(lumen_kv_stager* stager, uint64_t ticket, void* stream);
LUMEN_KV_API int lumen_kv_stager_sync(lumen_kv_stager* stager, uint64_t ticket);

/* number of chunks a staged call on this plan would be cut into for the given slot size
 * (host arithmetic only; ESIZE if a run does not fit a slot) */
LUMEN_KV_API int64_t lumen_kv_plan_num_chunks(const lumen_kv_plan* plan, int64_t slot_bytes);
/* The chunks themselves, for inspection: chunk i = runs [run_begin, run_end) replicated over
 * planes [plane_begin, plane_end) = buffer bytes [byte_begin, byte_end).  Writes at most cap
 * entries to out (may be NULL when cap == 0); returns the number of chunks or a status. */
typedef struct {
    int64_t run_begin, run_end;
    int32_t plane_begin, plane_end;
    int64_t byte_begin, byte_end;
} lumen_kv_chunk_info;
LUMEN_KV_API int64_t lumen_kv_plan_get_chunks(const lumen_kv_plan* plan, int64_t slot_bytes,
                                              lumen_kv_chunk_info* out, int64_t cap);

/*
 * Page tags (section 4.2): "each transferred page carries a page tag: a hash
 * value of the token IDs stored in page i, paired with the page's end position in the request
 * token sequence (i.e., the cumulative token length after page i)", regenerated from the
 * token history at recovery to find "the longest contiguous checkpointed prefix"
 * (PAPER.md:157).  The paper does not name the hash; this library uses 64-bit FNV-1a over
 * the little-endian bytes of the page's int32 token IDs, of that page only (DESIGN.md
 * reading A12).  A last page that is not full is hashed over the tokens it holds.
 */
typedef struct {
    uint64_t hash;     /* FNV-1a 64 of the token IDs stored in the page        */
    int64_t  end_pos;  /* cumulative token length after the page               */
} lumen_kv_tag;

/* pages of all requests = sum_r ceil((tok_offset[r+1] - tok_offset[r]) / page_size); host arithmetic.
 * EINVAL for null / decreasing offsets / page_size < 1. */
LUMEN_KV_API int64_t lumen_kv_tags_num_pages(const int64_t* tok_offset, int32_t num_reqs,
                                             int32_t page_size);
/*
 * lumen_kv_page_tags -- tags of every page of num_reqs requests, on the device.
 *   token_ids  : DEVICE array; request r's token IDs are [tok_offset[r], tok_offset[r+1]).
 *   tok_offset : HOST array of num_reqs + 1 non-decreasing offsets (read during the call).
 *   tags_out   : DEVICE array, 16-byte aligned, of tags_cap >= lumen_kv_tags_num_pages(..)
 *                entries; request r's tags follow request r-1's, in page order.
 * Asynchronous on `stream`.  Errors: EINVAL, ESIZE (tags_cap too small), ECUDA.
 */
LUMEN_KV_API int lumen_kv_page_tags(const int32_t* token_ids, const int64_t* tok_offset,
                                    int32_t num_reqs, int32_t page_size, lumen_kv_tag* tags_out,
                                    int64_t tags_cap, void* stream);
/*
 * lumen_kv_page_tags_host -- the same tags on the host, for the sender of a delta: the tags of
 * the pages touched by [t_begin, t_end) as of a history of t_end tokens (so the last page's end
 * position is min(page end, t_end)).  token_ids points at token `first_token`, which must be
 * a multiple of page_size and <= t_begin rounded down to a page.  Writes at most cap tags;
 * returns their number ((t_end-1)/S - t_begin/S + 1, or 0 for an empty range) or EINVAL.
 */
LUMEN_KV_API int64_t lumen_kv_page_tags_host(const int32_t* token_ids, int64_t first_token,
                                             int64_t t_begin, int64_t t_end, int32_t page_size,
                                             lumen_kv_tag* out, int64_t cap);
/*
 * lumen_kv_longest_prefix -- host lookup: walk the regenerated tags of one request in page
 * order and halt at the first that is not among `stored` (any order, duplicates allowed);
 * returns the end position of the last tag found = tokens of the longest contiguous
 * checkpointed prefix (0 if none), or EINVAL / ENOMEM.  Both arrays are HOST memory.
 */
LUMEN_KV_API int64_t lumen_kv_longest_prefix(const lumen_kv_tag* regen, int64_t n_regen,
                                             const lumen_kv_tag* stored, int64_t n_stored);

/*
 * Checkpoint store: the host-memory region of a worker that
 * persists "incoming remote KV pages".  One checkpoint per request; a request's footprint
 * is RESERVED at assignment from its maximum context length ("a conservative allocation
 * derived from the maximum context length rather than the current dynamic KV size") and
 * released at completion, so a holder can never run out of host memory; the per-worker
 * limit is the arena size (80 / 160 GB in the paper's deployments).  Deltas are appended as
 * they arrive, each with the page tags it carries, and become visible to lookups only when
 * the append has completed ("pages become visible in the checkpoint store only upon complete
 * reception").  Pure host code; thread-safe; the library allocates no payload memory:
 *   arena : caller's host memory (pin it if the GPU is to restore from it), 16-byte aligned.
 *   token_bytes = 2 * num_layers * row : bytes of one token over all planes.
 * A delta is the dense pack buffer of one request's range [t_begin, t_end)
 * ([plane][token][head][dim], what lumen_kv_checkpoint_pack writes for a 1-request plan);
 * deltas of a request must arrive in order (t_begin == tokens stored so far).
 * Status codes: EINVAL (unknown / duplicate request, out-of-order or oversized delta, bad
 * tag), ENOMEM (no contiguous room for the reservation), ESIZE (delta_bytes mismatch).
 */
typedef struct lumen_kv_store lumen_kv_store;
LUMEN_KV_API int lumen_kv_store_create(void* arena, int64_t arena_bytes, int64_t token_bytes,
                                       int32_t page_size, int32_t copy_threads,
                                       lumen_kv_store** out);
LUMEN_KV_API void lumen_kv_store_destroy(lumen_kv_store* store);
/* bytes not reserved: the "available checkpoint-store capacity" of the load table */
LUMEN_KV_API int64_t lumen_kv_store_available(const lumen_kv_store* store);
/* reserved footprint of all requests held, in bytes */
LUMEN_KV_API int64_t lumen_kv_store_reserved(const lumen_kv_store* store);
LUMEN_KV_API int lumen_kv_store_reserve(lumen_kv_store* store, uint64_t request_id,
                                        int64_t max_tokens);
LUMEN_KV_API int lumen_kv_store_release(lumen_kv_store* store, uint64_t request_id);
/* tags: the tags of the pages this delta touches, any order; every end_pos must lie in
 * (t_begin, t_end].  n_tags may be 0. */
LUMEN_KV_API int lumen_kv_store_append(lumen_kv_store* store, uint64_t request_id,
                                       int64_t t_begin, int64_t t_end, const void* delta,
                                       int64_t delta_bytes, const lumen_kv_tag* tags,
                                       int32_t n_tags);
/* tokens stored for the request (its "actual checkpointed size"), or EINVAL */
LUMEN_KV_API int64_t lumen_kv_store_tokens(const lumen_kv_store* store, uint64_t request_id);
/* longest contiguous checkpointed prefix, in tokens, for the tags regenerated from the
 * request's token history (lumen_kv_page_tags / lumen_kv_longest_prefix over the stored tags) */
LUMEN_KV_API int64_t lumen_kv_store_lookup(const lumen_kv_store* store, uint64_t request_id,
                                           const lumen_kv_tag* regen, int64_t n_regen);
/* The stored deltas that cover [0, prefix_tokens), in order: segment i holds tokens
 * [t_begin, t_end) at byte offset buf_offset of the arena with plane stride
 * plane_stride_tokens -- exactly a lumen_kv_req range + lumen_kv_req_layout for
 * lumen_kv_plan_build_layout, so the prefix is restored straight out of the arena.
 * Writes at most cap entries; returns the number of segments or a status. */
typedef struct {
    int64_t t_begin, t_end;
    int64_t buf_offset;
    int64_t plane_stride_tokens;
} lumen_kv_segment;
/* A ready-made sink for lumen_kv_ckpt_create (user = the lumen_kv_store*): appends the delta
 * with the tags it carries -- a holder on the same host, or the receiving end of the
 * transport in tests.  Returns the append's status; failed appends are counted as well. */
LUMEN_KV_API int lumen_kv_store_sink(void* store, uint64_t request_id, int64_t t_begin,
                                      int64_t t_end, const void* delta, int64_t delta_bytes,
                                      const lumen_kv_tag* tags, int32_t n_tags);
LUMEN_KV_API int64_t lumen_kv_store_sink_errors(const lumen_kv_store* store);
/*
 * Reserve-then-commit into the store (for lumen_kv_ckpt_set_direct; user = the lumen_kv_store*).
 * acquire claims [t_begin, t_end) at the tail of the request's reservation and returns the
 * position inside the arena where its delta belongs (layout of lumen_kv_store_append:
 * [plane][token][head][dim]), or NULL if the request is unknown, the range does not continue
 * what is stored plus what is already claimed, the reservation is too small, or a copying
 * append is in progress.  Claims of one request stack up in order.  The writer fills the bytes,
 * then calls lumen_kv_store_append / lumen_kv_store_sink with delta == that position: nothing
 * is copied, and the delta and its tags become visible to lookups only then.
 * abort voids every outstanding claim of the request; what they covered stays invisible.
 * lumen_kv_store_arena returns the arena the store was created on.
 */
LUMEN_KV_API void* lumen_kv_store_acquire(void* store, uint64_t request_id, int64_t t_begin,
                                          int64_t t_end, int64_t delta_bytes);
LUMEN_KV_API void lumen_kv_store_abort(void* store, uint64_t request_id);
LUMEN_KV_API void* lumen_kv_store_arena(const lumen_kv_store* store, int64_t* arena_bytes);
LUMEN_KV_API int64_t lumen_kv_store_segments(const lumen_kv_store* store, uint64_t request_id,
                                             int64_t prefix_tokens, lumen_kv_segment* out,
                                             int64_t cap);

/*
 * Background checkpointer -- the worker side of the incremental checkpoint pipeline
 * (PAPER.md:145): "workers track checkpoint progress and transmit only newly generated KV
 * pages after each prefill or decode batch. A background thread copies these pages from GPU
 * memory to the local pinned buffer (3), then streams them over the network to the designated
 * checkpoint store (4). This two-stage pipeline completely overlaps with normal inference".
 *
 * One object = one worker's thread.  It keeps t_prev per tracked request (step a1), and for
 * every notification builds ONE plan over all pending deltas [t_prev, t_cur) (a2), waits for
 * the batch's ready event on its own stream (A10), packs through the two-stage path with
 * per-chunk commit flags into the caller's pinned buffer (a3-a5) and hands each request's
 * delta to `sink` as soon as the chunks that hold it have committed -- while later chunks are
 * still in flight -- then advances t_prev.  The sink stands in for step (4); it runs on the
 * checkpointer's thread, must not keep the pointer, and sees for each request exactly the
 * dense pack buffer of its range: [plane][token][head][dim], with the tags of the pages it
 * touches when the caller supplied token IDs.  The sink returns 0 if it took the delta; on
 * any other value the request's progress stays where it was (lumen_kv_ckpt_progress does not
 * advance), what is pending or already in flight for that request is dropped, flush() reports
 * LUMEN_KV_ESINK, and the request's next notification packs again from its last delivered token.
 *   k_planes, v_planes : device pointers of the pool (copied).
 *   staging / slot_bytes / n_slots : device staging ring as for lumen_kv_stager_create.
 *   pinned / pinned_bytes : pinned host buffer (a multiple of 32 bytes), used as two halves:
 *                 while the sink drains one, the copy engine fills the other.  Deltas are
 *                 batched up to one half; a delta larger than a half is delivered in pieces.
 * notify() copies the page tables and returns at once; deltas of one request are delivered
 * in order; a later notification for a request extends an earlier one that has not started, and
 * each keeps its own ready event: the checkpointer packs what is ready now, up to the newest
 * notification whose event has fired.
 * ready_event: a cudaEvent_t recorded after the batch that produced the tokens (NULL: they
 * already exist); it must stay valid until the delta has been delivered.
 * flush() blocks until everything notified before the call has been delivered and returns
 * the first error the thread met (0 if none).  Errors: EINVAL, ESIZE, ENOMEM, ECUDA.
 */
typedef struct lumen_kv_ckpt lumen_kv_ckpt;
typedef int (*lumen_kv_sink_fn)(void* user, uint64_t request_id, int64_t t_begin, int64_t t_end,
                                 const void* delta, int64_t delta_bytes,
                                 const lumen_kv_tag* tags, int32_t n_tags);
LUMEN_KV_API int lumen_kv_ckpt_create(const lumen_kv_geom* geom, const void* const* k_planes,
                                      const void* const* v_planes, void* staging,
                                      int64_t slot_bytes, int32_t n_slots, void* pinned,
                                      int64_t pinned_bytes, lumen_kv_sink_fn sink, void* user,
                                      lumen_kv_ckpt** out);
LUMEN_KV_API void lumen_kv_ckpt_destroy(lumen_kv_ckpt* ckpt);          /* flushes, joins the thread */
/*
 * Reserve-then-commit delivery: the copy engine writes each delta straight to its final place.
 * By default a delta crosses host memory twice -- copy engine -> the checkpointer's pinned
 * halves, then the sink copies it to wherever it keeps checkpoints (for the store: 0.65-0.75 of
 * the D2H peak end to end).  With set_direct, the checkpointer asks `acquire(user, id, t_begin,
 * t_end, delta_bytes)` for the delta's destination before it packs a batch; if every delta of
 * the batch gets one (a pointer inside the PINNED region [region, region + region_bytes),
 * a multiple of one plane row from its base), the batch is packed to those positions and the
 * sink is then called with delta == that pointer, as the commit.  A claim that will not be
 * committed (rejected, failed or voided delta) is returned through `abort(user, id)` once no
 * copy can still be writing it.  Batches whose average delta is below min_avg_delta_bytes, or
 * for which any acquire returns NULL, go the default way.  acquire == NULL switches it off.
 * Both callbacks run on the checkpointer's thread.  For a lumen_kv_store: region =
 * lumen_kv_store_arena, acquire = lumen_kv_store_acquire, abort = lumen_kv_store_abort.
 * Errors: EINVAL (null, misaligned, region not pinned).
 */
typedef void* (*lumen_kv_acquire_fn)(void* user, uint64_t request_id, int64_t t_begin,
                                      int64_t t_end, int64_t delta_bytes);
typedef void (*lumen_kv_abort_fn)(void* user, uint64_t request_id);
LUMEN_KV_API int lumen_kv_ckpt_set_direct(lumen_kv_ckpt* ckpt, void* region, int64_t region_bytes,
                                          lumen_kv_acquire_fn acquire, lumen_kv_abort_fn abort,
                                          int64_t min_avg_delta_bytes);
LUMEN_KV_API int lumen_kv_ckpt_track(lumen_kv_ckpt* ckpt, uint64_t request_id, int64_t t_prev);
LUMEN_KV_API int lumen_kv_ckpt_untrack(lumen_kv_ckpt* ckpt, uint64_t request_id);
/* reqs[i].page_table / page_table_len: request ids[i]'s current table; reqs[i].t_end = t_cur;
 * reqs[i].t_begin is ignored (the checkpointer knows t_prev).
 * token_ids: NULL, or for each request a HOST pointer to its token history [0, t_cur) (entries
 * may be NULL); the part the new delta needs is copied, and the sink then receives the page
 * tags of the pages each delta touches ("each transferred page carries a page tag",
 * PAPER.md:147), computed by lumen_kv_page_tags_host.  Without tokens n_tags is 0.  A request
 * whose pending delta carries token IDs must keep passing them (EINVAL otherwise: the tags of
 * the pending pages would be lost). */
LUMEN_KV_API int lumen_kv_ckpt_notify(lumen_kv_ckpt* ckpt, const uint64_t* ids,
                                      const lumen_kv_req* reqs, const int32_t* const* token_ids,
                                      int32_t n, void* ready_event);
LUMEN_KV_API int lumen_kv_ckpt_flush(lumen_kv_ckpt* ckpt);
/* tokens of the request delivered to the sink so far (its t_prev), or EINVAL */
LUMEN_KV_API int64_t lumen_kv_ckpt_progress(lumen_kv_ckpt* ckpt, uint64_t request_id);

/*
 * lumen_kv_store_restore -- KV-reuse recovery of one request on its checkpoint holder
 * (PAPER.md:157): "From the request's token history, the holder deterministically regenerates
 * page tags to locate the longest contiguous checkpointed prefix within its local store,
 * subsequently loading the matching KV pages into GPU memory."  One call: regenerate the tags
 * of token_ids[0, n_tokens) (host), look the prefix up in the store, build an explicit-layout
 * plan over the stored deltas that cover it (lumen_kv_store_segments) with the fresh
 * page_table, and restore it out of the store's arena through the two-stage path.
 *   arena must be pinned (it is the source of the H2D copies); page_table must cover the
 *   prefix; k_planes / v_planes / stager / stream as for lumen_kv_restore_unpack_staged.
 *   *restored_tokens receives the prefix length P; the suffix [P, n_tokens) is the caller's to
 *   recompute ("partial prefill on the uncheckpointed suffix").
 * Asynchronous on `stream` like the restore itself.  Errors: EINVAL (unknown request, table too
 * short), ERANGE, EOVERLAP, ESIZE, ENOMEM, ECUDA.
 */
LUMEN_KV_API int lumen_kv_store_restore(const lumen_kv_store* store, uint64_t request_id,
                                        const int32_t* token_ids, int64_t n_tokens,
                                        const lumen_kv_geom* geom, const int32_t* page_table,
                                        int64_t page_table_len, void* const* k_planes,
                                        void* const* v_planes, lumen_kv_stager* stager,
                                        void* stream, int64_t* restored_tokens);

/*
 * Controller logic (host arithmetic only; section 4.2 Eq. (1), section 4.3).
 *
 * lumen_kv_choose_holder -- checkpoint placement, Eq. (1):
 *     h(r) = argmin over w in F(r) of  q_w + lambda * p_w(r)
 *   q[w]        : queueing delay of worker w;
 *   p_w(r)      : mean reserved footprint of the checkpoints w would hold after assigning r
 *                 (held[held_begin[w] .. held_begin[w+1]) plus footprint), divided by bandwidth;
 *   F(r)        : workers other than `serving` with available[w] >= footprint.
 *   Evaluated in double, in the order ((sum / count) / bandwidth) * lambda + q; ties go to
 *   the lowest worker id (reading F1).  *holder = h(r), or -1 if F(r) is empty.
 * lumen_kv_recover -- recovery dispatch + greedy load rebalancing:
 *   load[w]     : queued + running requests of worker w (ignored where alive[w] == 0);
 *   holder[i], ckpt_size[i] : checkpoint holder and checkpointed size of interrupted request i;
 *   assign[i]   : worker that takes request i;  reuse[i] : 1 if it restores its checkpoint
 *                 there, 0 if it recomputes;  final_load[w] : loads after rebalancing.
 *   Interrupted requests go to their holder (reuse) or, if the holder is dead, to the
 *   least-loaded survivor (recompute); then, while a survivor holding reusable requests has
 *   load > ceil(average load after dispatch), the most loaded such worker sheds its
 *   smallest checkpoint to the least-loaded other survivor (readings F2-F4).
 * Errors: EINVAL (null, no worker alive, negative sizes, bad ids).
 */
LUMEN_KV_API int lumen_kv_choose_holder(const double* q, const int64_t* held,
                                        const int32_t* held_begin, const int64_t* available,
                                        int32_t num_workers, int32_t serving, int64_t footprint,
                                        double lambda, double bandwidth, int32_t* holder);
LUMEN_KV_API int lumen_kv_recover(const int64_t* load, const uint8_t* alive, int32_t num_workers,
                                  const int32_t* holder, const int64_t* ckpt_size,
                                  int32_t num_interrupted, int32_t* assign, uint8_t* reuse,
                                  int64_t* final_load);

/* Release a plan.  Safe to call while work using the plan is still in flight on a
 * stream, or still queued in a stager's thread: the descriptors are recycled only after
 * that work has completed.  Never frees device or pinned memory (no implicit device
 * synchronisation on the caller's thread): descriptor memory goes back to a cache that
 * only lumen_kv_trim() empties.                                                      */
LUMEN_KV_API void lumen_kv_plan_free(lumen_kv_plan* plan);

/* Release cached descriptor memory held by the library (synchronises the device). */
LUMEN_KV_API void lumen_kv_trim(void);

/* One-time initialisation of the current device (SM count, load of every kernel variant);
 * done implicitly by the first launch on a device.  Errors: ECUDA.                     */
LUMEN_KV_API int lumen_kv_init(void);

/*
 * Tuning knobs.  They exist to reproduce the A/B measurements of DESIGN.md; the defaults are
 * the measured best and nothing needs them.  Each is also read once from the environment
 * (LUMEN_KV_<NAME in capitals>) at the library's first use.  Process-wide; do not change them
 * while another thread is inside pack/unpack.
 *   "pdl"         1 (default) / 0 : programmatic dependent launch of the SIMT kernel
 *   "wide"        1 (default) / 0 : 32-byte accesses where every address allows them, else 16-byte
 *   "warp_unroll" 4 (default) / 8 : loads in flight per lane of the 16-byte kernel
 *   "host_kernel" 2 (default, TMA bulk kernel) / 1 (SIMT kernel): what AUTO picks for a host buffer
 *   "host_ctas"   0 (default: 24..96 by item size) / n : grid of the bulk kernel on a host buffer
 *   "inline_max_runs" 1024 (default) / n : plans of more than n runs upload their descriptors
 *   "fail_after_chunks" -1 (default, off) / n >= 0 : TEST HOOK -- every staged call fails with ECUDA
 *                 (cudaErrorUnknown) in front of its chunk n; used to test the error paths
 *   "prefetch"    16 (default) / d >= 0 / -1 : the SIMT kernel asks L2 for the 4 KiB a warp d CTAs
 *                 further on will copy (parameter-resident plans; larger plans announce their own
 *                 4 KiB, whatever d) / no prefetch.  A hint: the bytes moved are the same.
 * Errors: EINVAL (unknown name).
 */
LUMEN_KV_API int lumen_kv_set_option(const char* name, int value);

LUMEN_KV_API const char* lumen_kv_strerror(int status);
/* last cudaError_t seen by the calling thread inside the library (0 if none) */
LUMEN_KV_API int lumen_kv_last_cuda_error(void);
LUMEN_KV_API int lumen_kv_version(void);

#ifdef __cplusplus
}
#endif
#endif /* LUMEN_KV_H */
