// Internal descriptor formats shared by the host plan builder and the kernels.
// Not part of the public ABI (include/lumen_kv.h is).
#pragma once
#include <cstdint>
#include <vector>

#include "lumen_kv.h"

namespace lumen {

// One token-run: `count` consecutive tokens that are contiguous in the pool
// (inside one page, or across physically adjacent pages when merged) and in the
// checkpoint buffer.  16 bytes so a warp fetches it with one vector load.
//   pool byte offset inside any plane   = src_off16 * 16
//   buffer row (plane p)                = req.row_base + p * req.n + dst_tok
// (the run is described once and replicated over the
//  2L planes by the grid, never materialised per plane.)
struct alignas(16) RunDesc {
    uint32_t src_lo;    // low 32 bits of src_off16
    uint32_t dst_tok;   // request-relative first token j
    uint32_t req;       // request index
    uint16_t count;     // tokens in the run, 1..65535
    uint16_t src_hi;    // high 16 bits of src_off16
};
static_assert(sizeof(RunDesc) == 16, "RunDesc must be 16 bytes");

struct alignas(16) ReqDesc {
    int64_t row_base;   // first row of the request's block in the buffer (dense: sum of n * 2L)
    int64_t n;          // rows between consecutive planes (dense: tokens of this request)
};
static_assert(sizeof(ReqDesc) == 16, "ReqDesc must be 16 bytes");

constexpr int64_t kChunkBytes = 32768;  // a run never exceeds this unless one row does

// Result of the host-side flattening; plain memory, no CUDA.
struct HostPlan {
    lumen_kv_geom geom{};
    int64_t row_bytes = 0;
    int64_t page_stride = 0;
    int64_t total_bytes = 0;
    int64_t total_tokens = 0;
    int32_t max_count = 0;            // longest run, tokens
    std::vector<RunDesc> runs;
    std::vector<ReqDesc> reqs;
    std::vector<int64_t> req_offset;  // num_reqs + 1 byte offsets (last = total_bytes)
    std::vector<int64_t> req_tokens;  // num_reqs: n_r
    std::vector<int64_t> req_stride;  // num_reqs: plane stride in tokens (dense: n_r)
    std::vector<int64_t> req_run_begin;  // num_reqs + 1: runs of request r are [begin[r], begin[r+1])
};

// A piece of a plan that is contiguous in the checkpoint buffer: runs [ra, rb) replicated
// over planes [p0, p1) cover exactly the buffer bytes [b0, b1).  Either whole requests over
// all planes, or one request over a plane range, or one plane of one request over a token
// range (buffer layout [req][plane][token], include/lumen_kv.h).
struct Chunk {
    int64_t ra, rb;
    int32_t p0, p1;
    int64_t b0, b1;
};

// Cuts the plan into chunks of at most slot_bytes each (the two-stage host path).  `runs` are
// the plan's run descriptors on the host.  ESIZE if a single run is larger than slot_bytes.
int build_chunks(const HostPlan& hp, const RunDesc* runs, int64_t slot_bytes,
                 std::vector<Chunk>* out);

// Validates and flattens.  Returns a lumen_kv_status.
int build_host_plan(const lumen_kv_geom* geom, const lumen_kv_req* reqs,
                    const lumen_kv_req_layout* layouts /* nullptr: dense */,
                    int32_t num_reqs, uint32_t flags, HostPlan* out);

}  // namespace lumen
