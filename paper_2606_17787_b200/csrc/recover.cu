// KV-reuse recovery of one request on its checkpoint holder (include/lumen_kv.h):
// tags from the token history -> longest checkpointed prefix -> explicit-layout plan over the
// stored deltas -> restore out of the store's arena.  Composition of the public C ABI.
#include <cuda_runtime.h>

#include <vector>

#include "lumen_kv.h"

// the store's arena base, needed as the source pointer of the restore (store.cpp)
extern "C" const void* lumen_kv_store_arena_(const lumen_kv_store* store, int64_t* bytes);

extern "C" int lumen_kv_store_restore(const lumen_kv_store* store, uint64_t id,
                                      const int32_t* token_ids, int64_t n_tokens,
                                      const lumen_kv_geom* geom, const int32_t* page_table,
                                      int64_t page_table_len, void* const* k_planes,
                                      void* const* v_planes, lumen_kv_stager* stager, void* stream,
                                      int64_t* restored_tokens) {
    if (restored_tokens) *restored_tokens = 0;
    if (!store || !geom || !restored_tokens || n_tokens < 0 || (n_tokens > 0 && !token_ids) ||
        geom->page_size < 1)
        return LUMEN_KV_EINVAL;
    const int32_t S = geom->page_size;
    // 1. regenerate the page tags of the whole history
    std::vector<lumen_kv_tag> regen(static_cast<size_t>((n_tokens + S - 1) / S));
    if (n_tokens > 0) {
        const int64_t n = lumen_kv_page_tags_host(token_ids, 0, 0, n_tokens, S, regen.data(),
                                                  static_cast<int64_t>(regen.size()));
        if (n < 0) return static_cast<int>(n);
    }
    // 2. longest contiguous checkpointed prefix
    const int64_t prefix = lumen_kv_store_lookup(store, id, regen.data(),
                                                 static_cast<int64_t>(regen.size()));
    if (prefix < 0) return static_cast<int>(prefix);
    *restored_tokens = prefix;
    if (prefix == 0) return LUMEN_KV_OK;
    if ((prefix + S - 1) / S > page_table_len || !page_table) return LUMEN_KV_EINVAL;
    // 3. the stored deltas that cover it, as plan entries with their layout in the arena
    const int64_t n_seg = lumen_kv_store_segments(store, id, prefix, nullptr, 0);
    if (n_seg < 0) return static_cast<int>(n_seg);
    std::vector<lumen_kv_segment> segs(static_cast<size_t>(n_seg));
    lumen_kv_store_segments(store, id, prefix, segs.data(), n_seg);
    std::vector<lumen_kv_req> reqs(segs.size());
    std::vector<lumen_kv_req_layout> lays(segs.size());
    for (size_t i = 0; i < segs.size(); ++i) {
        reqs[i].page_table = page_table;
        reqs[i].page_table_len = page_table_len;
        reqs[i].t_begin = segs[i].t_begin;
        reqs[i].t_end = segs[i].t_end;
        lays[i].buf_offset = segs[i].buf_offset;
        lays[i].plane_stride_tokens = segs[i].plane_stride_tokens;
    }
    lumen_kv_plan* plan = nullptr;
    int rc = lumen_kv_plan_build_layout(geom, reqs.data(), lays.data(), static_cast<int32_t>(reqs.size()),
                                        LUMEN_KV_VALIDATE_UNIQUE_DST, stream, &plan);
    if (rc != LUMEN_KV_OK) return rc;
    // 4. load the pages into GPU memory, straight out of the arena
    int64_t arena_bytes = 0;
    const void* arena = lumen_kv_store_arena_(store, &arena_bytes);
    rc = lumen_kv_restore_unpack_staged(plan, k_planes, v_planes, arena, arena_bytes, stager, stream);
    lumen_kv_plan_free(plan);               // safe while the restore is in flight
    return rc;
}
