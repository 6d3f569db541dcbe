// Page tags (include/lumen_kv.h): 64-bit FNV-1a of each page's token IDs,
// paired with the page's end position, and the longest-contiguous-prefix lookup.
//
// One thread per page.  A page is S int32 token IDs (64 B at S = 16) against 2L*S*row bytes
// of KV (4 MiB for the Qwen3-32B shape), so this kernel moves 1/65,536 of what the pack
// moves; it is bound by the 4 dependent 64-bit multiplies per token, not by memory.
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdint>
#include <new>
#include <vector>

#include "internal.hpp"
#include "lumen_kv.h"

namespace {

constexpr int kReqsPerLaunch = 480;   // offsets travel as kernel parameters (2 x 481 x 8 B)

struct TagParams {
    int64_t tok_off[kReqsPerLaunch + 1];    // token offsets of this batch's requests
    int64_t page_off[kReqsPerLaunch + 1];   // page offsets, relative to the batch's first tag
};

__global__ void __launch_bounds__(128)
page_tags_kernel(const __grid_constant__ TagParams p, const int32_t* __restrict__ tokens,
                 lumen_kv_tag* __restrict__ out, int32_t S) {
    const int r = blockIdx.y;
    const int64_t page = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    const int64_t pages = p.page_off[r + 1] - p.page_off[r];
    if (page >= pages) return;
    const int64_t len = p.tok_off[r + 1] - p.tok_off[r];
    const int64_t first = page * S;
    const int64_t end = (first + S < len) ? first + S : len;
    const int32_t* t = tokens + p.tok_off[r];
    uint64_t h = 0xcbf29ce484222325ull;
    for (int64_t i = first; i < end; ++i) {
        const uint32_t v = static_cast<uint32_t>(__ldg(t + i));
#pragma unroll
        for (int b = 0; b < 4; ++b) {                 // little-endian bytes of the token ID
            h ^= (v >> (8 * b)) & 0xffu;
            h *= 0x100000001b3ull;
        }
    }
    lumen_kv_tag tag;
    tag.hash = h;
    tag.end_pos = end;
    // one 16-byte store per tag
    *reinterpret_cast<ulonglong2*>(out + p.page_off[r] + page) =
        make_ulonglong2(tag.hash, static_cast<unsigned long long>(tag.end_pos));
}

inline bool tag_less(const lumen_kv_tag& a, const lumen_kv_tag& b) {
    return a.hash != b.hash ? a.hash < b.hash : a.end_pos < b.end_pos;
}

}  // namespace

extern "C" {

int64_t lumen_kv_tags_num_pages(const int64_t* tok_offset, int32_t num_reqs, int32_t page_size) {
    if (num_reqs < 0 || page_size < 1 || !tok_offset) return LUMEN_KV_EINVAL;
    int64_t pages = 0;
    for (int32_t r = 0; r < num_reqs; ++r) {
        const int64_t len = tok_offset[r + 1] - tok_offset[r];
        if (len < 0) return LUMEN_KV_EINVAL;
        pages += (len + page_size - 1) / page_size;
    }
    return pages;
}

int lumen_kv_page_tags(const int32_t* token_ids, const int64_t* tok_offset, int32_t num_reqs,
                       int32_t page_size, lumen_kv_tag* tags_out, int64_t tags_cap, void* stream) {
    const int64_t total = lumen_kv_tags_num_pages(tok_offset, num_reqs, page_size);
    if (total < 0) return static_cast<int>(total);
    if (total == 0) return LUMEN_KV_OK;
    if (!token_ids || !tags_out || (reinterpret_cast<uintptr_t>(tags_out) & 15) ||
        (reinterpret_cast<uintptr_t>(token_ids) & 3))
        return LUMEN_KV_EINVAL;
    if (tags_cap < total) return LUMEN_KV_ESIZE;
    int64_t tag_base = 0;
    for (int32_t r0 = 0; r0 < num_reqs; r0 += kReqsPerLaunch) {
        const int32_t nr = std::min<int32_t>(kReqsPerLaunch, num_reqs - r0);
        TagParams p;
        int64_t max_pages = 0;
        p.page_off[0] = 0;
        for (int32_t i = 0; i <= nr; ++i) p.tok_off[i] = tok_offset[r0 + i];
        for (int32_t i = 0; i < nr; ++i) {
            const int64_t pages = (p.tok_off[i + 1] - p.tok_off[i] + page_size - 1) / page_size;
            p.page_off[i + 1] = p.page_off[i] + pages;
            max_pages = std::max(max_pages, pages);
        }
        if (max_pages > 0) {
            const int64_t gx = (max_pages + 127) / 128;
            if (gx > 0x7fffffffLL) return LUMEN_KV_EINVAL;
            dim3 grid(static_cast<unsigned>(gx), static_cast<unsigned>(nr), 1);
            page_tags_kernel<<<grid, 128, 0, static_cast<cudaStream_t>(stream)>>>(
                p, token_ids, tags_out + tag_base, page_size);
            const cudaError_t e = cudaGetLastError();
            if (e != cudaSuccess) return lumen::cuda_fail(e);
        }
        tag_base += p.page_off[nr];
    }
    return LUMEN_KV_OK;
}

int64_t lumen_kv_page_tags_host(const int32_t* token_ids, int64_t first_token, int64_t t_begin,
                                int64_t t_end, int32_t S, lumen_kv_tag* out, int64_t cap) {
    if (S < 1 || t_begin < 0 || t_end < t_begin || cap < 0 || first_token < 0 ||
        first_token % S != 0)
        return LUMEN_KV_EINVAL;
    if (t_end == t_begin) return 0;
    const int64_t p0 = t_begin / S, p1 = (t_end - 1) / S;
    if (!token_ids || first_token > p0 * S || (cap > 0 && !out)) return LUMEN_KV_EINVAL;
    for (int64_t p = p0; p <= p1 && p - p0 < cap; ++p) {
        const int64_t end = (p + 1) * S < t_end ? (p + 1) * S : t_end;
        uint64_t h = 0xcbf29ce484222325ull;
        for (int64_t t = p * S; t < end; ++t) {
            const uint32_t v = static_cast<uint32_t>(token_ids[t - first_token]);
            for (int b = 0; b < 4; ++b) {             // little-endian bytes of the token ID
                h ^= (v >> (8 * b)) & 0xffu;
                h *= 0x100000001b3ull;
            }
        }
        out[p - p0].hash = h;
        out[p - p0].end_pos = end;
    }
    return p1 - p0 + 1;
}

int64_t lumen_kv_longest_prefix(const lumen_kv_tag* regen, int64_t n_regen,
                                const lumen_kv_tag* stored, int64_t n_stored) {
    if (n_regen < 0 || n_stored < 0 || (n_regen > 0 && !regen) || (n_stored > 0 && !stored))
        return LUMEN_KV_EINVAL;
    std::vector<lumen_kv_tag> sorted;
    try {
        sorted.assign(stored, stored + n_stored);
    } catch (const std::bad_alloc&) {
        return LUMEN_KV_ENOMEM;
    }
    std::sort(sorted.begin(), sorted.end(), tag_less);
    int64_t prefix = 0;
    for (int64_t i = 0; i < n_regen; ++i) {
        if (!std::binary_search(sorted.begin(), sorted.end(), regen[i], tag_less)) break;
        prefix = regen[i].end_pos;
    }
    return prefix;
}

}  // extern "C"
