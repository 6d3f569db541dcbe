// kvfill.cu -- TEST / BENCH TOOLING, not the path under test.
// CUDA twin of workloads/content.py: fills a device plane with the counter-based
// pattern g(seed, plane, word index) and computes a per-page 64-bit checksum used to
// prove "all other pages untouched" at sizes where the pool cannot be cloned
// (SURVEY.md section 8(c) C4/C5).  Built into workloads/libkvfill.so; it shares
// nothing with paper_2606_17787_b200/csrc.
#include <cuda_runtime.h>
#include <stdint.h>

namespace {

__device__ __forceinline__ uint64_t mix64(uint64_t x) {
    uint64_t z = x + 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

// one 64-bit hash = 4 little-endian 16-bit words; n_q = number of 8-byte groups
__global__ void fill_kernel(uint64_t* __restrict__ out, int64_t n_q, uint64_t base, int64_t q0) {
    const int64_t stride = static_cast<int64_t>(gridDim.x) * blockDim.x;
    for (int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x; i < n_q; i += stride)
        out[i] = mix64(base + static_cast<uint64_t>(q0 + i));
}

// checksum of page p = sum over its 8-byte groups i of mix64(value ^ mix64(i)); one CTA per page
__global__ void checksum_kernel(const uint64_t* __restrict__ plane, int64_t q_per_page,
                                uint64_t* __restrict__ out) {
    const uint64_t* page = plane + static_cast<int64_t>(blockIdx.x) * q_per_page;
    uint64_t acc = 0;
    for (int64_t i = threadIdx.x; i < q_per_page; i += blockDim.x)
        acc += mix64(page[i] ^ mix64(static_cast<uint64_t>(i)));
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, o);
    __shared__ uint64_t warp_sum[32];
    if ((threadIdx.x & 31) == 0) warp_sum[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        uint64_t t = 0;
        for (unsigned w = 0; w < (blockDim.x + 31) / 32; ++w) t += warp_sum[w];
        out[blockIdx.x] = t;
    }
}

}  // namespace

extern "C" {

// Fill words [first_word, first_word + n_words) of plane `plane` at dst (dst points at
// first_word).  first_word and n_words must be multiples of 4 and dst 8-byte aligned.
__attribute__((visibility("default")))
int kvfill_fill(void* dst, int64_t first_word, int64_t n_words, uint64_t seed, uint64_t plane,
                void* stream) {
    if ((first_word | n_words) & 3 || (reinterpret_cast<uintptr_t>(dst) & 7)) return -1;
    if (n_words == 0) return 0;
    const int64_t n_q = n_words / 4;
    const uint64_t base = seed ^ (plane << 40);
    int64_t blocks = (n_q + 255) / 256;
    if (blocks > 148 * 16) blocks = 148 * 16;
    fill_kernel<<<static_cast<unsigned>(blocks), 256, 0, static_cast<cudaStream_t>(stream)>>>(
        static_cast<uint64_t*>(dst), n_q, base, first_word / 4);
    return cudaGetLastError() == cudaSuccess ? 0 : -2;
}

// out[p] = checksum of page p for p in [0, n_pages); page_bytes % 8 == 0; out is device memory.
__attribute__((visibility("default")))
int kvfill_page_checksums(const void* plane, int64_t n_pages, int64_t page_bytes, void* out,
                          void* stream) {
    if (page_bytes % 8 || (reinterpret_cast<uintptr_t>(plane) & 7)) return -1;
    if (n_pages == 0) return 0;
    checksum_kernel<<<static_cast<unsigned>(n_pages), 256, 0, static_cast<cudaStream_t>(stream)>>>(
        static_cast<const uint64_t*>(plane), page_bytes / 8, static_cast<uint64_t*>(out));
    return cudaGetLastError() == cudaSuccess ? 0 : -2;
}

}  // extern "C"
