// Host-side helpers shared by the tensor-core translation units: TMA tensor-map encoding for the
// [tokens, heads, 128] bf16 tensors of the path.
#pragma once
#include <atomic>

#include "cas_internal.h"

namespace cas {

typedef CUresult (*TmaEncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

TmaEncodeFn tma_encoder();

// Map over a row-major [tokens, heads, 128] bf16 tensor; box = 64 (d) x 1 (head) x box_tokens,
// 128-byte swizzle: one box lands as [box_tokens][64] with 128-byte rows, the layout the UMMA
// descriptors in cas_sm100.cuh describe.  Rows past `tokens` read as zero.
int make_thd_map(CUtensorMap* out, const void* base, int64_t tokens, int heads, int box_tokens);

// cudaFuncAttributeMaxDynamicSharedMemorySize is a PER-DEVICE attribute: raise it once on every device the
// kernel is launched on (a process-wide flag would leave a second device at the 48 KB default).
struct SmemAttrOnce {
  std::atomic<uint64_t> done[2] = {{0}, {0}};
  int set(const void* func, int bytes) {
    int dev = 0;
    CAS_CUDA(cudaGetDevice(&dev));
    if (dev >= 0 && dev < 128 && ((done[dev >> 6].load(std::memory_order_acquire) >> (dev & 63)) & 1ull)) return CAS_OK;
    CAS_CUDA(cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
    if (dev >= 0 && dev < 128) done[dev >> 6].fetch_or(1ull << (dev & 63), std::memory_order_release);
    return CAS_OK;
  }
};

}  // namespace cas
