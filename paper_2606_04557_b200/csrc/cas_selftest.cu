// Hardware self-test of the CTA-pair (tcgen05 cta_group::2) primitives in cas_sm100.cuh -- the building block
// DESIGN.md section 10 names as the next step against the shared-memory-bandwidth limit of the attention kernels.
// D[256 x 128] = A[256 x 64] * B[128 x 64]^T (bf16 in, fp32 out) on a 2-CTA cluster: each CTA holds 128 rows of
// A and 64 rows of B; the leader issues the MMAs for both SMs.  Not on the hot path.
#include "cas_internal.h"
#include "cas_sm100.cuh"

namespace cas {
using namespace sm100;

__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(128, 1)
pair_mma_selftest_kernel(const __nv_bfloat16* __restrict__ A, const __nv_bfloat16* __restrict__ B, float* __restrict__ D) {
  extern __shared__ __align__(1024) uint8_t smem[];
  const uint32_t sbase = smem_u32(smem);
  const uint32_t rank = cluster_ctarank();
  const int tid = threadIdx.x, warp = tid >> 5;
  uint32_t* slot = reinterpret_cast<uint32_t*>(smem + 24576 + 64);
  const uint32_t bar = sbase + 24576;
  // A_r (rows 128r.., 64 bf16 = one 128-byte swizzle atom per row) at 0; B_r (rows 64r..) at 16384
  for (int i = tid; i < 128 * 8; i += 128) {
    const int row = i >> 3, c = i & 7;
    *reinterpret_cast<uint4*>(smem + row * 128 + ((c ^ (row & 7)) << 4)) =
        *reinterpret_cast<const uint4*>(A + (size_t)(128 * rank + row) * 64 + c * 8);
  }
  for (int i = tid; i < 64 * 8; i += 128) {
    const int row = i >> 3, c = i & 7;
    *reinterpret_cast<uint4*>(smem + 16384 + row * 128 + ((c ^ (row & 7)) << 4)) =
        *reinterpret_cast<const uint4*>(B + (size_t)(64 * rank + row) * 64 + c * 8);
  }
  if (tid == 0) {
    mbar_init(bar, 1);
    fence_mbar_init();
  }
  fence_proxy_async();
  if (warp == 0) tmem_alloc_pair(smem_u32(slot), 128);
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();                       // both CTAs: operands written, barrier initialised, TMEM allocated
  tc_fence_after();
  const uint32_t tbase = *slot;
  if (rank == 0 && tid == 0) {
    constexpr uint32_t idesc = make_idesc(256, 128, 0, 0);
#pragma unroll
    for (int kk = 0; kk < 4; ++kk)
      mma_ss_pair(tbase, desc_kmajor(sbase + kk * 32), desc_kmajor(sbase + 16384 + kk * 32), idesc, kk > 0);
    mma_commit_pair(bar, 3);
  }
  mbar_wait(bar, 0);
  tc_fence_after();
  float* out = D + (size_t)(128 * rank + tid) * 128;
  for (int c = 0; c < 4; ++c) {
    uint32_t d[32];
    tmem_ld32(tbase + ((uint32_t)(warp * 32) << 16) + c * 32, d);
    tc_wait_ld();
    for (int i = 0; i < 32; ++i) out[c * 32 + i] = __uint_as_float(d[i]);
  }
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();
  if (warp == 0) tmem_dealloc_pair(tbase, 128);
}

}  // namespace cas

extern "C" int cas_selftest_cta_pair_mma(const void* A, const void* B, float* D, void* stream) {
  using namespace cas;
  if (!A || !B || !D) { set_error("null arg"); return CAS_ERR_INVALID_ARG; }
  CAS_CUDA(cudaFuncSetAttribute(pair_mma_selftest_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 25600));
  pair_mma_selftest_kernel<<<2, 128, 25600, (cudaStream_t)stream>>>((const __nv_bfloat16*)A, (const __nv_bfloat16*)B, D);
  cudaError_t e = cudaGetLastError();
  return e == cudaSuccess ? CAS_OK : cuda_fail(e, "pair mma selftest launch");
}
