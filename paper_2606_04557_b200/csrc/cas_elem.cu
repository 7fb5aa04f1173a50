// HBM-bound elementwise kernels: fused Adam (sec. 2.2), arrival refresh (derive the
// working copy + zero the gradient slot after a swap-in), zero fill.
//
// Roofline: HBM.  Adam moves 30 B per element of a slot that holds gradients (read g,p,m,v = 16 B; write p,m,v
// = 12 B + bf16 working copy 2 B) and 26 B per element of a clean slot (g = 0 is not read).  Gradients are not
// zeroed: consuming them = clearing the slot's dirty flag; the next backward pass overwrites a clean slot.  All accesses are 16-byte vectors,
// fully coalesced, one (slot, chunk) per block; grid.y enumerates the slots.
#include <algorithm>

#include "cas_internal.h"

namespace cas {

__device__ __forceinline__ float4 ld4(const float* p) { return *reinterpret_cast<const float4*>(p); }
__device__ __forceinline__ void st4(float* p, float4 v) { *reinterpret_cast<float4*>(p) = v; }

__device__ __forceinline__ void store_work4(void* w, int64_t i, float4 p, bool bf16) {
  if (bf16) {
    __nv_bfloat162 a = __floats2bfloat162_rn(p.x, p.y);
    __nv_bfloat162 b = __floats2bfloat162_rn(p.z, p.w);
    uint2 u;
    u.x = *reinterpret_cast<uint32_t*>(&a);
    u.y = *reinterpret_cast<uint32_t*>(&b);
    *reinterpret_cast<uint2*>(reinterpret_cast<__nv_bfloat16*>(w) + i) = u;
  } else {
    st4(reinterpret_cast<float*>(w) + i, p);
  }
}

constexpr int kAdamThreads = 256;
constexpr int kAdamUnroll = 2;   // float4 per thread per tensor (8 independent 16-byte loads in flight)

template <bool BF16>
__global__ void __launch_bounds__(kAdamThreads)
adam_kernel(const __grid_constant__ AdamBatch batch, float lr, float b1, float b2, float eps, int zero_grad) {
  const AdamSlotDesc& d = batch.d[blockIdx.y];
  const float step = lr * d.step_size_scale;
  const float ibc1 = 1.0f / d.bc1, ibc2 = 1.0f / d.bc2;
  const int64_t chunk = (int64_t)kAdamThreads * 4 * kAdamUnroll;
  for (int which = 0; which < 2; ++which) {
    float* __restrict__ p = d.state + (int64_t)which * d.cap_elems;
    float* __restrict__ m = d.state + (int64_t)(2 + which) * d.cap_elems;
    float* __restrict__ v = d.state + (int64_t)(4 + which) * d.cap_elems;
    float* __restrict__ g = which ? d.gV : d.gK;
    void* w = which ? d.wV : d.wK;
    // frozen tokens are not updated; gradients are consumed by clearing the slot's dirty flag on
    // the host (a clean slot's buffer is undefined and overwritten by the next backward pass): nothing is zeroed
    for (int64_t base = d.frozen_elems + (int64_t)blockIdx.x * chunk; base < d.n_elems;
         base += (int64_t)gridDim.x * chunk) {
      float4 G[kAdamUnroll], P[kAdamUnroll], M[kAdamUnroll], V[kAdamUnroll];
#pragma unroll
      for (int u = 0; u < kAdamUnroll; ++u) {
        const int64_t i = base + ((int64_t)u * kAdamThreads + threadIdx.x) * 4;
        if (i < d.n_elems) {
          G[u] = d.has_grad ? ld4(g + i) : make_float4(0.f, 0.f, 0.f, 0.f);   // clean slot: g = 0, not read
          P[u] = ld4(p + i); M[u] = ld4(m + i); V[u] = ld4(v + i);
        }
      }
#pragma unroll
      for (int u = 0; u < kAdamUnroll; ++u) {
        const int64_t i = base + ((int64_t)u * kAdamThreads + threadIdx.x) * 4;
        if (i >= d.n_elems) continue;
        float* gp = reinterpret_cast<float*>(&G[u]);
        float* pp = reinterpret_cast<float*>(&P[u]);
        float* mp = reinterpret_cast<float*>(&M[u]);
        float* vp = reinterpret_cast<float*>(&V[u]);
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          const float gg = gp[k];
          const float mm = b1 * mp[k] + (1.0f - b1) * gg;
          const float vv = b2 * vp[k] + (1.0f - b2) * gg * gg;
          // m_hat = m/(1-b1^t), v_hat = v/(1-b2^t) as multiplications by the reciprocals; the one
          // remaining division is the fast one (2 ulp; IEEE division made this kernel ALU-bound and
          // takes a slow path once m, v decay to denormals).  Denominator >= eps > 0.
          pp[k] = pp[k] - __fdividef(step * (mm * ibc1), sqrtf(vv * ibc2) + eps);
          mp[k] = mm;
          vp[k] = vv;
        }
        st4(p + i, P[u]);
        st4(m + i, M[u]);
        st4(v + i, V[u]);
        store_work4(w, i, P[u], BF16);
      }
    }
  }
}

// The slot descriptors travel as KERNEL PARAMETERS (<= 256 slots = 20 KB per launch): no descriptor
// upload, so an Adam step never queues behind the 48 MiB swap copies on the host-to-device copy engine.
int launch_adam(const AdamSlotDesc* h_desc, int n, const cas_adam_cfg& cfg, int dtype, cudaStream_t st) {
  const int64_t chunk = (int64_t)kAdamThreads * 4 * kAdamUnroll;
  for (int i0 = 0; i0 < n; i0 += kAdamBatch) {
    const int cnt = std::min(kAdamBatch, n - i0);
    AdamBatch batch;
    int64_t max_elems = 0;
    for (int i = 0; i < cnt; ++i) {
      batch.d[i] = h_desc[i0 + i];
      max_elems = std::max(max_elems, h_desc[i0 + i].n_elems);
    }
    if (max_elems <= 0) continue;
    int64_t gx = (max_elems + chunk - 1) / chunk;
    if (gx > 65535) gx = 65535;
    dim3 grid((unsigned)gx, (unsigned)cnt);
    if (dtype == CAS_BF16)
      adam_kernel<true><<<grid, kAdamThreads, 0, st>>>(batch, cfg.lr, cfg.beta1, cfg.beta2, cfg.eps, cfg.zero_grad);
    else
      adam_kernel<false><<<grid, kAdamThreads, 0, st>>>(batch, cfg.lr, cfg.beta1, cfg.beta2, cfg.eps, cfg.zero_grad);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "adam_kernel launch");
  }
  return CAS_OK;
}

template <bool BF16>
__global__ void __launch_bounds__(256)
refresh_kernel(const float* __restrict__ pK, const float* __restrict__ pV, void* wK, void* wV,
               float* __restrict__ gK, float* __restrict__ gV, int64_t n) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x * 4;
  for (int64_t i = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) * 4; i < n; i += stride) {
    store_work4(wK, i, ld4(pK + i), BF16);
    store_work4(wV, i, ld4(pV + i), BF16);
  }
}

int launch_refresh(float* pK, float* pV, void* wK, void* wV, float* gK, float* gV, int64_t n, int dtype,
                   cudaStream_t st) {
  if (n <= 0) return CAS_OK;
  int64_t gx = (n / 4 + 255) / 256;
  if (gx > 148 * 8) gx = 148 * 8;
  if (dtype == CAS_BF16) refresh_kernel<true><<<(unsigned)gx, 256, 0, st>>>(pK, pV, wK, wV, gK, gV, n);
  else refresh_kernel<false><<<(unsigned)gx, 256, 0, st>>>(pK, pV, wK, wV, gK, gV, n);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return cuda_fail(e, "refresh_kernel launch");
  return CAS_OK;
}

// Zero the gradient rows of many (small) slots in ONE launch: the descriptors travel as kernel parameters, like Adam's
// (a cudaMemsetAsync per slot costs more than the attention itself when the cartridges are 16-64 tokens long).
__global__ void __launch_bounds__(256)
zero_slots_kernel(const __grid_constant__ ZeroBatch batch) {
  const ZeroDesc& d = batch.d[blockIdx.y];
  const float4 z = make_float4(0.f, 0.f, 0.f, 0.f);
  for (int64_t i = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) * 4; i < d.n; i += (int64_t)gridDim.x * blockDim.x * 4) {
    st4(d.a + i, z);
    st4(d.b + i, z);
  }
}

int launch_zero_slots(const ZeroDesc* h, int n, cudaStream_t st) {
  for (int i0 = 0; i0 < n; i0 += kZeroBatch) {
    const int cnt = std::min(kZeroBatch, n - i0);
    ZeroBatch batch;
    int64_t mx = 0;
    for (int i = 0; i < cnt; ++i) { batch.d[i] = h[i0 + i]; mx = std::max(mx, h[i0 + i].n); }
    if (mx <= 0) continue;
    const int64_t gx = std::min<int64_t>((mx / 4 + 255) / 256, 148 * 4);
    zero_slots_kernel<<<dim3((unsigned)gx, (unsigned)cnt), 256, 0, st>>>(batch);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "zero_slots_kernel launch");
  }
  return CAS_OK;
}

int launch_zero(float* p, int64_t n, cudaStream_t st) {
  cudaError_t e = cudaMemsetAsync(p, 0, (size_t)n * 4, st);
  if (e != cudaSuccess) return cuda_fail(e, "zero");
  return CAS_OK;
}

}  // namespace cas
