// CUDA-core (SIMT) prefix attention, forward and backward, fp32 accumulate, any storage dtype.
// Serves config 1 (fp32, D=64: tensor cores cannot hold 1e-4 with tf32) and every shape the
// tcgen05 path does not cover; also selectable with cas_set_impl(CAS_IMPL_SIMT).
//
// Definition implemented: include/cas.h cas_prefix_attn_fwd / _bwd.
// Mapping: 128 threads = 32 rows x 4 lanes; a lane owns the float4 columns {c, c+4, c+8, ...} of
// its row so that smem tile reads are conflict-free broadcasts.  KV (fwd, dQ) or query rows
// (dK/dV) stream through shared memory in 32-row tiles read IN PLACE from the pool through the
// slot table.  dK/dV are KV-stationary: one block owns 32 keys of one KV head and walks the
// inverted table, so each gradient element is written once, without atomics.
#include "cas_internal.h"

namespace cas {

template <typename T> struct Io;
template <> struct Io<float> {
  static __device__ __forceinline__ float4 ld4(const float* p) { return *reinterpret_cast<const float4*>(p); }
  static __device__ __forceinline__ void st4(float* p, float4 v) { *reinterpret_cast<float4*>(p) = v; }
};
template <> struct Io<__nv_bfloat16> {
  static __device__ __forceinline__ float4 ld4(const __nv_bfloat16* p) {
    uint2 u = *reinterpret_cast<const uint2*>(p);
    __nv_bfloat162 a = *reinterpret_cast<__nv_bfloat162*>(&u.x);
    __nv_bfloat162 b = *reinterpret_cast<__nv_bfloat162*>(&u.y);
    float2 fa = __bfloat1622float2(a), fb = __bfloat1622float2(b);
    return make_float4(fa.x, fa.y, fb.x, fb.y);
  }
  static __device__ __forceinline__ void st4(__nv_bfloat16* p, float4 v) {
    __nv_bfloat162 a = __floats2bfloat162_rn(v.x, v.y), b = __floats2bfloat162_rn(v.z, v.w);
    uint2 u;
    u.x = *reinterpret_cast<uint32_t*>(&a);
    u.y = *reinterpret_cast<uint32_t*>(&b);
    *reinterpret_cast<uint2*>(p) = u;
  }
};

__device__ __forceinline__ float quad_sum(float x) {
  x += __shfl_xor_sync(0xffffffffu, x, 1);
  x += __shfl_xor_sync(0xffffffffu, x, 2);
  return x;
}
__device__ __forceinline__ float dot4(float4 a, float4 b) { return a.x * b.x + a.y * b.y + a.z * b.z + a.w * b.w; }
__device__ __forceinline__ void fma4(float4& acc, float s, float4 v) {
  acc.x += s * v.x; acc.y += s * v.y; acc.z += s * v.z; acc.w += s * v.w;
}

struct SimtTab {
  const int32_t *seq_off, *sel_off, *sel_base, *sel_len, *inv_off, *inv_seq;
  const FwdItem* items;
  const BwdItem* bitems;
};

constexpr int TR = 32;   // rows per tile

// Load a [TR x D] tile (rows beyond n_valid are zero-filled) from a [tokens, H, D] tensor.
template <typename T, int D>
__device__ __forceinline__ void load_tile(float* sm, const T* base, int64_t tok0, int n_valid, int H, int head) {
  constexpr int V4 = D / 4;
  for (int i = threadIdx.x; i < TR * V4; i += blockDim.x) {
    const int r = i / V4, c = i % V4;
    float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
    if (r < n_valid) v = Io<T>::ld4(base + ((tok0 + r) * H + head) * D + c * 4);
    reinterpret_cast<float4*>(sm)[i] = v;
  }
}

// ------------------------------------------------------------------------------------------ fwd
// MODE 0: forward (O, LSE).  MODE 1: dQ (needs dO, LSE, delta).
template <typename T, int D, int MODE>
__global__ void __launch_bounds__(128)
simt_rowwise_kernel(SimtTab tab, const T* __restrict__ Q, const T* __restrict__ poolK, const T* __restrict__ poolV,
                    const T* __restrict__ Ks, const T* __restrict__ Vs, const T* __restrict__ dO,
                    const float* __restrict__ LSE_in, const float* __restrict__ delta, T* __restrict__ Out,
                    float* __restrict__ LSE_out, int Hq, int Hkv, float scale) {
  constexpr int NV = D / 16;
  __shared__ float sK[TR * D];
  __shared__ float sV[TR * D];
  const FwdItem it = tab.items[blockIdx.x];
  const int h = blockIdx.y, g = h / (Hq / Hkv);
  const int r = threadIdx.x >> 2, c = threadIdx.x & 3;
  const int t0 = tab.seq_off[it.seq];
  const int row = it.row0 + r;                 // row inside the sequence
  const bool row_ok = r < it.rows;
  const int64_t t = t0 + (row_ok ? row : it.row0);

  float4 q[NV], acc[NV], go[NV];
#pragma unroll
  for (int i = 0; i < NV; ++i) {
    q[i] = Io<T>::ld4(Q + (t * Hq + h) * D + (c + 4 * i) * 4);
    acc[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    if (MODE == 1) go[i] = Io<T>::ld4(dO + (t * Hq + h) * D + (c + 4 * i) * 4);
  }
  float m = -INFINITY, l = 0.f;
  float lse = 0.f, dl = 0.f;
  if (MODE == 1) { lse = LSE_in[t * Hq + h]; dl = delta[t * Hq + h]; }

  auto process = [&](const T* Kb, const T* Vb, int64_t tok0, int nkeys, int causal_first) {
    // causal_first >= 0: key index inside the sequence of the tile's first key (self tile)
    __syncthreads();
    load_tile<T, D>(sK, Kb, tok0, nkeys, Hkv, g);
    load_tile<T, D>(sV, Vb, tok0, nkeys, Hkv, g);
    __syncthreads();
    int nvis = nkeys;
    if (causal_first >= 0) nvis = min(nkeys, row - causal_first + 1);   // may be <= 0
    if (MODE == 0) {
      float s[TR];
      float mt = -INFINITY;
#pragma unroll
      for (int j = 0; j < TR; ++j) {
        float p = 0.f;
#pragma unroll
        for (int i = 0; i < NV; ++i) p += dot4(q[i], reinterpret_cast<const float4*>(sK)[j * (D / 4) + c + 4 * i]);
        p = quad_sum(p) * scale;
        s[j] = (j < nvis) ? p : -INFINITY;
        mt = fmaxf(mt, s[j]);
      }
      const float mn = fmaxf(m, mt);
      if (mn > -INFINITY) {
        const float corr = expf(m - mn);
        l *= corr;
#pragma unroll
        for (int i = 0; i < NV; ++i) { acc[i].x *= corr; acc[i].y *= corr; acc[i].z *= corr; acc[i].w *= corr; }
#pragma unroll
        for (int j = 0; j < TR; ++j) {
          const float p = expf(s[j] - mn);
          l += p;
#pragma unroll
          for (int i = 0; i < NV; ++i) fma4(acc[i], p, reinterpret_cast<const float4*>(sV)[j * (D / 4) + c + 4 * i]);
        }
        m = mn;
      }
    } else {
#pragma unroll 4
      for (int j = 0; j < TR; ++j) {
        float s = 0.f, dp = 0.f;
#pragma unroll
        for (int i = 0; i < NV; ++i) {
          s += dot4(q[i], reinterpret_cast<const float4*>(sK)[j * (D / 4) + c + 4 * i]);
          dp += dot4(go[i], reinterpret_cast<const float4*>(sV)[j * (D / 4) + c + 4 * i]);
        }
        s = quad_sum(s) * scale;
        dp = quad_sum(dp);
        const float p = (j < nvis) ? expf(s - lse) : 0.f;
        const float ds = p * (dp - dl);
#pragma unroll
        for (int i = 0; i < NV; ++i) fma4(acc[i], ds, reinterpret_cast<const float4*>(sK)[j * (D / 4) + c + 4 * i]);
      }
    }
  };

  for (int k = tab.sel_off[it.seq]; k < tab.sel_off[it.seq + 1]; ++k) {
    const int base = tab.sel_base[k], len = tab.sel_len[k];
    for (int j = 0; j < len; j += TR) process(poolK, poolV, base + j, min(TR, len - j), -1);
  }
  if (Ks != nullptr) {
    const int last = it.row0 + it.rows - 1;    // keys 0..last are visible to some row of the block
    for (int j = 0; j <= last; j += TR) process(Ks, Vs, (int64_t)t0 + j, min(TR, last + 1 - j), j);
  }
  if (!row_ok) return;
  if (MODE == 0) {
    const float inv = 1.f / l;
#pragma unroll
    for (int i = 0; i < NV; ++i) {
      float4 o = make_float4(acc[i].x * inv, acc[i].y * inv, acc[i].z * inv, acc[i].w * inv);
      Io<T>::st4(Out + (t * Hq + h) * D + (c + 4 * i) * 4, o);
    }
    if (c == 0) LSE_out[t * Hq + h] = m + logf(l);
  } else {
#pragma unroll
    for (int i = 0; i < NV; ++i) {
      float4 o = make_float4(acc[i].x * scale, acc[i].y * scale, acc[i].z * scale, acc[i].w * scale);
      Io<T>::st4(Out + (t * Hq + h) * D + (c + 4 * i) * 4, o);
    }
  }
}

// delta[t,h] = sum_d dO*O   (B1).  One warp per (t,h).
template <typename T>
__global__ void delta_kernel(const T* __restrict__ O, const T* __restrict__ dO, float* __restrict__ delta,
                             int64_t n_rows, int D) {
  const int64_t w = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  if (w >= n_rows) return;
  float s = 0.f;
  for (int d = lane * 4; d < D; d += 128) s += dot4(Io<T>::ld4(O + w * D + d), Io<T>::ld4(dO + w * D + d));
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if (lane == 0) delta[w] = s;
}

// ------------------------------------------------------------------------------- dK/dV (B5,B6)
// grid = (4 * n_bwd_items, Hkv): block owns 32 keys of a 128-key tile for one KV head.
template <typename T, int D>
__global__ void __launch_bounds__(128)
simt_dkdv_kernel(SimtTab tab, const T* __restrict__ Q, const T* __restrict__ poolK, const T* __restrict__ poolV,
                 const T* __restrict__ Ks, const T* __restrict__ Vs, const T* __restrict__ dO,
                 const float* __restrict__ LSE, const float* __restrict__ delta, float* __restrict__ gradK,
                 float* __restrict__ gradV, T* __restrict__ dKs, T* __restrict__ dVs, int Hq, int Hkv, float scale) {
  constexpr int NV = D / 16;
  __shared__ float sQ[TR * D];
  __shared__ float sG[TR * D];
  __shared__ float sL[TR], sD[TR];
  const BwdItem it = tab.bitems[blockIdx.x >> 2];
  const int sub = (blockIdx.x & 3) * TR;
  if (sub >= it.len) return;
  if (it.kind == 1 && Ks == nullptr) return;
  const int g = blockIdx.y, G = Hq / Hkv;
  const int r = threadIdx.x >> 2, c = threadIdx.x & 3;
  const bool key_ok = sub + r < it.len;
  const int64_t ktok = (int64_t)it.tok + sub + (key_ok ? r : 0);
  const T* Kb = it.kind == 0 ? poolK : Ks;
  const T* Vb = it.kind == 0 ? poolV : Vs;
  float4 k[NV], v[NV], dk[NV], dv[NV];
#pragma unroll
  for (int i = 0; i < NV; ++i) {
    k[i] = Io<T>::ld4(Kb + (ktok * Hkv + g) * D + (c + 4 * i) * 4);
    v[i] = Io<T>::ld4(Vb + (ktok * Hkv + g) * D + (c + 4 * i) * 4);
    dk[i] = dv[i] = make_float4(0.f, 0.f, 0.f, 0.f);
  }
  const int e0 = it.kind == 0 ? tab.inv_off[it.id] : 0;
  const int e1 = it.kind == 0 ? tab.inv_off[it.id + 1] : 1;
  for (int e = e0; e < e1; ++e) {
    const int b = it.kind == 0 ? tab.inv_seq[e] : it.id;
    const int t0 = tab.seq_off[b], lq = tab.seq_off[b + 1] - t0;
    // self tile: only rows >= key index matter; key index inside the sequence:
    const int kidx = it.kind == 1 ? (it.tok - t0) + sub + r : -1;
    const int row_begin = it.kind == 1 ? ((it.tok - t0) + sub) / TR * TR : 0;
    for (int h = g * G; h < (g + 1) * G; ++h) {
      for (int r0 = row_begin; r0 < lq; r0 += TR) {
        const int nrow = min(TR, lq - r0);
        __syncthreads();
        load_tile<T, D>(sQ, Q, (int64_t)t0 + r0, nrow, Hq, h);
        load_tile<T, D>(sG, dO, (int64_t)t0 + r0, nrow, Hq, h);
        if (threadIdx.x < TR) {
          const bool ok = threadIdx.x < nrow;
          sL[threadIdx.x] = ok ? LSE[(int64_t)(t0 + r0 + threadIdx.x) * Hq + h] : INFINITY;
          sD[threadIdx.x] = ok ? delta[(int64_t)(t0 + r0 + threadIdx.x) * Hq + h] : 0.f;
        }
        __syncthreads();
#pragma unroll 4
        for (int j = 0; j < TR; ++j) {
          float s = 0.f, dp = 0.f;
#pragma unroll
          for (int i = 0; i < NV; ++i) {
            const float4 qv = reinterpret_cast<const float4*>(sQ)[j * (D / 4) + c + 4 * i];
            const float4 gv = reinterpret_cast<const float4*>(sG)[j * (D / 4) + c + 4 * i];
            s += dot4(k[i], qv);
            dp += dot4(v[i], gv);
          }
          s = quad_sum(s) * scale;
          dp = quad_sum(dp);
          const bool vis = key_ok && (j < nrow) && (kidx < 0 || kidx <= r0 + j);
          const float p = vis ? expf(s - sL[j]) : 0.f;
          const float ds = p * (dp - sD[j]) * scale;
#pragma unroll
          for (int i = 0; i < NV; ++i) {
            fma4(dk[i], ds, reinterpret_cast<const float4*>(sQ)[j * (D / 4) + c + 4 * i]);
            fma4(dv[i], p, reinterpret_cast<const float4*>(sG)[j * (D / 4) + c + 4 * i]);
          }
        }
      }
    }
  }
  if (!key_ok) return;
#pragma unroll
  for (int i = 0; i < NV; ++i) {
    const int64_t o = (ktok * Hkv + g) * D + (c + 4 * i) * 4;
    if (it.kind == 0) {
      float4 a = *reinterpret_cast<float4*>(gradK + o), bq = *reinterpret_cast<float4*>(gradV + o);
      a.x += dk[i].x; a.y += dk[i].y; a.z += dk[i].z; a.w += dk[i].w;
      bq.x += dv[i].x; bq.y += dv[i].y; bq.z += dv[i].z; bq.w += dv[i].w;
      *reinterpret_cast<float4*>(gradK + o) = a;
      *reinterpret_cast<float4*>(gradV + o) = bq;
    } else if (dKs != nullptr) {
      Io<T>::st4(dKs + o, dk[i]);
      Io<T>::st4(dVs + o, dv[i]);
    }
  }
}

size_t simt_bwd_workspace(const cas_slot_table* t, int Hq) { return (size_t)t->T * Hq * 4 + 256; }

template <typename T, int D>
static int run_fwd(const AttnArgs& a) {
  const cas_slot_table* t = a.tab;
  SimtTab tab{t->d_seq_off, t->d_sel_off, t->d_sel_base, t->d_sel_len, t->d_inv_off, t->d_inv_seq,
              t->d_simt_items, t->d_simt_bwd_items};
  dim3 grid((unsigned)t->simt_items.size(), (unsigned)a.Hq);
  simt_rowwise_kernel<T, D, 0><<<grid, 128, 0, a.stream>>>(
      tab, (const T*)a.Q, (const T*)a.L->pool_K, (const T*)a.L->pool_V, (const T*)a.Ks, (const T*)a.Vs,
      nullptr, nullptr, nullptr, (T*)a.O_out, a.LSE_out, a.Hq, a.Hkv, a.scale);
  cudaError_t e = cudaGetLastError();
  return e == cudaSuccess ? CAS_OK : cuda_fail(e, "simt fwd launch");
}

template <typename T, int D>
static int run_bwd(const AttnArgs& a) {
  const cas_slot_table* t = a.tab;
  SimtTab tab{t->d_seq_off, t->d_sel_off, t->d_sel_base, t->d_sel_len, t->d_inv_off, t->d_inv_seq,
              t->d_simt_items, t->d_simt_bwd_items};
  float* delta = (float*)a.workspace;
  const int64_t rows = (int64_t)t->T * a.Hq;
  delta_kernel<T><<<(unsigned)((rows * 32 + 255) / 256), 256, 0, a.stream>>>((const T*)a.O, (const T*)a.dO, delta, rows, D);
  dim3 grid((unsigned)t->simt_items.size(), (unsigned)a.Hq);
  simt_rowwise_kernel<T, D, 1><<<grid, 128, 0, a.stream>>>(
      tab, (const T*)a.Q, (const T*)a.L->pool_K, (const T*)a.L->pool_V, (const T*)a.Ks, (const T*)a.Vs,
      (const T*)a.dO, a.LSE_in, delta, (T*)a.dQ, nullptr, a.Hq, a.Hkv, a.scale);
  dim3 grid2((unsigned)(4 * t->simt_bwd_items.size()), (unsigned)a.Hkv);
  simt_dkdv_kernel<T, D><<<grid2, 128, 0, a.stream>>>(
      tab, (const T*)a.Q, (const T*)a.L->pool_K, (const T*)a.L->pool_V, (const T*)a.Ks, (const T*)a.Vs,
      (const T*)a.dO, a.LSE_in, delta, a.L->grad_K, a.L->grad_V, (T*)a.dKs, (T*)a.dVs, a.Hq, a.Hkv, a.scale);
  cudaError_t e = cudaGetLastError();
  return e == cudaSuccess ? CAS_OK : cuda_fail(e, "simt bwd launch");
}

#define CAS_SIMT_DISPATCH(FN)                                                         \
  if (a.dtype == CAS_F32) {                                                           \
    switch (a.D) {                                                                    \
      case 32: return FN<float, 32>(a);                                               \
      case 64: return FN<float, 64>(a);                                               \
      case 96: return FN<float, 96>(a);                                               \
      case 128: return FN<float, 128>(a);                                             \
    }                                                                                 \
  } else {                                                                            \
    switch (a.D) {                                                                    \
      case 32: return FN<__nv_bfloat16, 32>(a);                                       \
      case 64: return FN<__nv_bfloat16, 64>(a);                                       \
      case 96: return FN<__nv_bfloat16, 96>(a);                                       \
      case 128: return FN<__nv_bfloat16, 128>(a);                                     \
    }                                                                                 \
  }                                                                                   \
  set_error("unsupported head dim %d", a.D);                                          \
  return CAS_ERR_SHAPE;

int simt_attn_fwd(const AttnArgs& a) { CAS_SIMT_DISPATCH(run_fwd) }
int simt_attn_bwd(const AttnArgs& a) { CAS_SIMT_DISPATCH(run_bwd) }

}  // namespace cas
