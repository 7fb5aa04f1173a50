// RoPE with the cartridge position offset ("query token position IDs
// must be offset by the total number of active cartridge KV tokens"; RoFormer Eq. 34).  In place on a
// packed [T, H, D] tensor (Q or K_self, before cas_prefix_attn_fwd; inverse = 1 is the transpose, i.e. the
// backward pass applied to dQ / dK_self).
//
// Roofline: HBM (read + write of X).  One thread owns one 16-byte chunk position of a token row and
// walks a group of 4 heads: the cos/sin of its dimension pairs are computed ONCE per token in double precision
// (position ids reach 10^5..10^6 with large pools, where a float angle is off by 10^-2 rad) and reused
// for the heads of the group, so the kernel stays memory-bound.  Consecutive lanes hold consecutive chunks of the
// same head row: every access is a fully used 128/256-byte segment.  The per-sequence (first token,
// position offset) table travels as kernel parameters.
#include <algorithm>
#include <cmath>

#include "cas_internal.h"

namespace cas {

constexpr int kRopeSeqs = 128;    // sequences per launch (the table is a kernel parameter: keep it small)
constexpr int kRopeHeads = 4;     // heads per thread (the angles of a token are recomputed per group of heads)
struct RopeSeqs {
  int32_t seq_off[kRopeSeqs + 1];   // packed-token offsets of this launch's sequences
  int64_t pos_off[kRopeSeqs];
  double theta[128];                // base^(-2k/D), k < D/2 <= 128, formed in double on the host
  int32_t n;
};

template <typename T> struct Vec16;                       // 16 bytes of T
template <> struct Vec16<float> { static constexpr int N = 4; };
template <> struct Vec16<__nv_bfloat16> { static constexpr int N = 8; };

template <typename T>
__device__ __forceinline__ void load16(const T* p, float* f) {
  const uint4 u = *reinterpret_cast<const uint4*>(p);
  if constexpr (sizeof(T) == 4) {
    f[0] = __uint_as_float(u.x); f[1] = __uint_as_float(u.y); f[2] = __uint_as_float(u.z); f[3] = __uint_as_float(u.w);
  } else {
    const uint32_t w[4] = {u.x, u.y, u.z, u.w};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const float2 v = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&w[i]));
      f[2 * i] = v.x;
      f[2 * i + 1] = v.y;
    }
  }
}
template <typename T>
__device__ __forceinline__ void store16(T* p, const float* f) {
  uint4 u;
  if constexpr (sizeof(T) == 4) {
    u = make_uint4(__float_as_uint(f[0]), __float_as_uint(f[1]), __float_as_uint(f[2]), __float_as_uint(f[3]));
  } else {
    uint32_t w[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const __nv_bfloat162 v = __floats2bfloat162_rn(f[2 * i], f[2 * i + 1]);
      w[i] = *reinterpret_cast<const uint32_t*>(&v);
    }
    u = make_uint4(w[0], w[1], w[2], w[3]);
  }
  *reinterpret_cast<uint4*>(p) = u;
}

// LAYOUT 0: pairs (2k, 2k+1): a thread owns N consecutive dims = N/2 pairs of one chunk.
// LAYOUT 1: pairs (k, k + D/2): a thread owns chunk c of the first half and the same chunk of the second
//           half = N pairs.
template <typename T, int LAYOUT>
__global__ void __launch_bounds__(256)
rope_kernel(const __grid_constant__ RopeSeqs sq, T* __restrict__ X, int H, int D, int inverse) {
  constexpr int N = Vec16<T>::N;
  constexpr int P = LAYOUT == 0 ? N / 2 : N;                  // pairs per thread
  const int chunks = LAYOUT == 0 ? D / N : D / (2 * N);       // threads per token
  // the parameter tables are indexed per lane below: stage them in shared memory once per block (a
  // constant-bank read with 32 different addresses is replayed 32 times)
  extern __shared__ __align__(16) unsigned char s_raw[];      // [128] theta | [n] pos_off | [n+1] seq_off
  double* s_theta = reinterpret_cast<double*>(s_raw);
  int64_t* s_pos = reinterpret_cast<int64_t*>(s_raw + 1024);
  int32_t* s_off = reinterpret_cast<int32_t*>(s_raw + 1024 + 8 * sq.n);
  for (int i = threadIdx.x; i <= sq.n; i += blockDim.x) s_off[i] = sq.seq_off[i];
  for (int i = threadIdx.x; i < sq.n; i += blockDim.x) s_pos[i] = sq.pos_off[i];
  for (int i = threadIdx.x; i < D / 2; i += blockDim.x) s_theta[i] = sq.theta[i];
  __syncthreads();
  const int64_t gid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int c = (int)(gid % chunks);
  const int64_t tl = gid / chunks;                            // token inside this launch's range
  const int t_first = s_off[0], n_tok = s_off[sq.n] - t_first;
  if (tl >= n_tok) return;
  const int t = t_first + (int)tl;
  int lo = 0, hi = sq.n - 1;                                  // sequence of token t
  while (lo < hi) {
    const int mid = (lo + hi + 1) >> 1;
    if (s_off[mid] <= t) lo = mid; else hi = mid - 1;
  }
  const double m = (double)(s_pos[lo] + (int64_t)(t - s_off[lo]));
  float cs[P], sn[P];
#pragma unroll
  for (int i = 0; i < P; ++i) {
    const int k = c * P + i;                                  // pair index 0..D/2-1
    // angle in double (m * theta reaches 10^5..10^6 rad), reduced to [-pi, pi] in double, then the float
    // sincos: absolute error ~1e-7, the resolution of the fp32 products below
    const double a = m * s_theta[k];
    const double r = fma(-rint(a * 0.15915494309189535), 6.283185307179586, a);
    float s, co;
    sincosf((float)r, &s, &co);
    cs[i] = co;
    sn[i] = inverse ? -s : s;
  }
  // blockIdx.y owns a group of kRopeHeads heads: enough threads to fill the machine and kRopeHeads
  // independent 16-byte loads in flight per thread (the head loop is unrolled)
  const int h0 = blockIdx.y * kRopeHeads, nh = min(H - h0, kRopeHeads);
  T* row = X + ((int64_t)t * H + h0) * D;
  for (int hh = 0; hh < nh; ++hh, row += D) {
    if constexpr (LAYOUT == 0) {
      float f[N];
      load16(row + c * N, f);
#pragma unroll
      for (int i = 0; i < P; ++i) {
        const float a = f[2 * i], b = f[2 * i + 1];
        f[2 * i] = a * cs[i] - b * sn[i];
        f[2 * i + 1] = a * sn[i] + b * cs[i];
      }
      store16(row + c * N, f);
    } else {
      float fa[N], fb[N];
      load16(row + c * N, fa);
      load16(row + D / 2 + c * N, fb);
#pragma unroll
      for (int i = 0; i < P; ++i) {
        const float a = fa[i], b = fb[i];
        fa[i] = a * cs[i] - b * sn[i];
        fb[i] = a * sn[i] + b * cs[i];
      }
      store16(row + c * N, fa);
      store16(row + D / 2 + c * N, fb);
    }
  }
}

template <typename T>
static int rope_launch(const RopeSeqs& sq, void* X, int H, int D, int layout, int inverse, cudaStream_t st) {
  constexpr int N = Vec16<T>::N;
  const int chunks = layout == 0 ? D / N : D / (2 * N);
  const int64_t n_thr = (int64_t)(sq.seq_off[sq.n] - sq.seq_off[0]) * chunks;
  if (n_thr <= 0) return CAS_OK;
  const dim3 grid((unsigned)((n_thr + 255) / 256), (unsigned)((H + kRopeHeads - 1) / kRopeHeads));
  const size_t smem = 1024 + 8 * (size_t)sq.n + 4 * ((size_t)sq.n + 1);
  if (layout == 0) rope_kernel<T, 0><<<grid, 256, smem, st>>>(sq, (T*)X, H, D, inverse);
  else rope_kernel<T, 1><<<grid, 256, smem, st>>>(sq, (T*)X, H, D, inverse);
  cudaError_t err = cudaGetLastError();
  return err == cudaSuccess ? CAS_OK : cuda_fail(err, "rope_kernel launch");
}

// ---- fused path: a cos/sin table per packed batch, shared by every head and every layer -----------------------
// cs[t][k] = (cos, sin)(m_t * base^(-2k/D)), angles formed and reduced in double as above.  The forward kernel
// rotates a Q tile in shared memory with it, dq_convert_kernel applies the transpose to dQ; K_self / dK_self (1/G of
// the bytes) go through rope_table_rotate_kernel.
__global__ void __launch_bounds__(256)
rope_table_kernel(const __grid_constant__ RopeSeqs sq, float2* __restrict__ cs, int half) {
  const int64_t gid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int k = (int)(gid % half);
  const int64_t tl = gid / half;
  const int t_first = sq.seq_off[0], n_tok = sq.seq_off[sq.n] - t_first;
  if (tl >= n_tok) return;
  const int t = t_first + (int)tl;
  int lo = 0, hi = sq.n - 1;
  while (lo < hi) {
    const int mid = (lo + hi + 1) >> 1;
    if (sq.seq_off[mid] <= t) lo = mid; else hi = mid - 1;
  }
  const double m = (double)(sq.pos_off[lo] + (int64_t)(t - sq.seq_off[lo]));
  const double a = m * sq.theta[k];
  const double r = fma(-rint(a * 0.15915494309189535), 6.283185307179586, a);
  float s, co;
  sincosf((float)r, &s, &co);
  cs[(int64_t)t * half + k] = make_float2(co, s);
}

// dst[t, h, :] = R(t) src[t, h, :] (or its transpose), bf16, D = 128; one thread = one 16-byte chunk position of a
// row (8 chunks per half): layout 0 rotates the four pairs inside each of its two chunks, layout 1 pairs chunk c of
// the first half with chunk c of the second.
__global__ void __launch_bounds__(256)
rope_table_rotate_kernel(const __nv_bfloat16* __restrict__ src, __nv_bfloat16* __restrict__ dst,
                         const float2* __restrict__ cs, int64_t n_rows, int H, int layout, int inverse) {
  const int64_t gid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int c = (int)(gid & 7);
  const int64_t row = gid >> 3;                      // (t, h)
  if (row >= n_rows) return;
  const int64_t t = row / H;
  const float2* tab = cs + t * 64;
  float fa[8], fb[8];
  load16(src + row * 128 + c * 8, fa);
  load16(src + row * 128 + 64 + c * 8, fb);
  const float sg = inverse ? -1.f : 1.f;
  if (layout == 0) {
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const float2 w0 = tab[4 * c + i], w1 = tab[32 + 4 * c + i];
      const float a0 = fa[2 * i], b0 = fa[2 * i + 1], a1 = fb[2 * i], b1 = fb[2 * i + 1];
      fa[2 * i] = a0 * w0.x - b0 * sg * w0.y;
      fa[2 * i + 1] = a0 * sg * w0.y + b0 * w0.x;
      fb[2 * i] = a1 * w1.x - b1 * sg * w1.y;
      fb[2 * i + 1] = a1 * sg * w1.y + b1 * w1.x;
    }
  } else {
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const float2 w = tab[8 * c + i];
      const float a = fa[i], b = fb[i];
      fa[i] = a * w.x - b * sg * w.y;
      fb[i] = a * sg * w.y + b * w.x;
    }
  }
  store16(dst + row * 128 + c * 8, fa);
  store16(dst + row * 128 + 64 + c * 8, fb);
}

int rope_table_rotate(const void* src, void* dst, const float* cs, int64_t T, int H, int layout, int inverse,
                      cudaStream_t st) {
  const int64_t n_rows = T * H;
  if (n_rows <= 0) return CAS_OK;
  rope_table_rotate_kernel<<<(unsigned)((n_rows * 8 + 255) / 256), 256, 0, st>>>(
      (const __nv_bfloat16*)src, (__nv_bfloat16*)dst, (const float2*)cs, n_rows, H, layout, inverse);
  cudaError_t err = cudaGetLastError();
  return err == cudaSuccess ? CAS_OK : cuda_fail(err, "rope_table_rotate_kernel launch");
}

}  // namespace cas

extern "C" int cas_rope_table(int32_t B, const int32_t* seq_off, const int64_t* pos_off, int32_t D, double base,
                              float* cs, void* stream) {
  using namespace cas;
  if (!seq_off || !pos_off || !cs || B < 1) { set_error("null / empty args"); return CAS_ERR_INVALID_ARG; }
  if (!(base > 1.0)) { set_error("RoPE base must be > 1"); return CAS_ERR_INVALID_ARG; }
  if (D < 2 || D > 256 || D % 2) { set_error("D = %d", D); return CAS_ERR_SHAPE; }
  if (seq_off[0] != 0) { set_error("offsets must start at 0"); return CAS_ERR_INVALID_ARG; }
  for (int b = 0; b < B; ++b) {
    if (seq_off[b + 1] < seq_off[b]) { set_error("seq_off not monotone"); return CAS_ERR_INVALID_ARG; }
    if (pos_off[b] < 0) { set_error("negative position offset"); return CAS_ERR_INVALID_ARG; }
  }
  for (int b0 = 0; b0 < B; b0 += kRopeSeqs) {
    RopeSeqs sq;
    for (int k = 0; k < D / 2; ++k) sq.theta[k] = pow(base, -2.0 * (double)k / (double)D);
    sq.n = std::min(kRopeSeqs, B - b0);
    for (int i = 0; i <= sq.n; ++i) sq.seq_off[i] = seq_off[b0 + i];
    for (int i = 0; i < sq.n; ++i) sq.pos_off[i] = pos_off[b0 + i];
    const int64_t n_thr = (int64_t)(sq.seq_off[sq.n] - sq.seq_off[0]) * (D / 2);
    if (n_thr <= 0) continue;
    rope_table_kernel<<<(unsigned)((n_thr + 255) / 256), 256, 0, (cudaStream_t)stream>>>(sq, (float2*)cs, D / 2);
    cudaError_t err = cudaGetLastError();
    if (err != cudaSuccess) return cuda_fail(err, "rope_table_kernel launch");
  }
  return CAS_OK;
}

extern "C" int cas_rope_apply(int32_t dtype, int32_t B, const int32_t* seq_off, const int64_t* pos_off, int32_t H,
                              int32_t D, double base, int32_t layout, int32_t inverse, void* X, void* stream) {
  using namespace cas;
  if (!seq_off || !pos_off || !X || B < 1 || H < 1) { set_error("null / empty args"); return CAS_ERR_INVALID_ARG; }
  if (dtype != CAS_BF16 && dtype != CAS_F32) { set_error("bad dtype"); return CAS_ERR_INVALID_ARG; }
  if (layout != 0 && layout != 1) { set_error("layout must be 0 (interleaved) or 1 (half-split)"); return CAS_ERR_INVALID_ARG; }
  if (!(base > 1.0)) { set_error("RoPE base must be > 1"); return CAS_ERR_INVALID_ARG; }
  const int n16 = dtype == CAS_BF16 ? 8 : 4;
  if (D < 2 || D > 256 || D % (layout == 0 ? n16 : 2 * n16)) { set_error("D = %d is not a whole number of 16-byte chunks per half", D); return CAS_ERR_SHAPE; }
  if (seq_off[0] != 0) { set_error("offsets must start at 0"); return CAS_ERR_INVALID_ARG; }
  for (int b = 0; b < B; ++b) {
    if (seq_off[b + 1] < seq_off[b]) { set_error("seq_off not monotone"); return CAS_ERR_INVALID_ARG; }
    if (pos_off[b] < 0) { set_error("negative position offset"); return CAS_ERR_INVALID_ARG; }
  }
  for (int b0 = 0; b0 < B; b0 += kRopeSeqs) {
    RopeSeqs sq;
    for (int k = 0; k < D / 2; ++k) sq.theta[k] = pow(base, -2.0 * (double)k / (double)D);
    sq.n = std::min(kRopeSeqs, B - b0);
    for (int i = 0; i <= sq.n; ++i) sq.seq_off[i] = seq_off[b0 + i];
    for (int i = 0; i < sq.n; ++i) sq.pos_off[i] = pos_off[b0 + i];
    const int rc = dtype == CAS_BF16
                       ? rope_launch<__nv_bfloat16>(sq, X, H, D, layout, inverse, (cudaStream_t)stream)
                       : rope_launch<float>(sq, X, H, D, layout, inverse, (cudaStream_t)stream);
    if (rc) return rc;
  }
  return CAS_OK;
}
