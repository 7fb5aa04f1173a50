// Prefix-attention BACKWARD on tcgen05 + TMEM + TMA, bf16, head_dim 128.
//
// Definition: include/cas.h cas_prefix_attn_bwd (PAPER.md:44 only the cartridge K/V receive
// gradients; :176 all active cartridges are back-propagated simultaneously; :75 unselected ones get
// none).  KV-stationary: one CTA owns one 128-key tile of one KV head -- a tile of a cartridge slot
// (read in place from the pool) or of a sequence's own keys -- and walks, through the INVERTED slot
// table, every (sequence that selected the slot) x (query head of the group) x (128-row Q tile).
// dK/dV of the tile accumulate in TMEM over that whole loop and are written ONCE ("+=" into the
// slot's fp32 gradient buffer, no atomics, deterministic).  dQ tiles are reduced into an fp32
// scratch with vector red.global.add and converted to bf16 (x scale) by a small epilogue kernel.
//
// Per inner iteration i (Q tile, dO tile, LSE, delta of 128 query rows), five MMAs, keys on lanes:
//   S^T  = K  Q^T        (SS)            dP^T = V  dO^T      (SS)
//   dV  += P^T dO        (P^T from TMEM) dK  += dS^T Q       (dS^T from SMEM, K-major)
//   dQ   = dS  K         (the same dS^T bytes in SMEM read as an MN-major A operand)
// TMEM (512 cols): [S^T / P^T] [dP^T / dQ] [dV] [dK].   SMEM (224 KB): K,V | 2 x (Q,dO) | dS^T.
// Warps: 0-3 softmax-backward (thread = key), 4-7 dQ reducers (thread = query), 8 TMA, 9 MMA.
// Issue order:  dV(i)  S(i+1)  dK(i) dQ(i)  [dQ drained]  dP(i+1)   -- exp of tile i+1 overlaps
// dK/dQ of tile i; the dQ drain overlaps the exp as well.
#include "cas_sm100.cuh"
#include "cas_tc_common.cuh"

namespace cas {
using namespace sm100;

constexpr float kLog2e = 1.4426950408889634f;

// delta[t,h] = sum_d dO*O (B1), stored head-major and padded per sequence to whole 128-row tiles
// (so each (head, Q tile) is one aligned 512-byte run): auxD[h][tile*128 + r]; auxL = LSE*log2(e).
__global__ void __launch_bounds__(256)
bwd_prep_kernel(const __nv_bfloat16* __restrict__ O, const __nv_bfloat16* __restrict__ dO,
                const float* __restrict__ LSE, const int32_t* __restrict__ seq_off,
                const int32_t* __restrict__ qtile_off, int B, int Hq, int64_t aux_stride,
                float* __restrict__ auxL, float* __restrict__ auxD, int64_t n_rows) {
  const int64_t w = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;   // (t, h) row
  const int lane = threadIdx.x & 31;
  if (w >= n_rows) return;
  const int t = (int)(w / Hq), h = (int)(w % Hq);
  const uint2 a = *reinterpret_cast<const uint2*>(O + w * 128 + lane * 4);
  const uint2 b = *reinterpret_cast<const uint2*>(dO + w * 128 + lane * 4);
  const float2 a0 = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&a.x));
  const float2 a1 = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&a.y));
  const float2 b0 = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&b.x));
  const float2 b1 = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&b.y));
  float s = a0.x * b0.x + a0.y * b0.y + a1.x * b1.x + a1.y * b1.y;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if (lane == 0) {
    int lo = 0, hi = B - 1;                      // sequence of token t
    while (lo < hi) {
      const int mid = (lo + hi + 1) >> 1;
      if (seq_off[mid] <= t) lo = mid; else hi = mid - 1;
    }
    const int64_t pos = (int64_t)h * aux_stride + (int64_t)qtile_off[lo] * 128 + (t - seq_off[lo]);
    auxD[pos] = s;
    auxL[pos] = LSE[w] * kLog2e;
  }
}

// dQ = bf16(scale * dQ_acc)
__global__ void __launch_bounds__(256)
dq_convert_kernel(const float* __restrict__ acc, __nv_bfloat16* __restrict__ dQ, float scale, int64_t n4) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += stride) {
    const float4 v = reinterpret_cast<const float4*>(acc)[i];
    uint2 u;
    u.x = pack_bf16(v.x * scale, v.y * scale);
    u.y = pack_bf16(v.z * scale, v.w * scale);
    reinterpret_cast<uint2*>(dQ)[i] = u;
  }
}

// ------------------------------------------------------------------------------- main kernel
constexpr int kBwdThreads = 384;   // warps 10,11 idle: whole warpgroups for setmaxnreg
constexpr uint32_t kT = 32768, kH = 16384;
constexpr uint32_t oK = 0, oV = kT, oQ = 2 * kT, oDO = 4 * kT, oDS = 6 * kT, oAuxL = 7 * kT, oAuxD = 7 * kT + 1024,
                   oBar = 7 * kT + 2048;
constexpr uint32_t kBwdSmem = oBar + 256;
enum { C_KV = 0, C_QF = 1, C_DOF = 3, C_STE = 5, C_SF = 7, C_DPF = 8, C_PF = 9, C_DSF = 10, C_DQF = 11, C_DQD = 12,
       C_DONE = 13, C_N = 14 };

struct BwdParams {
  const int32_t *seq_off, *inv_off, *inv_seq, *qtile_off;
  const BwdItem* items;
  const float *auxL, *auxD;
  float* dQacc;
  float *gradK, *gradV;
  __nv_bfloat16 *dKs, *dVs;
  int64_t aux_stride;
  int Hq, Hkv, has_self;
  float scale, scale_log2;
};

// Enumerates the inner iterations of an item: for e in inverted list: for h in group: for qt.
struct Walk {
  const BwdParams& p;
  const BwdItem& it;
  int g, G, e, e1, h, qt, b, t0, lq, nqt, qbeg;
  __device__ Walk(const BwdParams& p_, const BwdItem& it_, int g_) : p(p_), it(it_), g(g_) {
    G = p.Hq / p.Hkv;
    e = it.kind == 0 ? p.inv_off[it.id] : 0;
    e1 = it.kind == 0 ? p.inv_off[it.id + 1] : 1;
    load();
    h = g * G;
    qt = qbeg;
  }
  __device__ void load() {
    b = it.kind == 0 ? p.inv_seq[e] : it.id;
    t0 = p.seq_off[b];
    lq = p.seq_off[b + 1] - t0;
    nqt = (lq + 127) >> 7;
    qbeg = it.kind == 1 ? it.jt : 0;
  }
  __device__ int total() const {
    int n = 0;
    for (int x = e; x < e1; ++x) {
      const int bb = it.kind == 0 ? p.inv_seq[x] : it.id;
      const int l = p.seq_off[bb + 1] - p.seq_off[bb];
      n += G * (((l + 127) >> 7) - (it.kind == 1 ? it.jt : 0));
    }
    return n;
  }
  __device__ void next() {
    if (++qt < nqt) return;
    if (++h < (g + 1) * G) { qt = qbeg; return; }
    if (++e < e1) { load(); h = g * G; qt = qbeg; }
  }
  __device__ int tok() const { return t0 + 128 * qt; }                       // first packed token
  __device__ int rows() const { return min(128, lq - 128 * qt); }            // valid query rows
  __device__ int64_t aux() const { return (int64_t)h * p.aux_stride + (int64_t)(p.qtile_off[b] + qt) * 128; }
};

template <int N>
__device__ __forceinline__ void setmaxnreg_inc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(N)); }
template <int N>
__device__ __forceinline__ void setmaxnreg_dec() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(N)); }

__global__ void __launch_bounds__(kBwdThreads, 1)
tc_bwd_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmdO,
              const __grid_constant__ CUtensorMap tmKp, const __grid_constant__ CUtensorMap tmVp,
              const __grid_constant__ CUtensorMap tmKs, const __grid_constant__ CUtensorMap tmVs,
              const BwdParams prm) {
  extern __shared__ __align__(1024) uint8_t smem[];
  const uint32_t sbase = smem_u32(smem);
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + oBar + C_N * 8);
  auto bar = [&](int i) { return sbase + oBar + 8u * i; };
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int g = blockIdx.x % prm.Hkv;
  const BwdItem it = prm.items[blockIdx.x / prm.Hkv];
  if (it.kind == 1 && !prm.has_self) return;     // prefix-only call: no self tiles (block-uniform)

  if (threadIdx.x == 0) {
    if (sbase & 1023u) __trap();
    for (int i = 0; i < C_N; ++i) mbar_init(bar(i), (i == C_PF || i == C_DSF || i == C_DQD) ? 128 : 1);
    fence_mbar_init();
  }
  if (warp == 8) {
    tmem_alloc(smem_u32(tmem_slot), 512);
    tmem_relinquish();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tbase = *tmem_slot;
  const uint32_t tS = tbase, tdP = tbase + 128, tdV = tbase + 256, tdK = tbase + 384;

  if (warp >= 8) {
    setmaxnreg_dec<64>();
    if (warp == 8 && lane == 0) {
      // ================================================================= TMA producer
      const CUtensorMap* mk = it.kind == 0 ? &tmKp : &tmKs;
      const CUtensorMap* mv = it.kind == 0 ? &tmVp : &tmVs;
      mbar_expect_tx(bar(C_KV), 2 * kT);
      tma_load_3d(sbase + oK, mk, bar(C_KV), 0, g, it.tok);
      tma_load_3d(sbase + oK + kH, mk, bar(C_KV), 64, g, it.tok);
      tma_load_3d(sbase + oV, mv, bar(C_KV), 0, g, it.tok);
      tma_load_3d(sbase + oV + kH, mv, bar(C_KV), 64, g, it.tok);
      Walk w(prm, it, g);
      const int n = w.total();
      for (int i = 0; i < n; ++i) {
        const int st = i & 1;
        mbar_wait(bar(C_STE + st), ((i >> 1) & 1) ^ 1);
        mbar_expect_tx(bar(C_QF + st), kT + 512);
        tma_load_3d(sbase + oQ + st * kT, &tmQ, bar(C_QF + st), 0, w.h, w.tok());
        tma_load_3d(sbase + oQ + st * kT + kH, &tmQ, bar(C_QF + st), 64, w.h, w.tok());
        bulk_load(sbase + oAuxL + st * 512, prm.auxL + w.aux(), 512, bar(C_QF + st));
        mbar_expect_tx(bar(C_DOF + st), kT + 512);
        tma_load_3d(sbase + oDO + st * kT, &tmdO, bar(C_DOF + st), 0, w.h, w.tok());
        tma_load_3d(sbase + oDO + st * kT + kH, &tmdO, bar(C_DOF + st), 64, w.h, w.tok());
        bulk_load(sbase + oAuxD + st * 512, prm.auxD + w.aux(), 512, bar(C_DOF + st));
        w.next();
      }
    } else if (warp == 9 && lane == 0) {
      // ================================================================= MMA issuer
      constexpr uint32_t id_kk = make_idesc(128, 128, 0, 0), id_kmn = make_idesc(128, 128, 0, 1),
                         id_mnmn = make_idesc(128, 128, 1, 1);
      Walk w(prm, it, g);
      const int n = w.total();
      auto kmaj = [&](uint32_t base, int kk) { return desc_kmajor(base + (kk >> 2) * kH + (kk & 3) * 32); };
      auto mnmaj = [&](uint32_t base, int kk) { return desc_mnmajor(base + kk * 2048, kH); };
      auto mma_S = [&](int st) {
#pragma unroll
        for (int kk = 0; kk < 8; ++kk) mma_ss(tS, kmaj(sbase + oK, kk), kmaj(sbase + oQ + st * kT, kk), id_kk, kk > 0);
      };
      auto mma_dP = [&](int st) {
#pragma unroll
        for (int kk = 0; kk < 8; ++kk) mma_ss(tdP, kmaj(sbase + oV, kk), kmaj(sbase + oDO + st * kT, kk), id_kk, kk > 0);
      };
      mbar_wait(bar(C_KV), 0);
      mbar_wait(bar(C_QF), 0);
      tc_fence_after();
      mma_S(0);
      mma_commit(bar(C_SF));
      mbar_wait(bar(C_DOF), 0);
      tc_fence_after();
      mma_dP(0);
      mma_commit(bar(C_DPF));
      for (int i = 0; i < n; ++i) {
        const int st = i & 1, st1 = st ^ 1;
        const uint32_t ph1 = ((i + 1) >> 1) & 1;
        mbar_wait(bar(C_PF), i & 1);
        tc_fence_after();
#pragma unroll
        for (int kk = 0; kk < 8; ++kk)     // dV += P^T dO
          mma_ts(tdV, tS + kk * 8, mnmaj(sbase + oDO + st * kT, kk), id_kmn, (i > 0 || kk > 0) ? 1u : 0u);
        if (i + 1 < n) {
          mbar_wait(bar(C_QF + st1), ph1);
          tc_fence_after();
          mma_S(st1);
          mma_commit(bar(C_SF));
        }
        mbar_wait(bar(C_DSF), i & 1);
        tc_fence_after();
#pragma unroll
        for (int kk = 0; kk < 8; ++kk)     // dK += dS^T Q
          mma_ss(tdK, kmaj(sbase + oDS, kk), mnmaj(sbase + oQ + st * kT, kk), id_kmn, (i > 0 || kk > 0) ? 1u : 0u);
#pragma unroll
        for (int kk = 0; kk < 8; ++kk)     // dQ = dS K
          mma_ss(tdP, mnmaj(sbase + oDS, kk), mnmaj(sbase + oK, kk), id_mnmn, kk > 0);
        mma_commit(bar(C_DQF));
        mma_commit(bar(C_STE + st));
        if (i + 1 < n) {
          mbar_wait(bar(C_DOF + st1), ph1);
          mbar_wait(bar(C_DQD), i & 1);
          tc_fence_after();
          mma_dP(st1);
          mma_commit(bar(C_DPF));
        }
      }
      mma_commit(bar(C_DONE));
    }
  } else if (warp < 4) {
    // =================================================================== softmax backward
    setmaxnreg_inc<232>();
    const int k = threadIdx.x;                       // key lane
    const uint32_t lane_base = (uint32_t)(warp * 32) << 16;
    const bool key_ok = k < it.len;
    Walk w(prm, it, g);
    const int n = w.total();
    for (int i = 0; i < n; ++i) {
      const int st = i & 1;
      const uint32_t ph = (i >> 1) & 1;
      const int rows = w.rows();
      // valid query columns: qlo <= q < qhi
      const int qlo = (it.kind == 1 && w.qt == it.jt) ? k : 0;
      const int qhi = key_ok ? rows : 0;
      const float* aL = reinterpret_cast<const float*>(smem + oAuxL + st * 512);
      const float* aD = reinterpret_cast<const float*>(smem + oAuxD + st * 512);
      mbar_wait(bar(C_QF + st), ph);
      mbar_wait(bar(C_SF), i & 1);
      tc_fence_after();
      float p[128];
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        uint32_t s[32];
        tmem_ld32(tS + lane_base + c * 32, s);
        tc_wait_ld();
#pragma unroll
        for (int q = 0; q < 32; ++q) {
          const int qq = c * 32 + q;
          const float e = ex2_approx(__uint_as_float(s[q]) * prm.scale_log2 - aL[qq]);
          p[qq] = (qq >= qlo && qq < qhi) ? e : 0.f;
        }
      }
#pragma unroll
      for (int c = 0; c < 2; ++c) {
        uint32_t pk[32];
#pragma unroll
        for (int q = 0; q < 32; ++q) pk[q] = pack_bf16(p[c * 64 + 2 * q], p[c * 64 + 2 * q + 1]);
        tmem_st32(tS + lane_base + c * 32, pk);
      }
      tc_wait_st();
      tc_fence_before();
      mbar_arrive(bar(C_PF));
      mbar_wait(bar(C_DOF + st), ph);
      mbar_wait(bar(C_DPF), i & 1);
      tc_fence_after();
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        uint32_t d[32];
        tmem_ld32(tdP + lane_base + c * 32, d);
        tc_wait_ld();
#pragma unroll
        for (int q8 = 0; q8 < 4; ++q8) {
          uint32_t pk[4];
#pragma unroll
          for (int x = 0; x < 4; ++x) {
            const int q = q8 * 8 + 2 * x, qq = c * 32 + q;
            const float d0 = p[qq] * (__uint_as_float(d[q]) - aD[qq]);
            const float d1 = p[qq + 1] * (__uint_as_float(d[q + 1]) - aD[qq + 1]);
            pk[x] = pack_bf16(d0, d1);
          }
          const int q0 = c * 32 + q8 * 8;
          const uint32_t addr = sbase + oDS + (q0 >> 6) * kH + k * 128 + ((((q0 >> 3) & 7) ^ (k & 7)) << 4);
          asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(pk[0]), "r"(pk[1]), "r"(pk[2]), "r"(pk[3]) : "memory");
        }
      }
      tc_fence_before();
      fence_proxy_async();
      mbar_arrive(bar(C_DSF));
      w.next();
    }
  } else {
    // =================================================================== dQ reducers
    setmaxnreg_dec<96>();
    const int q = threadIdx.x - 128;                 // query lane
    const uint32_t lane_base = (uint32_t)((warp & 3) * 32) << 16;
    Walk w(prm, it, g);
    const int n = w.total();
    for (int i = 0; i < n; ++i) {
      const bool ok = q < w.rows();
      float* dst = prm.dQacc + ((int64_t)(w.tok() + q) * prm.Hq + w.h) * 128;
      mbar_wait(bar(C_DQF), i & 1);
      tc_fence_after();
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        uint32_t d[32];
        tmem_ld32(tdP + lane_base + c * 32, d);
        tc_wait_ld();
        if (c == 3) {
          tc_fence_before();
          mbar_arrive(bar(C_DQD));
        }
        if (ok) {
#pragma unroll
          for (int x = 0; x < 8; ++x)
            red_add_v4(dst + c * 32 + x * 4, __uint_as_float(d[4 * x]), __uint_as_float(d[4 * x + 1]),
                       __uint_as_float(d[4 * x + 2]), __uint_as_float(d[4 * x + 3]));
        }
      }
      w.next();
    }
  }
  // ===================================================================== dK / dV write-out
  if (warp < 8) {
    const int k = threadIdx.x & 127;
    const uint32_t lane_base = (uint32_t)((warp & 3) * 32) << 16;
    const bool isK = warp >= 4;
    mbar_wait(bar(C_DONE), 0);
    tc_fence_after();
    const uint32_t src = (isK ? tdK : tdV) + lane_base;
    const float mul = isK ? prm.scale : 1.f;
    const int64_t row = ((int64_t)(it.tok + k) * prm.Hkv + g) * 128;
    const bool ok = k < it.len;
#pragma unroll
    for (int c = 0; c < 4; ++c) {
      uint32_t d[32];
      tmem_ld32(src + c * 32, d);
      tc_wait_ld();
      if (!ok) continue;
      if (it.kind == 0) {
        float* dst = (isK ? prm.gradK : prm.gradV) + row + c * 32;
#pragma unroll
        for (int x = 0; x < 8; ++x) {
          float4 a = *reinterpret_cast<float4*>(dst + 4 * x);
          a.x += __uint_as_float(d[4 * x]) * mul;
          a.y += __uint_as_float(d[4 * x + 1]) * mul;
          a.z += __uint_as_float(d[4 * x + 2]) * mul;
          a.w += __uint_as_float(d[4 * x + 3]) * mul;
          *reinterpret_cast<float4*>(dst + 4 * x) = a;
        }
      } else if (prm.dKs != nullptr) {
        __nv_bfloat16* dst = (isK ? prm.dKs : prm.dVs) + row + c * 32;
#pragma unroll
        for (int x = 0; x < 4; ++x) {
          uint4 u;
          u.x = pack_bf16(__uint_as_float(d[8 * x]) * mul, __uint_as_float(d[8 * x + 1]) * mul);
          u.y = pack_bf16(__uint_as_float(d[8 * x + 2]) * mul, __uint_as_float(d[8 * x + 3]) * mul);
          u.z = pack_bf16(__uint_as_float(d[8 * x + 4]) * mul, __uint_as_float(d[8 * x + 5]) * mul);
          u.w = pack_bf16(__uint_as_float(d[8 * x + 6]) * mul, __uint_as_float(d[8 * x + 7]) * mul);
          *reinterpret_cast<uint4*>(dst + 8 * x) = u;
        }
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 8) tmem_dealloc(tbase, 512);
}

static inline size_t up1k(size_t x) { return (x + 1023) / 1024 * 1024; }

size_t tc_bwd_workspace(const cas_slot_table* t, int Hq, int D) {
  if (D != 128) return 0;
  const size_t nqt = (size_t)t->qtile_off[t->B];
  return up1k((size_t)t->T * Hq * 128 * 4) + 2 * up1k((size_t)Hq * nqt * 128 * 4) + 1024;
}

int tc_attn_bwd(const AttnArgs& a) {
  const cas_slot_table* t = a.tab;
  static bool attr_set = false;
  if (!attr_set) {
    CAS_CUDA(cudaFuncSetAttribute(tc_bwd_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kBwdSmem));
    attr_set = true;
  }
  const size_t nqt = (size_t)t->qtile_off[t->B];
  const size_t b_acc = up1k((size_t)t->T * a.Hq * 128 * 4), b_aux = up1k((size_t)a.Hq * nqt * 128 * 4);
  char* ws = (char*)(((uintptr_t)a.workspace + 1023) & ~(uintptr_t)1023);
  float* dQacc = (float*)ws;
  float* auxL = (float*)(ws + b_acc);
  float* auxD = (float*)(ws + b_acc + b_aux);
  CAS_CUDA(cudaMemsetAsync(ws, 0, b_acc + 2 * b_aux, a.stream));
  const int64_t n_rows = (int64_t)t->T * a.Hq;
  bwd_prep_kernel<<<(unsigned)((n_rows * 32 + 255) / 256), 256, 0, a.stream>>>(
      (const __nv_bfloat16*)a.O, (const __nv_bfloat16*)a.dO, a.LSE_in, t->d_seq_off, t->d_qtile_off, t->B, a.Hq,
      (int64_t)nqt * 128, auxL, auxD, n_rows);
  CUtensorMap tmQ, tmdO, tmKs, tmVs;
  int rc = make_thd_map(&tmQ, a.Q, t->T, a.Hq, 128);
  if (rc) return rc;
  rc = make_thd_map(&tmdO, a.dO, t->T, a.Hq, 128);
  if (rc) return rc;
  if (a.Ks) {
    rc = make_thd_map(&tmKs, a.Ks, t->T, a.Hkv, 128);
    if (rc) return rc;
    rc = make_thd_map(&tmVs, a.Vs, t->T, a.Hkv, 128);
    if (rc) return rc;
  } else {
    tmKs = a.pool->tm_K;
    tmVs = a.pool->tm_V;
  }
  BwdParams prm{t->d_seq_off, t->d_inv_off, t->d_inv_seq, t->d_qtile_off, t->d_bwd_items, auxL, auxD, dQacc,
                a.pool->grad_K, a.pool->grad_V, (__nv_bfloat16*)a.dKs, (__nv_bfloat16*)a.dVs, (int64_t)nqt * 128,
                a.Hq, a.Hkv, a.Ks ? 1 : 0, a.scale, a.scale * kLog2e};
  const unsigned grid = (unsigned)(t->bwd_items.size() * a.Hkv);
  tc_bwd_kernel<<<grid, kBwdThreads, kBwdSmem, a.stream>>>(tmQ, tmdO, a.pool->tm_K, a.pool->tm_V, tmKs, tmVs, prm);
  const int64_t n4 = n_rows * 32;
  dq_convert_kernel<<<(unsigned)std::min<int64_t>((n4 + 255) / 256, 148 * 16), 256, 0, a.stream>>>(
      dQacc, (__nv_bfloat16*)a.dQ, a.scale, n4);
  cudaError_t e = cudaGetLastError();
  return e == cudaSuccess ? CAS_OK : cuda_fail(e, "tc bwd launch");
}

}  // namespace cas
