// Prefix-attention BACKWARD on tcgen05 + TMEM + TMA, bf16, head_dim 128.
//
// Definition: include/cas.h cas_prefix_attn_bwd (PAPER.md:44 only the cartridge K/V receive
// gradients; :176 all active cartridges are back-propagated simultaneously; :75 unselected ones get
// none).  KV-stationary: one CTA owns one 128-key tile of one KV head -- a tile of a cartridge slot
// (read in place from the pool) or of a sequence's own keys -- and walks, through the INVERTED slot
// table, every (sequence that selected the slot) x (query head of the group) x (128-row Q tile).
// dK/dV of the tile accumulate in TMEM over that whole loop and are written ONCE ("+=" into the
// slot's fp32 gradient buffer, no atomics, deterministic).  dQ tiles are staged through shared
// memory and added to an fp32 scratch with bulk reductions (cp.reduce.async.bulk ... add.f32: one
// 16 KB contiguous L2 reduction per quarter tile), then converted to bf16 (x scale) by an epilogue
// kernel.
//
// Per inner iteration i (Q tile, dO tile, LSE, delta of 128 query rows), five MMAs, keys on lanes:
//   S^T  = K  Q^T        (SS)            dP^T = V  dO^T      (SS)
//   dV  += P^T dO        (P^T from TMEM) dK  += dS^T Q       (dS^T from SMEM, K-major)
//   dQ   = dS  K         (the same dS^T bytes in SMEM read as an MN-major A operand)
// TMEM (512 cols): [S^T / P^T] [dP^T / dQ] [dV] [dK].   SMEM (226 KB): K,V | 2 x Q | dO | dQ staging | dS^T.
// dO needs ONE stage: its readers are dP(i) (issued at the end of iteration i-1) and dV(i) (start of iteration
// i), so dO(i+1) can be fetched while S(i+1), dQ(i), dK(i) run.
// Warps: 0-3 / 4-7 two compute warpgroups (thread = key; group w owns query columns [64w, 64w+64)):
// exp -> P^T, then dS^T; 8-11 dQ reducers (thread = query); 12 TMA producer; 13 MMA issuer.
// Issue order:  dV(i)  S(i+1)  dQ(i) dK(i)  [dQ drained]  dP(i+1)   -- the exp of tile i+1 overlaps
// dQ/dK of tile i, the dQ drain overlaps dK.  dQ is staged in its own 32 KB (two 16 KB quarter-tile buffers): the
// bulk-reduction engine drains shared memory at only ~20 B/clk per SM (measured), so a staging buffer stays
// busy for most of an iteration and must not be one of the pipeline stages.
#include <cstdlib>

#include "cas_sm100.cuh"
#include "cas_tc_common.cuh"

namespace cas {
using namespace sm100;

constexpr float kLog2e = 1.4426950408889634f;


// delta[t,h] = sum_d dO*O (B1), stored head-major and padded per sequence to whole 128-row tiles
// (so each (head, Q tile) is one aligned 512-byte run): auxD[h][tile*128 + r] = -delta; auxL = -LSE*log2(e).
// The same pass ZEROES the fp32 dQ scratch row of every (t, h) (no separate 100 MB memset launch) and the padding
// entries of auxL / auxD behind the last token of every sequence (they are multiplied by masked zeros in the main
// kernel and must be finite).  Eight lanes per (t, h) row, 16 columns = two 16-byte loads per tensor and lane: a
// warp covers four consecutive rows = 1 KB contiguous of O and of dO.
__global__ void __launch_bounds__(256)
bwd_prep_kernel(const __nv_bfloat16* __restrict__ O, const __nv_bfloat16* __restrict__ dO,
                const float* __restrict__ LSE, const int32_t* __restrict__ seq_off,
                const int32_t* __restrict__ qtile_off, int B, int Hq, int64_t aux_stride,
                float* __restrict__ auxL, float* __restrict__ auxD, float* __restrict__ dQacc, int64_t n_rows) {
  const int64_t w = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 3;   // (t, h) row
  const int sub = threadIdx.x & 7;
  const bool live = w < n_rows;
  const int64_t wr = live ? w : 0;
  const int t = (int)(wr / Hq), h = (int)(wr % Hq);
  const uint4* po = reinterpret_cast<const uint4*>(O + wr * 128 + sub * 16);
  const uint4* pd = reinterpret_cast<const uint4*>(dO + wr * 128 + sub * 16);
  const uint4 a0 = po[0], a1 = po[1], b0 = pd[0], b1 = pd[1];
  const uint32_t av[8] = {a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w};
  const uint32_t bv[8] = {b0.x, b0.y, b0.z, b0.w, b1.x, b1.y, b1.z, b1.w};
  float s = 0.f;
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const float2 x = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&av[i]));
    const float2 y = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&bv[i]));
    s += x.x * y.x + x.y * y.y;
  }
#pragma unroll
  for (int o = 4; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if (!live) return;
  int lo = 0, hi = B - 1;                        // sequence of token t
  while (lo < hi) {
    const int mid = (lo + hi + 1) >> 1;
    if (seq_off[mid] <= t) lo = mid; else hi = mid - 1;
  }
  const int row = t - seq_off[lo];
  const int64_t u = qtile_off[lo] + (row >> 7);
  const int r = row & 127;
  // this row's 512 bytes of the dQ scratch: quarter c = sub >> 1 holds 128 bytes of it, this lane zeroes one half
  {
    float4* z = reinterpret_cast<float4*>(dQacc + (((int64_t)h * (aux_stride >> 7) + u) * 4 + (sub >> 1)) * 4096 + r * 32 +
                                          (sub & 1) * 16);
    const float4 zero = make_float4(0.f, 0.f, 0.f, 0.f);
    z[0] = zero; z[1] = zero; z[2] = zero; z[3] = zero;
  }
  const int64_t pos = (int64_t)h * aux_stride + u * 128 + r;
  if (sub == 0) {
    auxD[pos] = -s;                    // negated: the main kernel adds them with packed FADD2 / FFMA2
    auxL[pos] = -LSE[wr] * kLog2e;
  }
  // the last token of a sequence also clears the padding of its last tile (<= 127 entries per head)
  if (t + 1 == seq_off[lo + 1]) {
    for (int x = r + 1 + sub; x < 128; x += 8) {
      auxD[pos - r + x] = 0.f;
      auxL[pos - r + x] = 0.f;
    }
  }
}

// dQ scratch layout (written by the bulk reductions of tc_bwd_kernel): per (head h, global Q tile u)
// four quarter tiles of 32 columns, each [128 rows][32 fp32] = 16 KB contiguous; inside a 128-byte
// row the 16-byte chunk j sits at position j ^ (row & 7) (bank-conflict-free staging stores).
// dQ[t,h,:] = bf16(scale * scratch);  one warp per (t, h) row, lane = 4 columns.
__global__ void __launch_bounds__(256)
dq_convert_kernel(const float* __restrict__ acc, __nv_bfloat16* __restrict__ dQ, const int32_t* __restrict__ seq_off,
                  const int32_t* __restrict__ qtile_off, int B, int Hq, int64_t nqt, float scale, int64_t n_rows,
                  const float2* __restrict__ rope_cs, int rope_layout) {
  const int64_t w = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  if (w >= n_rows) return;
  const int t = (int)(w / Hq), h = (int)(w % Hq);
  int lo = 0, hi = B - 1;
  while (lo < hi) {
    const int mid = (lo + hi + 1) >> 1;
    if (seq_off[mid] <= t) lo = mid; else hi = mid - 1;
  }
  const int row = t - seq_off[lo];
  const int64_t u = qtile_off[lo] + (row >> 7);
  const int r = row & 127, c = lane >> 3, j = lane & 7;
  const float4 v = *reinterpret_cast<const float4*>(acc + (((int64_t)h * nqt + u) * 4 + c) * 4096 + r * 32 +
                                                    ((j ^ (r & 7)) << 2));
  float x0 = v.x * scale, x1 = v.y * scale, x2 = v.z * scale, x3 = v.w * scale;     // columns 4*lane .. 4*lane+3
  if (rope_cs) {
    // fused RoPE backward: dQ w.r.t. the un-rotated queries = R(t)^T dQ_rot, in fp32 before the one
    // rounding to bf16.  The whole warp is here (a warp = one row), so the shuffles are safe.
    const float2* tab = rope_cs + (int64_t)t * 64;
    if (rope_layout == 0) {                       // pairs (2k, 2k+1): k = 2*lane, 2*lane+1
      const float2 w0 = __ldg(tab + 2 * lane), w1 = __ldg(tab + 2 * lane + 1);
      const float a0 = x0, b0 = x1, a1 = x2, b1 = x3;
      x0 = a0 * w0.x + b0 * w0.y;  x1 = -a0 * w0.y + b0 * w0.x;
      x2 = a1 * w1.x + b1 * w1.y;  x3 = -a1 * w1.y + b1 * w1.x;
    } else {                                      // pairs (k, k + 64): lanes l and l + 16 hold the two halves
      const float y0 = __shfl_xor_sync(0xffffffffu, x0, 16), y1 = __shfl_xor_sync(0xffffffffu, x1, 16);
      const float y2 = __shfl_xor_sync(0xffffffffu, x2, 16), y3 = __shfl_xor_sync(0xffffffffu, x3, 16);
      const int k = 4 * (lane & 15);
      const float2 w0 = __ldg(tab + k), w1 = __ldg(tab + k + 1), w2 = __ldg(tab + k + 2), w3 = __ldg(tab + k + 3);
      if (lane < 16) {                            // own = a, partner = b:  a' = a cos + b sin
        x0 = x0 * w0.x + y0 * w0.y;  x1 = x1 * w1.x + y1 * w1.y;  x2 = x2 * w2.x + y2 * w2.y;  x3 = x3 * w3.x + y3 * w3.y;
      } else {                                    // own = b, partner = a:  b' = -a sin + b cos
        x0 = -y0 * w0.y + x0 * w0.x;  x1 = -y1 * w1.y + x1 * w1.x;  x2 = -y2 * w2.y + x2 * w2.x;  x3 = -y3 * w3.y + x3 * w3.x;
      }
    }
  }
  uint2 o;
  o.x = pack_bf16(x0, x1);
  o.y = pack_bf16(x2, x3);
  *reinterpret_cast<uint2*>(dQ + w * 128 + lane * 4) = o;
}

// ------------------------------------------------------------------------------- main kernel
constexpr int kBwdThreads = 512;   // 4 warpgroups (setmaxnreg works on whole warpgroups); warps 14,15 idle
constexpr uint32_t kT = 32768, kH = 16384;
constexpr uint32_t oK = 0, oV = kT, oQ = 2 * kT, oDO = 4 * kT, oStg = 5 * kT, oDS = 6 * kT, oAuxL = 7 * kT, oAuxD = 7 * kT + 1024,
                   oBar = 7 * kT + 2048;
constexpr uint32_t kBwdSmem = oBar + 256;
enum { C_KV = 0, C_QF = 1, C_DOF = 3, C_QE = 5, C_DOE = 7, C_SF = 9, C_DPF = 10, C_PF = 11, C_DSF = 12, C_DQF = 13,
       C_DQD = 14, C_DONE = 15, C_N = 16 };

struct BwdParams {
  const int32_t *seq_off, *inv_off, *inv_seq, *qtile_off;
  const BwdItem* items;
  const PackedTile* ptiles;     // packed prefix tiles (kind 2 items)
  const float *auxL, *auxD;
  float* dQacc;
  float *gradK, *gradV;
  __nv_bfloat16 *dKs, *dVs;
  int64_t aux_stride;     // nqt * 128
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
  __device__ int64_t utile() const { return p.qtile_off[b] + qt; }           // global Q tile index
  __device__ int64_t aux() const { return (int64_t)h * p.aux_stride + utile() * 128; }
};

template <int N>
__device__ __forceinline__ void setmaxnreg_inc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(N)); }
template <int N>
__device__ __forceinline__ void setmaxnreg_dec() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(N)); }

__global__ void __launch_bounds__(kBwdThreads, 1)
tc_bwd_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmdO,
              const __grid_constant__ CUtensorMap tmKp, const __grid_constant__ CUtensorMap tmVp,
              const __grid_constant__ CUtensorMap tmKs, const __grid_constant__ CUtensorMap tmVs,
              const __grid_constant__ CUtensorMap tmKp16, const __grid_constant__ CUtensorMap tmVp16,
              const BwdParams prm, const __grid_constant__ SlotMask dirty) {
  extern __shared__ __align__(1024) uint8_t smem[];
  const uint32_t sbase = smem_u32(smem);
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + oBar + C_N * 8);
  auto bar = [&](int i) { return sbase + oBar + 8u * i; };
  const int warp = warp_id_uniform(), lane = threadIdx.x & 31;
  // KV-head-major block order: the CTAs in flight share one KV group, so the Q / dO / LSE / delta rows they
  // re-read (G heads of every selecting sequence) stay in L2
  const int n_items = gridDim.x / prm.Hkv;
  const int g = blockIdx.x / n_items;
  const BwdItem it = prm.items[blockIdx.x % n_items];
  if (it.kind == 1 && !prm.has_self) return;     // prefix-only call: no self tiles (block-uniform)
  const PackedTile* pt = it.kind == 2 ? prm.ptiles + it.tok : nullptr;   // a sequence's packed 16-token pages

  if (threadIdx.x == 0) {
    if (sbase & 1023u) __trap();
    for (int i = 0; i < C_N; ++i)
      mbar_init(bar(i), (i == C_PF || i == C_DSF) ? 256 : (i == C_DQD ? 128 : 1));
    fence_mbar_init();
  }
  if (warp == 12) {
    tmem_alloc(smem_u32(tmem_slot), 512);
    tmem_relinquish();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tbase = *tmem_slot;
  const uint32_t tS = tbase, tdP = tbase + 128, tdV = tbase + 256, tdK = tbase + 384;

  if (warp >= 12) {
    setmaxnreg_dec<56>();
    if (warp == 12) { if (elect_one()) {
      // ================================================================= TMA producer
      const CUtensorMap* mk = it.kind == 0 ? &tmKp : &tmKs;
      const CUtensorMap* mv = it.kind == 0 ? &tmVp : &tmVs;
      mbar_expect_tx(bar(C_KV), 2 * kT);
      if (pt) {
        for (int u = 0; u < 8; ++u) {
          tma_load_3d(sbase + oK + u * 2048, &tmKp16, bar(C_KV), 0, g, pt->tok[u]);
          tma_load_3d(sbase + oK + kH + u * 2048, &tmKp16, bar(C_KV), 64, g, pt->tok[u]);
          tma_load_3d(sbase + oV + u * 2048, &tmVp16, bar(C_KV), 0, g, pt->tok[u]);
          tma_load_3d(sbase + oV + kH + u * 2048, &tmVp16, bar(C_KV), 64, g, pt->tok[u]);
        }
      } else {
        tma_load_3d(sbase + oK, mk, bar(C_KV), 0, g, it.tok);
        tma_load_3d(sbase + oK + kH, mk, bar(C_KV), 64, g, it.tok);
        tma_load_3d(sbase + oV, mv, bar(C_KV), 0, g, it.tok);
        tma_load_3d(sbase + oV + kH, mv, bar(C_KV), 64, g, it.tok);
      }
      Walk w(prm, it, g);
      const int n = w.total();
      for (int i = 0; i < n; ++i) {
        const int st = i & 1;
        const uint32_t eph = ((i >> 1) & 1) ^ 1;
        mbar_wait(bar(C_QE + st), eph);
        mbar_expect_tx(bar(C_QF + st), kT + 512);
        tma_load_3d(sbase + oQ + st * kT, &tmQ, bar(C_QF + st), 0, w.h, w.tok());
        tma_load_3d(sbase + oQ + st * kT + kH, &tmQ, bar(C_QF + st), 64, w.h, w.tok());
        bulk_load(sbase + oAuxL + st * 512, prm.auxL + w.aux(), 512, bar(C_QF + st));
        if (i > 0) mbar_wait(bar(C_DOE), (i - 1) & 1);   // dV(i-1) has read dO(i-1): the single dO stage is free
        mbar_expect_tx(bar(C_DOF), kT + 512);
        tma_load_3d(sbase + oDO, &tmdO, bar(C_DOF), 0, w.h, w.tok());
        tma_load_3d(sbase + oDO + kH, &tmdO, bar(C_DOF), 64, w.h, w.tok());
        bulk_load(sbase + oAuxD + st * 512, prm.auxD + w.aux(), 512, bar(C_DOF));
        w.next();
      }
    } } else if (warp == 13) { if (elect_one()) {
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
        for (int kk = 0; kk < 8; ++kk) mma_ss(tdP, kmaj(sbase + oV, kk), kmaj(sbase + oDO, kk), id_kk, kk > 0);
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
        // dV += P^T dO ; P^T (bf16) of query columns [0,64) sits at tS+[0,32), of [64,128) at tS+64+[0,32)
#pragma unroll
        for (int kk = 0; kk < 8; ++kk)
          mma_ts(tdV, tS + (kk >> 2) * 64 + (kk & 3) * 8, mnmaj(sbase + oDO, kk), id_kmn,
                 (i > 0 || kk > 0) ? 1u : 0u);
        mma_commit(bar(C_DOE));               // dO(i) is dead: dP(i) was issued before, dV(i) is its last reader
        if (i + 1 < n) {
          mbar_wait(bar(C_QF + st1), ph1);
          tc_fence_after();
          mma_S(st1);
          mma_commit(bar(C_SF));
        }
        mbar_wait(bar(C_DSF), i & 1);
        tc_fence_after();
#pragma unroll
        for (int kk = 0; kk < 8; ++kk)     // dQ = dS K
          mma_ss(tdP, mnmaj(sbase + oDS, kk), mnmaj(sbase + oK, kk), id_mnmn, kk > 0);
        mma_commit(bar(C_DQF));
#pragma unroll
        for (int kk = 0; kk < 8; ++kk)     // dK += dS^T Q
          mma_ss(tdK, kmaj(sbase + oDS, kk), mnmaj(sbase + oQ + st * kT, kk), id_kmn, (i > 0 || kk > 0) ? 1u : 0u);
        mma_commit(bar(C_QE + st));
        if (i + 1 < n) {
          mbar_wait(bar(C_DOF), (i + 1) & 1);
          mbar_wait(bar(C_DQD), i & 1);
          tc_fence_after();
          mma_dP(st1);
          mma_commit(bar(C_DPF));
        }
      }
      mma_commit(bar(C_DONE));
    } }
  } else if (warp < 8) {
    // =================================================================== compute: P^T, dS^T
    setmaxnreg_inc<152>();
    const int wg = warp >> 2;                        // query-column half owned by this warpgroup
    const int k = threadIdx.x & 127;                 // key lane
    const uint32_t lane_base = (uint32_t)((warp & 3) * 32) << 16;
    const uint32_t tSw = tS + lane_base + wg * 64, tdPw = tdP + lane_base + wg * 64;
    const bool key_ok = pt ? ((pt->mask[k >> 5] >> (k & 31)) & 1u) != 0 : k < it.len;
    const bool tile_full = it.len == 128;            // (a packed tile with 128 valid keys has every mask bit set)
    const uint32_t ds_row = sbase + oDS + wg * kH + k * 128;
    Walk w(prm, it, g);
    const int n = w.total();
    for (int i = 0; i < n; ++i) {
      const int st = i & 1;
      const uint32_t ph = (i >> 1) & 1;
      const int rows = w.rows();
      const bool diag = it.kind == 1 && w.qt == it.jt;
      const bool masked = diag || rows < 128 || !tile_full;            // block-uniform
      // valid query columns of this key: qlo <= q < qhi
      const int qlo = diag ? k : 0;
      const int qhi = key_ok ? rows : 0;
      const float4* aL = reinterpret_cast<const float4*>(smem + oAuxL + st * 512 + wg * 256);
      const float4* aD = reinterpret_cast<const float4*>(smem + oAuxD + st * 512 + wg * 256);
      mbar_wait(bar(C_QF + st), ph);
      mbar_wait(bar(C_SF), i & 1);
      tc_fence_after();
      float p[64];
      const uint64_t sc2 = pack2(prm.scale_log2, prm.scale_log2);
#pragma unroll
      uint32_t sall[64];
      tmem_ld32(tSw, sall);                           // both 32-column loads in flight, one wait
      tmem_ld32(tSw + 32, sall + 32);
      tc_wait_ld();
#pragma unroll
      for (int c = 0; c < 2; ++c) {
        const uint32_t* s = sall + c * 32;
#pragma unroll
        for (int q4 = 0; q4 < 8; ++q4) {
          const float4 L = aL[c * 8 + q4];          // -LSE*log2(e) of four query columns
          float e0, e1, e2, e3;
          unpack2(fma2(pack2(__uint_as_float(s[4 * q4 + 0]), __uint_as_float(s[4 * q4 + 1])), sc2, pack2(L.x, L.y)), e0, e1);
          unpack2(fma2(pack2(__uint_as_float(s[4 * q4 + 2]), __uint_as_float(s[4 * q4 + 3])), sc2, pack2(L.z, L.w)), e2, e3);
          p[c * 32 + 4 * q4 + 0] = ex2_approx(e0);
          p[c * 32 + 4 * q4 + 1] = ex2_approx(e1);
          p[c * 32 + 4 * q4 + 2] = ex2_approx(e2);
          p[c * 32 + 4 * q4 + 3] = ex2_approx(e3);
        }
      }
      if (masked) {
#pragma unroll
        for (int q = 0; q < 64; ++q) {
          const int qq = wg * 64 + q;
          p[q] = (qq >= qlo && qq < qhi) ? p[q] : 0.f;
        }
      }
      {
        uint32_t pk[32];
#pragma unroll
        for (int q = 0; q < 32; ++q) pk[q] = pack_bf16(p[2 * q], p[2 * q + 1]);
        tmem_st32(tSw, pk);
      }
      tc_wait_st();
      tc_fence_before();
      mbar_arrive(bar(C_PF));
      mbar_wait(bar(C_DOF), i & 1);
      mbar_wait(bar(C_DPF), i & 1);
      tc_fence_after();
#pragma unroll
      uint32_t dall[64];
      tmem_ld32(tdPw, dall);
      tmem_ld32(tdPw + 32, dall + 32);
      tc_wait_ld();
#pragma unroll
      for (int c = 0; c < 2; ++c) {
        const uint32_t* d = dall + c * 32;
#pragma unroll
        for (int q8 = 0; q8 < 4; ++q8) {
          const float4 D0 = aD[c * 8 + q8 * 2], D1 = aD[c * 8 + q8 * 2 + 1];   // -delta of eight query columns
          const int q = c * 32 + q8 * 8;
          uint32_t pk[4];
          float x0, x1;
          // dS = P * (dP - delta): packed FADD2 + FMUL2 on two columns at a time
          unpack2(mul2(pack2(p[q + 0], p[q + 1]), add2(pack2(__uint_as_float(d[q8 * 8 + 0]), __uint_as_float(d[q8 * 8 + 1])), pack2(D0.x, D0.y))), x0, x1);
          pk[0] = pack_bf16(x0, x1);
          unpack2(mul2(pack2(p[q + 2], p[q + 3]), add2(pack2(__uint_as_float(d[q8 * 8 + 2]), __uint_as_float(d[q8 * 8 + 3])), pack2(D0.z, D0.w))), x0, x1);
          pk[1] = pack_bf16(x0, x1);
          unpack2(mul2(pack2(p[q + 4], p[q + 5]), add2(pack2(__uint_as_float(d[q8 * 8 + 4]), __uint_as_float(d[q8 * 8 + 5])), pack2(D1.x, D1.y))), x0, x1);
          pk[2] = pack_bf16(x0, x1);
          unpack2(mul2(pack2(p[q + 6], p[q + 7]), add2(pack2(__uint_as_float(d[q8 * 8 + 6]), __uint_as_float(d[q8 * 8 + 7])), pack2(D1.z, D1.w))), x0, x1);
          pk[3] = pack_bf16(x0, x1);
          const uint32_t addr = ds_row + ((uint32_t)((c * 4 + q8) ^ (k & 7)) << 4);
          asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(pk[0]), "r"(pk[1]), "r"(pk[2]), "r"(pk[3]) : "memory");
        }
      }
      tc_fence_before();
      fence_proxy_async();
      mbar_arrive(bar(C_DSF));
      w.next();
    }
  } else {
    // =================================================================== dQ reducers (warps 8-11)
    setmaxnreg_inc<152>();
    const int q = threadIdx.x - 256;                 // query lane
    const uint32_t lane_base = (uint32_t)((warp & 3) * 32) << 16;
    Walk w(prm, it, g);
    const int n = w.total();
    for (int i = 0; i < n; ++i) {
      const int st = i & 1;
      const uint32_t stage = sbase + oStg;           // dedicated staging: two 16 KB quarter-tile buffers
      float* dst = prm.dQacc + ((int64_t)w.h * (prm.aux_stride >> 7) + w.utile()) * 16384;
      mbar_wait(bar(C_DQF), i & 1);
      tc_fence_after();
      uint32_t d[128];
#pragma unroll
      for (int c = 0; c < 4; ++c) tmem_ld32(tdP + lane_base + c * 32, d + c * 32);
      tc_wait_ld();
      tc_fence_before();
      mbar_arrive(bar(C_DQD));                       // TMEM is free for dP(i+1)
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        const uint32_t buf = stage + (c & 1) * kH;
        if (c >= 2 || i > 0) {                       // the quarter staged two steps ago must have left this buffer
          if (q == 0) asm volatile("cp.async.bulk.wait_group.read 1;" ::: "memory");
          asm volatile("bar.sync 1, 128;" ::: "memory");
        }
#pragma unroll
        for (int j = 0; j < 8; ++j) {
          const uint32_t addr = buf + q * 128 + ((uint32_t)(j ^ (q & 7)) << 4);
          asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(d[c * 32 + 4 * j]),
                       "r"(d[c * 32 + 4 * j + 1]), "r"(d[c * 32 + 4 * j + 2]), "r"(d[c * 32 + 4 * j + 3]) : "memory");
        }
        fence_proxy_async();
        asm volatile("bar.sync 1, 128;" ::: "memory");
        if (q == 0) {
          asm volatile("cp.reduce.async.bulk.global.shared::cta.bulk_group.add.f32 [%0], [%1], %2;"
                       ::"l"(dst + c * 4096), "r"(buf), "r"(16384u) : "memory");
          asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        }
      }
      w.next();
    }
    if (q == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
  }
  // ===================================================================== dK / dV write-out
  // Every stage buffer is dead after the last MMA.  Thread = key row: TMEM -> registers -> its own
  // padded row in shared memory -> ONE bulk operation per row: "+=" into the slot's fp32 gradient
  // row (cp.reduce.async.bulk add.f32, 512 B; each row is owned by exactly one CTA, so the sum is
  // deterministic) or, for a self tile, a 256 B bf16 bulk store into dK_self/dV_self.
  if (warp < 8) {
    const int k = threadIdx.x & 127;
    const uint32_t lane_base = (uint32_t)((warp & 3) * 32) << 16;
    const bool isK = warp >= 4;
    mbar_wait(bar(C_DONE), 0);
    tc_fence_after();
    const uint32_t src = (isK ? tdK : tdV) + lane_base;
    const float mul = isK ? prm.scale : 1.f;
    const int key_tok = pt ? pt->tok[k >> 4] + (k & 15) : it.tok + k;       // packed: the key's own cartridge row
    const int64_t row = ((int64_t)key_tok * prm.Hkv + g) * 128;
    const bool ok = pt ? ((pt->mask[k >> 5] >> (k & 31)) & 1u) != 0 : k < it.len;
    if (it.kind != 1) {
      const uint32_t srow = sbase + (isK ? 67584u : 0u) + k * 528;     // 528 B row pitch: conflict-free v4 stores
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        uint32_t d[32];
        tmem_ld32(src + c * 32, d);
        tc_wait_ld();
#pragma unroll
        for (int x = 0; x < 8; ++x)
          asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(srow + c * 128 + x * 16),
                       "f"(__uint_as_float(d[4 * x]) * mul), "f"(__uint_as_float(d[4 * x + 1]) * mul),
                       "f"(__uint_as_float(d[4 * x + 2]) * mul), "f"(__uint_as_float(d[4 * x + 3]) * mul) : "memory");
      }
      fence_proxy_async();
      if (ok) {
        // a slot that already holds gradients is added to; a clean slot's buffer is undefined and is overwritten
        // a packed tile always ADDS: other sequences' CTAs write the same cartridge rows (the host has zeroed the
        // clean slots it touches)
        if (pt || ((dirty.w[it.id >> 5] >> (it.id & 31)) & 1u))
          asm volatile("cp.reduce.async.bulk.global.shared::cta.bulk_group.add.f32 [%0], [%1], %2;"
                       ::"l"((isK ? prm.gradK : prm.gradV) + row), "r"(srow), "r"(512u) : "memory");
        else
          asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;"
                       ::"l"((isK ? prm.gradK : prm.gradV) + row), "r"(srow), "r"(512u) : "memory");
        asm volatile("cp.async.bulk.commit_group;" ::: "memory");
      }
    } else if (prm.dKs != nullptr) {
      const uint32_t srow = sbase + (isK ? 34816u : 0u) + k * 272;
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        uint32_t d[32];
        tmem_ld32(src + c * 32, d);
        tc_wait_ld();
#pragma unroll
        for (int x = 0; x < 4; ++x)
          asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(srow + c * 64 + x * 16),
                       "r"(pack_bf16(__uint_as_float(d[8 * x]) * mul, __uint_as_float(d[8 * x + 1]) * mul)),
                       "r"(pack_bf16(__uint_as_float(d[8 * x + 2]) * mul, __uint_as_float(d[8 * x + 3]) * mul)),
                       "r"(pack_bf16(__uint_as_float(d[8 * x + 4]) * mul, __uint_as_float(d[8 * x + 5]) * mul)),
                       "r"(pack_bf16(__uint_as_float(d[8 * x + 6]) * mul, __uint_as_float(d[8 * x + 7]) * mul)) : "memory");
      }
      fence_proxy_async();
      if (ok) {
        asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;"
                     ::"l"((isK ? prm.dKs : prm.dVs) + row), "r"(srow), "r"(256u) : "memory");
        asm volatile("cp.async.bulk.commit_group;" ::: "memory");
      }
    }
    asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 12) tmem_dealloc(tbase, 512);
}

static inline size_t up1k(size_t x) { return (x + 1023) / 1024 * 1024; }

size_t tc_bwd_workspace(const cas_slot_table* t, int Hq, int D) {
  if (D != 128) return 0;
  const size_t nqt = (size_t)t->qtile_off[t->B];
  return up1k((size_t)Hq * nqt * 65536) + 2 * up1k((size_t)Hq * nqt * 128 * 4) + 1024;
}

int tc_attn_bwd(const AttnArgs& a) {
  const cas_slot_table* t = a.tab;
  static SmemAttrOnce attr;
  {
    const int rc_attr = attr.set((const void*)tc_bwd_kernel, (int)kBwdSmem);
    if (rc_attr) return rc_attr;
  }
  const size_t nqt = (size_t)t->qtile_off[t->B];
  const size_t b_acc = up1k((size_t)a.Hq * nqt * 65536), b_aux = up1k((size_t)a.Hq * nqt * 128 * 4);
  char* ws = (char*)(((uintptr_t)a.workspace + 1023) & ~(uintptr_t)1023);
  float* dQacc = (float*)ws;
  float* auxL = (float*)(ws + b_acc);
  float* auxD = (float*)(ws + b_acc + b_aux);
  // no memset: bwd_prep_kernel zeroes the dQ scratch rows of every real (t, h) and the aux padding; the scratch rows of
  // padding tokens are only ever added to (masked zeros) and never read
  const int64_t n_rows = (int64_t)t->T * a.Hq;
  bwd_prep_kernel<<<(unsigned)((n_rows * 8 + 255) / 256), 256, 0, a.stream>>>(
      (const __nv_bfloat16*)a.O, (const __nv_bfloat16*)a.dO, a.LSE_in, t->d_seq_off, t->d_qtile_off, t->B, a.Hq,
      (int64_t)nqt * 128, auxL, auxD, dQacc, n_rows);
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
    tmKs = a.L->tm_K;
    tmVs = a.L->tm_V;
  }
  BwdParams prm{t->d_seq_off, t->d_inv_off, t->d_inv_seq, t->d_qtile_off, t->d_bwd_items, t->d_ptiles, auxL, auxD, dQacc,
                a.L->grad_K, a.L->grad_V, (__nv_bfloat16*)a.dKs, (__nv_bfloat16*)a.dVs, (int64_t)nqt * 128,
                a.Hq, a.Hkv, a.Ks ? 1 : 0, a.scale, a.scale * kLog2e};
  const unsigned grid = (unsigned)(t->bwd_items.size() * a.Hkv);
  SlotMask dirty{};
  const int32_t* gd = a.pool->grad_dirty.data() + (size_t)a.layer * a.pool->desc.n_slots;   // this layer's flags
  for (int sl = 0; sl < a.pool->desc.n_slots; ++sl)
    if (gd[sl]) dirty.w[sl >> 5] |= 1u << (sl & 31);
  if (a.pool->pack)   // paged pool: the clean slots of this table were zeroed by the caller, every tile adds
    for (int sl : t->used_slots) dirty.w[sl >> 5] |= 1u << (sl & 31);
  tc_bwd_kernel<<<grid, kBwdThreads, kBwdSmem, a.stream>>>(tmQ, tmdO, a.L->tm_K, a.L->tm_V, tmKs, tmVs, a.L->tm_K16,
                                                           a.L->tm_V16, prm, dirty);
  dq_convert_kernel<<<(unsigned)((n_rows * 32 + 255) / 256), 256, 0, a.stream>>>(
      dQacc, (__nv_bfloat16*)a.dQ, t->d_seq_off, t->d_qtile_off, t->B, a.Hq, (int64_t)nqt, a.scale, n_rows,
      (const float2*)a.rope_cs, a.rope_layout);
  cudaError_t e = cudaGetLastError();
  return e == cudaSuccess ? CAS_OK : cuda_fail(e, "tc bwd launch");
}

}  // namespace cas

