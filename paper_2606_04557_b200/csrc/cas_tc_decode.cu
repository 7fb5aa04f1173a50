// Prefix-attention FORWARD for decode-shaped batches: every sequence has exactly ONE query token whose keys are
// the selected cartridges (read in place from the pool) plus the sequence's own cache of self keys -- the tokens
// generated so far ("2048 maximum completion tokens"; BASELINE.json configs[4]; PAPER.md:111 inference
// over all loaded cartridges, :142 retrieval-selected variant).  bf16, head_dim 128, tcgen05 + TMEM + TMA.
//
// The work is HBM-bound (each K/V byte is used by G query heads of a few sequences), so the kernel reads every
// selected K/V tile from HBM as few times as possible and keeps every SM streaming:
//  * KV-stationary batching through the INVERTED slot table: slots with the same set of selecting sequences form a
//    group; the rows of an MMA tile are (sequence, head-of-group) pairs -- up to 128/G sequences x G heads -- so one
//    pass over a K/V tile serves all of them.
//  * PERSISTENT CTAs, one per SM.  The host cuts every (group, row block, KV head) tile list into segments of about
//    total/#SM tiles and deals them to the CTAs in order (the row blocks that share a chunk of tiles run at the same
//    time, so the second read of a tile hits L2); a CTA then draws the self-cache units -- one per (sequence, KV
//    head), whose length is only known at launch -- from a device ticket counter, which also evens out the tail.
//  * One segment = one (row block, KV head, run of tiles).  Two softmax warpgroups take alternate tiles (even tiles:
//    S0/O0, odd tiles: S1/O1 in TMEM), each with its own running max and sum, so the exp work of tile j+1 overlaps
//    the MMAs of tiles j and j+2; at the end of the segment the two accumulators are merged and written as ONE
//    un-normalised partial (O, m, l) per row.  A group with MORE rows than one block (c5 "all loaded": 64 sequences
//    x 4 heads = 256 rows) runs PAIRED segments (kind 2): two resident Q tiles, warpgroup w owns row block w and
//    takes every tile, so a K/V tile is fetched once for both blocks (4 MMAs per tile) and each block writes its
//    own partial.  Measured: same time as two separate segments (the period is the softmax -> PV -> QK chain of
//    one warpgroup either way, and at 256 rows x 256 k keys the step is as tensor-bound as it is HBM-bound:
//    0.27 PFLOP against 1.05 GB), but half the L2 -> SMEM traffic.
//  * MERGE of a row's split-KV partials (plus the few self keys of a young cache, dotted on the CUDA cores),
//    normalisation, O and LSE: small batches (<= 256 output rows, row blocks <= 32 rows, no paired segment) are merged
//    IN this launch by warp 11 -- every row has a counter, the CTA that writes a row's last partial merges it --
//    which saves the second launch of a latency-bound step; bigger batches by decode_combine_kernel (one warp per
//    output row; measured 2x faster than the in-kernel merge at 2048 rows).
// Warps: 0-3 / 4-7 softmax warpgroups (thread = row = TMEM lane), 8 scheduler + TMA producer (descriptors published
// one segment ahead through a 4-deep ring), 9 MMA issuer, 10 query gather (the rows of the next segment while the
// current one drains), 11 row counters + fused merge.
// SMEM: two Q tiles 64 KB + K/V ring of five 32 KB slots (unit 2t = K(t), 2t+1 = V(t)).  TMEM (512 cols): S0 | S1 | O0 | O1.
#include <algorithm>
#include <cstring>
#include <map>
#include <type_traits>

#include "cas_sm100.cuh"
#include "cas_tc_common.cuh"

namespace cas {
using namespace sm100;

constexpr int kDecThreads = 384;
constexpr int kRing = 5;           // K/V ring: five 32 KB slots filled in the order K(0) V(0) K(1) V(1) ...
constexpr int kDescRing = 4;
constexpr int kInlineSelf = 4;     // caches up to this length are dotted on the CUDA cores inside the merge
constexpr int kMaxDecB = 1024;     // sequences per decode call with a self cache (their lengths travel as kernel parameters)
constexpr uint32_t dT = 32768, dH = 16384;
constexpr uint32_t dOffQ = 0, dOffKV = 2 * dT, dOffBar = 2 * dT + kRing * dT;   // Q tile A | Q tile B | ring
enum { D_RF = 0, D_RE = 5, D_SF = 10, D_PF = 12, D_OV = 14, D_QF = 16, D_QE = 17, D_DF = 18, D_DE = 22, D_PW = 26, D_N = 30 };
constexpr uint32_t dOffDesc = dOffBar + D_N * 8 + 32;                       // after the barriers and the TMEM slot
constexpr uint32_t dOffML = dOffDesc + kDescRing * 32;                      // (m, l) of both warpgroups: 2 x 128 x 8 B
constexpr uint32_t kDecSmem = dOffML + 2048;
static_assert(kDecSmem <= 232448, "decode kernel shared memory");
static_assert(sizeof(DecSeg) == 32, "descriptor ring entry");
constexpr int kPartStride = 132;   // 128 O + m + l + pad (16-byte aligned rows)

struct SelfLens {
  int32_t v[kMaxDecB];       // cached tokens per sequence
  int32_t useq[kMaxDecB];    // the sequences whose cache gets a tensor-core segment (has_self_unit)
  int32_t n_useq;
};

struct DecParams {
  const DecSeg* segs;
  const int32_t* cta_seg_off;   // [grid + 1]
  const int32_t* seqs;          // row-block sequence lists
  const KvTile* tiles;
  const PackedTile* ptiles;     // packed prefix tiles (16-token pages), named by KvTile.tok < 0
  const int32_t* seq_off;       // packed token index of every sequence (one token each)
  const int32_t* comb_off;      // [B + 1] partial rows (in units of sequences) of the prefix segments covering sequence b
  const int32_t* comb_row;
  const __nv_bfloat16* Q;
  const __nv_bfloat16 *Kc, *Vc; // self cache [B, cache_cap, Hkv, 128] or null
  __nv_bfloat16* O;
  float* LSE;
  float* part;
  int32_t* cnt;                 // [Hkv * B * G] partials written per row so far (self-resetting)
  int32_t* ticket;              // [2]: next self unit, CTAs done (self-resetting)
  int64_t rows_total;           // partial rows per KV head
  int32_t self_row_base;        // first partial row (in units of sequences) of the self units
  int32_t cache_cap;
  int B, Hq, Hkv;
  int fused;                    // 1: warp 11 counts and merges in this launch; 0: decode_combine_kernel follows
  float scale_log2;
};

// A sequence's cache gets its own tensor-core segment when it is longer than the merge can dot inline, or when it is
// the sequence's only source of keys (someone has to trigger the merge).
__host__ __device__ __forceinline__ bool has_self_unit(int len, int n_prefix_partials) {
  return len > kInlineSelf || (len > 0 && n_prefix_partials == 0);
}

// End of a segment (both softmax warpgroups, 256 threads): merge the two TMEM accumulators and write ONE partial per
// row; thread (w, r) writes columns [64w, 64w + 64) of row r.  The partials are counted and merged by warps 10-11.
__device__ __forceinline__ void dec_segment_epilogue(const DecParams& prm, const DecSeg d, const int w, const int r,
                                                     const uint32_t tbase, const uint32_t lane_base, const float m,
                                                     const float l, const int c0, const int c1, const uint32_t bar_ov,
                                                     float2* ml) {
  const int G = prm.Hq / prm.Hkv;
  const int n = d.n_tiles;
  const int n1 = n >> 1;                                           // tiles of warpgroup 1 (warpgroup 0 has >= 1)
  ml[w * 128 + r] = make_float2(m, l);
  asm volatile("bar.sync 2, 256;" ::: "memory");                   // both warpgroups are past their last tile ...
  mbar_wait(bar_ov, (c0 - 1) & 1);                                 // ... so these waits are at most one phase behind
  if (n1) mbar_wait(bar_ov + 8, (c1 - 1) & 1);
  tc_fence_after();
  const float2 a = ml[r], b = ml[128 + r];
  const float M = n1 ? fmaxf(a.x, b.x) : a.x;
  const float f0 = ex2_approx(a.x - M), f1 = n1 ? ex2_approx(b.x - M) : 0.f;
  const float L = f0 * a.y + f1 * b.y;
  const int n_rows = d.n_seqs * G;
  float* prow = prm.part + ((int64_t)d.g * prm.rows_total + (int64_t)d.part_row * G + r) * kPartStride;
  const uint32_t tO0 = tbase + 256 + lane_base + w * 64, tO1 = tO0 + 128;
#pragma unroll
  for (int cc = 0; cc < 2; ++cc) {
    uint32_t o0[32], o1[32];
    tmem_ld32(tO0 + cc * 32, o0);
    if (n1) tmem_ld32(tO1 + cc * 32, o1);
    tc_wait_ld();
    if (r < n_rows) {
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        float4 v;
        v.x = f0 * __uint_as_float(o0[4 * i]); v.y = f0 * __uint_as_float(o0[4 * i + 1]);
        v.z = f0 * __uint_as_float(o0[4 * i + 2]); v.w = f0 * __uint_as_float(o0[4 * i + 3]);
        if (n1) {
          v.x += f1 * __uint_as_float(o1[4 * i]); v.y += f1 * __uint_as_float(o1[4 * i + 1]);
          v.z += f1 * __uint_as_float(o1[4 * i + 2]); v.w += f1 * __uint_as_float(o1[4 * i + 3]);
        }
        __stcg(reinterpret_cast<float4*>(prow + w * 64 + cc * 32 + 4 * i), v);
      }
    }
  }
  if (w == 0 && r < n_rows) __stcg(reinterpret_cast<float2*>(prow + 128), make_float2(M, L));
  // BOTH warpgroups have read O0 and O1 (each its column half) before either goes on: the next segment's first PV
  // overwrites an accumulator as soon as ONE warpgroup has posted its next P tile
  tc_fence_before();
  asm volatile("bar.sync 2, 256;" ::: "memory");
  // no fence here: the partial is published by the thread that counts it (warp 11 fences after its barrier wait;
  // a wide table is merged by the next launch)
}

// End of a PAIRED segment: warpgroup w owns row block w (its own S_w / O_w); thread r writes the whole partial row.
__device__ __forceinline__ void dec_paired_epilogue(const DecParams& prm, const DecSeg d, const int w, const int r,
                                                    const uint32_t tbase, const uint32_t lane_base, const float m,
                                                    const float l, const int c_own, const uint32_t bar_ov) {
  const int G = prm.Hq / prm.Hkv;
  mbar_wait(bar_ov, (c_own - 1) & 1);                              // this warpgroup's last PV
  tc_fence_after();
  const int n_rows = (w ? d.self_len : d.n_seqs) * G;
  float* prow = prm.part + ((int64_t)d.g * prm.rows_total + (int64_t)(d.part_row + (w ? d.n_seqs : 0)) * G + r) * kPartStride;
  const uint32_t tO = tbase + 256 + w * 128 + lane_base;
#pragma unroll
  for (int cc = 0; cc < 4; ++cc) {
    uint32_t o[32];
    tmem_ld32(tO + cc * 32, o);
    tc_wait_ld();
    if (r < n_rows) {
#pragma unroll
      for (int i = 0; i < 8; ++i)
        __stcg(reinterpret_cast<float4*>(prow + cc * 32 + 4 * i),
               make_float4(__uint_as_float(o[4 * i]), __uint_as_float(o[4 * i + 1]), __uint_as_float(o[4 * i + 2]),
                           __uint_as_float(o[4 * i + 3])));
    }
  }
  if (r < n_rows) __stcg(reinterpret_cast<float2*>(prow + 128), make_float2(m, l));
  tc_fence_before();
}

// Merge of ONE output row (sequence seq, query head g*G + hh): all split-KV partials of the row -- the prefix segments
// that cover the sequence (comb lists), its self-cache segment if it has one -- plus the few self keys of a young cache
// dotted here, normalised, written as O (bf16) and LSE.  LPR lanes cooperate on a row (lane `sub` owns 128/LPR
// columns); the caller guarantees that the LPR lanes of a row are converged and that every partial is visible.
// One pass with a running maximum; the partials are fetched four at a time (their loads are independent, so a
// row costs about two L2 round trips per four partials instead of two per partial).
template <int LPR>
__device__ __forceinline__ void dec_merge_row(const DecParams& prm, const SelfLens& slen, const int g, const int seq,
                                              const int hh, const int sub, const bool valid) {
  constexpr int NC = 128 / LPR;                                    // columns per lane
  const int G = prm.Hq / prm.Hkv;
  const int h = g * G + hh;
  const int e0 = valid ? prm.comb_off[seq] : 0, e1 = valid ? prm.comb_off[seq + 1] : 0;
  const int len = (valid && prm.Kc) ? slen.v[seq] : 0;
  const bool self_unit = has_self_unit(len, e1 - e0);
  const int n_inline = self_unit ? 0 : len;
  const int e_end = e1 + (self_unit ? 1 : 0);
  const int64_t pbase = (int64_t)g * prm.rows_total * kPartStride;
  const int64_t tq = valid ? prm.seq_off[seq] : 0;
  float Mx = -INFINITY, Ls = 0.f;
  float acc[NC];
#pragma unroll
  for (int i = 0; i < NC; ++i) acc[i] = 0.f;
  auto fold = [&](float m_p, float l_p, const float* v) {          // (acc, Ls, Mx) += one partial
    const float Mn = fmaxf(Mx, m_p);
    const float sc = ex2_approx(Mx - Mn), f = ex2_approx(m_p - Mn);
    Mx = Mn;
    Ls = Ls * sc + f * l_p;
#pragma unroll
    for (int i = 0; i < NC; ++i) acc[i] = acc[i] * sc + f * v[i];
  };
  for (int e = e0; e < e_end; e += 4) {
    const float* p[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int ee = e + u;
      p[u] = nullptr;
      if (ee < e_end) {
        const int pr = ee < e1 ? prm.comb_row[ee] : prm.self_row_base + seq;
        p[u] = prm.part + pbase + ((int64_t)pr * G + hh) * kPartStride;
      }
    }
    float2 mlp[4];
    float v[4][NC];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      mlp[u] = make_float2(-INFINITY, 0.f);
      if (p[u]) {
        mlp[u] = __ldcg(reinterpret_cast<const float2*>(p[u] + 128));
#pragma unroll
        for (int i = 0; i < NC; i += 4) {
          const float4 x = __ldcg(reinterpret_cast<const float4*>(p[u] + sub * NC + i));
          v[u][i] = x.x; v[u][i + 1] = x.y; v[u][i + 2] = x.z; v[u][i + 3] = x.w;
        }
      }
    }
#pragma unroll
    for (int u = 0; u < 4; ++u)
      if (p[u]) fold(mlp[u].x, mlp[u].y, v[u]);
  }
#pragma unroll
  for (int i = 0; i < kInlineSelf; ++i) {
    // the shuffles run with the full mask on every lane, whatever its row's n_inline
    float dot = 0.f;
    float vv[NC];
    if (i < n_inline) {
      const __nv_bfloat16* qp = prm.Q + (tq * prm.Hq + h) * 128 + sub * NC;
      const __nv_bfloat16* kp = prm.Kc + (((int64_t)seq * prm.cache_cap + i) * prm.Hkv + g) * 128 + sub * NC;
      const __nv_bfloat16* vp = prm.Vc + (((int64_t)seq * prm.cache_cap + i) * prm.Hkv + g) * 128 + sub * NC;
#pragma unroll
      for (int x = 0; x < NC; x += 4) {
        const uint2 qa = *reinterpret_cast<const uint2*>(qp + x), ka = *reinterpret_cast<const uint2*>(kp + x);
        const uint2 va = *reinterpret_cast<const uint2*>(vp + x);
        const float2 q0 = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&qa.x));
        const float2 q1 = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&qa.y));
        const float2 k0 = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&ka.x));
        const float2 k1 = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&ka.y));
        const float2 v0 = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&va.x));
        const float2 v1 = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&va.y));
        dot += q0.x * k0.x + q0.y * k0.y + q1.x * k1.x + q1.y * k1.y;
        vv[x] = v0.x; vv[x + 1] = v0.y; vv[x + 2] = v1.x; vv[x + 3] = v1.y;
      }
    }
#pragma unroll
    for (int o = LPR / 2; o > 0; o >>= 1) dot += __shfl_xor_sync(0xffffffffu, dot, o);
    if (i < n_inline) fold(dot * prm.scale_log2, 1.f, vv);
  }
  if (!valid) return;
  const float inv = 1.f / Ls;
  __nv_bfloat16* orow = prm.O + (tq * prm.Hq + h) * 128 + sub * NC;
#pragma unroll
  for (int x = 0; x < NC; x += 4) {
    uint2 o;
    o.x = pack_bf16(acc[x] * inv, acc[x + 1] * inv);
    o.y = pack_bf16(acc[x + 2] * inv, acc[x + 3] * inv);
    *reinterpret_cast<uint2*>(orow + x) = o;
  }
  if (sub == 0) prm.LSE[tq * prm.Hq + h] = Mx * 0.6931471805599453f + logf(Ls);
}

// Fused merge (small batches only -- a few sequences generating: at most kFusedOut output rows in all and row blocks of
// at most 32 rows): warp 11, after a segment's partials are written, counts them per row and merges the rows whose
// LAST partial this was, two rows at a time (sixteen lanes per row).  It saves the second launch of a latency-bound
// step.  Measured on the full-size top-8 config (2048 rows, 3-9 partials each) the same scheme is 2x SLOWER than a
// separate launch: one warp per CTA walks ~3 dependent L2 round trips per row, and the descriptor ring makes the
// whole pipeline wait for it -- so bigger batches use decode_combine_kernel (one warp per row, 2048 warps at once).
constexpr int kFusedRows = 32;
constexpr int kFusedOut = 256;
__device__ __forceinline__ void dec_count_and_merge(const DecParams& prm, const SelfLens& slen, const DecSeg d, const int lane) {
  const int G = prm.Hq / prm.Hkv;
  const int n_rows = d.n_seqs * G;
  __threadfence();     // after the barrier wait: covers the partial rows the softmax warpgroups have written
  int last = 0, seq = 0;
  if (lane < n_rows) {
    seq = d.kind == 0 ? prm.seqs[d.seq_off + lane / G] : d.seq_off;
    const int len = prm.Kc ? slen.v[seq] : 0;
    const int npre = prm.comb_off[seq + 1] - prm.comb_off[seq];
    const int expected = npre + (has_self_unit(len, npre) ? 1 : 0);
    last = atomicAdd(prm.cnt + ((int64_t)d.g * prm.B + seq) * G + lane % G, 1) == expected - 1;
    if (last) prm.cnt[((int64_t)d.g * prm.B + seq) * G + lane % G] = 0;      // re-arm for the next launch on this table
  }
  uint32_t todo = __ballot_sync(0xffffffffu, last);
  if (todo) __threadfence();
  while (todo) {
    // the (lane / 16)-th pending row goes to this half warp (sixteen lanes per row: eight columns each keep the
    // warp within its small register budget)
    uint32_t t = todo;
    int mine = -1;
    for (int q = 0; q < 2 && t; ++q) {
      const int bit = __ffs(t) - 1;
      if (q == (lane >> 4)) mine = bit;
      t &= t - 1;
    }
    todo = t;
    const int rseq = __shfl_sync(0xffffffffu, seq, mine < 0 ? 0 : mine);
    dec_merge_row<16>(prm, slen, d.g, rseq, (mine < 0 ? 0 : mine) % G, lane & 15, mine >= 0);
  }
}

// Tables with wider row blocks (c5 "all loaded": 128 rows with a dozen partials each, all finishing together) are
// merged by a second, massively parallel launch instead: one warp per output row.
__global__ void __launch_bounds__(256)
decode_combine_kernel(const __grid_constant__ DecParams prm, const __grid_constant__ SelfLens slen) {
  const int wrow = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (wrow >= prm.B * prm.Hq) return;
  const int G = prm.Hq / prm.Hkv;
  const int b = wrow / prm.Hq, h = wrow % prm.Hq;
  dec_merge_row<32>(prm, slen, h / G, b, h % G, lane, true);
}

__global__ void __launch_bounds__(kDecThreads, 1)
tc_decode_kernel(const __grid_constant__ CUtensorMap tmK, const __grid_constant__ CUtensorMap tmV,
                 const __grid_constant__ CUtensorMap tmKc, const __grid_constant__ CUtensorMap tmVc,
                 const __grid_constant__ CUtensorMap tmK16, const __grid_constant__ CUtensorMap tmV16,
                 const __grid_constant__ DecParams prm, const __grid_constant__ SelfLens slen) {
  extern __shared__ __align__(1024) uint8_t smem[];
  const uint32_t sbase = smem_u32(smem);
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + dOffBar + D_N * 8);
  auto bar = [&](int i) { return sbase + dOffBar + 8u * i; };
  const DecSeg* dring = reinterpret_cast<const DecSeg*>(smem + dOffDesc);
  const int warp = warp_id_uniform();
  const int G = prm.Hq / prm.Hkv;

  if (threadIdx.x == 0) {
    if (sbase & 1023u) __trap();
    for (int i = 0; i < D_N; ++i) {
      uint32_t c = 1;
      if (i == D_PF || i == D_PF + 1) c = 128;
      if (i == D_QF) c = 32;
      if (i >= D_DE) c = 3;
      if (i >= D_PW) c = 256;
      mbar_init(bar(i), c);
    }
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

  if (warp >= 8) {
    if (warp == 8) {
      // ===================================================================== scheduler + TMA producer
      if (elect_one()) {
        tma_prefetch_desc(&tmK);
        tma_prefetch_desc(&tmV);
        DecSeg* wring = reinterpret_cast<DecSeg*>(smem + dOffDesc);
        int nseg = 0, t = 0;
        // descriptors are published ONE SEGMENT AHEAD of the tile loads, so that warp 10 gathers the next segment's
        // query rows while the current segment still computes
        auto publish = [&](const DecSeg& d) {
          const int k = nseg & (kDescRing - 1);
          mbar_wait(bar(D_DE + k), ((nseg / kDescRing) & 1) ^ 1);
          wring[k] = d;
          mbar_arrive(bar(D_DF + k));
          ++nseg;
        };
        auto load_tiles = [&](const DecSeg& d) {
          const CUtensorMap* mk = d.kind != 1 ? &tmK : &tmKc;
          const CUtensorMap* mv = d.kind != 1 ? &tmV : &tmVc;
          for (int j = 0; j < d.n_tiles; ++j, ++t) {
            const int uk = 2 * t, uv = 2 * t + 1;                    // ring units of this tile's K and V
            const int sk = uk % kRing, sv = uv % kRing;
            const uint32_t kb = sbase + dOffKV + sk * dT, vb = sbase + dOffKV + sv * dT;
            const int tok = d.kind != 1 ? prm.tiles[d.tile_off + j].tok : d.seq_off * prm.cache_cap + 128 * j;
            const PackedTile* pt = (d.kind != 1 && tok < 0) ? prm.ptiles + (-1 - tok) : nullptr;
            mbar_wait(bar(D_RE + sk), ((uk / kRing) & 1) ^ 1);
            mbar_expect_tx(bar(D_RF + sk), dT);
            if (pt) {
              for (int u = 0; u < 8; ++u) {
                tma_load_3d(kb + u * 2048, &tmK16, bar(D_RF + sk), 0, d.g, pt->tok[u]);
                tma_load_3d(kb + dH + u * 2048, &tmK16, bar(D_RF + sk), 64, d.g, pt->tok[u]);
              }
            } else {
              tma_load_3d(kb, mk, bar(D_RF + sk), 0, d.g, tok);
              tma_load_3d(kb + dH, mk, bar(D_RF + sk), 64, d.g, tok);
            }
            mbar_wait(bar(D_RE + sv), ((uv / kRing) & 1) ^ 1);
            mbar_expect_tx(bar(D_RF + sv), dT);
            if (pt) {
              for (int u = 0; u < 8; ++u) {
                tma_load_3d(vb + u * 2048, &tmV16, bar(D_RF + sv), 0, d.g, pt->tok[u]);
                tma_load_3d(vb + dH + u * 2048, &tmV16, bar(D_RF + sv), 64, d.g, pt->tok[u]);
              }
            } else {
              tma_load_3d(vb, mv, bar(D_RF + sv), 0, d.g, tok);
              tma_load_3d(vb + dH, mv, bar(D_RF + sv), 64, d.g, tok);
            }
          }
        };
        // source of segments: this CTA's static list, then self-cache units (one per (sequence with a long cache, KV
        // head)) drawn from the ticket counter
        int sidx = prm.cta_seg_off[blockIdx.x];
        const int send = prm.cta_seg_off[blockIdx.x + 1];
        const int n_units = slen.n_useq * prm.Hkv;
        bool tickets_open = n_units > 0;
        auto next = [&](DecSeg& out) -> bool {
          if (sidx < send) { out = prm.segs[sidx++]; return true; }
          if (tickets_open) {
            const int u = atomicAdd(prm.ticket, 1);
            if (u < n_units) {
              const int b = slen.useq[u / prm.Hkv], len = slen.v[b];
              out = DecSeg{1, 0, (len + 127) >> 7, u % prm.Hkv, b, 1, prm.self_row_base + b, len};
              return true;
            }
            tickets_open = false;
            __threadfence();
            if (atomicAdd(prm.ticket + 1, 1) == (int)gridDim.x - 1) {   // every CTA has left the queue: re-arm
              prm.ticket[0] = 0;
              prm.ticket[1] = 0;
            }
          }
          return false;
        };
        const DecSeg stop{-1, 0, 0, 0, 0, 0, 0, 0};
        DecSeg cur, nxt;
        bool has_cur = next(cur);
        publish(has_cur ? cur : stop);
        while (has_cur) {
          const bool has_nxt = next(nxt);
          publish(has_nxt ? nxt : stop);
          load_tiles(cur);
          cur = nxt;
          has_cur = has_nxt;
        }
      }
    } else if (warp == 9) {
      // ===================================================================== MMA issuer
      if (elect_one()) {
        constexpr uint32_t idesc_qk = make_idesc(128, 128, 0, 0);
        constexpr uint32_t idesc_pv = make_idesc(128, 128, 0, 1);
        int t = 0, c0 = 0, c1 = 0;
        // S_w = Q_q K(tt)^T; K(tt) sits in ring unit 2 tt.  `release`: the K slot is free once this MMA is done.
        auto issue_qk = [&](int tt, int w, int q, bool wait_k, bool release) {
          const int u = 2 * tt, sl = u % kRing;
          if (wait_k) {
            mbar_wait(bar(D_RF + sl), (u / kRing) & 1);
            tc_fence_after();
          }
          const uint32_t qa = sbase + dOffQ + q * dT, ka = sbase + dOffKV + sl * dT;
#pragma unroll
          for (int kk = 0; kk < 8; ++kk) {
            const uint32_t o = (kk >> 2) * dH + (kk & 3) * 32;
            mma_ss(tbase + w * 128, desc_kmajor(qa + o), desc_kmajor(ka + o), idesc_qk, kk > 0);
          }
          mma_commit(bar(D_SF + w));
          if (release) mma_commit(bar(D_RE + sl));
        };
        // O_w (+)= P_w V(tt); V(tt) sits in ring unit 2 tt + 1
        auto issue_pv = [&](int tt, int w, bool wait_v, bool release, bool accum) {
          const int u = 2 * tt + 1, sl = u % kRing;
          if (wait_v) mbar_wait(bar(D_RF + sl), (u / kRing) & 1);
          tc_fence_after();
          const uint32_t va = sbase + dOffKV + sl * dT;
#pragma unroll
          for (int kk = 0; kk < 8; ++kk)
            mma_ts(tbase + 256 + w * 128, tbase + w * 128 + kk * 8, desc_mnmajor(va + kk * 2048, dH), idesc_pv,
                   (accum || kk > 0) ? 1u : 0u);
          if (release) mma_commit(bar(D_RE + sl));
          mma_commit(bar(D_OV + w));
        };
        for (int nseg = 0;; ++nseg) {
          const int k = nseg & (kDescRing - 1);
          mbar_wait(bar(D_DF + k), (nseg / kDescRing) & 1);
          const int n = dring[k].n_tiles;
          const int kind = dring[k].kind;
          if (kind < 0) break;
          mbar_wait(bar(D_QF), nseg & 1);
          tc_fence_after();
          if (kind == 2) {
            // PAIRED row blocks: Q tile A -> S0/O0 (warpgroup 0), Q tile B -> S1/O1 (warpgroup 1), every K/V tile is
            // fetched once and used by both:  PV_a(j) QK_a(j+1) PV_b(j) QK_b(j+1)
            issue_qk(t, 0, 0, true, false);
            issue_qk(t, 1, 1, false, true);
            if (n == 1) mma_commit(bar(D_QE));
            for (int j = 0; j < n; ++j) {
              mbar_wait(bar(D_PF), c0 & 1);
              ++c0;
              issue_pv(t + j, 0, true, false, j > 0);
              if (j + 1 < n) issue_qk(t + j + 1, 0, 0, true, false);
              mbar_wait(bar(D_PF + 1), c1 & 1);
              ++c1;
              issue_pv(t + j, 1, false, true, j > 0);
              if (j + 1 < n) {
                issue_qk(t + j + 1, 1, 1, false, true);
                if (j + 1 == n - 1) mma_commit(bar(D_QE));
              }
            }
          } else {
            // ONE row block: the warpgroups take alternate tiles
            issue_qk(t, 0, 0, true, true);
            if (n > 1) issue_qk(t + 1, 1, 0, true, true);
            if (n <= 2) mma_commit(bar(D_QE));
            for (int j = 0; j < n; ++j) {
              const int w = j & 1;
              mbar_wait(bar(D_PF + w), (w ? c1 : c0) & 1);
              if (w) ++c1; else ++c0;
              issue_pv(t + j, w, true, true, j >= 2);
              if (j + 2 < n) {
                issue_qk(t + j + 2, w, 0, true, true);
                if (j + 2 == n - 1) mma_commit(bar(D_QE));
              }
            }
          }
          t += n;
        }
      }
    } else {
      // ===================================================================== query gather + partial merge (warps 10, 11)
      const int lane = threadIdx.x & 31;
      if (warp == 10) {
        // ------------------------------------------------------------------- query gather: rows lane + 32 rr
        for (int nseg = 0;; ++nseg) {
          const int k = nseg & (kDescRing - 1);
          mbar_wait(bar(D_DF + k), (nseg / kDescRing) & 1);
          const DecSeg d = dring[k];
          if (d.kind < 0) break;
          mbar_wait(bar(D_QE), (nseg & 1) ^ 1);                      // the previous segment's last QK has read the tile
          // a paired segment (kind 2) has a second row block: sequences seq_off + n_seqs .., self_len of them -> Q tile B
          const int n_tiles_q = d.kind == 2 ? 2 : 1;
#pragma unroll 1
          for (int rr = 0; rr < 4 * n_tiles_q; ++rr) {
            const int qt = rr >> 2, r = lane + 32 * (rr & 3);
            const int n_rows = (qt ? d.self_len : d.n_seqs) * G;
            const uint4* src = nullptr;
            if (r < n_rows) {
              const int seq = d.kind != 1 ? prm.seqs[d.seq_off + (qt ? d.n_seqs : 0) + r / G] : d.seq_off, h = d.g * G + r % G;
              src = reinterpret_cast<const uint4*>(prm.Q + ((int64_t)prm.seq_off[seq] * prm.Hq + h) * 128);
            }
#pragma unroll
            for (int half = 0; half < 2; ++half) {
              uint4 q[8];
#pragma unroll
              for (int c = 0; c < 8; ++c) q[c] = src ? src[half * 8 + c] : make_uint4(0, 0, 0, 0);
#pragma unroll
              for (int c = 0; c < 8; ++c) {
                const uint32_t addr = sbase + dOffQ + qt * dT + half * dH + r * 128 + ((uint32_t)(c ^ (r & 7)) << 4);
                asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(q[c].x), "r"(q[c].y), "r"(q[c].z), "r"(q[c].w) : "memory");
              }
            }
          }
          fence_proxy_async();
          mbar_arrive(bar(D_QF));
        }
      } else {
        // ------------------------------------------------------------------- warp 11: count + merge (fused tables)
        for (int nseg = 0;; ++nseg) {
          const int k = nseg & (kDescRing - 1);
          mbar_wait(bar(D_DF + k), (nseg / kDescRing) & 1);
          const DecSeg d = dring[k];
          if (d.kind < 0) break;
          // one barrier per descriptor-ring slot: the writers cannot lap this wait (the slot is released below)
          mbar_wait(bar(D_PW + k), (nseg / kDescRing) & 1);
          if (prm.fused) dec_count_and_merge(prm, slen, d, lane);
          if (lane == 0) mbar_arrive(bar(D_DE + k));                 // last reader of the descriptor
        }
      }
    }
  } else {
    // ======================================================================= softmax warpgroups
    const int w = warp >> 2;                                         // warpgroup: tiles j = w, w + 2, ...
    const int r = threadIdx.x & 127;                                 // row = TMEM lane
    const uint32_t lane_base = (uint32_t)((warp & 3) * 32) << 16;
    const uint32_t tS = tbase + w * 128 + lane_base, tOw = tbase + 256 + w * 128 + lane_base;
    float2* ml = reinterpret_cast<float2*>(smem + dOffML);           // [2][128]
    int cme = 0, cother = 0;                                         // tiles this / the other warpgroup has handled
    for (int nseg = 0;; ++nseg) {
      const int k = nseg & (kDescRing - 1);
      mbar_wait(bar(D_DF + k), (nseg / kDescRing) & 1);
      const DecSeg d = dring[k];
      if (d.kind < 0) break;
      const int n = d.n_tiles;
      const bool paired = d.kind == 2;               // two row blocks: this warpgroup owns ONE of them and takes EVERY tile
      const int jstep = paired ? 1 : 2;
      float m = -INFINITY, l = 0.f;
      for (int j = paired ? 0 : w; j < n; j += jstep) {
        // key-valid bits of the tile, one word per 32-column chunk: a prefix of `limit` keys, or a packed tile's pages
        uint32_t mw[4];
        {
          const KvTile tl = d.kind != 1 ? prm.tiles[d.tile_off + j] : KvTile{0, min(128, d.self_len - 128 * j)};
          if (d.kind != 1 && tl.tok < 0) {
            const uint4 mk = *reinterpret_cast<const uint4*>(prm.ptiles[-1 - tl.tok].mask);
            mw[0] = mk.x; mw[1] = mk.y; mw[2] = mk.z; mw[3] = mk.w;
          } else {
#pragma unroll
            for (int c = 0; c < 4; ++c)
              mw[c] = tl.len >= 32 * (c + 1) ? 0xffffffffu : (tl.len > 32 * c ? (1u << (tl.len - 32 * c)) - 1u : 0u);
          }
        }
        const bool ragged = (mw[0] & mw[1] & mw[2] & mw[3]) != 0xffffffffu;
        mbar_wait(bar(D_SF + w), cme & 1);
        tc_fence_after();
        // Two passes over the 128 scores (row max, then exp) in 32-column chunks with the NEXT chunk's TMEM load in
        // flight while the current one is processed: 64 live registers instead of 128, no exposed TMEM latency.
        uint32_t buf[2][32];
        float mx0 = -INFINITY, mx1 = -INFINITY, mx2 = -INFINITY, mx3 = -INFINITY;   // four independent chains
        tmem_ld32(tS, buf[0]);
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          tc_wait_ld();
          if (c < 3) tmem_ld32(tS + 32 * (c + 1), buf[(c + 1) & 1]);
          uint32_t* s = buf[c & 1];
          if (ragged) {
#pragma unroll
            for (int cc = 0; cc < 32; ++cc)
              if (!((mw[c] >> cc) & 1u)) s[cc] = 0xff800000u;
          }
#pragma unroll
          for (int cc = 0; cc < 32; cc += 8) {
            mx0 = max3(mx0, __uint_as_float(s[cc]), __uint_as_float(s[cc + 1]));
            mx1 = max3(mx1, __uint_as_float(s[cc + 2]), __uint_as_float(s[cc + 3]));
            mx2 = max3(mx2, __uint_as_float(s[cc + 4]), __uint_as_float(s[cc + 5]));
            mx3 = max3(mx3, __uint_as_float(s[cc + 6]), __uint_as_float(s[cc + 7]));
          }
        }
        const float m_new = fmaxf(m, fmaxf(fmaxf(mx0, mx1), fmaxf(mx2, mx3)) * prm.scale_log2);
        if (j < jstep) {                             // this warpgroup's first tile of the segment
          m = m_new;
        } else if (__any_sync(0xffffffffu, m_new > m + 8.f)) {
          mbar_wait(bar(D_OV + w), (cme - 1) & 1);                   // this warpgroup's previous PV has updated O
          tc_fence_after();
          const float f = ex2_approx(m - m_new);
          m = m_new;
          l *= f;
#pragma unroll
          for (int cc = 0; cc < 4; ++cc) {
            uint32_t o[32];
            tmem_ld32(tOw + cc * 32, o);
            tc_wait_ld();
#pragma unroll
            for (int i = 0; i < 32; ++i) o[i] = __float_as_uint(__uint_as_float(o[i]) * f);
            tmem_st32(tOw + cc * 32, o);
            tc_wait_st();                            // the store has read o[] before the next chunk's load reuses it
          }
        }
        const uint64_t sc2 = pack2(prm.scale_log2, prm.scale_log2), nm2 = pack2(-m, -m);
        uint64_t sum2a = pack2(0.f, 0.f), sum2b = sum2a;
        tmem_ld32(tS, buf[0]);
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          tc_wait_ld();
          // buf[(c+1)&1] was the SOURCE of the P store of chunk c-1: that store must have read its registers before
          // the next load overwrites them
          if (c > 0) tc_wait_st();
          if (c < 3) tmem_ld32(tS + 32 * (c + 1), buf[(c + 1) & 1]);
          uint32_t* s = buf[c & 1];
          // the masked form is a separate copy of the loop: selects inside the common one cost the full tiles (all of
          // c5) a third of their exp phase
          auto exp_chunk = [&](auto masked_tag) {
            constexpr bool kMasked = decltype(masked_tag)::value;
#pragma unroll
            for (int i = 0; i < 16; i += 2) {
              float a0, a1, b0, b1;
              unpack2(fma2(pack2(__uint_as_float(s[2 * i]), __uint_as_float(s[2 * i + 1])), sc2, nm2), a0, a1);
              unpack2(fma2(pack2(__uint_as_float(s[2 * i + 2]), __uint_as_float(s[2 * i + 3])), sc2, nm2), b0, b1);
              a0 = ex2_approx(a0); a1 = ex2_approx(a1);
              if ((i & 6) != 6) exp2_poly2(b0, b1, b0, b1);    // 3 of every 8 scores on the FMA pipe
              else { b0 = ex2_approx(b0); b1 = ex2_approx(b1); }
              if (kMasked) {
                // a masked key weighs EXACTLY 0 (its raw score may be anything; its V row may be a stale cache row)
                a0 = (mw[c] >> (2 * i)) & 1u ? a0 : 0.f;
                a1 = (mw[c] >> (2 * i + 1)) & 1u ? a1 : 0.f;
                b0 = (mw[c] >> (2 * i + 2)) & 1u ? b0 : 0.f;
                b1 = (mw[c] >> (2 * i + 3)) & 1u ? b1 : 0.f;
              }
              sum2a = add2(sum2a, pack2(a0, a1));
              sum2b = add2(sum2b, pack2(b0, b1));
              s[i] = pack_bf16(a0, a1);
              s[i + 1] = pack_bf16(b0, b1);
            }
          };
          if (ragged) exp_chunk(std::true_type{});
          else exp_chunk(std::false_type{});
          tmem_st16(tS + 16 * c, s);                         // P of keys [32c, 32c+32) -> columns [16c, 16c+16)
        }
        {
          float x0, x1;
          unpack2(add2(sum2a, sum2b), x0, x1);
          l += x0 + x1;
        }
        tc_wait_st();
        tc_fence_before();
        mbar_arrive(bar(D_PF + w));
        ++cme;
      }
      cother += paired ? n : (n - (w ^ 1) + 1) >> 1;                // the other warpgroup's tiles of this segment
      if (paired) dec_paired_epilogue(prm, d, w, r, tbase, lane_base, m, l, cme, bar(D_OV + w));
      else dec_segment_epilogue(prm, d, w, r, tbase, lane_base, m, l, w ? cother : cme, w ? cme : cother, bar(D_OV), ml);
      mbar_arrive(bar(D_PW + k));                                    // warp 11 counts and merges (fused tables)
      if ((threadIdx.x & 127) == 0) mbar_arrive(bar(D_DE + k));
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 8) tmem_dealloc(tbase, 512);
}

// ------------------------------------------------------------------------------- host side
bool tc_decode_supported(const cas_pool* p, const cas_slot_table* t, int Hq) {
  if (!(p->desc.dtype == CAS_BF16 && p->desc.D == 128 && p->has_tma)) return false;
  if (t->max_lq != 1) return false;
  const int G = Hq / p->desc.Hkv;
  return G >= 1 && G <= 128;
}

// Groups the used slots by their set of selecting sequences, cuts every (group, row block, KV head) tile list into
// chunks of about total/#SM tiles, deals the resulting segments to the persistent CTAs and uploads the lists
// (asynchronously, through a pinned mirror) together with the partial-result scratch, the row counters and the
// ticket -- all library-owned, part of the slot table, freed with it.
static int decode_prepare(cas_slot_table* t, int Hq) {
  if (t->dec_Hq == Hq && t->d_dec_blob) return CAS_OK;
  if (t->d_dec_blob) {
    cudaDeviceSynchronize();
    cudaFree(t->d_dec_blob);
    cudaFreeHost(t->h_dec_blob);
    t->d_dec_blob = nullptr;
    t->h_dec_blob = nullptr;
  }
  const cas_pool* p = t->pool;
  const int Hkv = p->desc.Hkv, G = Hq / Hkv, R = 128 / G;
  int dev = 0, n_sm = 148;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
  std::map<std::vector<int32_t>, std::vector<int32_t>> groups;   // sequence set -> slots (ascending)
  for (int s : t->used_slots)
    groups[std::vector<int32_t>(t->inv_seq.begin() + t->inv_off[s], t->inv_seq.begin() + t->inv_off[s + 1])].push_back(s);
  int64_t units = 0;
  std::vector<std::vector<KvTile>> gtiles;
  std::vector<PackedTile> ptiles;
  for (auto& kv : groups) {
    std::vector<KvTile> tl;
    std::vector<std::pair<int32_t, int32_t>> pages;   // 16-token pages left over (pools with tile_tokens == 16)
    for (int s : kv.second) {
      const int len = p->cart_len[p->cart_in[s]], whole = p->pack ? len / 128 * 128 : len;
      for (int j = 0; j < whole; j += 128) tl.push_back({p->slot_base[s] + j, std::min(128, len - j)});
      for (int j = whole; j < len; j += 16) pages.push_back({p->slot_base[s] + j, std::min(16, len - j)});
    }
    for (size_t i = 0; i < pages.size(); i += 8) {      // the group's remainders share packed tiles
      PackedTile pt{};
      int nvalid = 0;
      for (int u = 0; u < 8; ++u) {
        const bool have = i + u < pages.size();
        pt.tok[u] = have ? pages[i + u].first : pages[i].first;
        const int cnt = have ? pages[i + u].second : 0;
        for (int x = 0; x < cnt; ++x) pt.mask[(16 * u + x) >> 5] |= 1u << ((16 * u + x) & 31);
        nvalid += cnt;
      }
      tl.push_back({-1 - (int32_t)ptiles.size(), nvalid});
      ptiles.push_back(pt);
    }
    // cost in tile times: a PAIR of row blocks shares every K/V tile in one CTA (4 MMAs per tile, ~1.5 tile times)
    const int64_t nrb = (int64_t)(kv.first.size() + R - 1) / R;
    units += ((nrb / 2) * 3 + (nrb & 1) * 2) * (int64_t)tl.size() * Hkv / 2;
    gtiles.push_back(std::move(tl));
  }
  const int64_t quota = std::max<int64_t>(1, (units + n_sm - 1) / n_sm);   // tiles per CTA
  std::vector<DecSeg> segs;
  std::vector<int32_t> seqs;
  std::vector<KvTile> tiles;
  std::vector<std::vector<int32_t>> comb(t->B);
  int32_t row_off = 0;
  size_t gi = 0;
  for (auto& kv : groups) {
    const std::vector<KvTile>& tl = gtiles[gi++];
    const int nt = (int)tl.size();
    // whole chunks of about `quota` tiles: the row blocks of one chunk land on CTAs that start together and walk the
    // same tiles at the same time, so a tile that several row blocks need is fetched from HBM once
    const bool pairs = kv.first.size() > (size_t)R;                 // two or more row blocks: pair them
    const int nchunk = (int)std::min<int64_t>(nt, std::max<int64_t>(1, (pairs ? (int64_t)nt * 3 / 2 : nt) / quota));   // rounded down: never more segments than CTAs' worth of work, never an empty one
    std::vector<int> seq_offs;
    for (size_t r0 = 0; r0 < kv.first.size(); r0 += R) {
      const int ns = (int)std::min<size_t>(R, kv.first.size() - r0);
      seq_offs.push_back((int)seqs.size());
      seqs.insert(seqs.end(), kv.first.begin() + r0, kv.first.begin() + r0 + ns);
    }
    const int to = (int)tiles.size();
    tiles.insert(tiles.end(), tl.begin(), tl.end());
    for (int c = 0; c < nchunk; ++c) {
      const int a = (int)((int64_t)nt * c / nchunk), b = (int)((int64_t)nt * (c + 1) / nchunk);
      for (size_t rb = 0; rb < seq_offs.size(); ++rb) {
        const size_t r0 = rb * R;
        const int ns = (int)std::min<size_t>(R, kv.first.size() - r0);
        if (rb + 1 < seq_offs.size()) {
          // row blocks rb and rb + 1 as ONE paired segment: both Q tiles resident, every K/V tile fetched once
          // (their sequences are consecutive in `seqs`, their partial rows consecutive from row_off)
          const int ns2 = (int)std::min<size_t>(R, kv.first.size() - r0 - R);
          for (int g = 0; g < Hkv; ++g) segs.push_back(DecSeg{2, to + a, b - a, g, seq_offs[rb], ns, row_off, ns2});
          for (int j = 0; j < ns + ns2; ++j) comb[kv.first[r0 + j]].push_back(row_off + j);
          row_off += ns + ns2;
          ++rb;
          continue;
        }
        for (int g = 0; g < Hkv; ++g) segs.push_back(DecSeg{0, to + a, b - a, g, seq_offs[rb], ns, row_off, 0});
        for (int j = 0; j < ns; ++j) comb[kv.first[r0 + j]].push_back(row_off + j);
        row_off += ns;
      }
    }
  }
  // deal the segments to the CTAs in order: a CTA is closed once it holds its share of what is left.  A segment
  // costs its tiles plus a fixed part (pipeline fill and drain, query gather, partial write: about two tile times)
  const int grid = n_sm;
  constexpr int64_t kSegCost = 2;    // measured at c5 top-8: 0.134 / 0.131 / 0.130 / 0.141 / 0.149 ms with 0 / 1 / 2 / 3 / 6
  std::vector<int32_t> cta_seg_off(grid + 1, 0);
  {
    int64_t total = 0;
    auto cost = [&](const DecSeg& sg) { return (sg.kind == 2 ? (int64_t)sg.n_tiles * 3 / 2 : sg.n_tiles) + kSegCost; };
    for (const DecSeg& sg : segs) total += cost(sg);
    int64_t load = 0, done = 0;
    int cta = 0;
    for (size_t i = 0; i < segs.size(); ++i) {
      const int64_t c = cost(segs[i]);
      const int64_t share = (total - done + (grid - cta) - 1) / std::max(1, grid - cta);
      if (load > 0 && load + c / 2 >= share && cta < grid - 1) {
        cta_seg_off[++cta] = (int32_t)i;
        done += load;
        load = 0;
      }
      load += c;
    }
    for (int c = cta + 1; c <= grid; ++c) cta_seg_off[c] = (int32_t)segs.size();
  }
  std::vector<int32_t> comb_off(t->B + 1, 0), comb_row;
  for (int b = 0; b < t->B; ++b) {
    comb_row.insert(comb_row.end(), comb[b].begin(), comb[b].end());
    comb_off[b + 1] = (int32_t)comb_row.size();
  }
  auto up = [](size_t x) { return (x + 255) / 256 * 256; };
  const size_t o_sg = 0, o_cs = up(segs.size() * sizeof(DecSeg) + 32), o_sq = o_cs + up(cta_seg_off.size() * 4),
               o_tl = o_sq + up(seqs.size() * 4 + 4), o_co = o_tl + up(tiles.size() * sizeof(KvTile) + 8),
               o_cr = o_co + up(comb_off.size() * 4), o_cn = o_cr + up(comb_row.size() * 4 + 4),
               o_tk = o_cn + up((size_t)t->B * Hq * 4), o_pk = o_tk + 256,
               o_pt = o_pk + up(ptiles.size() * sizeof(PackedTile) + 16);
  const int64_t part_rows = (int64_t)row_off + t->B;               // prefix partial rows + one self row per sequence
  const size_t part_bytes = (size_t)Hkv * part_rows * G * kPartStride * 4;
  cudaError_t e = cudaMalloc((void**)&t->d_dec_blob, o_pt + part_bytes + 256);
  if (e == cudaSuccess) e = cudaHostAlloc((void**)&t->h_dec_blob, o_pt, cudaHostAllocDefault);
  if (e == cudaSuccess && !t->dec_ready) e = cudaEventCreateWithFlags(&t->dec_ready, cudaEventDisableTiming);
  if (e != cudaSuccess) {
    if (t->d_dec_blob) cudaFree(t->d_dec_blob);
    if (t->h_dec_blob) cudaFreeHost(t->h_dec_blob);
    t->d_dec_blob = nullptr;
    t->h_dec_blob = nullptr;
    return cuda_fail(e, "decode table allocation");
  }
  char* h = t->h_dec_blob;
  memset(h, 0, o_pt);                                              // row counters and ticket start at zero
  if (!segs.empty()) memcpy(h + o_sg, segs.data(), segs.size() * sizeof(DecSeg));
  memcpy(h + o_cs, cta_seg_off.data(), cta_seg_off.size() * 4);
  if (!seqs.empty()) memcpy(h + o_sq, seqs.data(), seqs.size() * 4);
  if (!tiles.empty()) memcpy(h + o_tl, tiles.data(), tiles.size() * sizeof(KvTile));
  memcpy(h + o_co, comb_off.data(), comb_off.size() * 4);
  if (!comb_row.empty()) memcpy(h + o_cr, comb_row.data(), comb_row.size() * 4);
  if (!ptiles.empty()) memcpy(h + o_pk, ptiles.data(), ptiles.size() * sizeof(PackedTile));
  cudaStream_t up_st = t->pool->st_upload;
  e = cudaMemcpyAsync(t->d_dec_blob, h, o_pt, cudaMemcpyHostToDevice, up_st);
  if (e == cudaSuccess) e = cudaEventRecord(t->dec_ready, up_st);
  if (e != cudaSuccess) return cuda_fail(e, "decode table upload");
  char* d = t->d_dec_blob;
  t->d_dec_segs = (DecSeg*)(d + o_sg);
  t->d_dec_cta_off = (int32_t*)(d + o_cs);
  t->d_dec_seqs = (int32_t*)(d + o_sq);
  t->d_dec_tiles = (KvTile*)(d + o_tl);
  t->d_comb_off = (int32_t*)(d + o_co);
  t->d_comb_row = (int32_t*)(d + o_cr);
  t->d_dec_cnt = (int32_t*)(d + o_cn);
  t->d_dec_ticket = (int32_t*)(d + o_tk);
  t->d_dec_ptiles = (PackedTile*)(d + o_pk);
  t->d_dec_part = (float*)(d + o_pt);
  t->dec_comb_off = comb_off;
  t->dec_grid = grid;
  t->dec_rows = part_rows * G;
  t->dec_self_row_base = row_off;
  t->dec_n_segs = (int32_t)segs.size();
  t->dec_fused = t->B * Hq <= kFusedOut ? 1 : 0;
  for (const DecSeg& sg : segs)
    if (sg.n_seqs * G > kFusedRows || sg.kind == 2) t->dec_fused = 0;
  t->dec_Hq = Hq;
  return CAS_OK;
}

int tc_decode_fwd(const AttnArgs& a, const void* Kc, const void* Vc, int cache_cap, const int32_t* self_len) {
  cas_slot_table* t = const_cast<cas_slot_table*>(a.tab);
  if (Kc && t->B > kMaxDecB) { set_error("decode with a self cache takes at most %d sequences per call", kMaxDecB); return CAS_ERR_CAPACITY; }
  int rc = decode_prepare(t, a.Hq);
  if (rc) return rc;
  SelfLens sl;
  sl.n_useq = 0;
  for (int b = 0; b < t->B; ++b) {
    const int len = Kc ? self_len[b] : 0;
    const int npre = t->dec_comb_off[b + 1] - t->dec_comb_off[b];
    if (len < 0 || len > cache_cap) { set_error("self_len[%d] = %d outside [0, cache_cap]", b, len); return CAS_ERR_INVALID_ARG; }
    if (len == 0 && npre == 0) { set_error("sequence %d sees no key at all", b); return CAS_ERR_SHAPE; }
    if (b < kMaxDecB) {
      sl.v[b] = len;
      if (has_self_unit(len, npre)) sl.useq[sl.n_useq++] = b;
    }
  }
  static SmemAttrOnce attr;
  rc = attr.set((const void*)tc_decode_kernel, (int)kDecSmem);
  if (rc) return rc;
  CAS_CUDA(cudaStreamWaitEvent(a.stream, t->dec_ready, 0));
  CUtensorMap tmKc = a.L->tm_K, tmVc = a.L->tm_V;
  if (Kc) {
    rc = make_thd_map(&tmKc, Kc, (int64_t)t->B * cache_cap, a.Hkv, 128);
    if (rc) return rc;
    rc = make_thd_map(&tmVc, Vc, (int64_t)t->B * cache_cap, a.Hkv, 128);
    if (rc) return rc;
  }
  const float scale_log2 = a.scale * 1.4426950408889634f;
  DecParams prm{t->d_dec_segs, t->d_dec_cta_off, t->d_dec_seqs, t->d_dec_tiles, t->d_dec_ptiles, t->d_seq_off, t->d_comb_off,
                t->d_comb_row, (const __nv_bfloat16*)a.Q, (const __nv_bfloat16*)Kc, (const __nv_bfloat16*)Vc,
                (__nv_bfloat16*)a.O_out, a.LSE_out, t->d_dec_part, t->d_dec_cnt, t->d_dec_ticket, t->dec_rows,
                t->dec_self_row_base, cache_cap, t->B, a.Hq, a.Hkv, t->dec_fused, scale_log2};
  tc_decode_kernel<<<(unsigned)t->dec_grid, kDecThreads, kDecSmem, a.stream>>>(a.L->tm_K, a.L->tm_V, tmKc, tmVc, a.L->tm_K16,
                                                                               a.L->tm_V16, prm, sl);
  if (!t->dec_fused) {
    const int n_w = t->B * a.Hq;
    decode_combine_kernel<<<(n_w * 32 + 255) / 256, 256, 0, a.stream>>>(prm, sl);
  }
  cudaError_t e = cudaGetLastError();
  return e == cudaSuccess ? CAS_OK : cuda_fail(e, "tc decode launch");
}

}  // namespace cas
