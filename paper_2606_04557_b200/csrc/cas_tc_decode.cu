// Prefix-attention FORWARD for decode-shaped batches (every sequence has exactly ONE query token;
// BASELINE.json configs[4], PAPER.md:111 inference over all loaded cartridges, :142 retrieval-selected
// variant), bf16, head_dim 128, tcgen05 + TMEM + TMA.
//
// The work is HBM-bound (each K/V byte is used by G query heads of a few sequences), so the kernel
// is organised to read every selected K/V tile from HBM as few times as possible and to keep every
// SM streaming:
//  * KV-stationary batching through the INVERTED slot table: slots with the same set of selecting
//    sequences form a group; the rows of an MMA tile are (sequence, head-of-group) pairs -- up to
//    128/G sequences x G heads -- so one pass over a K/V tile serves all of them (c5 "all loaded":
//    64 sequences x 4 heads = two 128-row blocks share each tile; the second read hits L2).
//  * split-KV: a group's tile list is cut into chunks so that the grid has a few CTAs per SM; each
//    CTA writes an un-normalised partial (O, m, l) per row and decode_combine_kernel merges the
//    partials of a (sequence, head) and adds the query's own key/value (the 1-token causal block).
// CTA: warps 0-3 softmax (thread = row = TMEM lane), 4 TMA producer, 5 MMA issuer.
// SMEM: Q tile 32 KB (gathered rows, written by the softmax warps) + 3-stage K/V ring 192 KB.
// TMEM: S0 | S1 | O (fp32, 128 columns each); QK(j+1) is issued before PV(j) into the other S buffer.
#include <algorithm>
#include <map>

#include "cas_sm100.cuh"
#include "cas_tc_common.cuh"

namespace cas {
using namespace sm100;

constexpr int kDecThreads = 192;
constexpr int kDecStages = 3;
constexpr uint32_t dT = 32768, dH = 16384;
constexpr uint32_t dOffQ = 0, dOffKV = dT, dOffBar = dT + kDecStages * 2 * dT;
constexpr uint32_t kDecSmem = dOffBar + 256;
enum { D_KF = 0, D_KE = 3, D_VF = 6, D_VE = 9, D_SF = 12, D_PF = 14, D_QR = 16, D_OV = 17, D_OD = 18, D_N = 19 };
constexpr int kPartStride = 132;   // 128 O + m + l + pad (16-byte aligned rows)

struct DecParams {
  const DecItem* items;
  const int32_t* seqs;          // row-block sequence lists
  const KvTile* tiles;
  const int32_t* seq_off;
  const __nv_bfloat16* Q;
  float* part;
  int64_t rows_total;           // partial rows per KV head
  int Hq, Hkv;
  float scale_log2;
};

__global__ void __launch_bounds__(kDecThreads, 1)
tc_decode_kernel(const __grid_constant__ CUtensorMap tmK, const __grid_constant__ CUtensorMap tmV, const DecParams prm) {
  extern __shared__ __align__(1024) uint8_t smem[];
  const uint32_t sbase = smem_u32(smem);
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + dOffBar + D_N * 8);
  auto bar = [&](int i) { return sbase + dOffBar + 8u * i; };
  const int warp = warp_id_uniform(), lane = threadIdx.x & 31;
  const int g = blockIdx.x % prm.Hkv, G = prm.Hq / prm.Hkv;
  const DecItem it = prm.items[blockIdx.x / prm.Hkv];
  const KvTile* tiles = prm.tiles + it.tile_off;
  const int n = it.n_tiles;

  if (threadIdx.x == 0) {
    if (sbase & 1023u) __trap();
    for (int i = 0; i < D_N; ++i) mbar_init(bar(i), (i == D_PF || i == D_PF + 1 || i == D_QR) ? 128 : 1);
    fence_mbar_init();
  }
  if (warp == 4) {
    tmem_alloc(smem_u32(tmem_slot), 512);
    tmem_relinquish();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tbase = *tmem_slot;
  const uint32_t tO = tbase + 256;

  if (warp == 4) {
    // ===================================================================== TMA producer
    if (elect_one()) {
      tma_prefetch_desc(&tmK);
      tma_prefetch_desc(&tmV);
      for (int j = 0; j < n; ++j) {
        const int s = j % kDecStages;
        const uint32_t ph = (j / kDecStages) & 1;
        const uint32_t kb = sbase + dOffKV + s * 2 * dT, vb = kb + dT;
        const int tok = tiles[j].tok;
        mbar_wait(bar(D_KE + s), ph ^ 1);
        mbar_expect_tx(bar(D_KF + s), dT);
        tma_load_3d(kb, &tmK, bar(D_KF + s), 0, g, tok);
        tma_load_3d(kb + dH, &tmK, bar(D_KF + s), 64, g, tok);
        mbar_wait(bar(D_VE + s), ph ^ 1);
        mbar_expect_tx(bar(D_VF + s), dT);
        tma_load_3d(vb, &tmV, bar(D_VF + s), 0, g, tok);
        tma_load_3d(vb + dH, &tmV, bar(D_VF + s), 64, g, tok);
      }
    }
  } else if (warp == 5) {
    // ===================================================================== MMA issuer
    if (elect_one()) {
      constexpr uint32_t idesc_qk = make_idesc(128, 128, 0, 0);
      constexpr uint32_t idesc_pv = make_idesc(128, 128, 0, 1);
      auto issue_qk = [&](int j) {
        const uint32_t qa = sbase + dOffQ, ka = sbase + dOffKV + (j % kDecStages) * 2 * dT;
#pragma unroll
        for (int kk = 0; kk < 8; ++kk) {
          const uint32_t o = (kk >> 2) * dH + (kk & 3) * 32;
          mma_ss(tbase + (j & 1) * 128, desc_kmajor(qa + o), desc_kmajor(ka + o), idesc_qk, kk > 0);
        }
      };
      mbar_wait(bar(D_QR), 0);
      mbar_wait(bar(D_KF), 0);
      tc_fence_after();
      issue_qk(0);
      mma_commit(bar(D_SF));
      mma_commit(bar(D_KE));
      for (int j = 0; j < n; ++j) {
        if (j + 1 < n) {
          const int s1 = (j + 1) % kDecStages;
          mbar_wait(bar(D_KF + s1), ((j + 1) / kDecStages) & 1);
          tc_fence_after();
          issue_qk(j + 1);
          mma_commit(bar(D_SF + ((j + 1) & 1)));
          mma_commit(bar(D_KE + s1));
        }
        const int s = j % kDecStages;
        mbar_wait(bar(D_PF + (j & 1)), (j >> 1) & 1);
        mbar_wait(bar(D_VF + s), (j / kDecStages) & 1);
        tc_fence_after();
        const uint32_t va = sbase + dOffKV + s * 2 * dT + dT;
#pragma unroll
        for (int kk = 0; kk < 8; ++kk)
          mma_ts(tO, tbase + (j & 1) * 128 + kk * 8, desc_mnmajor(va + kk * 2048, dH), idesc_pv, (j > 0 || kk > 0) ? 1u : 0u);
        mma_commit(bar(D_VE + s));
        mma_commit(bar(D_OV));
      }
      mma_commit(bar(D_OD));
    }
  } else {
    // ===================================================================== softmax + partial write
    const int r = threadIdx.x;                                   // row = TMEM lane
    const int n_rows = it.n_seqs * G;
    const uint32_t lane_base = (uint32_t)(warp * 32) << 16;
    {
      // gather this row's query: (sequence j, head g*G + h') -> 256 bytes into the swizzled K-major tile
      uint4 q[16];
      if (r < n_rows) {
        const int seq = prm.seqs[it.seq_off + r / G], h = g * G + r % G;
        const uint4* src = reinterpret_cast<const uint4*>(prm.Q + ((int64_t)prm.seq_off[seq] * prm.Hq + h) * 128);
#pragma unroll
        for (int c = 0; c < 16; ++c) q[c] = src[c];
      } else {
#pragma unroll
        for (int c = 0; c < 16; ++c) q[c] = make_uint4(0, 0, 0, 0);
      }
#pragma unroll
      for (int c = 0; c < 16; ++c) {
        const uint32_t addr = sbase + dOffQ + (c >> 3) * dH + r * 128 + ((uint32_t)((c & 7) ^ (r & 7)) << 4);
        asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(q[c].x), "r"(q[c].y), "r"(q[c].z), "r"(q[c].w) : "memory");
      }
      fence_proxy_async();
      mbar_arrive(bar(D_QR));
    }
    float m = -INFINITY, l = 0.f;
    for (int j = 0; j < n; ++j) {
      const uint32_t tS = tbase + (j & 1) * 128 + lane_base;
      const int limit = tiles[j].len;
      mbar_wait(bar(D_SF + (j & 1)), (j >> 1) & 1);
      tc_fence_after();
      uint32_t s[128];
      tmem_ld32(tS, s);
      tmem_ld32(tS + 32, s + 32);
      tmem_ld32(tS + 64, s + 64);
      tmem_ld32(tS + 96, s + 96);
      tc_wait_ld();
      if (limit < 128) {
#pragma unroll
        for (int c = 0; c < 128; ++c)
          if (c >= limit) s[c] = 0xff800000u;
      }
      float mx0 = -INFINITY, mx1 = -INFINITY, mx2 = -INFINITY, mx3 = -INFINITY;   // four independent chains
#pragma unroll
      for (int c = 0; c < 128; c += 8) {
        mx0 = max3(mx0, __uint_as_float(s[c]), __uint_as_float(s[c + 1]));
        mx1 = max3(mx1, __uint_as_float(s[c + 2]), __uint_as_float(s[c + 3]));
        mx2 = max3(mx2, __uint_as_float(s[c + 4]), __uint_as_float(s[c + 5]));
        mx3 = max3(mx3, __uint_as_float(s[c + 6]), __uint_as_float(s[c + 7]));
      }
      const float m_new = fmaxf(m, fmaxf(fmaxf(mx0, mx1), fmaxf(mx2, mx3)) * prm.scale_log2);
      if (j == 0) {
        m = m_new;
      } else if (__any_sync(0xffffffffu, m_new > m + 8.f)) {
        mbar_wait(bar(D_OV), (j - 1) & 1);                       // PV(j-1) has finished updating O
        tc_fence_after();
        const float f = ex2_approx(m - m_new);
        m = m_new;
        l *= f;
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          uint32_t o[32];
          tmem_ld32(tO + lane_base + c * 32, o);
          tc_wait_ld();
#pragma unroll
          for (int i = 0; i < 32; ++i) o[i] = __float_as_uint(__uint_as_float(o[i]) * f);
          tmem_st32(tO + lane_base + c * 32, o);
        }
      }
      const uint64_t sc2 = pack2(prm.scale_log2, prm.scale_log2), nm2 = pack2(-m, -m);
      uint64_t sum2a = pack2(0.f, 0.f), sum2b = sum2a;
#pragma unroll
      for (int i = 0; i < 64; i += 2) {
        float a0, a1, b0, b1;
        unpack2(fma2(pack2(__uint_as_float(s[2 * i]), __uint_as_float(s[2 * i + 1])), sc2, nm2), a0, a1);
        unpack2(fma2(pack2(__uint_as_float(s[2 * i + 2]), __uint_as_float(s[2 * i + 3])), sc2, nm2), b0, b1);
        a0 = ex2_approx(a0); a1 = ex2_approx(a1);
        if ((i & 6) != 6) exp2_poly2(b0, b1, b0, b1);    // 3 of every 8 scores on the FMA pipe
        else { b0 = ex2_approx(b0); b1 = ex2_approx(b1); }
        sum2a = add2(sum2a, pack2(a0, a1));
        sum2b = add2(sum2b, pack2(b0, b1));
        s[i] = pack_bf16(a0, a1);
        s[i + 1] = pack_bf16(b0, b1);
      }
      {
        float x0, x1;
        unpack2(add2(sum2a, sum2b), x0, x1);
        l += x0 + x1;
      }
      tmem_st32(tS, s);
      tmem_st32(tS + 32, s + 32);
      tc_wait_st();
      tc_fence_before();
      mbar_arrive(bar(D_PF + (j & 1)));
    }
    mbar_wait(bar(D_OD), 0);
    tc_fence_after();
    float* prow = prm.part + ((int64_t)g * prm.rows_total + (int64_t)it.row_off * G + r) * kPartStride;
#pragma unroll
    for (int c = 0; c < 4; ++c) {
      uint32_t o[32];
      tmem_ld32(tO + lane_base + c * 32, o);
      tc_wait_ld();
      if (r < n_rows) {
#pragma unroll
        for (int i = 0; i < 8; ++i)
          *reinterpret_cast<float4*>(prow + c * 32 + 4 * i) =
              make_float4(__uint_as_float(o[4 * i]), __uint_as_float(o[4 * i + 1]), __uint_as_float(o[4 * i + 2]),
                          __uint_as_float(o[4 * i + 3]));
      }
    }
    if (r < n_rows) *reinterpret_cast<float2*>(prow + 128) = make_float2(m, l);
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 4) tmem_dealloc(tbase, 512);
}

// Merges the split-KV partials of one (sequence, head) and adds the query's own key/value (the
// causal self block of a 1-token sequence).  One warp per (sequence, head); lane = 4 columns.
__global__ void __launch_bounds__(256)
decode_combine_kernel(const float* __restrict__ part, const int32_t* __restrict__ comb_off,
                      const int32_t* __restrict__ comb_row, const int32_t* __restrict__ seq_off,
                      const __nv_bfloat16* __restrict__ Q, const __nv_bfloat16* __restrict__ Ks,
                      const __nv_bfloat16* __restrict__ Vs, __nv_bfloat16* __restrict__ O, float* __restrict__ LSE,
                      int64_t rows_total, int B, int Hq, int Hkv, float scale_log2) {
  const int w = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (w >= B * Hq) return;
  const int b = w / Hq, h = w % Hq, G = Hq / Hkv, g = h / G;
  const int64_t t = seq_off[b];
  const int e0 = comb_off[b], e1 = comb_off[b + 1];
  float M = -INFINITY, s_self = -INFINITY;
  if (Ks != nullptr) {
    const uint2 qa = *reinterpret_cast<const uint2*>(Q + (t * Hq + h) * 128 + lane * 4);
    const uint2 ka = *reinterpret_cast<const uint2*>(Ks + (t * Hkv + g) * 128 + lane * 4);
    const float2 q0 = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&qa.x));
    const float2 q1 = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&qa.y));
    const float2 k0 = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&ka.x));
    const float2 k1 = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&ka.y));
    float d = q0.x * k0.x + q0.y * k0.y + q1.x * k1.x + q1.y * k1.y;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) d += __shfl_xor_sync(0xffffffffu, d, o);
    s_self = d * scale_log2;
    M = s_self;
  }
  for (int e = e0; e < e1; ++e)
    M = fmaxf(M, part[((int64_t)g * rows_total + (int64_t)comb_row[e] * G + h % G) * kPartStride + 128]);
  float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
  float L = 0.f;
  for (int e = e0; e < e1; ++e) {
    const float* p = part + ((int64_t)g * rows_total + (int64_t)comb_row[e] * G + h % G) * kPartStride;
    const float f = ex2_approx(p[128] - M);
    const float4 v = *reinterpret_cast<const float4*>(p + lane * 4);
    acc.x += f * v.x; acc.y += f * v.y; acc.z += f * v.z; acc.w += f * v.w;
    L += f * p[129];
  }
  if (Ks != nullptr) {
    const float f = ex2_approx(s_self - M);
    const uint2 va = *reinterpret_cast<const uint2*>(Vs + (t * Hkv + g) * 128 + lane * 4);
    const float2 v0 = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&va.x));
    const float2 v1 = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&va.y));
    acc.x += f * v0.x; acc.y += f * v0.y; acc.z += f * v1.x; acc.w += f * v1.y;
    L += f;
  }
  const float inv = 1.f / L;
  uint2 o;
  o.x = pack_bf16(acc.x * inv, acc.y * inv);
  o.y = pack_bf16(acc.z * inv, acc.w * inv);
  *reinterpret_cast<uint2*>(O + (t * Hq + h) * 128 + lane * 4) = o;
  if (lane == 0) LSE[t * Hq + h] = M * 0.6931471805599453f + logf(L);
}

// ------------------------------------------------------------------------------- host side
bool tc_decode_supported(const cas_pool* p, const cas_slot_table* t, int Hq) {
  if (!(p->desc.dtype == CAS_BF16 && p->desc.D == 128 && p->has_tma)) return false;
  if (t->max_lq != 1 || t->nsel == 0) return false;
  const int G = Hq / p->desc.Hkv;
  return G >= 1 && G <= 128;
}

// Groups the used slots by their set of selecting sequences, cuts every group into row blocks of
// 128/G sequences and chunks of KV tiles, and uploads the item / sequence / tile / combine lists plus
// the partial-result scratch (library-owned, part of the slot table, freed with it).
static int decode_prepare(cas_slot_table* t, int Hq) {
  if (t->dec_Hq == Hq && t->d_dec_blob) return CAS_OK;
  if (t->d_dec_blob) { cudaDeviceSynchronize(); cudaFree(t->d_dec_blob); t->d_dec_blob = nullptr; }
  const cas_pool* p = t->pool;
  const int Hkv = p->desc.Hkv, G = Hq / Hkv, R = 128 / G;
  std::map<std::vector<int32_t>, std::vector<int32_t>> groups;   // sequence set -> slots (ascending)
  for (int s : t->used_slots)
    groups[std::vector<int32_t>(t->inv_seq.begin() + t->inv_off[s], t->inv_seq.begin() + t->inv_off[s + 1])].push_back(s);
  int64_t units = 0;
  std::vector<std::vector<KvTile>> gtiles;
  for (auto& kv : groups) {
    std::vector<KvTile> tl;
    for (int s : kv.second) {
      const int len = p->cart_len[p->cart_in[s]];
      for (int j = 0; j < len; j += 128) tl.push_back({p->slot_base[s] + j, std::min(128, len - j)});
    }
    units += (int64_t)((kv.first.size() + R - 1) / R) * (int64_t)tl.size();
    gtiles.push_back(std::move(tl));
  }
  const int64_t target = std::max<int64_t>(1, (148 * 4) / Hkv);          // CTAs per KV head: ~4 per SM in total
  const int64_t C = std::max<int64_t>(4, (units + target - 1) / target);  // tiles per chunk
  std::vector<DecItem> items;
  std::vector<int32_t> seqs;
  std::vector<KvTile> tiles;
  std::vector<std::vector<int32_t>> comb(t->B);
  int32_t row_off = 0;
  size_t gi = 0;
  for (auto& kv : groups) {
    const std::vector<KvTile>& tl = gtiles[gi++];
    const int nt = (int)tl.size();
    const int nchunk = (int)((nt + C - 1) / C);
    // chunk-major: the row blocks that share a chunk of tiles get adjacent block indices, so they run in the
    // same wave and the second read of a K/V tile hits L2 instead of HBM
    std::vector<int> seq_offs;
    for (size_t r0 = 0; r0 < kv.first.size(); r0 += R) {
      const int ns = (int)std::min<size_t>(R, kv.first.size() - r0);
      seq_offs.push_back((int)seqs.size());
      seqs.insert(seqs.end(), kv.first.begin() + r0, kv.first.begin() + r0 + ns);
    }
    for (int c = 0; c < nchunk; ++c) {
      const int a = (int)((int64_t)nt * c / nchunk), b = (int)((int64_t)nt * (c + 1) / nchunk);
      const int to = (int)tiles.size();
      tiles.insert(tiles.end(), tl.begin() + a, tl.begin() + b);
      for (size_t rb = 0; rb < seq_offs.size(); ++rb) {
        const size_t r0 = rb * R;
        const int ns = (int)std::min<size_t>(R, kv.first.size() - r0);
        items.push_back({seq_offs[rb], ns, to, b - a, row_off, {0, 0, 0}});
        for (int j = 0; j < ns; ++j) comb[kv.first[r0 + j]].push_back(row_off + j);
        row_off += ns;
      }
    }
  }
  std::stable_sort(items.begin(), items.end(), [](const DecItem& a, const DecItem& b) { return a.n_tiles > b.n_tiles; });
  std::vector<int32_t> comb_off(t->B + 1, 0), comb_row;
  for (int b = 0; b < t->B; ++b) {
    comb_row.insert(comb_row.end(), comb[b].begin(), comb[b].end());
    comb_off[b + 1] = (int32_t)comb_row.size();
  }
  auto up = [](size_t x) { return (x + 255) / 256 * 256; };
  const size_t o_it = 0, o_sq = up(items.size() * sizeof(DecItem)), o_tl = o_sq + up(seqs.size() * 4),
               o_co = o_tl + up(tiles.size() * sizeof(KvTile)), o_cr = o_co + up(comb_off.size() * 4),
               o_pt = o_cr + up(comb_row.size() * 4 + 4);
  const size_t part_bytes = (size_t)Hkv * row_off * G * kPartStride * 4;
  std::vector<char> h(o_pt, 0);
  memcpy(h.data() + o_it, items.data(), items.size() * sizeof(DecItem));
  memcpy(h.data() + o_sq, seqs.data(), seqs.size() * 4);
  memcpy(h.data() + o_tl, tiles.data(), tiles.size() * sizeof(KvTile));
  memcpy(h.data() + o_co, comb_off.data(), comb_off.size() * 4);
  if (!comb_row.empty()) memcpy(h.data() + o_cr, comb_row.data(), comb_row.size() * 4);
  cudaError_t e = cudaMalloc((void**)&t->d_dec_blob, o_pt + part_bytes + 256);
  if (e == cudaSuccess) e = cudaMemcpy(t->d_dec_blob, h.data(), o_pt, cudaMemcpyHostToDevice);
  if (e != cudaSuccess) { if (t->d_dec_blob) cudaFree(t->d_dec_blob); t->d_dec_blob = nullptr; return cuda_fail(e, "decode table upload"); }
  char* d = t->d_dec_blob;
  t->d_dec_items = (DecItem*)(d + o_it);
  t->d_dec_seqs = (int32_t*)(d + o_sq);
  t->d_dec_tiles = (KvTile*)(d + o_tl);
  t->d_comb_off = (int32_t*)(d + o_co);
  t->d_comb_row = (int32_t*)(d + o_cr);
  t->d_dec_part = (float*)(d + o_pt);
  t->dec_items = std::move(items);
  t->dec_rows = (int64_t)row_off * G;
  t->dec_Hq = Hq;
  return CAS_OK;
}

int tc_decode_fwd(const AttnArgs& a) {
  cas_slot_table* t = const_cast<cas_slot_table*>(a.tab);
  int rc = decode_prepare(t, a.Hq);
  if (rc) return rc;
  static SmemAttrOnce attr;
  {
    const int rc_attr = attr.set((const void*)tc_decode_kernel, (int)kDecSmem);
    if (rc_attr) return rc_attr;
  }
  const float scale_log2 = a.scale * 1.4426950408889634f;
  DecParams prm{t->d_dec_items, t->d_dec_seqs, t->d_dec_tiles, t->d_seq_off, (const __nv_bfloat16*)a.Q,
                t->d_dec_part, t->dec_rows, a.Hq, a.Hkv, scale_log2};
  const unsigned grid = (unsigned)(t->dec_items.size() * a.Hkv);
  tc_decode_kernel<<<grid, kDecThreads, kDecSmem, a.stream>>>(a.pool->tm_K, a.pool->tm_V, prm);
  const int n_w = t->B * a.Hq;
  decode_combine_kernel<<<(n_w * 32 + 255) / 256, 256, 0, a.stream>>>(
      t->d_dec_part, t->d_comb_off, t->d_comb_row, t->d_seq_off, (const __nv_bfloat16*)a.Q,
      (const __nv_bfloat16*)a.Ks, (const __nv_bfloat16*)a.Vs, (__nv_bfloat16*)a.O_out, a.LSE_out, t->dec_rows, t->B,
      a.Hq, a.Hkv, scale_log2);
  cudaError_t e = cudaGetLastError();
  return e == cudaSuccess ? CAS_OK : cuda_fail(e, "tc decode launch");
}

}  // namespace cas
