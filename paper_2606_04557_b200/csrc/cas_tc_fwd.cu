// Prefix-attention FORWARD on the 5th-gen tensor cores (tcgen05 + TMEM + TMA), bf16, head_dim 128.
//
// Definition: include/cas.h cas_prefix_attn_fwd.  The selected cartridges
// are never concatenated: the TMA producer walks the per-sequence KV tile list (slot table) and
// fetches 128-key tiles IN PLACE from the pool, then the sequence's own K/V tiles up to the
// diagonal.
//
// CTA = (256 query rows of one sequence) x (one query head) = two 128-row Q tiles that ping-pong on
// the tensor pipe.  Warps: 0-3 softmax of tile 0, 4-7 softmax of tile 1 (thread = row = TMEM lane),
// 8 TMA producer, 9 MMA issuer (one elected lane).
// TMEM (512 cols): S0 | S1 | O0 | O1, fp32 128 columns each; P (bf16, 64 cols) overwrites S in place
// and is fed back as the A operand of O += P*V straight from TMEM.
// SMEM (192 KB): Q0 Q1 | K ring x2 | V ring x2, all 128x128 bf16 tiles in two 128B-swizzled halves.
// Issue order per KV tile j:  PV0(j) QK0(j+1) PV1(j) QK1(j+1)  so that the softmax of one Q tile
// runs under the MMAs of the other.  Online softmax in the log2 domain with lazy rescaling (O is only
// rescaled when the running max grows by more than 2^8).
#include "cas_sm100.cuh"
#include "cas_tc_common.cuh"
#include <algorithm>
#include <cstdlib>
#include <mutex>
#include <vector>

namespace cas {
using namespace sm100;

// ------------------------------------------------------------------------------- host helpers
TmaEncodeFn tma_encoder() {
  static TmaEncodeFn fn = nullptr;
  if (!fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = (TmaEncodeFn)p;
  }
  return fn;
}

int make_thd_map(CUtensorMap* out, const void* base, int64_t tokens, int heads, int box_tokens) {
  TmaEncodeFn enc = tma_encoder();
  if (!enc) { set_error("cuTensorMapEncodeTiled unavailable"); return CAS_ERR_CUDA; }
  cuuint64_t dims[3] = {128, (cuuint64_t)heads, (cuuint64_t)tokens};
  cuuint64_t strides[2] = {128 * 2, (cuuint64_t)heads * 128 * 2};
  cuuint32_t box[3] = {64, 1, (cuuint32_t)box_tokens};
  cuuint32_t es[3] = {1, 1, 1};
  CUresult r = enc(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(base), dims, strides, box, es,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) { set_error("cuTensorMapEncodeTiled failed (%d)", (int)r); return CAS_ERR_CUDA; }
  return CAS_OK;
}

int tc_make_pool_maps(cas_pool* p) {
  for (PoolLayer& L : p->layers) {
    int rc = make_thd_map(&L.tm_K, L.pool_K, p->pool_tokens, p->desc.Hkv, 128);
    if (rc) return rc;
    rc = make_thd_map(&L.tm_V, L.pool_V, p->pool_tokens, p->desc.Hkv, 128);
    if (rc) return rc;
    rc = make_thd_map(&L.tm_K16, L.pool_K, p->pool_tokens, p->desc.Hkv, 16);
    if (rc) return rc;
    rc = make_thd_map(&L.tm_V16, L.pool_V, p->pool_tokens, p->desc.Hkv, 16);
    if (rc) return rc;
  }
  p->has_tma = true;
  return CAS_OK;
}

bool tc_supported(const cas_pool* p, const cas_slot_table*, int) {
  return p->desc.dtype == CAS_BF16 && p->desc.D == 128 && p->has_tma;
}

// ------------------------------------------------------------------------------- kernel
constexpr int kFwdThreads = 384;   // 3 warpgroups: two softmax groups + (TMA, MMA, 2 idle warps)
constexpr uint32_t kTile = 32768, kHalf = 16384;
constexpr uint32_t kOffQ = 0, kOffK = 2 * kTile, kOffV = 4 * kTile, kOffBar = 6 * kTile;
constexpr uint32_t kFwdSmem = 6 * kTile + 256 + 1024;   // + barriers + alignment slack
enum { B_QF = 0, B_KF = 2, B_KE = 4, B_VF = 6, B_VE = 8, B_SF = 10, B_PF = 12, B_OD = 14, B_QR = 15, B_N = 17 };

struct FwdParams {
  const int32_t* seq_off;
  const int32_t* kv_tile_off;
  const KvTile* kv_tiles;
  const PackedTile* ptiles;      // packed prefix tiles (16-token pages), named by KvTile.tok < 0
  const FwdItem* items;
  __nv_bfloat16* O;
  float* LSE;
  float* part;                   // split-KV partials of the tail blocks: [tail block][part][256 rows][kFwdPartStride]
  const float2* rope_cs;         // fused RoPE: (cos, sin) per [token][pair] or null
  __nv_bfloat16* Q_rot;          // the rotated Q rows (the backward pass reads them)
  int rope_layout;
  int Hq, Hkv, has_self;
  int n_blocks;                  // (item, head) blocks = items x Hq, in KV-group-major order
  int n_whole;                   // blocks [0, n_whole) run whole; each later one is cut into n_parts CTAs
  int n_parts;
  float scale_log2;
};
constexpr int kFwdPartStride = 132;   // 128 O + m + l + pad (16-byte aligned rows)

__device__ __forceinline__ float ex2(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

__global__ void __launch_bounds__(kFwdThreads, 1)
tc_fwd_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmKp,
              const __grid_constant__ CUtensorMap tmVp, const __grid_constant__ CUtensorMap tmKs,
              const __grid_constant__ CUtensorMap tmVs, const __grid_constant__ CUtensorMap tmKp16,
              const __grid_constant__ CUtensorMap tmVp16, const FwdParams prm) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t sbase = (smem_u32(smem_raw) + 1023u) & ~1023u;
  uint8_t* sptr = smem_raw + (sbase - smem_u32(smem_raw));
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(sptr + kOffBar + B_N * 8);
  auto bar = [&](int i) { return sbase + kOffBar + 8u * i; };

  const int warp = warp_id_uniform(), lane = threadIdx.x & 31;
  // KV-group-major block order (inside a group: items longest first, the G heads of an item adjacent): the CTAs
  // in flight work on one KV group at a time, so its K/V tiles (shared by the G heads and by every sequence that
  // selected the cartridge) stay in L2
  const int Gq = prm.Hq / prm.Hkv, per_group = prm.n_blocks / prm.Hkv;    // blocks of one KV group: items x G heads
  // TAIL SPLIT: the last blocks of the launch order (the ones that would run alone in a part-filled last wave) are
  // cut along the KV axis into n_parts CTAs each, which write un-normalised partials merged by fwd_combine_kernel
  const bool split = (int)blockIdx.x >= prm.n_whole;
  const int tail_idx = split ? ((int)blockIdx.x - prm.n_whole) / prm.n_parts : 0;
  const int part = split ? ((int)blockIdx.x - prm.n_whole) % prm.n_parts : 0;
  const int blk = split ? prm.n_whole + tail_idx : (int)blockIdx.x;
  const int g = blk / per_group, rem = blk % per_group;
  const int item_idx = rem / Gq, h = g * Gq + rem % Gq;
  const FwdItem it = prm.items[item_idx];
  const int t0 = prm.seq_off[it.seq], lq = prm.seq_off[it.seq + 1] - t0;
  const int n_pre = prm.kv_tile_off[it.seq + 1] - prm.kv_tile_off[it.seq];
  const KvTile* tiles = prm.kv_tiles + prm.kv_tile_off[it.seq];
  const int nq = it.rows > 128 ? 2 : 1;
  const int diag0 = it.row0 >> 7;
  const int n_all = n_pre + (prm.has_self ? diag0 + nq : 0);      // KV tiles of the block (tile 1 sees one more)
  // this CTA's run of KV tiles [ja, jb): every part has >= 2 tiles (host), so Q tile 0 always has work
  const int ja = split ? (int)((int64_t)part * n_all / prm.n_parts) : 0;
  const int jb = split ? (int)((int64_t)(part + 1) * n_all / prm.n_parts) : n_all;
  const int nkv0 = min(jb, n_pre + (prm.has_self ? diag0 + 1 : 0)) - ja;     // tiles of Q tile 0 / 1, counted from ja
  const int nkv1 = jb - ja;
  const int n_max = nq == 2 ? nkv1 : nkv0;

  if (threadIdx.x == 0) {
    for (int i = 0; i < B_N; ++i) mbar_init(bar(i), (i == B_PF || i == B_PF + 1 || i == B_QR || i == B_QR + 1) ? 128 : 1);
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
  asm volatile("setmaxnreg.dec.sync.aligned.u32 56;");
  if (warp == 8) {
    // ===================================================================== TMA producer
    if (elect_one()) {
      tma_prefetch_desc(&tmQ);
      tma_prefetch_desc(&tmKp);
      tma_prefetch_desc(&tmVp);
      for (int t = 0; t < nq; ++t) {
        mbar_expect_tx(bar(B_QF + t), kTile);
        tma_load_3d(sbase + kOffQ + t * kTile, &tmQ, bar(B_QF + t), 0, h, t0 + it.row0 + 128 * t);
        tma_load_3d(sbase + kOffQ + t * kTile + kHalf, &tmQ, bar(B_QF + t), 64, h, t0 + it.row0 + 128 * t);
      }
      for (int j = 0; j < n_max; ++j) {
        const int s = j & 1;
        const uint32_t ph = (j >> 1) & 1;
        const bool pre = ja + j < n_pre;
        const int tok = pre ? tiles[ja + j].tok : t0 + 128 * (ja + j - n_pre);
        const CUtensorMap* mk = pre ? &tmKp : &tmKs;
        const CUtensorMap* mv = pre ? &tmVp : &tmVs;
        const PackedTile* pt = (pre && tok < 0) ? prm.ptiles + (-1 - tok) : nullptr;
        mbar_wait(bar(B_KE + s), ph ^ 1);
        mbar_expect_tx(bar(B_KF + s), kTile);
        if (pt) {   // eight 16-token pages, each in place from its own cartridge
          for (int u = 0; u < 8; ++u) {
            tma_load_3d(sbase + kOffK + s * kTile + u * 2048, &tmKp16, bar(B_KF + s), 0, g, pt->tok[u]);
            tma_load_3d(sbase + kOffK + s * kTile + kHalf + u * 2048, &tmKp16, bar(B_KF + s), 64, g, pt->tok[u]);
          }
        } else {
          tma_load_3d(sbase + kOffK + s * kTile, mk, bar(B_KF + s), 0, g, tok);
          tma_load_3d(sbase + kOffK + s * kTile + kHalf, mk, bar(B_KF + s), 64, g, tok);
        }
        mbar_wait(bar(B_VE + s), ph ^ 1);
        mbar_expect_tx(bar(B_VF + s), kTile);
        if (pt) {
          for (int u = 0; u < 8; ++u) {
            tma_load_3d(sbase + kOffV + s * kTile + u * 2048, &tmVp16, bar(B_VF + s), 0, g, pt->tok[u]);
            tma_load_3d(sbase + kOffV + s * kTile + kHalf + u * 2048, &tmVp16, bar(B_VF + s), 64, g, pt->tok[u]);
          }
        } else {
          tma_load_3d(sbase + kOffV + s * kTile, mv, bar(B_VF + s), 0, g, tok);
          tma_load_3d(sbase + kOffV + s * kTile + kHalf, mv, bar(B_VF + s), 64, g, tok);
        }
      }
    }
  } else if (warp == 9) {
    // ===================================================================== MMA issuer
    if (elect_one()) {
      constexpr uint32_t idesc_qk = make_idesc(128, 128, 0, 0);
      constexpr uint32_t idesc_pv = make_idesc(128, 128, 0, 1);
      auto issue_qk = [&](int t, int j) {
        const uint32_t qa = sbase + kOffQ + t * kTile, ka = sbase + kOffK + (j & 1) * kTile;
#pragma unroll
        for (int kk = 0; kk < 8; ++kk) {
          const uint32_t o = (kk >> 2) * kHalf + (kk & 3) * 32;
          mma_ss(tbase + t * 128, desc_kmajor(qa + o), desc_kmajor(ka + o), idesc_qk, kk > 0);
        }
      };
      auto issue_pv = [&](int t, int j) {
        const uint32_t va = sbase + kOffV + (j & 1) * kTile;
#pragma unroll
        for (int kk = 0; kk < 8; ++kk)
          mma_ts(tbase + 256 + t * 128, tbase + t * 128 + kk * 8, desc_mnmajor(va + kk * 2048, kHalf), idesc_pv,
                 (j > 0 || kk > 0) ? 1u : 0u);
      };
      // with fused RoPE the softmax warpgroups rotate the Q tiles in shared memory first
      mbar_wait(bar(prm.rope_cs ? B_QR : B_QF), 0);
      if (nq == 2) mbar_wait(bar((prm.rope_cs ? B_QR : B_QF) + 1), 0);
      mbar_wait(bar(B_KF), 0);
      tc_fence_after();
      issue_qk(0, 0);
      mma_commit(bar(B_SF));
      if (nq == 2) {
        issue_qk(1, 0);
        mma_commit(bar(B_SF + 1));
      }
      mma_commit(bar(B_KE));
      for (int j = 0; j < n_max; ++j) {
        const int s = j & 1;
        const bool act0 = j < nkv0, act1 = nq == 2;
        const bool nxt0 = j + 1 < nkv0, nxt1 = nq == 2 && j + 1 < n_max;
        mbar_wait(bar(B_VF + s), (j >> 1) & 1);
        // K(j+1) is waited for HERE, before P0(j): every mbarrier wait of this thread costs ~250 clk even when the
        // phase is long complete, and this one would otherwise sit between PV0(j) and QK0(j+1) on tile 0's chain
        if (nxt0 || nxt1) mbar_wait(bar(B_KF + ((j + 1) & 1)), ((j + 1) >> 1) & 1);
        if (act0) {
          mbar_wait(bar(B_PF), j & 1);
          tc_fence_after();
          issue_pv(0, j);
        }
        if (nxt0) {
          issue_qk(0, j + 1);
          mma_commit(bar(B_SF));
        }
        if (act1) {
          mbar_wait(bar(B_PF + 1), j & 1);
          tc_fence_after();
          issue_pv(1, j);
        }
        mma_commit(bar(B_VE + s));
        if (nxt1) {
          issue_qk(1, j + 1);
          mma_commit(bar(B_SF + 1));
        }
        if (nxt0 || nxt1) mma_commit(bar(B_KE + ((j + 1) & 1)));
      }
      mma_commit(bar(B_OD));
    }
  }
  } else {
    // ===================================================================== softmax + epilogue
    asm volatile("setmaxnreg.inc.sync.aligned.u32 208;");
    const int t = warp >> 2;
    if (t < nq) {
      const int r = threadIdx.x - 128 * t;
      const int row = it.row0 + 128 * t + r;          // row inside the sequence
      const uint32_t lane_base = (uint32_t)((warp & 3) * 32) << 16;
      const uint32_t tS = tbase + t * 128 + lane_base, tO = tbase + 256 + t * 128 + lane_base;
      const int nkv = t == 0 ? nkv0 : nkv1;
      if (prm.rope_cs) {
        // FUSED RoPE: thread = query row.  The row's 16-byte chunk c of half hh sits at chunk position
        // c ^ (r & 7) of its 128-byte line (TMA 128B swizzle); rotate in place for the MMAs and write the rotated row
        // to Q_rot for the backward pass (each (row, head) belongs to one block; of a split block, part 0 writes).
        // the cos/sin of chunk c+1 are fetched (four 16-byte loads, L2) while chunk c is rotated, those of chunk 0
        // before the Q tile has even arrived: the rotation sits in front of the block's first MMA
        const bool live = row < lq;
        const float4* tab4 = reinterpret_cast<const float4*>(prm.rope_cs + (int64_t)(t0 + (live ? row : 0)) * 64);
        const int lay = prm.rope_layout;
        auto fetch = [&](int c, float4 (&w)[4]) {       // layout 0: pairs 4c..4c+3 and 32+4c..; layout 1: pairs 8c..8c+7
          const int i0 = lay == 0 ? 2 * c : 4 * c, i1 = lay == 0 ? 16 + 2 * c : 4 * c + 2;
          w[0] = __ldg(tab4 + i0); w[1] = __ldg(tab4 + i0 + 1); w[2] = __ldg(tab4 + i1); w[3] = __ldg(tab4 + i1 + 1);
        };
        float4 wn[4];
        fetch(0, wn);
        mbar_wait(bar(B_QF + t), 0);
        if (live) {
          __nv_bfloat16* qrow = prm.Q_rot + ((int64_t)(t0 + row) * prm.Hq + h) * 128;
          const uint32_t qb = sbase + kOffQ + t * kTile + r * 128;
#pragma unroll
          for (int c = 0; c < 8; ++c) {
            const float4 w4[4] = {wn[0], wn[1], wn[2], wn[3]};
            if (c < 7) fetch(c + 1, wn);
            const float2 w[8] = {{w4[0].x, w4[0].y}, {w4[0].z, w4[0].w}, {w4[1].x, w4[1].y}, {w4[1].z, w4[1].w},
                                 {w4[2].x, w4[2].y}, {w4[2].z, w4[2].w}, {w4[3].x, w4[3].y}, {w4[3].z, w4[3].w}};
            const uint32_t pos = (uint32_t)((c ^ (r & 7)) << 4);
            uint32_t ua[4], ub[4];
            asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(ua[0]), "=r"(ua[1]), "=r"(ua[2]), "=r"(ua[3]) : "r"(qb + pos));
            asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(ub[0]), "=r"(ub[1]), "=r"(ub[2]), "=r"(ub[3]) : "r"(qb + kHalf + pos));
            float fa[8], fb[8];
#pragma unroll
            for (int i = 0; i < 4; ++i) {
              const float2 x = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&ua[i]));
              const float2 y = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&ub[i]));
              fa[2 * i] = x.x; fa[2 * i + 1] = x.y; fb[2 * i] = y.x; fb[2 * i + 1] = y.y;
            }
            if (lay == 0) {                        // pairs (2k, 2k+1): four inside each chunk (w[0..3]: first half)
#pragma unroll
              for (int i = 0; i < 4; ++i) {
                const float2 w0 = w[i], w1 = w[4 + i];
                const float a0 = fa[2 * i], b0 = fa[2 * i + 1], a1 = fb[2 * i], b1 = fb[2 * i + 1];
                fa[2 * i] = a0 * w0.x - b0 * w0.y;  fa[2 * i + 1] = a0 * w0.y + b0 * w0.x;
                fb[2 * i] = a1 * w1.x - b1 * w1.y;  fb[2 * i + 1] = a1 * w1.y + b1 * w1.x;
              }
            } else {                               // pairs (k, k + 64): chunk c of both halves
#pragma unroll
              for (int i = 0; i < 8; ++i) {
                const float a = fa[i], b = fb[i];
                fa[i] = a * w[i].x - b * w[i].y;
                fb[i] = a * w[i].y + b * w[i].x;
              }
            }
#pragma unroll
            for (int i = 0; i < 4; ++i) {
              ua[i] = pack_bf16(fa[2 * i], fa[2 * i + 1]);
              ub[i] = pack_bf16(fb[2 * i], fb[2 * i + 1]);
            }
            asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(qb + pos), "r"(ua[0]), "r"(ua[1]), "r"(ua[2]), "r"(ua[3]) : "memory");
            asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(qb + kHalf + pos), "r"(ub[0]), "r"(ub[1]), "r"(ub[2]), "r"(ub[3]) : "memory");
            if (part == 0) {
              *reinterpret_cast<uint4*>(qrow + 8 * c) = make_uint4(ua[0], ua[1], ua[2], ua[3]);
              *reinterpret_cast<uint4*>(qrow + 64 + 8 * c) = make_uint4(ub[0], ub[1], ub[2], ub[3]);
            }
          }
        }
        fence_proxy_async();
        mbar_arrive(bar(B_QR + t));
      }
      float m = -INFINITY, l = 0.f;
      for (int j = 0; j < nkv; ++j) {
        int limit;
        const PackedTile* pt = nullptr;
        if (ja + j < n_pre) {
          limit = tiles[ja + j].len;
          if (tiles[ja + j].tok < 0) { pt = prm.ptiles + (-1 - tiles[ja + j].tok); limit = 128; }
        } else {
          const int k0 = 128 * (ja + j - n_pre);
          limit = min(min(128, lq - k0), row - k0 + 1);
        }
        mbar_wait(bar(B_SF + t), j & 1);
        tc_fence_after();
        uint32_t s[128];
        tmem_ld32(tS, s);
        tmem_ld32(tS + 32, s + 32);
        tmem_ld32(tS + 64, s + 64);
        tmem_ld32(tS + 96, s + 96);
        tc_wait_ld();
        if (!__all_sync(0xffffffffu, limit >= 128)) {
#pragma unroll
          for (int c = 0; c < 128; ++c)
            if (c >= limit) s[c] = 0xff800000u;      // -inf: masked key
        }
        if (pt) {                                    // packed tile: the valid keys are those of its pages (warp-uniform)
          const uint4 mk = *reinterpret_cast<const uint4*>(pt->mask);
          const uint32_t mw[4] = {mk.x, mk.y, mk.z, mk.w};
          if ((mk.x & mk.y & mk.z & mk.w) != 0xffffffffu) {
#pragma unroll
            for (int c = 0; c < 128; ++c)
              if (!((mw[c >> 5] >> (c & 31)) & 1u)) s[c] = 0xff800000u;
          }
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
          const float f = ex2(m - m_new);
          m = m_new;
          l *= f;
#pragma unroll
          for (int c = 0; c < 4; ++c) {
            uint32_t o[32];
            tmem_ld32(tO + c * 32, o);
            tc_wait_ld();
#pragma unroll
            for (int i = 0; i < 32; ++i) o[i] = __float_as_uint(__uint_as_float(o[i]) * f);
            tmem_st32(tO + c * 32, o);
            tc_wait_st();                            // the store has read o[] before the next chunk's load reuses it
          }
        }
        // p = 2^(s*scale_log2 - m): one packed FFMA per two scores, one MUFU each, packed row sum
        const uint64_t sc2 = pack2(prm.scale_log2, prm.scale_log2), nm2 = pack2(-m, -m);
        uint64_t sum2a = pack2(0.f, 0.f), sum2b = sum2a;
#pragma unroll
        for (int i = 0; i < 64; i += 2) {
          float a0, a1, b0, b1;
          unpack2(fma2(pack2(__uint_as_float(s[2 * i]), __uint_as_float(s[2 * i + 1])), sc2, nm2), a0, a1);
          unpack2(fma2(pack2(__uint_as_float(s[2 * i + 2]), __uint_as_float(s[2 * i + 3])), sc2, nm2), b0, b1);
          a0 = ex2(a0); a1 = ex2(a1);
          if ((i & 6) != 6) exp2_poly2(b0, b1, b0, b1);    // 3 of every 8 scores on the FMA pipe (exp phase 1410 -> 1090 clk)
          else { b0 = ex2(b0); b1 = ex2(b1); }
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
        mbar_arrive(bar(B_PF + t));
      }
      // epilogue: O = acc / l, LSE = ln2 * m + ln(l)
      mbar_wait(bar(B_OD), 0);
      tc_fence_after();
      if (split) {
        // un-normalised partial (O, m, l) of this row over the CTA's run of tiles
        float* prow = prm.part + ((((int64_t)tail_idx * prm.n_parts + part) * 256) + 128 * t + r) * kFwdPartStride;
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          uint32_t o[32];
          tmem_ld32(tO + c * 32, o);
          tc_wait_ld();
#pragma unroll
          for (int i = 0; i < 8; ++i)
            __stcg(reinterpret_cast<float4*>(prow + c * 32 + 4 * i),
                   make_float4(__uint_as_float(o[4 * i]), __uint_as_float(o[4 * i + 1]), __uint_as_float(o[4 * i + 2]),
                               __uint_as_float(o[4 * i + 3])));
        }
        __stcg(reinterpret_cast<float2*>(prow + 128), make_float2(m, l));
      } else {
      const float inv = 1.f / l;
      const bool ok = row < lq && r < it.rows - 128 * t;
      __nv_bfloat16* orow = prm.O + ((int64_t)(t0 + row) * prm.Hq + h) * 128;
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        uint32_t o[32];
        tmem_ld32(tO + c * 32, o);
        tc_wait_ld();
        if (ok) {
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            uint4 u;
            u.x = pack_bf16(__uint_as_float(o[8 * i + 0]) * inv, __uint_as_float(o[8 * i + 1]) * inv);
            u.y = pack_bf16(__uint_as_float(o[8 * i + 2]) * inv, __uint_as_float(o[8 * i + 3]) * inv);
            u.z = pack_bf16(__uint_as_float(o[8 * i + 4]) * inv, __uint_as_float(o[8 * i + 5]) * inv);
            u.w = pack_bf16(__uint_as_float(o[8 * i + 6]) * inv, __uint_as_float(o[8 * i + 7]) * inv);
            *reinterpret_cast<uint4*>(orow + c * 32 + i * 8) = u;
          }
        }
      }
      if (ok) prm.LSE[(int64_t)(t0 + row) * prm.Hq + h] = m * 0.6931471805599453f + logf(l);
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 8) tmem_dealloc(tbase, 512);
}

// Merge of the tail blocks' split-KV partials: one warp per (tail block, row); lane = 4 output columns.
__global__ void __launch_bounds__(256)
fwd_combine_kernel(const FwdParams prm, int n_tail) {
  const int w = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (w >= n_tail * 256) return;
  const int tail_idx = w >> 8, rr = w & 255;
  const int Gq = prm.Hq / prm.Hkv, per_group = prm.n_blocks / prm.Hkv;
  const int blk = prm.n_whole + tail_idx;
  const int g = blk / per_group, rem = blk % per_group;
  const FwdItem it = prm.items[rem / Gq];
  const int h = g * Gq + rem % Gq;
  const int t0 = prm.seq_off[it.seq], lq = prm.seq_off[it.seq + 1] - t0;
  const int row = it.row0 + rr;
  if (rr >= it.rows || row >= lq) return;
  const float* p0 = prm.part + (((int64_t)tail_idx * prm.n_parts) * 256 + rr) * kFwdPartStride;
  float M = -INFINITY;
  for (int q = 0; q < prm.n_parts; ++q) M = fmaxf(M, __ldcg(p0 + (int64_t)q * 256 * kFwdPartStride + 128));
  float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
  float L = 0.f;
  for (int q = 0; q < prm.n_parts; ++q) {
    const float* pr = p0 + (int64_t)q * 256 * kFwdPartStride;
    const float2 ml = __ldcg(reinterpret_cast<const float2*>(pr + 128));
    const float4 v = __ldcg(reinterpret_cast<const float4*>(pr + 4 * lane));
    const float f = ex2(ml.x - M);
    L += f * ml.y;
    acc.x += f * v.x; acc.y += f * v.y; acc.z += f * v.z; acc.w += f * v.w;
  }
  const float inv = 1.f / L;
  uint2 o;
  o.x = pack_bf16(acc.x * inv, acc.y * inv);
  o.y = pack_bf16(acc.z * inv, acc.w * inv);
  *reinterpret_cast<uint2*>(prm.O + ((int64_t)(t0 + row) * prm.Hq + h) * 128 + 4 * lane) = o;
  if (lane == 0) prm.LSE[(int64_t)(t0 + row) * prm.Hq + h] = M * 0.6931471805599453f + logf(L);
}

// How many blocks at the end of the launch order to cut, and into how many parts.  Greedy list schedule of the
// blocks (cost = KV tiles + a constant for prologue and epilogue) on the SMs, in launch order, the way the
// hardware block scheduler deals them; the blocks that end later than the balanced makespan are the tail.
static void plan_tail_split(const cas_slot_table* t, int Hq, int Hkv, bool has_self, int n_sm, int* n_tail, int* n_parts) {
  *n_tail = 0;
  *n_parts = 1;
  const int Gq = Hq / Hkv;
  const size_t n_items = t->fwd_items.size(), n_blocks = n_items * Hq;
  if (n_blocks <= (size_t)n_sm || getenv("CAS_FWD_NO_SPLIT")) return;
  std::vector<int> cost(n_items), tiles(n_items);
  double total = 0;
  for (size_t i = 0; i < n_items; ++i) {
    const FwdItem& it = t->fwd_items[i];
    const int n_pre = t->kv_tile_off[it.seq + 1] - t->kv_tile_off[it.seq];
    tiles[i] = n_pre + (has_self ? (it.row0 >> 7) + (it.rows > 128 ? 2 : 1) : 0);
    cost[i] = (it.rows > 128 ? 2 : 1) * tiles[i] + 3;
    total += (double)cost[i] * Hq;
  }
  std::vector<int64_t> heap(n_sm, 0);               // min-heap of SM free times
  auto cmp = [](int64_t a, int64_t b) { return a > b; };
  std::vector<int64_t> finish(n_blocks);
  for (size_t b = 0; b < n_blocks; ++b) {
    const size_t item = (b % (n_items * Gq)) / Gq;
    std::pop_heap(heap.begin(), heap.end(), cmp);
    heap.back() += cost[item];
    finish[b] = heap.back();
    std::push_heap(heap.begin(), heap.end(), cmp);
  }
  const double balanced = total / n_sm * 1.03;
  int r = 0;
  while ((size_t)r < n_blocks && finish[n_blocks - 1 - r] > balanced) ++r;
  if (r == 0 || 2 * r > n_sm) return;               // nothing sticks out, or the last wave is at least half full
  int parts = std::min(n_sm / r, 8);
  for (int i = 0; i < r; ++i) {
    const size_t b = n_blocks - 1 - i;
    parts = std::min(parts, tiles[(b % (n_items * Gq)) / Gq] / 2);      // every part keeps >= 2 KV tiles
  }
  if (parts < 2) return;
  *n_tail = r;
  *n_parts = parts;
}

// ---- cas_prefix_attn_fwd_noalloc: the tail blocks' split-KV partials in a file-scope device array --------------
// For callers that may not allocate (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc).  Every GPU
// that loads the library holds these 20,004,864 bytes until exit.  In host code the array's NAME is a host-side
// stand-in, not a device address: the kernels get the address cudaGetSymbolAddress returns, looked up once per device
// with that device current.  All calls share the array (calls that overlap on the GPU race); nothing in it has to
// start at zero: a call reads only the partial rows its own CTAs have written.
constexpr int kNoAllocPartBlocks = 148;      // split CTAs (tail blocks x parts) one call may use
static __device__ __align__(256) float g_fwd_part_static[(size_t)kNoAllocPartBlocks * 256 * kFwdPartStride];

static int fwd_static_scratch(float** out) {
  constexpr int kMaxDev = 64;
  static float* addr[kMaxDev] = {};
  static std::mutex mu;
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return cuda_fail(e, "cudaGetDevice");
  if (dev < 0 || dev >= kMaxDev) { set_error("device ordinal %d not supported by the static scratch", dev); return CAS_ERR_INVALID_ARG; }
  std::lock_guard<std::mutex> lk(mu);
  if (!addr[dev]) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_fwd_part_static);      // the address on the CURRENT device
    if (e != cudaSuccess) return cuda_fail(e, "cudaGetSymbolAddress(g_fwd_part_static)");
    addr[dev] = (float*)p;
  }
  *out = addr[dev];
  return CAS_OK;
}

int tc_attn_fwd(const AttnArgs& a) {
  const cas_slot_table* t = a.tab;
  const FwdItem* items = t->d_fwd_items;
  const size_t n_items = t->fwd_items.size();
  static SmemAttrOnce attr;
  int rc = attr.set((const void*)tc_fwd_kernel, (int)kFwdSmem);
  if (rc) return rc;
  CUtensorMap tmQ, tmKs, tmVs;
  rc = make_thd_map(&tmQ, a.Q, t->T, a.Hq, 128);
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
  // tail split (cached per table and head count: a table serves every layer of a step)
  cas_slot_table* tm = const_cast<cas_slot_table*>(t);
  const int has_self = a.Ks ? 1 : 0;
  if (tm->fwd_plan_key != a.Hq * 2 + has_self) {
    plan_tail_split(t, a.Hq, a.Hkv, has_self != 0, a.pool->n_sm, &tm->fwd_n_tail, &tm->fwd_n_parts);
    tm->fwd_plan_key = a.Hq * 2 + has_self;
  }
  const int n_blocks = (int)(n_items * a.Hq), n_tail = t->fwd_n_tail, n_parts = t->fwd_n_parts;
  float* part = nullptr;
  if (n_tail && a.static_scratch) {
    if (n_tail * n_parts > kNoAllocPartBlocks) {
      set_error("cas_prefix_attn_fwd_noalloc: this table splits %d tail blocks into %d parts = %d split CTAs; the static "
                "scratch holds %d (%zu bytes): use cas_prefix_attn_fwd", n_tail, n_parts, n_tail * n_parts,
                kNoAllocPartBlocks, sizeof(float) * kNoAllocPartBlocks * 256 * kFwdPartStride);
      return CAS_ERR_CAPACITY;
    }
    rc = fwd_static_scratch(&part);
    if (rc) return rc;
  } else if (n_tail) {
    // pool-owned, grow-only: forward calls on one pool are ordered by the caller's stream (cas.h)
    const size_t need = (size_t)n_tail * n_parts * 256 * kFwdPartStride * sizeof(float);
    cas_pool* pm = const_cast<cas_pool*>(a.pool);
    if (pm->fwd_part_bytes < need) {
      if (pm->fwd_part) {
        cudaError_t e = cudaStreamSynchronize(a.stream);     // the old buffer may still be read by an earlier call
        if (e != cudaSuccess) return cuda_fail(e, "fwd partial scratch sync");
        cudaFree(pm->fwd_part);
        pm->fwd_part = nullptr;
        pm->fwd_part_bytes = 0;
      }
      cudaError_t e = cudaMalloc(&pm->fwd_part, need);
      if (e != cudaSuccess) return cuda_fail(e, "fwd partial scratch");
      pm->fwd_part_bytes = need;
    }
    part = (float*)pm->fwd_part;
  }
  FwdParams prm{t->d_seq_off, t->d_kv_tile_off, t->d_kv_tiles, t->d_ptiles, items, (__nv_bfloat16*)a.O_out, a.LSE_out,
                part, (const float2*)a.rope_cs, (__nv_bfloat16*)a.Q_rot, a.rope_layout,
                a.Hq, a.Hkv, has_self, n_blocks, n_blocks - n_tail, n_parts, a.scale * 1.4426950408889634f};
  const unsigned grid = (unsigned)(n_blocks - n_tail + n_tail * n_parts);
  tc_fwd_kernel<<<grid, kFwdThreads, kFwdSmem, a.stream>>>(tmQ, a.L->tm_K, a.L->tm_V, tmKs, tmVs, a.L->tm_K16, a.L->tm_V16, prm);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return cuda_fail(e, "tc fwd launch");
  if (n_tail) {
    fwd_combine_kernel<<<(n_tail * 256 * 32 + 255) / 256, 256, 0, a.stream>>>(prm, n_tail);
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "fwd combine launch");
  }
  return CAS_OK;
}

}  // namespace cas

