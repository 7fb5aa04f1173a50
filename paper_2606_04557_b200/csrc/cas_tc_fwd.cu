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
#include <cstdlib>

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
enum { B_QF = 0, B_KF = 2, B_KE = 4, B_VF = 6, B_VE = 8, B_SF = 10, B_PF = 12, B_OD = 14, B_N = 15 };

struct FwdParams {
  const int32_t* seq_off;
  const int32_t* kv_tile_off;
  const KvTile* kv_tiles;
  const PackedTile* ptiles;      // packed prefix tiles (16-token pages), named by KvTile.tok < 0
  const FwdItem* items;
  __nv_bfloat16* O;
  float* LSE;
  int Hq, Hkv, has_self;
  float scale_log2;
};

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
  const int Gq = prm.Hq / prm.Hkv, per_group = gridDim.x / prm.Hkv;      // blocks of one KV group: items x G heads
  const int g = blockIdx.x / per_group, rem = blockIdx.x % per_group;
  const int item_idx = rem / Gq, h = g * Gq + rem % Gq;
  const FwdItem it = prm.items[item_idx];
  const int t0 = prm.seq_off[it.seq], lq = prm.seq_off[it.seq + 1] - t0;
  const int n_pre = prm.kv_tile_off[it.seq + 1] - prm.kv_tile_off[it.seq];
  const KvTile* tiles = prm.kv_tiles + prm.kv_tile_off[it.seq];
  const int nq = it.rows > 128 ? 2 : 1;
  const int diag0 = it.row0 >> 7;
  const int nkv0 = n_pre + (prm.has_self ? diag0 + 1 : 0);
  const int nkv1 = n_pre + (prm.has_self ? diag0 + 2 : 0);
  const int n_max = nq == 2 ? nkv1 : nkv0;

  if (threadIdx.x == 0) {
    for (int i = 0; i < B_N; ++i) mbar_init(bar(i), (i == B_PF || i == B_PF + 1) ? 128 : 1);
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
        const bool pre = j < n_pre;
        const int tok = pre ? tiles[j].tok : t0 + 128 * (j - n_pre);
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
      mbar_wait(bar(B_QF), 0);
      if (nq == 2) mbar_wait(bar(B_QF + 1), 0);
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
        if (act0) {
          mbar_wait(bar(B_PF), j & 1);
          tc_fence_after();
          issue_pv(0, j);
        }
        if (nxt0 || nxt1) {
          mbar_wait(bar(B_KF + ((j + 1) & 1)), ((j + 1) >> 1) & 1);
          tc_fence_after();
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
      float m = -INFINITY, l = 0.f;
      for (int j = 0; j < nkv; ++j) {
        int limit;
        const PackedTile* pt = nullptr;
        if (j < n_pre) {
          limit = tiles[j].len;
          if (tiles[j].tok < 0) { pt = prm.ptiles + (-1 - tiles[j].tok); limit = 128; }
        } else {
          const int k0 = 128 * (j - n_pre);
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
  tc_fence_before();
  __syncthreads();
  if (warp == 8) tmem_dealloc(tbase, 512);
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
  FwdParams prm{t->d_seq_off, t->d_kv_tile_off, t->d_kv_tiles, t->d_ptiles, items, (__nv_bfloat16*)a.O_out, a.LSE_out,
                a.Hq, a.Hkv, a.Ks ? 1 : 0, a.scale * 1.4426950408889634f};
  const unsigned grid = (unsigned)(n_items * a.Hq);
  tc_fwd_kernel<<<grid, kFwdThreads, kFwdSmem, a.stream>>>(tmQ, a.L->tm_K, a.L->tm_V, tmKs, tmVs, a.L->tm_K16, a.L->tm_V16, prm);
  cudaError_t e = cudaGetLastError();
  return e == cudaSuccess ? CAS_OK : cuda_fail(e, "tc fwd launch");
}

}  // namespace cas

