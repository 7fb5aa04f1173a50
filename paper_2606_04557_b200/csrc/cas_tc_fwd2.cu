// Prefix-attention FORWARD on CTA PAIRS (tcgen05 cta_group::2), bf16, head_dim 128.
//
// Same definition and same per-CTA structure as cas_tc_fwd.cu (two 128-row Q tiles ping-ponging, P fed from
// TMEM, online softmax in the log2 domain), but two CTAs of a cluster share every K/V tile: the pair covers
// 512 query rows of one sequence and one head, each CTA loads HALF of each K tile (64 keys x 128 d) and half of
// each V tile (128 keys x 64 d) into its own shared memory, and the LEADER CTA issues every MMA for both SMs
// with M = 256 (the two CTAs' Q tiles t) -- the B operand halves are read by both tensor cores.  Per CTA and KV
// step the shared-memory pipe then carries 160 KB instead of 256 KB (the forward kernel is limited by that pipe,
// DESIGN.md section 10).
//
// Cross-CTA protocol.  TMA loads complete on barriers of the loading CTA; the peer's otherwise idle MMA warp
// relays "my half has landed" to leader-only barriers with remote mbarrier arrives, in the order in which the
// leader consumes them; the softmax threads of both CTAs arrive on the leader's "P is written" barriers directly.  MMA completions (S ready, O done, stage free) are
// multicast-committed to the same barrier offset in both CTAs.
//
// Used for 512-row blocks with more than 256 rows; the remaining blocks go to tc_fwd_kernel.
#include "cas_sm100.cuh"
#include "cas_tc_common.cuh"

namespace cas {
using namespace sm100;

#ifdef CAS_TRACE
__device__ long long cas_fwd2_trace_buf[4 * 32 * 8];
#define PTRACE(role, i, ev)                                                                                     \
  do {                                                                                                          \
    if (blockIdx.x == 300 && (i) < 32) cas_fwd2_trace_buf[((role) * 32 + (i)) * 8 + (ev)] = clock64();           \
    if (blockIdx.x == 301 && (i) < 32 && (role) >= 1) cas_fwd2_trace_buf[(3 * 32 + (i)) * 8 + 2 * ((role) - 1) + (ev)] = clock64(); \
  } while (0)
#else
#define PTRACE(role, i, ev) do {} while (0)
#endif

constexpr int kP2Threads = 384;
constexpr int kP2Stages = 4;                       // K-half / V-half ring depth (16 KB per stage each)
constexpr uint32_t pTile = 32768, pHalf = 16384, pQuart = 8192;
constexpr uint32_t pOffQ = 0, pOffK = 2 * pTile, pOffV = pOffK + kP2Stages * pHalf, pOffBar = pOffV + kP2Stages * pHalf;
enum { P_QF = 0, P_KF = 2, P_VF = 6, P_KE = 10, P_VE = 14, P_SF = 18, P_PF = 20, P_OD = 22,
       P_QFP = 23, P_KFP = 24, P_VFP = 28, P_PFP = 32, P_N = 34 };
constexpr uint32_t kP2Smem = pOffBar + 512;

struct Fwd2Params {
  const int32_t* seq_off;
  const int32_t* kv_tile_off;
  const KvTile* kv_tiles;
  const FwdItem* items;       // 512-row blocks
  __nv_bfloat16* O;
  float* LSE;
  int Hq, Hkv, has_self;
  float scale_log2;
};

__device__ __forceinline__ uint32_t mapa_rank(uint32_t addr, uint32_t rank) {
  uint32_t r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank));
  return r;
}
__device__ __forceinline__ void mbar_arrive_remote(uint32_t cluster_addr) {
  asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr) : "memory");
}
// Relaxed form for "my P is in TMEM": the data is not in memory, tcgen05.wait::st + fence::before_thread_sync
// have already completed it, and a cluster-scope release costs ~1200 clk on the softmax critical path (measured).
__device__ __forceinline__ void mbar_arrive_remote_relaxed(uint32_t cluster_addr) {
  asm volatile("mbarrier.arrive.relaxed.cluster.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr) : "memory");
}
// Spins on test_wait: a thread suspended in try_wait is not woken promptly by an arrival that comes from the
// other CTA of the cluster (measured: ~1800 clk late), so barriers with remote arrivals are polled.
__device__ __forceinline__ void mbar_wait_cluster(uint32_t bar, uint32_t parity) {   // acquire at cluster scope
  uint32_t ok = 0;
  while (!ok) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.test_wait.parity.acquire.cluster.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
  }
}
__device__ __forceinline__ void mma_ts_pair(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t idesc, uint32_t accum) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::2.kind::f16 [%0], [%1], %2, %3, p;\n\t}"
      ::"r"(d_tmem), "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accum)
      : "memory");
}
__device__ __forceinline__ float ex2f(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kP2Threads, 1)
tc_fwd2_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmKp64,
               const __grid_constant__ CUtensorMap tmVp, const __grid_constant__ CUtensorMap tmKs64,
               const __grid_constant__ CUtensorMap tmVs, const Fwd2Params prm) {
  extern __shared__ __align__(1024) uint8_t smem[];
  const uint32_t sbase = smem_u32(smem);
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + pOffBar + P_N * 8);
  auto bar = [&](int i) { return sbase + pOffBar + 8u * i; };
  const int warp = warp_id_uniform(), lane = threadIdx.x & 31;
  const uint32_t rank = cluster_ctarank();
  // KV-group-major cluster order (as tc_fwd_kernel): cluster id -> (g, item, head of group)
  const int cid = blockIdx.x >> 1, n_clusters = gridDim.x >> 1;
  const int Gq = prm.Hq / prm.Hkv, per_group = n_clusters / prm.Hkv;
  const int g = cid / per_group, rem = cid % per_group;
  const int item_idx = rem / Gq, h = g * Gq + rem % Gq;
  const FwdItem it = prm.items[item_idx];
  const int t0 = prm.seq_off[it.seq], lq = prm.seq_off[it.seq + 1] - t0;
  const int n_pre = prm.kv_tile_off[it.seq + 1] - prm.kv_tile_off[it.seq];
  const KvTile* tiles = prm.kv_tiles + prm.kv_tile_off[it.seq];
  const int row0 = it.row0 + 256 * (int)rank;                     // first row of this CTA inside the sequence
  // every tile of the pair runs the same number of KV steps: up to the diagonal tile of the pair's last row
  const int n = n_pre + (prm.has_self ? ((it.row0 + it.rows - 1) >> 7) + 1 : 0);

  if (threadIdx.x == 0) {
    if (sbase & 1023u) __trap();
    for (int i = 0; i < P_N; ++i) mbar_init(bar(i), (i == P_PF || i == P_PF + 1) ? 8 : 1);   // P ready: one arrival per softmax warp, 4 local + 4 remote
    fence_mbar_init();
  }
  if (warp == 8) tmem_alloc_pair(smem_u32(tmem_slot), 512);
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();                                              // both CTAs: barriers initialised, TMEM allocated
  tc_fence_after();
  const uint32_t tbase = *tmem_slot;

  if (warp >= 8) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 56;");
    if (warp == 8) {
      // =================================================================== TMA producer (each CTA: its halves)
      if (elect_one()) {
        tma_prefetch_desc(&tmQ);
        tma_prefetch_desc(&tmKp64);
        tma_prefetch_desc(&tmVp);
        for (int t = 0; t < 2; ++t) {
          mbar_expect_tx(bar(P_QF + t), pTile);
          tma_load_3d(sbase + pOffQ + t * pTile, &tmQ, bar(P_QF + t), 0, h, t0 + row0 + 128 * t);
          tma_load_3d(sbase + pOffQ + t * pTile + pHalf, &tmQ, bar(P_QF + t), 64, h, t0 + row0 + 128 * t);
        }
        for (int j = 0; j < n; ++j) {
          const int s = j % kP2Stages;
          const uint32_t ph = (j / kP2Stages) & 1;
          const bool pre = j < n_pre;
          const int tok = pre ? tiles[j].tok : t0 + 128 * (j - n_pre);
          const CUtensorMap* mk = pre ? &tmKp64 : &tmKs64;
          const CUtensorMap* mv = pre ? &tmVp : &tmVs;
          // K half: keys [64*rank, +64) x 128 d as two [64 x 64] blocks; V half: 128 keys x d [64*rank, +64)
          mbar_wait(bar(P_KE + s), ph ^ 1);
          mbar_expect_tx(bar(P_KF + s), pHalf);
          tma_load_3d(sbase + pOffK + s * pHalf, mk, bar(P_KF + s), 0, g, tok + 64 * (int)rank);
          tma_load_3d(sbase + pOffK + s * pHalf + pQuart, mk, bar(P_KF + s), 64, g, tok + 64 * (int)rank);
          mbar_wait(bar(P_VE + s), ph ^ 1);
          mbar_expect_tx(bar(P_VF + s), pHalf);
          tma_load_3d(sbase + pOffV + s * pHalf, mv, bar(P_VF + s), 64 * (int)rank, g, tok);
        }
      }
    } else if (warp == 9) { if (elect_one()) {
      if (rank == 0) {
        // ================================================================= MMA issuer (leader, both SMs)
        constexpr uint32_t idesc_qk = make_idesc(256, 128, 0, 0);
        constexpr uint32_t idesc_pv = make_idesc(256, 128, 0, 1);
        auto issue_qk = [&](int t, int j) {
          const uint32_t qa = sbase + pOffQ + t * pTile, ka = sbase + pOffK + (j % kP2Stages) * pHalf;
#pragma unroll
          for (int kk = 0; kk < 8; ++kk)
            mma_ss_pair(tbase + t * 128, desc_kmajor(qa + (kk >> 2) * pHalf + (kk & 3) * 32),
                        desc_kmajor(ka + (kk >> 2) * pQuart + (kk & 3) * 32), idesc_qk, kk > 0);
        };
        auto issue_pv = [&](int t, int j) {
          const uint32_t va = sbase + pOffV + (j % kP2Stages) * pHalf;
#pragma unroll
          for (int kk = 0; kk < 8; ++kk)
            mma_ts_pair(tbase + 256 + t * 128, tbase + t * 128 + kk * 8, desc_mnmajor(va + kk * 2048, pHalf), idesc_pv,
                        (j > 0 || kk > 0) ? 1u : 0u);
        };
        mbar_wait(bar(P_QF), 0);
        mbar_wait(bar(P_QF + 1), 0);
        mbar_wait_cluster(bar(P_QFP), 0);
        mbar_wait(bar(P_KF), 0);
        mbar_wait_cluster(bar(P_KFP), 0);
        tc_fence_after();
        issue_qk(0, 0);
        mma_commit_pair(bar(P_SF), 3);
        issue_qk(1, 0);
        mma_commit_pair(bar(P_SF + 1), 3);
        mma_commit_pair(bar(P_KE), 3);
        for (int j = 0; j < n; ++j) {
          const int s = j % kP2Stages, s1 = (j + 1) % kP2Stages;
          const uint32_t ph = (j / kP2Stages) & 1, ph1 = ((j + 1) / kP2Stages) & 1;
          const bool nxt = j + 1 < n;
          mbar_wait(bar(P_VF + s), ph);
          PTRACE(0, j, 0);
          mbar_wait_cluster(bar(P_VFP + s), ph);
          PTRACE(0, j, 1);
          mbar_wait_cluster(bar(P_PF), j & 1);
          PTRACE(0, j, 2);
          tc_fence_after();
          issue_pv(0, j);
          if (nxt) {
            mbar_wait(bar(P_KF + s1), ph1);
            mbar_wait_cluster(bar(P_KFP + s1), ph1);
            tc_fence_after();
            issue_qk(0, j + 1);
            mma_commit_pair(bar(P_SF), 3);
          }
          PTRACE(0, j, 3);
          mbar_wait_cluster(bar(P_PF + 1), j & 1);
          PTRACE(0, j, 4);
          tc_fence_after();
          issue_pv(1, j);
          mma_commit_pair(bar(P_VE + s), 3);
          if (nxt) {
            issue_qk(1, j + 1);
            mma_commit_pair(bar(P_SF + 1), 3);
            mma_commit_pair(bar(P_KE + s1), 3);
          }
          PTRACE(0, j, 5);
        }
        mma_commit_pair(bar(P_OD), 3);
      } else {
        // ================================================================= relay (peer): local -> leader barriers
        auto relay = [&](int i) { mbar_arrive_remote(mapa_rank(bar(i), 0)); };
        mbar_wait(bar(P_QF), 0);
        mbar_wait(bar(P_QF + 1), 0);
        relay(P_QFP);
        mbar_wait(bar(P_KF), 0);
        relay(P_KFP);
        for (int j = 0; j < n; ++j) {
          const int s = j % kP2Stages, s1 = (j + 1) % kP2Stages;
          const uint32_t ph = (j / kP2Stages) & 1, ph1 = ((j + 1) / kP2Stages) & 1;
          mbar_wait(bar(P_VF + s), ph);
          relay(P_VFP + s);
          if (j + 1 < n) {
            mbar_wait(bar(P_KF + s1), ph1);
            relay(P_KFP + s1);
          }
        }
      }
    } }
  } else {
    // ===================================================================== softmax + epilogue (as tc_fwd_kernel)
    asm volatile("setmaxnreg.inc.sync.aligned.u32 208;");
    const int t = warp >> 2;
    const int r = threadIdx.x - 128 * t;
    const int row = row0 + 128 * t + r;                 // row inside the sequence
    const uint32_t lane_base = (uint32_t)((warp & 3) * 32) << 16;
    const uint32_t tS = tbase + t * 128 + lane_base, tO = tbase + 256 + t * 128 + lane_base;
    // "P is written" goes straight to the LEADER's barrier (the leader issues the PV MMA of both CTAs)
    const uint32_t pf_leader = mapa_rank(bar(P_PF + t), 0);
    float m = -INFINITY, l = 0.f;
    for (int j = 0; j < n; ++j) {
      int limit;
      if (j < n_pre) {
        limit = tiles[j].len;
      } else {
        const int k0 = 128 * (j - n_pre);
        limit = min(min(128, lq - k0), row - k0 + 1);   // <= 0 beyond this tile's diagonal: fully masked step
      }
      mbar_wait(bar(P_SF + t), j & 1);
      if ((threadIdx.x & 127) == 0) PTRACE(1 + t, j, 0);
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
          if (c >= limit) s[c] = 0xff800000u;           // -inf: masked key
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
        const float f = ex2f(m - m_new);
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
      const uint64_t sc2 = pack2(prm.scale_log2, prm.scale_log2), nm2 = pack2(-m, -m);
      uint64_t sum2a = pack2(0.f, 0.f), sum2b = sum2a;
#pragma unroll
      for (int i = 0; i < 64; i += 2) {
        float a0, a1, b0, b1;
        unpack2(fma2(pack2(__uint_as_float(s[2 * i]), __uint_as_float(s[2 * i + 1])), sc2, nm2), a0, a1);
        unpack2(fma2(pack2(__uint_as_float(s[2 * i + 2]), __uint_as_float(s[2 * i + 3])), sc2, nm2), b0, b1);
        a0 = ex2f(a0); a1 = ex2f(a1); b0 = ex2f(b0); b1 = ex2f(b1);
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
      __syncwarp();                                     // every lane's P is in TMEM and fenced
      if (lane == 0) {
        if (rank == 0) mbar_arrive(bar(P_PF + t));
        else mbar_arrive_remote_relaxed(pf_leader);
      }
      if ((threadIdx.x & 127) == 0) PTRACE(1 + t, j, 1);
    }
    mbar_wait(bar(P_OD), 0);
    tc_fence_after();
    const float inv = 1.f / l;
    const bool ok = row < lq && row < it.row0 + it.rows;
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
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();                                             // the peer's MMAs / TMEM reads are finished too
  if (warp == 8) tmem_dealloc_pair(tbase, 512);
}

// Launches the pair kernel over `n_items` 512-row blocks (t->d_fwd2_items).
int tc_attn_fwd_pairs(const AttnArgs& a, int n_items) {
  const cas_slot_table* t = a.tab;
  static bool attr_set = false;
  if (!attr_set) {
    CAS_CUDA(cudaFuncSetAttribute(tc_fwd2_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kP2Smem));
    attr_set = true;
  }
  CUtensorMap tmQ, tmKs64, tmVs, tmKp64;
  int rc = make_thd_map(&tmQ, a.Q, t->T, a.Hq, 128);
  if (rc) return rc;
  rc = make_thd_map(&tmKp64, a.pool->pool_K, a.pool->pool_tokens, a.Hkv, 64);
  if (rc) return rc;
  if (a.Ks) {
    rc = make_thd_map(&tmKs64, a.Ks, t->T, a.Hkv, 64);
    if (rc) return rc;
    rc = make_thd_map(&tmVs, a.Vs, t->T, a.Hkv, 128);
    if (rc) return rc;
  } else {
    tmKs64 = tmKp64;
    tmVs = a.pool->tm_V;
  }
  Fwd2Params prm{t->d_seq_off, t->d_kv_tile_off, t->d_kv_tiles, t->d_fwd2_items, (__nv_bfloat16*)a.O_out, a.LSE_out,
                 a.Hq, a.Hkv, a.Ks ? 1 : 0, a.scale * 1.4426950408889634f};
  const unsigned grid = (unsigned)(n_items * a.Hq * 2);
  tc_fwd2_kernel<<<grid, kP2Threads, kP2Smem, a.stream>>>(tmQ, tmKp64, a.pool->tm_V, tmKs64, tmVs, prm);
  cudaError_t e = cudaGetLastError();
  return e == cudaSuccess ? CAS_OK : cuda_fail(e, "tc fwd pair launch");
}

}  // namespace cas

#ifdef CAS_TRACE
extern "C" int cas_debug_fwd2_trace_read(long long* out) {
  return (int)cudaMemcpyFromSymbol(out, cas::cas_fwd2_trace_buf, sizeof(cas::cas_fwd2_trace_buf));
}
#endif
