// Internal declarations shared by the host runtime (cas_host.cu) and the kernel translation units.
// Not part of the ABI.
#pragma once
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "../../include/cas.h"

namespace cas {

void set_error(const char* fmt, ...);
int cuda_fail(cudaError_t e, const char* what);

#define CAS_CUDA(expr)                                     \
  do {                                                     \
    cudaError_t _e = (expr);                               \
    if (_e != cudaSuccess) return cas::cuda_fail(_e, #expr); \
  } while (0)

struct Pending {
  cas_manifest_entry e;
  int64_t step;
};

// One KV tile (<= tile_tokens keys that never straddle two slots).
struct KvTile {
  int32_t tok;   // first pool token (prefix tile) / first packed token (self tile)
  int32_t len;   // valid keys in the tile, 1..128
};

// A KV tile PACKED from 16-token pages of several cartridges (pools with tile_tokens == 16; SURVEY.md 8(f) NEXT-2,
// cartridges are whole 16-token pages, down to ONE page at 50-100x compression): KvTile.tok < 0
// names packed tile -1 - tok.  Page i lands in rows [16 i, 16 i + 16) of the 128-row MMA tile; bit k of `mask` = key k
// is a real token (a cartridge's last page may be partly filled; unused page slots repeat page 0 with no bits set,
// so the tile always holds finite data).
struct PackedTile {
  int32_t tok[8];     // first pool token of each page
  uint32_t mask[4];   // 128 key-valid bits
};

// Backward work item: one KV tile of one KV head is owned by one CTA (deterministic dK/dV).
struct BwdItem {
  int32_t kind;     // 0 = prefix tile of a slot, 1 = self tile of a sequence, 2 = packed prefix tile of a sequence (tok = its index)
  int32_t id;       // slot (kind 0) or sequence (kind 1)
  int32_t tok;      // first key token of the tile (pool token / packed token)
  int32_t len;      // valid keys
  int32_t jt;       // tile index inside the slot / sequence
  int32_t cost;     // number of (q-tile, head) inner iterations (for longest-first ordering)
};

// Forward work item: one block of query rows of one sequence (all heads enumerated by the grid).
struct FwdItem {
  int32_t seq;
  int32_t row0;     // first row inside the sequence
  int32_t rows;     // rows in this block (<= block size)
  int32_t cost;
};

// Decode segment (cas_tc_decode.cu): one run of KV tiles for one row block (<= 128/G sequences with the same
// selection group, or ONE sequence's self cache) and one KV head; a persistent CTA walks a list of them.
struct DecSeg {
  int32_t kind;      // 0 = pool tiles (dec_tiles[tile_off ..]), 1 = self cache of sequence seq_off, -1 = stop
  int32_t tile_off;
  int32_t n_tiles;
  int32_t g;         // KV head
  int32_t seq_off;   // into dec_seqs (kind 0) / the sequence id (kind 1)
  int32_t n_seqs;
  int32_t part_row;  // first partial row of this segment, in units of sequences (x G rows per sequence)
  int32_t self_len;  // kind 1: keys in the cache
};

}  // namespace cas

// Device blob + pinned mirror of one slot table.  Blobs are recycled through the pool (no cudaMalloc /
// cudaFree / device-wide synchronisation per step): `done` marks the last kernel that read the blob,
// `ready` the end of its asynchronous upload.
struct TabBlob {
  char* d = nullptr;
  char* h = nullptr;
  size_t cap = 0;
  cudaEvent_t done = nullptr, ready = nullptr;
  bool has_done = false;
};

// One layer of the pool (Z in R^{L x p x d x 2} has a layer axis): the same slot layout repeated.
struct PoolLayer {
  void* pool_K = nullptr;
  void* pool_V = nullptr;
  float* grad_K = nullptr;
  float* grad_V = nullptr;
  float* state = nullptr;
  CUtensorMap tm_K, tm_V;        // [pool_tokens, Hkv, 128] bf16, 128-token boxes (bf16, D == 128 only)
  CUtensorMap tm_K16, tm_V16;    // the same tensors with 16-token boxes: one page of a packed tile
};

// Layout of cas_train_step_host's device scratch (byte offsets of the staged inputs, outputs and workspace).
// Device scratch of cas_train_step_host: TWO buffer sets (inputs Q, K_self, V_self, dO and results O, LSE, dQ,
// dK_self, dV_self; offsets relative to the set) used alternately by consecutive steps, then the backward workspace.
struct StepScratch {
  size_t oQ, oKs, oVs, odO, oO, oLSE, odQ, odKs, odVs, set_bytes, oWs, ws_bytes, total;
};

struct cas_pool {
  cas_pool_desc desc;
  std::vector<int32_t> cart_len;
  int32_t tile = 128;
  int64_t row_elems = 0;   // Hkv*D
  int elem_bytes = 2;
  std::vector<int32_t> slot_base, slot_cap;
  int64_t pool_tokens = 0;
  std::vector<int64_t> home_off;
  std::vector<int32_t> slot_of, cart_in, in_transit;
  std::vector<int32_t> grad_dirty;   // [n_layers * n_slots], layer-major
  std::vector<int64_t> opt_steps, last_used;
  std::vector<cas::Pending> pending;
  // data (caller-owned arenas)
  char* dev = nullptr;
  char* pinned = nullptr;
  cudaStream_t side = nullptr;
  int n_layers = 1;
  std::vector<PoolLayer> layers;
  // paged pool (desc.pool_tokens_budget > 0): pages of `tile` tokens, contiguous first-fit extents
  bool paged = false;
  int32_t n_pages = 0;
  std::vector<int32_t> page_owner;   // committed owner (cartridge id) of every page, -1 = free
  std::vector<int32_t> page_claim;   // arrival in flight that will own the page at commit, -1 = none
  cudaEvent_t ev_out_last = nullptr; // end of the most recent eviction copy (paged arrivals wait for it)
  bool pack = false;                 // tile == 16: remainders of the selected cartridges are packed into shared KV tiles
  int32_t pages_for(int c) const { return (cart_len[c] + tile - 1) / tile; }
  cudaEvent_t ev_side = nullptr, ev_main = nullptr;
  // arrivals (H2D) run on a second, library-owned stream so that they overlap the evictions (D2H) on
  // the caller's side stream (full-duplex host link); ev_slot[s] orders an arrival after the eviction
  // that frees its slot.
  cudaStream_t side_in = nullptr;
  cudaEvent_t ev_side_in = nullptr;
  std::vector<cudaEvent_t> ev_slot;
  std::vector<cudaEvent_t> ev_cart;   // end of a cartridge's last eviction copy (its pinned home is complete)
  std::vector<TabBlob> tab_free;     // recycled slot-table blobs
  cudaStream_t st_upload = nullptr;  // slot-table uploads
  // cas_train_step_host: input / output copies on their own streams so they overlap the kernels
  cudaStream_t st_h2d = nullptr, st_d2h = nullptr;
  // events of cas_train_step_host: [0] call begin; per buffer set k: [1+5k] Q/K_self/V_self in, [2+5k] dO in,
  // [3+5k] forward done, [4+5k] backward done, [5+5k] last read-back done
  cudaEvent_t ev_step[11] = {};
  int64_t step_count = 0;                // steps since the last layout change (buffer set = step_count & 1)
  void* fwd_part = nullptr;              // split-KV partials of the forward kernel's tail blocks (grow-only)
  size_t fwd_part_bytes = 0;
  int n_sm = 148;
  void* step_prev_scratch = nullptr;     // scratch / stream of the previous cas_train_step_host call
  cudaStream_t step_prev_stream = nullptr;
  StepScratch step_prev_layout{};
  bool has_tma = false;              // TMA descriptors over the working copies exist (bf16, D==128 only)

  float* slot_state(int l, int s, int which) const {  // which: 0..5 = pK,pV,mK,mV,vK,vV
    return layers[l].state + 6 * (int64_t)slot_base[s] * row_elems + (int64_t)which * slot_cap[s] * row_elems;
  }
  // pinned home of cartridge c: n_layers x six fp32 tensors of cart_len*Hkv*D elements, layer-major
  int64_t home_layer_bytes(int c) const { return 6 * (int64_t)cart_len[c] * row_elems * 4; }
  int64_t home_bytes(int c) const { return n_layers * home_layer_bytes(c); }
  float* home(int c, int l, int which) const {
    return (float*)(pinned + home_off[c] + l * home_layer_bytes(c)) + (int64_t)which * cart_len[c] * row_elems;
  }
  bool any_dirty(int s) const {
    for (int l = 0; l < n_layers; ++l) if (grad_dirty[(size_t)l * desc.n_slots + s]) return true;
    return false;
  }
};

struct cas_slot_table {
  cas_pool* pool = nullptr;
  int32_t B = 0, T = 0, nsel = 0;
  std::vector<int32_t> seq_off, sel_off, sel_cart, sel_slot, sel_base, sel_len, inv_off, inv_seq;
  std::vector<int64_t> P;
  std::vector<int32_t> used_slots;            // distinct selected slots, ascending
  std::vector<int32_t> kv_tile_off;           // [B+1] into kv_tiles (prefix tiles of sequence b)
  std::vector<int32_t> qtile_off;             // [B+1] 128-row query tiles before sequence b
  std::vector<cas::KvTile> kv_tiles;
  std::vector<cas::PackedTile> ptiles;        // packed prefix tiles (pools with 16-token pages)
  std::vector<int32_t> ptile_off;             // [B+1] packed tiles of sequence b
  std::vector<cas::FwdItem> fwd_items;        // 256-row blocks, longest first
  std::vector<cas::FwdItem> simt_items;       // 32-row blocks
  std::vector<cas::BwdItem> bwd_items;        // longest first
  std::vector<cas::BwdItem> simt_bwd_items;   // the CUDA-core path's tiles (never packed)
  int64_t pairs = 0, prefix_tokens = 0, unique_prefix_tokens = 0;
  int32_t max_lq = 0;
  // one device blob holding all the arrays above (recycled through the pool)
  TabBlob blob;
  char* d_blob = nullptr;
  mutable cudaStream_t last_stream = nullptr;   // stream of the last kernel that read the blob
  mutable bool used = false;
  int32_t *d_seq_off = nullptr, *d_sel_off = nullptr, *d_sel_base = nullptr, *d_sel_len = nullptr,
          *d_inv_off = nullptr, *d_inv_seq = nullptr, *d_kv_tile_off = nullptr,
          *d_used_slots = nullptr, *d_sel_slot = nullptr, *d_qtile_off = nullptr;
  cas::KvTile* d_kv_tiles = nullptr;
  cas::PackedTile* d_ptiles = nullptr;
  cas::FwdItem *d_fwd_items = nullptr, *d_simt_items = nullptr;
  cas::BwdItem* d_bwd_items = nullptr;
  cas::BwdItem* d_simt_bwd_items = nullptr;
  int32_t* d_counters = nullptr;              // persistent-scheduler tickets (zeroed per launch)
  int fwd_plan_key = -1, fwd_n_tail = 0, fwd_n_parts = 1;   // forward tail split, planned at the first forward call
  // decode-shaped batches: segments of the persistent split-KV kernel, built lazily for a given Hq by cas_tc_decode.cu
  int32_t dec_Hq = 0;
  int64_t dec_rows = 0;                       // partial rows per KV head (prefix segments + one self row per sequence) x G
  int32_t dec_grid = 0, dec_self_row_base = 0, dec_n_segs = 0;
  int32_t dec_fused = 1;                     // 1: every row block has <= 32 rows: partials are merged inside the decode launch
  std::vector<int32_t> dec_comb_off;          // [B+1] prefix partials per sequence
  char* d_dec_blob = nullptr;
  char* h_dec_blob = nullptr;                 // pinned mirror of the lists (asynchronous upload)
  cudaEvent_t dec_ready = nullptr;
  cas::DecSeg* d_dec_segs = nullptr;
  int32_t *d_dec_cta_off = nullptr, *d_dec_seqs = nullptr, *d_comb_off = nullptr, *d_comb_row = nullptr,
          *d_dec_cnt = nullptr, *d_dec_ticket = nullptr;
  cas::KvTile* d_dec_tiles = nullptr;
  cas::PackedTile* d_dec_ptiles = nullptr;
  float* d_dec_part = nullptr;
};

namespace cas {

// ---- kernel launchers (each returns CAS_OK / CAS_ERR_*) -------------------------------------
// Slots whose gradient buffer holds valid data at the time of a backward launch (grad-dirty).  A CLEAN slot's
// buffer is undefined: the first backward pass that touches it OVERWRITES, later ones accumulate.
constexpr int kMaxSlots = 8192;
struct SlotMask {
  uint32_t w[kMaxSlots / 32];
};

struct AttnArgs {
  const cas_pool* pool;
  const PoolLayer* L;            // the layer this call works on
  int layer;
  const cas_slot_table* tab;
  int Hq, Hkv, D, dtype;
  const void *Q, *Ks, *Vs, *O, *dO;
  const float* LSE_in;
  void *O_out, *dQ, *dKs, *dVs;
  float* LSE_out;
  float scale;
  void* workspace;
  size_t workspace_bytes;
  cudaStream_t stream;
  // RoPE fused into the tensor-core kernels (cas_prefix_attn_*_rope): cos/sin table [T, 64] of cas_rope_table;
  // forward: Q is rotated as its tile is loaded and written to Q_rot; backward: dQ leaves through the transpose
  const float* rope_cs = nullptr;
  int rope_layout = 0;
  void* Q_rot = nullptr;
  bool static_scratch = false;   // cas_prefix_attn_fwd_noalloc: split-KV partials in the library's static device array
};

int rope_table_rotate(const void* src, void* dst, const float* cs, int64_t T, int H, int layout, int inverse,
                      cudaStream_t st);
int simt_attn_fwd(const AttnArgs& a);
int simt_attn_bwd(const AttnArgs& a);
size_t simt_bwd_workspace(const cas_slot_table* t, int Hq);

bool tc_supported(const cas_pool* p, const cas_slot_table* t, int Hq);
int tc_attn_fwd(const AttnArgs& a);
int tc_attn_bwd(const AttnArgs& a);
size_t tc_bwd_workspace(const cas_slot_table* t, int Hq, int D);
int tc_make_pool_maps(cas_pool* p);
bool tc_decode_supported(const cas_pool* p, const cas_slot_table* t, int Hq);
int tc_decode_fwd(const AttnArgs& a, const void* Kc, const void* Vc, int cache_cap, const int32_t* self_len);

// Adam / refresh / zero
struct AdamSlotDesc {
  float* state;       // slot_state(s,0)
  void* wK;           // working copy of the slot (K), V is at wV
  void* wV;
  float* gK;
  float* gV;
  int64_t cap_elems;  // slot_cap*row_elems  (stride between the six state tensors)
  int64_t n_elems;    // cart_len*row_elems
  int64_t frozen_elems;
  float step_size_scale;  // lr_scale
  float bc1, bc2;     // 1-beta1^t, 1-beta2^t
  int32_t has_grad;   // 0: the slot's gradient buffer is not valid (clean slot): g = 0, nothing read or written
};
constexpr int kAdamBatch = 256;   // slot descriptors per launch, passed as kernel parameters (20 KB)
struct AdamBatch {
  AdamSlotDesc d[kAdamBatch];
};
int launch_adam(const AdamSlotDesc* h_desc, int n, const cas_adam_cfg& cfg, int dtype, cudaStream_t st);
int launch_refresh(float* pK, float* pV, void* wK, void* wV, float* gK, float* gV, int64_t n,
                   int dtype, cudaStream_t st);
int launch_zero(float* p, int64_t n, cudaStream_t st);
struct ZeroDesc {
  float *a, *b;     // gradient rows of one slot (K and V), 16-byte aligned
  int64_t n;        // elements (multiple of 4)
};
constexpr int kZeroBatch = 512;
struct ZeroBatch {
  ZeroDesc d[kZeroBatch];
};
int launch_zero_slots(const ZeroDesc* h, int n, cudaStream_t st);

}  // namespace cas
