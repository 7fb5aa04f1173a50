/* cas.h -- C ABI of libcas: the data-parallel hot path of "Cartridges at Scale" (CAS,
 * arxiv/paper_2606_04557) multi-cartridge training on one NVIDIA B200 (sm_100a).
 *
 * Citations are "PAPER.md:<line>" = the paper text this library was written from, plus the section.
 *
 * Conventions
 *   - plain C, no exceptions; every call returns an int: CAS_OK (0) or a negative CAS_ERR_* code;
 *     cas_last_error() returns the text of the last failure of the calling thread.
 *   - "device" pointers are CUDA device memory, "host" pointers ordinary host memory, "pinned"
 *     page-locked host memory (cudaHostAlloc).  THE CALLER OWNS every data buffer (pool arenas,
 *     Q/K/V/O/gradients, workspaces: allocate with PyTorch or cudaMalloc) and the main and side
 *     streams.  The library owns host metadata behind the opaque handles plus (a) device-side index
 *     tables (slot tables, tile lists, work lists) with pinned mirrors, kept in a small ring of blobs
 *     per pool that is recycled from table to table (cudaMalloc only while the ring warms up, freed in
 *     cas_pool_destroy); (b) for decode-shaped tables the split-KV work list and its partial-result
 *     scratch, allocated at the first forward call and freed with the table; (c) four internal
 *     non-blocking streams and their events: arrivals of a swap (high priority), slot-table uploads,
 *     and the input / output copies of cas_train_step_host.
 *   - compute calls are asynchronous on the caller's stream (cudaStream_t passed as void*): a
 *     stream that uses a slot table first waits (event) for the table's asynchronous upload.
 *     Evictions run on the side stream given at pool creation, arrivals on the library's own
 *     arrival stream (both directions of the host link are used at once).
 *   - destroy every slot table of a pool before the pool itself.
 *   - tensors are row-major, innermost dimension last:  Q/O/dO/dQ [T, Hq, D];  K_self/V_self and
 *     their grads [T, Hkv, D];  LSE [T, Hq] fp32;  pool tensors [pool_tokens, Hkv, D].
 *     T = total packed query tokens, sequence b owns tokens seq_off[b] .. seq_off[b+1]-1.
 *   - dtype CAS_BF16: Q,K,V,O,dO,dQ,dK_self,dV_self are bf16; CAS_F32: fp32.  Master params, Adam
 *     moments, gradient slots and LSE are fp32 in both.
 *   - query head h reads KV head h / (Hq/Hkv)  (consecutive query heads share a KV head).
 *   - all index arrays are int32 on the HOST; the library uploads what kernels need.
 */
#ifndef CAS_H_
#define CAS_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define CAS_OK 0
#define CAS_ERR_INVALID_ARG (-1)
#define CAS_ERR_SHAPE (-2)
#define CAS_ERR_NOT_RESIDENT (-3)
#define CAS_ERR_BUSY (-4)      /* slot/cartridge in transit, or gradients not yet consumed */
#define CAS_ERR_CAPACITY (-5)
#define CAS_ERR_CUDA (-6)

#define CAS_F32 0
#define CAS_BF16 1

#define CAS_DIR_OUT 0          /* HBM slot -> pinned host home */
#define CAS_DIR_IN 1           /* pinned host home -> HBM slot */

/* cas_set_impl(): which attention kernels serve the calls */
#define CAS_IMPL_AUTO 0        /* tcgen05/TMEM/TMA kernels when dtype==bf16 && D==128, else SIMT */
#define CAS_IMPL_SIMT 1        /* fp32-accumulate CUDA-core kernels (any dtype / D<=128, D%32==0) */
#define CAS_IMPL_TC 2          /* tensor-core kernels; CAS_ERR_SHAPE if the shape is unsupported */

typedef struct cas_pool cas_pool;
typedef struct cas_slot_table cas_slot_table;

/* The cartridge pool (sec. 2.1 "Budget Manager": "a fixed GPU pool of B <= N
 * cartridges, keeping the remaining N-B cartridges offloaded to CPU memory").  One layer's worth:
 * a cartridge is K and V of shape [cart_len, Hkv, D] (Z in R^{L x p x d x 2}, one L). */
typedef struct {
  int32_t dtype;            /* CAS_F32 | CAS_BF16: dtype of the working copy attention reads */
  int32_t Hkv;
  int32_t D;                /* head dim, multiple of 32, <= 128 */
  int32_t n_carts;          /* N */
  int32_t n_slots;          /* B <= N HBM slots.  n_slots == n_carts: slot s is sized for cartridge
                               s; otherwise all slots have the capacity of the longest cartridge */
  int32_t tile_tokens;      /* slot capacity granularity; 0 => 128 (the KV tile of the kernels;
                               the paper's own page is 16 tokens) */
  const int32_t* cart_len;  /* host [n_carts], tokens per cartridge, each >= 1 */
  int32_t n_layers;         /* L of Z in R^{L x p x d x 2}; 0 => 1.  Every layer has the same slot
                               layout; the device arena holds L carvings back to back, a cartridge's pinned home
                               L x (pK,pV,mK,mV,vK,vV).  Residency, step counts and rotation are per cartridge
                               (all layers move together); gradients-dirty is tracked per (layer, slot) */
  int64_t pool_tokens_budget; /* 0: static slots (above).  > 0: PAGED pool (PAPER.md:442-446:
                               cartridge sizes are multiples of the 16-token page of the paged KV cache, "enabling
                               efficient memory allocation and deallocation during ... pool rotation").  The pool holds
                               pool_tokens_budget tokens (a multiple of tile_tokens, which must then be given) = that many
                               pages of tile_tokens tokens; a resident cartridge owns a CONTIGUOUS run of
                               ceil(len/tile_tokens) pages chosen first-fit (lowest base) when it arrives and freed when
                               it leaves; the n_slots slots are handles (the most cartridges resident at once) whose
                               base and capacity follow their occupant.  Cartridges 0..n_slots-1 are placed first-fit
                               in order at creation (CAS_ERR_CAPACITY if they do not fit). */
} cas_pool_desc;

/* Device-side layout of the pool inside the caller's arena (all pointers are device pointers
 * into dev_arena; index arrays are host pointers owned by the pool, valid until destroy). */
typedef struct {
  void* pool_K;             /* working copy [pool_tokens,Hkv,D], dtype */
  void* pool_V;
  float* grad_K;            /* fp32 gradient slots [pool_tokens,Hkv,D]; the rows of a slot are defined only
                               while the slot is grad-dirty (see cas_prefix_attn_bwd); a clean slot's
                               gradient is zero by definition and its rows hold stale bytes */
  float* grad_V;
  float* state;             /* per slot s at state + 6*slot_base[s]*Hkv*D: six fp32 tensors of
                               slot_cap[s]*Hkv*D elements each: pK, pV, mK, mV, vK, vV */
  const int32_t* slot_base; /* host [n_slots] first pool token of slot s (paged pool: of its current occupant;
                               valid until the next cas_swap_in) */
  const int32_t* slot_cap;  /* host [n_slots] capacity in tokens (multiple of tile_tokens) */
  int64_t pool_tokens;
} cas_pool_layout;

typedef struct {
  int32_t cart;
  int32_t slot;
  int32_t dir;              /* CAS_DIR_OUT | CAS_DIR_IN */
  int32_t base_tok;         /* first pool token of the cartridge's extent: where it sits (OUT) / where it goes (IN).
                               Static slots: slot_base[slot]; paged pool: the first-fit run the planner chose */
  int64_t host_off;         /* byte offset of the cartridge's home in the pinned arena */
  int64_t nbytes;           /* 6 * cart_len * Hkv * D * 4 (params + both Adam moments, K and V) */
} cas_manifest_entry;

/* Adam (sec. 2.2 "Adam (Kingma and Ba, 2014) with fp32 precision, while we keep the
 * weights in bfloat16"; Table 5 PAPER.md:366-373, :390 "Num frozen tokens 1"). */
typedef struct {
  float lr, beta1, beta2, eps;
  int32_t n_frozen;         /* first n_frozen tokens of every cartridge are not updated */
  int32_t zero_grad;        /* 1: the step consumes the gradients: the slots become clean (gradient = 0) */
} cas_adam_cfg;

typedef struct {
  int32_t B, T, nsel, n_kv_tiles;
  int64_t pairs_per_head;   /* sum_b Lq_b*P_b + Lq_b(Lq_b+1)/2 : visible (query,key) pairs */
  int64_t prefix_tokens;    /* sum_b P_b */
  int64_t unique_prefix_tokens; /* tokens of distinct selected slots */
} cas_table_info;

const char* cas_version(void);
/* Copies the calling thread's last error text (NUL-terminated, truncated to n). */
void cas_last_error(char* buf, size_t n);
/* Select attention implementation (process-wide).  Returns CAS_ERR_INVALID_ARG on a bad value. */
int cas_set_impl(int impl);

/* ---- pool ---------------------------------------------------------------------------------- */
/* Bytes the caller must provide: dev_bytes of device memory (256-B aligned) and host_bytes of
 * pinned host memory for the homes of ALL n_carts cartridges (fp32 pK,pV,mK,mV,vK,vV packed). */
int cas_pool_query_bytes(const cas_pool_desc* desc, size_t* dev_bytes, size_t* host_bytes);
/* Carves the arenas, zero-fills the device arena (on side_stream, synchronised before return) and
 * places cartridges 0..n_slots-1 in slots 0..n_slots-1.  dev_arena == NULL creates a
 * bookkeeping-only pool (planning, tables and counters work; anything touching data returns
 * CAS_ERR_INVALID_ARG) -- used to test the host logic without a GPU.  pinned_arena may be NULL when
 * n_slots == n_carts (nothing can be swapped). */
int cas_pool_create(const cas_pool_desc* desc, void* dev_arena, void* pinned_arena,
                    void* side_stream, cas_pool** out);
int cas_pool_destroy(cas_pool* pool);
int cas_pool_layout_get(const cas_pool* pool, cas_pool_layout* out);
/* Initialise cartridge `cart` from host fp32 K,V [cart_len,Hkv,D]: master params <- K,V; moments
 * <- 0; resident: working copy <- cast(master), slot clean (gradient 0).  Synchronous. */
int cas_pool_load(cas_pool* pool, int32_t cart, const float* K, const float* V);
/* Read back one tensor of a cartridge into host memory.  Synchronous (device-wide). `what`:
 * 0..5 = pK,pV,mK,mV,vK,vV (fp32, from the slot if resident else from the pinned home);
 * 6,7 = grad_K, grad_V (fp32, resident only; zeros for a clean slot); 8,9 = working copy K,V (pool dtype,
 * resident only). */
int cas_pool_read(cas_pool* pool, int32_t cart, int32_t what, void* out);
/* The same for one layer of a multi-layer pool (cas_pool_load / cas_pool_read act on layer 0). */
int cas_pool_load_layer(cas_pool* pool, int32_t layer, int32_t cart, const float* K, const float* V);
int cas_pool_read_layer(cas_pool* pool, int32_t layer, int32_t cart, int32_t what, void* out);
/* Export integer state; any pointer may be NULL.  slot_of[n_carts] (-1 = not resident),
 * cart_in[n_slots] (-1 = free), opt_steps[n_carts], last_used[n_carts],
 * in_transit[n_carts] (0 stable, 1 leaving, 2 arriving), grad_dirty[n_slots]. */
int cas_pool_counters(const cas_pool* pool, int32_t* slot_of, int32_t* cart_in, int64_t* opt_steps,
                      int64_t* last_used, int32_t* in_transit, int32_t* grad_dirty);
/* Restore counters of one cartridge (checkpoint/resume, tests). */
int cas_pool_set_counters(cas_pool* pool, int32_t cart, int64_t opt_steps, int64_t last_used);

/* ---- slot table (sec. 2.1: per-sample subset Z~ = Z* U S, "each packed sample sees
 * a different subset via an attention mask") --------------------------------------------------- */
/* sel_cart[sel_off[b] .. sel_off[b+1]) = distinct cartridge ids visible to sequence b (target
 * first).  Validates (CAS_ERR_INVALID_ARG: bad offsets / ids / duplicates; CAS_ERR_SHAPE: an empty
 * sequence; CAS_ERR_NOT_RESIDENT; CAS_ERR_BUSY: cartridge in transit), maps ids to slots, builds
 * the inverted table (slot -> sequences, sorted by slot then sequence), the KV tile lists and
 * kernel work lists, uploads them, and stamps last_used = step on the selected cartridges. */
int cas_slot_table_build(cas_pool* pool, int32_t B, const int32_t* seq_off, const int32_t* sel_off,
                         const int32_t* sel_cart, int64_t step, cas_slot_table** out);
int cas_slot_table_destroy(cas_slot_table* table);
int cas_slot_table_info(const cas_slot_table* table, cas_table_info* out);
/* Any pointer may be NULL: sel_slot[nsel], inv_off[n_slots+1], inv_seq[nsel], P[B] (prefix
 * tokens visible to sequence b). */
int cas_slot_table_export(const cas_slot_table* table, int32_t* sel_slot, int32_t* inv_off,
                          int32_t* inv_seq, int64_t* P);
/* Diagnostic: the tail split the last tensor-core forward call planned for this table (0 blocks / 1 part before
 * the first call or when nothing is split).  The forward kernel runs one CTA per (256 query rows, head); when
 * the last wave of CTAs would fill less than half of the SMs, those n_tail blocks are cut along the KV axis into
 * n_parts CTAs each, whose un-normalised partials a small second kernel merges -- the result is the same
 * attention, summed in a different order. */
int cas_slot_table_fwd_split(const cas_slot_table* table, int32_t* n_tail, int32_t* n_parts);
/* "query token position IDs must be offset by the total number of active cartridge
 * KV tokens".  total_resident = tokens of all resident cartridges (the packed layout of
 * PAPER.md:71); P[b] = tokens visible to sequence b.  Either may be NULL. */
int cas_position_offsets(const cas_pool* pool, const cas_slot_table* table,
                         int64_t* total_resident, int64_t* P);

/* RoPE with that offset (RoFormer, Su et al. 2024, Eq. 34, cited at PAPER.md:77,
 * :320).  In place on X, device [T, H, D] dtype (Q with H = Hq, or K_self with H = Hkv; apply before
 * cas_prefix_attn_fwd -- the cartridge K in the pool are trained as they are and are not rotated).
 * Token i of sequence b gets position id m = pos_off[b] + i (host arrays; pos_off[b] = total_resident
 * or P[b] of cas_position_offsets, R7) and dimension pair k (k < D/2) is rotated by the angle
 * m * base^(-2k/D):  (a, b) -> (a cos - b sin, a sin + b cos).  layout 0: pair k = dims (2k, 2k+1)
 * (RoFormer's interleaved form); layout 1: pair k = dims (k, k + D/2) (the rotate-half storage of the
 * Qwen3 checkpoints).  inverse = 1 rotates by the negative angle = the transposed map: apply it to dQ and
 * dK_self to carry gradients back through the embedding.  Angles are formed in double precision.
 * D must be a multiple of 16 bytes of dtype per pair half (bf16: D % 8 == 0 for layout 0, D % 16 == 0 for
 * layout 1) and D <= 256, else CAS_ERR_SHAPE.  Asynchronous on `stream`. */
int cas_rope_apply(int32_t dtype, int32_t B, const int32_t* seq_off, const int64_t* pos_off, int32_t H,
                   int32_t D, double base, int32_t layout, int32_t inverse, void* X, void* stream);

/* ---- attention ------------------------------------------------------------------------------ */
/* Forward.  For every sequence b, query head h, row i (token t):
 *   visible keys = all tokens of the slots selected by b (read IN PLACE from the pool, no concat)
 *                  U own tokens seq_off[b]..t of K_self/V_self (causal, diagonal included);
 *   s_j = scale*q.k_j ; LSE[t,h] = ln sum_j exp(s_j) ; O[t,h,:] = sum_j exp(s_j-LSE) v_j.
 * Q,O device [T,Hq,D] dtype; K_self,V_self device [T,Hkv,D] dtype or both NULL (prefix only; then
 * every sequence must select >= 1 cartridge); LSE device [T,Hq] fp32.  scale must be positive and finite
 * (CAS_ERR_INVALID_ARG otherwise: the kernels take row maxima on the raw scores).  Forward calls on one pool must be
 * ordered by the caller (one stream, or events): they share the pool's split-KV partial scratch.  Pool rows past a cartridge's
 * length inside its slot are read by the tile loads and masked; they must stay finite (the arena is zero-filled at
 * creation and the library never writes there). */
int cas_prefix_attn_fwd(cas_pool* pool, const cas_slot_table* table, int32_t Hq, const void* Q,
                        const void* K_self, const void* V_self, float scale, void* O, float* LSE,
                        void* stream);
/* Decode step with a growing self cache (sec. 2.5 inference: the selected
 * cartridges' KV are concatenated before the prompt; :340 App. A "2048 maximum completion tokens").  `table` must
 * hold ONE query token per sequence (seq_off = 0,1,..,B); Q,O device [B,Hq,D] bf16, LSE device [B,Hq] fp32.  The
 * keys of sequence b are all tokens of its selected cartridges (read in place from the pool) plus rows
 * [0, self_len[b]) of ITS OWN cache K_cache/V_cache, device [B, cache_cap, Hkv, D] bf16: the caller appends the
 * current token's key/value at row self_len[b]-1 before the call, so the query sees itself (causal diagonal) and
 * every earlier token of the sequence.  self_len is a HOST array [B], 0 <= self_len[b] <= cache_cap.  K_cache and
 * V_cache may both be NULL (prefix only).  The result is cas_prefix_attn_fwd's for the last row of a sequence of
 * self_len[b] tokens.  Cache rows at and beyond self_len[b] are loaded with their tile and masked: they must hold
 * FINITE values (zero-initialise the cache).  bf16 pools with D = 128 only (CAS_ERR_SHAPE otherwise); at most 1024
 * sequences per call when a cache is given (CAS_ERR_CAPACITY).  One kernel launch: split-KV partials are merged by
 * the CTA that finishes a row last.  A slot table carries the scratch of ONE decode launch at a time: launches that
 * share a table must be ordered (same stream).  Asynchronous on `stream`. */
int cas_decode_attn(cas_pool* pool, const cas_slot_table* table, int32_t Hq, const void* Q, const void* K_cache,
                    const void* V_cache, int32_t cache_cap, const int32_t* self_len, float scale, void* O,
                    float* LSE, void* stream);
/* Retrieval-ordered cartridge selection (sec. 3 "Retrieval": "we map each retrieved chunk to a document
 * id, which in turn is associated with a cartridge.  The final list contains the unique cartridge ids in the order of
 * their retrieval").  chunk_ids[k]: retrieved chunks, best first; chunk_to_cart[n_chunks]: chunk -> cartridge id.
 * Writes at most max_carts distinct cartridge ids in order of first appearance.  Host only. */
int cas_select_retrieved(const int32_t* chunk_ids, int32_t k, const int32_t* chunk_to_cart, int32_t n_chunks,
                         int32_t max_carts, int32_t* out_carts, int32_t* n_out);

/* Device workspace bytes cas_prefix_attn_bwd needs for this table / Hq. */
int cas_prefix_attn_bwd_workspace_bytes(const cas_pool* pool, const cas_slot_table* table,
                                        int32_t Hq, size_t* bytes);
/* Backward (PAPER.md:44 "only the key-value vectors in Z receive gradients"; :176 all active
 * cartridges back-propagated simultaneously).  dQ [T,Hq,D] dtype is overwritten.  dK/dV of prefix
 * keys are ACCUMULATED (+=) into the pool's fp32 gradient slots of the selected slots, summed over
 * the Hq/Hkv heads of a group and over every sequence that selected the slot; slots selected by no
 * sequence are not touched.  dK_self/dV_self [T,Hkv,D] dtype are overwritten (may both be NULL).
 * Marks the selected slots grad-dirty.  "+=" is implemented without ever zeroing a buffer: a CLEAN slot
 * (never touched, or consumed by cas_adam_step / cas_grad_zero, or just arrived) has gradient zero by
 * definition, so the first backward pass that selects it OVERWRITES its rows and marks it dirty; later
 * passes add.  Read gradients through cas_pool_read (zeros for clean slots), not through the raw rows.
 * Determinism: dK/dV (pool slots and self) are bit-reproducible run to run -- every gradient row is produced by
 * exactly one CTA in a fixed order.  dQ on the tensor-core path is NOT: the per-KV-tile partial dQ tiles are summed
 * by fp32 reductions in L2 whose order depends on CTA scheduling, so two runs can differ in the last fp32 bits
 * before the final rounding to bf16 (within 1 bf16 ulp per element; CAS_IMPL_SIMT is deterministic). */
int cas_prefix_attn_bwd(cas_pool* pool, const cas_slot_table* table, int32_t Hq, const void* Q,
                        const void* K_self, const void* V_self, const void* O, const float* LSE,
                        const void* dO, float scale, void* dQ, void* dK_self, void* dV_self,
                        void* workspace, size_t workspace_bytes, void* stream);

/* ---- optimizer ------------------------------------------------------------------------------ */
/* One fused Adam step over the listed slots (slots == NULL: every resident slot whose cartridge
 * is not in transit).  Per cartridge: t = ++opt_steps; m = b1 m + (1-b1) g; v = b2 v + (1-b2) g^2;
 * p -= lr*lr_scale[i]*(m/(1-b1^t)) / (sqrt(v/(1-b2^t)) + eps); working copy = RNE(p); with zero_grad
 * the slot becomes clean (g = 0; nothing is written to the gradient rows).  A clean slot is updated with
 * g = 0 and its gradient rows are not read.  lr_scale: host [n] per listed slot (PAPER.md:85 per-cartridge warmup), NULL = 1. */
int cas_adam_step(cas_pool* pool, const cas_adam_cfg* cfg, const int32_t* slots, int32_t n,
                  const float* lr_scale, void* stream);
/* Discards the gradients of the listed slots (NULL: all): the slots become clean.  Host bookkeeping only. */
int cas_grad_zero(cas_pool* pool, const int32_t* slots, int32_t n, void* stream);

/* ---- rotation (sec. 2.1 "Pool rotation"; Table 5 :377-381) ------------------------ */
/* Pure integer planning, moves no data.  Evictees: the n_out resident, stable, unprotected
 * cartridges with the smallest last_used (ties: smaller id).  Arrivals: up to n_in non-resident
 * cartridges with the fewest opt_steps (ties: smaller mix64(seed,step,cart), then smaller id),
 * paired in that order with the free slots (free now or freed by the evictees) in ascending slot
 * order.  Writes all OUT entries (ascending slot) then all IN entries.  CAS_ERR_CAPACITY if
 * `capacity` entries do not suffice.  Paged pool: an arrival takes the lowest unused slot handle and the
 * first-fit run of pages that are free now or freed by this round's evictees and not taken by an earlier arrival of
 * the plan (entry.base_tok); a cartridge for which no run is long enough is skipped (fragmentation -- the paper's
 * own implementation empties its allocator cache every 5 rotations for the same reason). */
int cas_plan_rotation(const cas_pool* pool, int64_t step, int32_t n_in, int32_t n_out,
                      const int32_t* protect_carts, int32_t n_protect, uint64_t seed,
                      cas_manifest_entry* entries, int32_t capacity, int32_t* n_entries);
/* Enqueue the OUT entries of a manifest on the side stream (resp. the IN entries on the library's
 * arrival stream), in order, one cudaMemcpyAsync per contiguous piece.  An arrival into a slot that
 * an eviction of the same round frees waits (per-slot event) for that eviction only.  After all
 * arrival copies, one kernel per arrival derives the working copy; the slot starts clean (gradient 0).
 * swap_out first waits (event) for work already enqueued on `after_stream` (the stream whose Adam
 * last wrote the evictees; may be NULL).
 * CAS_ERR_BUSY: evictee has un-consumed gradients / cartridge already in transit / slot occupied. */
int cas_swap_out(cas_pool* pool, const cas_manifest_entry* entries, int32_t n, int64_t step,
                 void* after_stream);
int cas_swap_in(cas_pool* pool, const cas_manifest_entry* entries, int32_t n, int64_t step);
/* Makes main_stream wait for everything enqueued on the side and arrival streams and flips residency:
 * evictees leave, arrivals become selectable with last_used = the step of their swap_in. */
int cas_swap_commit(cas_pool* pool, void* main_stream);

/* ---- policy helpers (host only) ---------------------------------------- */
/* Eq. 1 mixture sampler: example b with target cartridge targets[b] sees only its target
 * with probability p_iso, else the target plus S ~ U(Z_dist, k), k ~ U{k_min..k_max} (inclusive), where
 * Z_dist = the resident, stable cartridges without the target; k is clamped to card(Z_dist); S is drawn
 * without replacement (partial Fisher-Yates over Z_dist in ascending id order).  Output in the layout
 * cas_slot_table_build takes: sel_off[B+1], sel_cart (target first, then the distractors in draw order).
 * Randomness is the counter-based generator of DESIGN.md R31 (seed, step, b, draw index), so a call is a
 * pure function of its arguments and the pool's residency.  CAS_ERR_NOT_RESIDENT: a target is not resident;
 * CAS_ERR_CAPACITY: sel_cart is too small. */
int cas_sample_selection(const cas_pool* pool, int32_t B, const int32_t* targets, double p_iso,
                         int32_t k_min, int32_t k_max, uint64_t seed, int64_t step, int32_t* sel_off,
                         int32_t* sel_cart, int32_t capacity);

/* Global learning rate ("slow linear decay schedule", Table 5 :366-373): linear from
 * warmup_min_lr at t = 0 to eta0 at t = warmup_steps, then linear down to alpha_f * eta0 at total_steps,
 * constant afterwards (R29). */
typedef struct cas_lr_cfg {
  double eta0;            /* peak learning rate (0.05 - 0.1) */
  int64_t warmup_steps;   /* W = 200 */
  double warmup_min_lr;   /* 0.002 */
  double alpha_f;         /* final LR multiplier 0.02 */
  int64_t total_steps;
} cas_lr_cfg;
int cas_lr_schedule(const cas_lr_cfg* cfg, int64_t t, double* eta);

/* Per-cartridge warmup: scale[i] for the cartridge in slots[i] with s optimizer steps =
 * ceil(min(1, (s+1)/w_c) * n_b) / n_b -- min(1, s/W_c) counted with the step being taken and rounded up to
 * one of n_b levels (N_b = 4 in the paper; R30).  Feed the result to cas_adam_step's lr_scale. */
int cas_warmup_scales(const cas_pool* pool, const int32_t* slots, int32_t n, int32_t w_c, int32_t n_b,
                      float* scale);

/* ---- the layer axis and micro-batches -----------------------------------------
 * a cartridge is Z in R^{L x p x d x 2} -- one K/V block per attention layer; PAPER.md:375-376 (Table 5):
 * global batch 128 of packed 8,192-token sequences, i.e. several micro-batches per optimizer step.  The *_layer
 * calls are cas_prefix_attn_fwd / _bwd / cas_decode_attn on layer `layer` of the pool (those act on layer 0); ONE
 * slot table serves every layer (the selection, and the residency it was built against, are per cartridge).
 * cas_adam_step updates every layer of the listed slots in one launch sequence, cas_swap_* move every layer. */
int cas_prefix_attn_fwd_layer(cas_pool* pool, const cas_slot_table* table, int32_t layer, int32_t Hq, const void* Q,
                              const void* K_self, const void* V_self, float scale, void* O, float* LSE, void* stream);
int cas_prefix_attn_bwd_layer(cas_pool* pool, const cas_slot_table* table, int32_t layer, int32_t Hq, const void* Q,
                              const void* K_self, const void* V_self, const void* O, const float* LSE,
                              const void* dO, float scale, void* dQ, void* dK_self, void* dV_self, void* workspace,
                              size_t workspace_bytes, void* stream);
int cas_decode_attn_layer(cas_pool* pool, const cas_slot_table* table, int32_t layer, int32_t Hq, const void* Q,
                          const void* K_cache, const void* V_cache, int32_t cache_cap, const int32_t* self_len,
                          float scale, void* O, float* LSE, void* stream);
/* ---- a forward call that allocates nothing ---------------------------------------------------------------
 * cas_prefix_attn_fwd_layer for callers that may not call cudaMalloc (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid it).  cas_prefix_attn_fwd keeps the split-KV partials of its tail blocks
 * (cas_slot_table_fwd_split) in a pool-owned buffer that it allocates, and may grow, inside a call; this variant keeps
 * them in a file-scope device array of the library instead -- 148 split CTAs x 256 rows x 132 floats = 20,004,864
 * bytes, held by every GPU that loads the library until the process exits -- and calls no cudaMalloc / cudaFree or
 * allocating library routine (the first forward call on a table plans the split with a few small host-heap vectors;
 * later calls reuse the plan).  Same arguments, same kernels, same result bits as cas_prefix_attn_fwd_layer.
 * Errors: CAS_ERR_SHAPE unless the tensor-core training kernel serves the call (bf16, D = 128, some sequence with
 * more than one query token); CAS_ERR_CAPACITY when the table's split needs more than 148 split CTAs (it never does
 * on a GPU with <= 148 SMs).  ALL calls on a device share the one array, which keeps the last call's contents
 * (nothing in it has to start at zero: a call reads only the partial rows its own CTAs wrote): calls of this entry
 * point that overlap on the GPU -- two streams, two pools, two host threads -- race; order them on one stream or
 * with events.  Asynchronous on `stream`. */
int cas_prefix_attn_fwd_noalloc(cas_pool* pool, const cas_slot_table* table, int32_t layer, int32_t Hq,
                                const void* Q, const void* K_self, const void* V_self, float scale, void* O,
                                float* LSE, void* stream);

/* ---- RoPE fused into the attention calls (PAPER.md:77 the offset is "recomputed at each
 * step") -----------------------------------------------------------------------------------------------------
 * cas_rope_table writes, once per packed batch (it serves every head and every layer), cs[t][k] = (cos, sin) of
 * m_t * base^(-2k/D) as device fp32 [T, D/2, 2]; position ids, angle arithmetic (double) and argument checks as
 * cas_rope_apply.  cas_prefix_attn_fwd_rope takes UN-rotated Q / K_self: the forward kernel rotates every Q tile
 * in shared memory as it arrives and writes the rotated rows to Q_rot (device [T, Hq, D] bf16) -- no separate pass
 * reads and re-writes Q -- and K_self (1/G of the query bytes) is rotated into K_self_rot by a small pass in the same
 * call; the attention is that of cas_prefix_attn_fwd on the rotated tensors.  cas_prefix_attn_bwd_rope takes Q_rot
 * and K_self_rot as left by the forward call and returns dQ and dK_self with respect to the UN-rotated inputs: the
 * transpose rotation is applied to dQ in fp32 inside the kernel that converts the dQ accumulators to bf16, and to
 * dK_self in place.  Cartridge K/V in the pool are not rotated (they are trained as they are).  Tensor-core path only
 * (bf16, D = 128, more than one query token per sequence somewhere): otherwise CAS_ERR_SHAPE -- use cas_rope_apply. */
typedef struct cas_rope {
  const float* cs;    /* device [T, D/2, 2], written by cas_rope_table for the SAME seq_off as the slot table */
  int32_t layout;     /* 0: pairs (2k, 2k+1); 1: pairs (k, k + D/2) -- as cas_rope_apply */
  int32_t reserved;
} cas_rope;
int cas_rope_table(int32_t B, const int32_t* seq_off, const int64_t* pos_off, int32_t D, double base, float* cs,
                   void* stream);
int cas_prefix_attn_fwd_rope(cas_pool* pool, const cas_slot_table* table, int32_t layer, int32_t Hq, const void* Q,
                             const void* K_self, const void* V_self, const cas_rope* rope, void* Q_rot,
                             void* K_self_rot, float scale, void* O, float* LSE, void* stream);
int cas_prefix_attn_bwd_rope(cas_pool* pool, const cas_slot_table* table, int32_t layer, int32_t Hq,
                             const void* Q_rot, const void* K_self_rot, const void* V_self, const void* O,
                             const float* LSE, const void* dO, const cas_rope* rope, float scale, void* dQ,
                             void* dK_self, void* dV_self, void* workspace, size_t workspace_bytes, void* stream);

/* Device buffers of one (micro-batch, layer): shapes as in cas_prefix_attn_fwd / _bwd.  rope != NULL: Q and K_self
 * are un-rotated, the step runs the *_rope calls with Q_rot / K_self_rot as scratch outputs (K_self_rot may be NULL
 * when K_self is). */
typedef struct {
  const void *Q, *K_self, *V_self, *dO;
  void* O;
  float* LSE;
  void *dQ, *dK_self, *dV_self;
  const cas_rope* rope;
  void *Q_rot, *K_self_rot;
} cas_layer_io;
/* One optimizer step: for every micro-batch m (its own slot table tables[m], all built against the current
 * residency) the forward pass of layers 0..L-1, then the backward pass of layers L-1..0 -- dK/dV ACCUMULATE into the
 * gradient slots across micro-batches -- and then ONE cas_adam_step over all stable resident slots (lr_scale as
 * there, per resident slot in ascending slot order, or NULL).  io[m * L + l].  In a real model each layer's Q and
 * dO come from the frozen network around the attention call; this driver takes them all up front (synthetic
 * benchmarks, tests).  workspace: cas_train_step_layers_workspace_bytes().  Asynchronous on `stream`. */
int cas_train_step_layers_workspace_bytes(const cas_pool* pool, const cas_slot_table* const* tables, int32_t n_micro,
                                          int32_t Hq, size_t* bytes);
int cas_train_step_layers(cas_pool* pool, const cas_slot_table* const* tables, int32_t n_micro, int32_t Hq,
                          const cas_layer_io* io, float scale, const cas_adam_cfg* cfg, const float* lr_scale,
                          void* workspace, size_t workspace_bytes, void* stream);

/* ---- end-to-end convenience: one training step from HOST buffers --------------------------------
 * H2D copies of hQ,hK_self,hV_self,hdO (pinned host, dtype), fwd, bwd, Adam over all stable
 * resident slots, D2H of O, LSE, dQ and (when hdK_self/hdV_self are given: both or neither) dK_self, dV_self --
 * every result of the backward pass that does not stay in the pool.  Kernels run on `stream`; the copies run on
 * two internal copy streams: dO arrives under the forward pass, O/LSE leave under the backward pass, dQ, dK_self,
 * dV_self leave under Adam.  dev_scratch must hold cas_train_step_host_scratch_bytes() (single-layer pools only):
 * TWO sets of input and result buffers, used alternately by consecutive calls, plus the backward workspace; it
 * belongs to the library between back-to-back calls that reuse it.  When the next call has the SAME scratch layout
 * (same scratch, stream, T, Hq, workspace size) its inputs are copied into the other set while this call still
 * computes (they wait only for the backward pass two calls back, the last reader of that set); with a different
 * layout (ragged batches) the call first waits for everything in flight, because the regions move.
 *   cas_train_step_host        `stream` finally waits for this call's last read-back: once `stream` has completed
 *                              the call, the host results are valid and the host inputs may be overwritten.
 *   cas_train_step_host_async  does NOT make `stream` wait for the read-back, so the next call's kernels start while
 *                              this call's dQ is still crossing the host link (steady state: a step costs
 *                              max(kernels, H2D bytes, D2H bytes) instead of their sum).  The host inputs may be
 *                              overwritten once `stream` has completed the call; the host RESULTS are valid only
 *                              after cas_train_step_host_wait.  Result buffers of calls in flight must be distinct
 *                              or the caller accepts that a later call overwrites them (copies run in call order).
 *   cas_train_step_host_wait   makes `stream` wait for the read-backs of all earlier calls (no host blocking).
 * In every variant the host inputs must hold their data when the call is MADE (the input copies are ordered after
 * earlier copies, not after the caller's stream).  Asynchronous. */
int cas_train_step_host_scratch_bytes(const cas_pool* pool, const cas_slot_table* table, int32_t Hq,
                                      size_t* bytes);
int cas_train_step_host(cas_pool* pool, const cas_slot_table* table, int32_t Hq, const void* hQ,
                        const void* hK_self, const void* hV_self, const void* hdO, float scale,
                        const cas_adam_cfg* cfg, void* hO, float* hLSE, void* hdQ, void* hdK_self,
                        void* hdV_self, void* dev_scratch, size_t scratch_bytes, void* stream);
int cas_train_step_host_async(cas_pool* pool, const cas_slot_table* table, int32_t Hq, const void* hQ,
                              const void* hK_self, const void* hV_self, const void* hdO, float scale,
                              const cas_adam_cfg* cfg, void* hO, float* hLSE, void* hdQ, void* hdK_self,
                              void* hdV_self, void* dev_scratch, size_t scratch_bytes, void* stream);
int cas_train_step_host_wait(cas_pool* pool, void* stream);

/* ---- hardware self-test (not on the hot path) --------------------------------------------------
 * D[256,128] fp32 = A[256,64] * B[128,64]^T (bf16, row-major, device) computed by ONE tcgen05.mma.cta_group::2
 * stream on a 2-CTA cluster: proves the CTA-pair primitives of csrc/cas_sm100.cuh on the GPU at hand. */
int cas_selftest_cta_pair_mma(const void* A, const void* B, float* D, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* CAS_H_ */
