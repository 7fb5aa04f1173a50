// Host runtime of libcas: pool carving, integer bookkeeping (slot tables, inverted tables, rotation
// planner, manifests, counters), swap engine, dispatch to the kernels.  C ABI: include/cas.h.
//
// The integer rules implemented here are DESIGN.md "Bookkeeping" K1-K4 (sec. 2.1);
// an independent pure-Python restatement lives in oracle/bookkeeping.py and is compared bit-exactly.
#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <numeric>
#include <set>

#include "cas_internal.h"

namespace cas {

static thread_local char g_err[512] = "";
static int g_impl = CAS_IMPL_AUTO;

void set_error(const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
}

int cuda_fail(cudaError_t e, const char* what) {
  set_error("CUDA error %d (%s) at %s", (int)e, cudaGetErrorString(e), what);
  return CAS_ERR_CUDA;
}

static inline int64_t round_up(int64_t x, int64_t m) { return (x + m - 1) / m * m; }

// DESIGN.md R15: SplitMix64 finaliser over seed + gamma*(step+1) + 0xD1B54A32D192ED03*(cart+1).
static inline uint64_t mix64(uint64_t seed, uint64_t step, uint64_t cart) {
  uint64_t z = seed + 0x9E3779B97F4A7C15ull * (step + 1) + 0xD1B54A32D192ED03ull * (cart + 1);
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}

struct Carve {
  int64_t off_K, off_V, off_gK, off_gV, off_state, total;
};

static Carve carve(int64_t pool_tokens, int64_t row_elems, int eb) {
  Carve c;
  int64_t o = 0;
  const int64_t A = 1024;
  c.off_K = o;      o = round_up(o + pool_tokens * row_elems * eb, A);
  c.off_V = o;      o = round_up(o + pool_tokens * row_elems * eb, A);
  c.off_gK = o;     o = round_up(o + pool_tokens * row_elems * 4, A);
  c.off_gV = o;     o = round_up(o + pool_tokens * row_elems * 4, A);
  c.off_state = o;  o = round_up(o + 6 * pool_tokens * row_elems * 4, A);
  c.total = o;
  return c;
}

static int check_desc(const cas_pool_desc* d) {
  if (!d || !d->cart_len) { set_error("null pool desc"); return CAS_ERR_INVALID_ARG; }
  if (d->dtype != CAS_F32 && d->dtype != CAS_BF16) { set_error("bad dtype"); return CAS_ERR_INVALID_ARG; }
  if (d->Hkv < 1 || d->D < 32 || d->D > 128 || d->D % 32) { set_error("Hkv>=1, D in {32,64,96,128}"); return CAS_ERR_SHAPE; }
  if (d->n_carts < 1 || d->n_slots < 1 || d->n_slots > d->n_carts) { set_error("need 1 <= n_slots <= n_carts"); return CAS_ERR_INVALID_ARG; }
  if (d->n_slots > kMaxSlots) { set_error("at most %d slots", kMaxSlots); return CAS_ERR_CAPACITY; }
  if (d->n_layers < 0 || d->n_layers > 1024) { set_error("n_layers must be in [0, 1024] (0 = 1)"); return CAS_ERR_INVALID_ARG; }
  if (d->pool_tokens_budget < 0 || (d->pool_tokens_budget > 0 && (d->tile_tokens == 0 || d->pool_tokens_budget % d->tile_tokens))) {
    set_error("pool_tokens_budget must be a positive multiple of an explicit tile_tokens");
    return CAS_ERR_INVALID_ARG;
  }
  if (d->tile_tokens < 0 || (d->tile_tokens && d->tile_tokens % 16)) { set_error("tile_tokens must be a multiple of 16"); return CAS_ERR_INVALID_ARG; }
  for (int i = 0; i < d->n_carts; ++i)
    if (d->cart_len[i] < 1) { set_error("cart_len[%d] < 1", i); return CAS_ERR_INVALID_ARG; }
  return CAS_OK;
}

// Lowest base page of a run of n pages that are all free per `ok(page)`; -1 if there is none (first fit).
template <typename F>
static int32_t first_fit(int32_t n_pages, int32_t n, F ok) {
  int32_t run = 0;
  for (int32_t q = 0; q < n_pages; ++q) {
    run = ok(q) ? run + 1 : 0;
    if (run == n) return q - n + 1;
  }
  return -1;
}

// returns false if the initial cartridges of a paged pool do not fit its budget
static bool layout_slots(const cas_pool_desc* d, std::vector<int32_t>& base, std::vector<int32_t>& cap,
                         int64_t& pool_tokens, std::vector<int32_t>* page_owner = nullptr) {
  const int tile = d->tile_tokens ? d->tile_tokens : 128;
  base.assign(d->n_slots, 0);
  cap.assign(d->n_slots, 0);
  if (d->pool_tokens_budget > 0) {
    const int32_t n_pages = (int32_t)(d->pool_tokens_budget / tile);
    std::vector<int32_t> owner(n_pages, -1);
    for (int c = 0; c < d->n_slots; ++c) {
      const int32_t n = (d->cart_len[c] + tile - 1) / tile;
      const int32_t b = first_fit(n_pages, n, [&](int32_t q) { return owner[q] < 0; });
      if (b < 0) return false;
      for (int32_t q = b; q < b + n; ++q) owner[q] = c;
      base[c] = b * tile;
      cap[c] = n * tile;
    }
    pool_tokens = d->pool_tokens_budget;
    if (page_owner) *page_owner = owner;
    return true;
  }
  if (d->n_slots == d->n_carts) {
    for (int s = 0; s < d->n_slots; ++s) cap[s] = (int32_t)round_up(d->cart_len[s], tile);
  } else {
    int32_t mx = 0;
    for (int i = 0; i < d->n_carts; ++i) mx = std::max(mx, d->cart_len[i]);
    for (int s = 0; s < d->n_slots; ++s) cap[s] = (int32_t)round_up(mx, tile);
  }
  int64_t o = 0;
  for (int s = 0; s < d->n_slots; ++s) { base[s] = (int32_t)o; o += cap[s]; }
  pool_tokens = o;
  return true;
}

template <typename T>
static size_t blob_add(size_t& off, const std::vector<T>& v, size_t extra = 0) {
  size_t o = off;
  off = (size_t)round_up((int64_t)(off + (v.size() + extra) * sizeof(T)), 256);
  return o;
}

}  // namespace cas

using namespace cas;

extern "C" {

const char* cas_version(void) { return "libcas 0.1 (sm_100a)"; }

void cas_last_error(char* buf, size_t n) {
  if (!buf || !n) return;
  strncpy(buf, g_err, n - 1);
  buf[n - 1] = 0;
}

int cas_set_impl(int impl) {
  if (impl < CAS_IMPL_AUTO || impl > CAS_IMPL_TC) { set_error("bad impl"); return CAS_ERR_INVALID_ARG; }
  g_impl = impl;
  return CAS_OK;
}

int cas_pool_query_bytes(const cas_pool_desc* desc, size_t* dev_bytes, size_t* host_bytes) {
  int rc = check_desc(desc);
  if (rc) return rc;
  std::vector<int32_t> base, cap;
  int64_t pool_tokens;
  if (!layout_slots(desc, base, cap, pool_tokens)) { set_error("the first n_slots cartridges do not fit pool_tokens_budget"); return CAS_ERR_CAPACITY; }
  if (pool_tokens >= (1ll << 31)) { set_error("pool too large for int32 token indices"); return CAS_ERR_CAPACITY; }
  const int64_t row = (int64_t)desc->Hkv * desc->D;
  Carve c = carve(pool_tokens, row, desc->dtype == CAS_BF16 ? 2 : 4);
  const int64_t L = desc->n_layers ? desc->n_layers : 1;
  if (dev_bytes) *dev_bytes = (size_t)(L * c.total);
  if (host_bytes) {
    int64_t h = 0;
    for (int i = 0; i < desc->n_carts; ++i) h += L * 6 * (int64_t)desc->cart_len[i] * row * 4;
    *host_bytes = (size_t)h;
  }
  return CAS_OK;
}

int cas_pool_create(const cas_pool_desc* desc, void* dev_arena, void* pinned_arena, void* side_stream,
                    cas_pool** out) {
  if (!out) { set_error("null out"); return CAS_ERR_INVALID_ARG; }
  int rc = check_desc(desc);
  if (rc) return rc;
  if (dev_arena && !pinned_arena && desc->n_slots != desc->n_carts) {
    set_error("pinned arena required when n_slots < n_carts");
    return CAS_ERR_INVALID_ARG;
  }
  cas_pool* p = new cas_pool();
  p->desc = *desc;
  p->cart_len.assign(desc->cart_len, desc->cart_len + desc->n_carts);
  p->desc.cart_len = p->cart_len.data();
  p->tile = desc->tile_tokens ? desc->tile_tokens : 128;
  p->n_layers = desc->n_layers ? desc->n_layers : 1;
  p->desc.n_layers = p->n_layers;
  p->row_elems = (int64_t)desc->Hkv * desc->D;
  p->elem_bytes = desc->dtype == CAS_BF16 ? 2 : 4;
  p->paged = desc->pool_tokens_budget > 0;
  p->pack = p->tile == 16;
  if (!layout_slots(desc, p->slot_base, p->slot_cap, p->pool_tokens, &p->page_owner)) {
    delete p;
    set_error("the first n_slots cartridges do not fit pool_tokens_budget");
    return CAS_ERR_CAPACITY;
  }
  if (p->paged) {
    p->n_pages = (int32_t)p->page_owner.size();
    p->page_claim.assign(p->n_pages, -1);
  }
  if (p->pool_tokens >= (1ll << 31)) { delete p; set_error("pool too large"); return CAS_ERR_CAPACITY; }
  p->home_off.assign(desc->n_carts, 0);
  for (int c = 1; c < desc->n_carts; ++c) p->home_off[c] = p->home_off[c - 1] + p->home_bytes(c - 1);
  p->slot_of.assign(desc->n_carts, -1);
  p->cart_in.assign(desc->n_slots, -1);
  for (int s = 0; s < desc->n_slots; ++s) { p->slot_of[s] = s; p->cart_in[s] = s; }
  p->in_transit.assign(desc->n_carts, 0);
  p->grad_dirty.assign((size_t)p->n_layers * desc->n_slots, 0);
  p->layers.assign(p->n_layers, PoolLayer());
  p->opt_steps.assign(desc->n_carts, 0);
  p->last_used.assign(desc->n_carts, -1);
  p->dev = (char*)dev_arena;
  p->pinned = (char*)pinned_arena;
  p->side = (cudaStream_t)side_stream;
  if (p->dev) {
    Carve c = carve(p->pool_tokens, p->row_elems, p->elem_bytes);
    for (int l = 0; l < p->n_layers; ++l) {        // the same carving repeated per layer
      char* base = p->dev + (int64_t)l * c.total;
      PoolLayer& L = p->layers[l];
      L.pool_K = base + c.off_K;
      L.pool_V = base + c.off_V;
      L.grad_K = (float*)(base + c.off_gK);
      L.grad_V = (float*)(base + c.off_gV);
      L.state = (float*)(base + c.off_state);
    }
    cudaError_t e = cudaMemsetAsync(p->dev, 0, (size_t)c.total * p->n_layers, p->side);
    if (e == cudaSuccess) e = cudaStreamSynchronize(p->side);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&p->ev_side, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&p->ev_main, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&p->ev_side_in, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&p->ev_out_last, cudaEventDisableTiming);
    if (e == cudaSuccess) {   // highest priority: its small refresh kernels must not queue behind the attention CTAs
      int lo = 0, hi = 0;
      cudaDeviceGetStreamPriorityRange(&lo, &hi);
      e = cudaStreamCreateWithPriority(&p->side_in, cudaStreamNonBlocking, hi);
    }
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&p->st_h2d, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&p->st_upload, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&p->st_d2h, cudaStreamNonBlocking);
    for (int i = 0; i < 11 && e == cudaSuccess; ++i) e = cudaEventCreateWithFlags(&p->ev_step[i], cudaEventDisableTiming);
    if (e == cudaSuccess) {
      int dev = 0;
      cudaGetDevice(&dev);
      cudaDeviceGetAttribute(&p->n_sm, cudaDevAttrMultiProcessorCount, dev);
    }
    p->ev_cart.assign(desc->n_carts, nullptr);   // created at a cartridge's first eviction
    p->ev_slot.assign(desc->n_slots, nullptr);
    for (int s2 = 0; s2 < desc->n_slots && e == cudaSuccess; ++s2)
      e = cudaEventCreateWithFlags(&p->ev_slot[s2], cudaEventDisableTiming);
    if (e != cudaSuccess) { delete p; return cuda_fail(e, "pool_create"); }
    if (desc->dtype == CAS_BF16 && desc->D == 128) {
      rc = tc_make_pool_maps(p);
      if (rc) { delete p; return rc; }
    }
  }
  *out = p;
  return CAS_OK;
}

int cas_pool_destroy(cas_pool* p) {
  if (!p) return CAS_OK;
  if (p->dev) {
    cudaDeviceSynchronize();
    if (p->ev_side) cudaEventDestroy(p->ev_side);
    if (p->ev_main) cudaEventDestroy(p->ev_main);
    if (p->ev_side_in) cudaEventDestroy(p->ev_side_in);
    if (p->ev_out_last) cudaEventDestroy(p->ev_out_last);
    if (p->side_in) cudaStreamDestroy(p->side_in);
    if (p->st_h2d) cudaStreamDestroy(p->st_h2d);
    if (p->st_upload) cudaStreamDestroy(p->st_upload);
    for (TabBlob& b : p->tab_free) {
      if (b.d) cudaFree(b.d);
      if (b.h) cudaFreeHost(b.h);
      if (b.done) cudaEventDestroy(b.done);
      if (b.ready) cudaEventDestroy(b.ready);
    }
    p->tab_free.clear();
    if (p->st_d2h) cudaStreamDestroy(p->st_d2h);
    if (p->fwd_part) cudaFree(p->fwd_part);
    for (cudaEvent_t ev : p->ev_step) if (ev) cudaEventDestroy(ev);
    for (cudaEvent_t ev : p->ev_slot) if (ev) cudaEventDestroy(ev);
    for (cudaEvent_t ev : p->ev_cart) if (ev) cudaEventDestroy(ev);
  }
  delete p;
  return CAS_OK;
}

int cas_pool_layout_get(const cas_pool* p, cas_pool_layout* out) {
  if (!p || !out) { set_error("null arg"); return CAS_ERR_INVALID_ARG; }
  const PoolLayer L0 = p->layers.empty() ? PoolLayer() : p->layers[0];
  out->pool_K = L0.pool_K;
  out->pool_V = L0.pool_V;
  out->grad_K = L0.grad_K;
  out->grad_V = L0.grad_V;
  out->state = L0.state;
  out->slot_base = p->slot_base.data();
  out->slot_cap = p->slot_cap.data();
  out->pool_tokens = p->pool_tokens;
  return CAS_OK;
}

static int need_data(const cas_pool* p) {
  if (!p) { set_error("null pool"); return CAS_ERR_INVALID_ARG; }
  if (!p->dev) { set_error("bookkeeping-only pool has no data"); return CAS_ERR_INVALID_ARG; }
  return CAS_OK;
}

int cas_pool_load_layer(cas_pool* p, int32_t layer, int32_t cart, const float* K, const float* V) {
  int rc = need_data(p);
  if (rc) return rc;
  if (layer < 0 || layer >= p->n_layers) { set_error("layer %d out of range", layer); return CAS_ERR_INVALID_ARG; }
  if (cart < 0 || cart >= p->desc.n_carts || !K || !V) { set_error("bad cart / null data"); return CAS_ERR_INVALID_ARG; }
  if (p->in_transit[cart]) { set_error("cartridge %d in transit", cart); return CAS_ERR_BUSY; }
  const int64_t n = (int64_t)p->cart_len[cart] * p->row_elems;
  const int s = p->slot_of[cart];
  const PoolLayer& L = p->layers[layer];
  if (s >= 0) {
    CAS_CUDA(cudaStreamSynchronize(p->side));
    CAS_CUDA(cudaMemcpy(p->slot_state(layer, s, 0), K, n * 4, cudaMemcpyHostToDevice));
    CAS_CUDA(cudaMemcpy(p->slot_state(layer, s, 1), V, n * 4, cudaMemcpyHostToDevice));
    for (int w = 2; w < 6; ++w) CAS_CUDA(cudaMemsetAsync(p->slot_state(layer, s, w), 0, n * 4, p->side));
    const int64_t o = (int64_t)p->slot_base[s] * p->row_elems;
    rc = launch_refresh(p->slot_state(layer, s, 0), p->slot_state(layer, s, 1), (char*)L.pool_K + o * p->elem_bytes,
                        (char*)L.pool_V + o * p->elem_bytes, L.grad_K + o, L.grad_V + o, n, p->desc.dtype, p->side);
    if (rc) return rc;
    CAS_CUDA(cudaStreamSynchronize(p->side));
    p->grad_dirty[(size_t)layer * p->desc.n_slots + s] = 0;
  } else {
    if (!p->pinned) { set_error("no pinned arena"); return CAS_ERR_INVALID_ARG; }
    CAS_CUDA(cudaStreamSynchronize(p->side));
    memcpy(p->home(cart, layer, 0), K, n * 4);
    memcpy(p->home(cart, layer, 1), V, n * 4);
    memset(p->home(cart, layer, 2), 0, 4 * n * 4);
  }
  return CAS_OK;
}

int cas_pool_load(cas_pool* p, int32_t cart, const float* K, const float* V) { return cas_pool_load_layer(p, 0, cart, K, V); }

int cas_pool_read_layer(cas_pool* p, int32_t layer, int32_t cart, int32_t what, void* out) {
  int rc = need_data(p);
  if (rc) return rc;
  if (layer < 0 || layer >= p->n_layers) { set_error("layer %d out of range", layer); return CAS_ERR_INVALID_ARG; }
  if (cart < 0 || cart >= p->desc.n_carts || what < 0 || what > 9 || !out) { set_error("bad args"); return CAS_ERR_INVALID_ARG; }
  const int64_t n = (int64_t)p->cart_len[cart] * p->row_elems;
  const int s = p->slot_of[cart];
  const PoolLayer& L = p->layers[layer];
  CAS_CUDA(cudaDeviceSynchronize());
  if (what < 6) {
    // in transit (either way) the pinned home is the valid copy after the device-wide synchronisation above: an
    // evictee's copy has landed, and in a paged pool its slot handle may already describe the arrival's extent
    if (s >= 0 && !p->in_transit[cart]) {
      CAS_CUDA(cudaMemcpy(out, p->slot_state(layer, s, what), n * 4, cudaMemcpyDeviceToHost));
    } else {
      if (!p->pinned) { set_error("no pinned arena"); return CAS_ERR_INVALID_ARG; }
      memcpy(out, p->home(cart, layer, what), n * 4);
    }
    return CAS_OK;
  }
  if (s < 0) { set_error("cartridge %d not resident", cart); return CAS_ERR_NOT_RESIDENT; }
  const int64_t o = (int64_t)p->slot_base[s] * p->row_elems;
  if ((what == 6 || what == 7) && !p->grad_dirty[(size_t)layer * p->desc.n_slots + s]) {
    memset(out, 0, (size_t)n * 4);   // a clean slot's buffer is undefined: its gradient is zero
    return CAS_OK;
  }
  if (what == 6) CAS_CUDA(cudaMemcpy(out, L.grad_K + o, n * 4, cudaMemcpyDeviceToHost));
  if (what == 7) CAS_CUDA(cudaMemcpy(out, L.grad_V + o, n * 4, cudaMemcpyDeviceToHost));
  if (what == 8) CAS_CUDA(cudaMemcpy(out, (char*)L.pool_K + o * p->elem_bytes, n * p->elem_bytes, cudaMemcpyDeviceToHost));
  if (what == 9) CAS_CUDA(cudaMemcpy(out, (char*)L.pool_V + o * p->elem_bytes, n * p->elem_bytes, cudaMemcpyDeviceToHost));
  return CAS_OK;
}

int cas_pool_read(cas_pool* p, int32_t cart, int32_t what, void* out) { return cas_pool_read_layer(p, 0, cart, what, out); }

int cas_pool_counters(const cas_pool* p, int32_t* slot_of, int32_t* cart_in, int64_t* opt_steps,
                      int64_t* last_used, int32_t* in_transit, int32_t* grad_dirty) {
  if (!p) { set_error("null pool"); return CAS_ERR_INVALID_ARG; }
  const int N = p->desc.n_carts, S = p->desc.n_slots;
  if (slot_of) memcpy(slot_of, p->slot_of.data(), N * 4);
  if (cart_in) memcpy(cart_in, p->cart_in.data(), S * 4);
  if (opt_steps) memcpy(opt_steps, p->opt_steps.data(), N * 8);
  if (last_used) memcpy(last_used, p->last_used.data(), N * 8);
  if (in_transit) memcpy(in_transit, p->in_transit.data(), N * 4);
  if (grad_dirty) for (int s2 = 0; s2 < S; ++s2) grad_dirty[s2] = p->any_dirty(s2) ? 1 : 0;   // any layer
  return CAS_OK;
}

int cas_pool_set_counters(cas_pool* p, int32_t cart, int64_t opt_steps, int64_t last_used) {
  if (!p || cart < 0 || cart >= p->desc.n_carts || opt_steps < 0) { set_error("bad args"); return CAS_ERR_INVALID_ARG; }
  p->opt_steps[cart] = opt_steps;
  p->last_used[cart] = last_used;
  return CAS_OK;
}

// ---------------------------------------------------------------------------------------------
// slot table (K1)
// ---------------------------------------------------------------------------------------------
int cas_slot_table_build(cas_pool* p, int32_t B, const int32_t* seq_off, const int32_t* sel_off,
                         const int32_t* sel_cart, int64_t step, cas_slot_table** out) {
  if (!p || !out || !seq_off || !sel_off || B < 1) { set_error("null / empty args"); return CAS_ERR_INVALID_ARG; }
  if (seq_off[0] != 0 || sel_off[0] != 0) { set_error("offsets must start at 0"); return CAS_ERR_INVALID_ARG; }
  for (int b = 0; b < B; ++b) {
    if (seq_off[b + 1] <= seq_off[b]) { set_error("sequence %d has no query tokens", b); return CAS_ERR_SHAPE; }
    if (sel_off[b + 1] < sel_off[b]) { set_error("sel_off not monotone"); return CAS_ERR_INVALID_ARG; }
  }
  const int nsel = sel_off[B];
  if (nsel > 0 && !sel_cart) { set_error("null sel_cart"); return CAS_ERR_INVALID_ARG; }
  const int N = p->desc.n_carts, S = p->desc.n_slots;
  cas_slot_table* t = new cas_slot_table();
  t->pool = p;
  t->B = B;
  t->T = seq_off[B];
  t->nsel = nsel;
  t->seq_off.assign(seq_off, seq_off + B + 1);
  t->sel_off.assign(sel_off, sel_off + B + 1);
  t->sel_cart.assign(sel_cart, sel_cart + nsel);
  t->sel_slot.resize(nsel);
  t->sel_base.resize(nsel);
  t->sel_len.resize(nsel);
  t->P.assign(B, 0);
  std::vector<int32_t> mark(N, -1);
  for (int b = 0; b < B; ++b) {
    for (int k = sel_off[b]; k < sel_off[b + 1]; ++k) {
      const int c = sel_cart[k];
      int rc = CAS_OK;
      if (c < 0 || c >= N) { set_error("cartridge id %d out of range", c); rc = CAS_ERR_INVALID_ARG; }
      else if (mark[c] == b) { set_error("duplicate cartridge %d in sequence %d", c, b); rc = CAS_ERR_INVALID_ARG; }
      else if (p->slot_of[c] < 0) { set_error("cartridge %d not resident", c); rc = CAS_ERR_NOT_RESIDENT; }
      else if (p->in_transit[c]) { set_error("cartridge %d in transit", c); rc = CAS_ERR_BUSY; }
      if (rc) { delete t; return rc; }
      mark[c] = b;
      t->sel_slot[k] = p->slot_of[c];
      t->sel_base[k] = p->slot_base[p->slot_of[c]];
      t->sel_len[k] = p->cart_len[c];
      t->P[b] += p->cart_len[c];
    }
  }
  for (int k = 0; k < nsel; ++k) p->last_used[sel_cart[k]] = step;
  // inverted CSR sorted by (slot, sequence): counting sort keeps sequences ascending per slot
  t->inv_off.assign(S + 1, 0);
  for (int k = 0; k < nsel; ++k) t->inv_off[t->sel_slot[k] + 1]++;
  for (int s = 0; s < S; ++s) t->inv_off[s + 1] += t->inv_off[s];
  t->inv_seq.resize(nsel);
  {
    std::vector<int32_t> cur(t->inv_off.begin(), t->inv_off.end() - 1);
    for (int b = 0; b < B; ++b)
      for (int k = sel_off[b]; k < sel_off[b + 1]; ++k) t->inv_seq[cur[t->sel_slot[k]]++] = b;
  }
  for (int s = 0; s < S; ++s)
    if (t->inv_off[s + 1] > t->inv_off[s]) {
      t->used_slots.push_back(s);
      t->unique_prefix_tokens += p->cart_len[p->cart_in[s]];
    }
  // KV tile lists + work lists
  const int tile = 128;
  const bool pack = p->pack;   // 16-token pages: the remainders of a sequence's cartridges share packed KV tiles
  t->kv_tile_off.assign(B + 1, 0);
  t->qtile_off.assign(B + 1, 0);
  t->ptile_off.assign(B + 1, 0);
  for (int b = 0; b < B; ++b) {
    std::vector<std::pair<int32_t, int32_t>> pages;   // (first token, valid keys) of the remainder pages
    for (int k = sel_off[b]; k < sel_off[b + 1]; ++k) {
      const int len = t->sel_len[k], whole = pack ? len / tile * tile : len;
      for (int j = 0; j < whole; j += tile)
        t->kv_tiles.push_back({t->sel_base[k] + j, std::min(tile, len - j)});
      for (int j = whole; j < len; j += 16) pages.push_back({t->sel_base[k] + j, std::min(16, len - j)});
    }
    for (size_t i = 0; i < pages.size(); i += 8) {
      PackedTile pt{};
      int nvalid = 0;
      for (int u = 0; u < 8; ++u) {
        const bool have = i + u < pages.size();
        pt.tok[u] = have ? pages[i + u].first : pages[i].first;
        const int cnt = have ? pages[i + u].second : 0;
        for (int x = 0; x < cnt; ++x) pt.mask[(16 * u + x) >> 5] |= 1u << ((16 * u + x) & 31);
        nvalid += cnt;
      }
      t->kv_tiles.push_back({-1 - (int32_t)t->ptiles.size(), nvalid});
      t->ptiles.push_back(pt);
    }
    t->ptile_off[b + 1] = (int32_t)t->ptiles.size();
    t->kv_tile_off[b + 1] = (int32_t)t->kv_tiles.size();
    const int64_t lq = seq_off[b + 1] - seq_off[b];
    t->qtile_off[b + 1] = t->qtile_off[b] + (int32_t)((lq + 127) / 128);
    t->max_lq = std::max<int32_t>(t->max_lq, (int32_t)lq);
    t->pairs += lq * t->P[b] + lq * (lq + 1) / 2;
    t->prefix_tokens += t->P[b];
    const int npre = t->kv_tile_off[b + 1] - t->kv_tile_off[b];
    for (int r = 0; r < lq; r += 256) {
      const int rows = (int)std::min<int64_t>(256, lq - r);
      const int nq = (rows + 127) / 128;
      t->fwd_items.push_back({b, r, rows, nq * npre + (r / 128) * nq + (nq == 2 ? 3 : 1)});
    }
    for (int r = 0; r < lq; r += 32) t->simt_items.push_back({b, r, (int)std::min<int64_t>(32, lq - r), 0});
  }
  std::stable_sort(t->fwd_items.begin(), t->fwd_items.end(), [](const FwdItem& a, const FwdItem& b) { return a.cost > b.cost; });
  for (int s : t->used_slots) {
    int cost = 0;
    for (int e = t->inv_off[s]; e < t->inv_off[s + 1]; ++e) {
      const int b = t->inv_seq[e];
      cost += (seq_off[b + 1] - seq_off[b] + 127) / 128;
    }
    const int len = p->cart_len[p->cart_in[s]], whole = pack ? len / tile * tile : len;
    for (int j = 0; j < whole; j += tile)
      t->bwd_items.push_back({0, s, p->slot_base[s] + j, std::min(tile, len - j), j / tile, cost});
    for (int j = 0; j < len; j += tile)      // the CUDA-core kernels never pack: every tile of the slot, ragged end included
      t->simt_bwd_items.push_back({0, s, p->slot_base[s] + j, std::min(tile, len - j), j / tile, cost});
  }
  // packed tiles belong to ONE sequence: their CTA walks that sequence only and ADDS its rows to the gradient slots
  for (int b = 0; b < B; ++b)
    for (int i = t->ptile_off[b]; i < t->ptile_off[b + 1]; ++i) {
      int nvalid = 0;
      for (uint32_t w : t->ptiles[i].mask) nvalid += __builtin_popcount(w);
      t->bwd_items.push_back({2, b, i, nvalid, 0, (seq_off[b + 1] - seq_off[b] + 127) / 128});
    }
  for (int b = 0; b < B; ++b) {
    const int lq = seq_off[b + 1] - seq_off[b];
    const int nt = (lq + tile - 1) / tile;
    for (int j = 0; j < nt; ++j) {
      t->bwd_items.push_back({1, b, seq_off[b] + j * tile, std::min(tile, lq - j * tile), j, nt - j});
      t->simt_bwd_items.push_back(t->bwd_items.back());
    }
  }
  std::stable_sort(t->bwd_items.begin(), t->bwd_items.end(),
                   [](const BwdItem& a, const BwdItem& b) { return a.cost > b.cost; });
  if (p->dev) {
    size_t off = 0;
    const size_t o_seq = blob_add(off, t->seq_off), o_sel = blob_add(off, t->sel_off),
                 o_base = blob_add(off, t->sel_base, 1), o_len = blob_add(off, t->sel_len, 1),
                 o_slot = blob_add(off, t->sel_slot, 1), o_ioff = blob_add(off, t->inv_off),
                 o_iseq = blob_add(off, t->inv_seq, 1), o_kto = blob_add(off, t->kv_tile_off),
                 o_kt = blob_add(off, t->kv_tiles, 1), o_fw = blob_add(off, t->fwd_items),
                 o_si = blob_add(off, t->simt_items), o_bw = blob_add(off, t->bwd_items),
                 o_us = blob_add(off, t->used_slots, 1), o_qt = blob_add(off, t->qtile_off),
                 o_pt = blob_add(off, t->ptiles, 1), o_sb = blob_add(off, t->simt_bwd_items);
    const size_t o_cnt = off;
    off += 256;
    // a recycled blob whose last reader has finished, else a new one (device memory + pinned mirror)
    TabBlob blob;
    for (size_t i = 0; i < p->tab_free.size(); ++i) {
      TabBlob& b = p->tab_free[i];
      if (b.cap >= off && (!b.has_done || cudaEventQuery(b.done) == cudaSuccess)) {
        blob = b;
        p->tab_free.erase(p->tab_free.begin() + i);
        break;
      }
    }
    (void)cudaGetLastError();   // cudaEventQuery reports "not ready" as an error code
    if (!blob.d && p->tab_free.size() >= 3) {
      // the host runs several steps ahead of the GPU: wait for the oldest blob instead of growing the ring
      for (size_t i = 0; i < p->tab_free.size(); ++i)
        if (p->tab_free[i].cap >= off) {
          blob = p->tab_free[i];
          p->tab_free.erase(p->tab_free.begin() + i);
          if (blob.has_done) cudaEventSynchronize(blob.done);
          break;
        }
    }
    if (!blob.d) {
      blob.cap = std::max<size_t>(off + off / 2, 1 << 20);
      cudaError_t e = cudaMalloc((void**)&blob.d, blob.cap);
      if (e == cudaSuccess) e = cudaHostAlloc((void**)&blob.h, blob.cap, cudaHostAllocDefault);
      if (e == cudaSuccess) e = cudaEventCreateWithFlags(&blob.done, cudaEventDisableTiming);
      if (e == cudaSuccess) e = cudaEventCreateWithFlags(&blob.ready, cudaEventDisableTiming);
      if (e != cudaSuccess) {
        if (blob.d) cudaFree(blob.d);
        if (blob.h) cudaFreeHost(blob.h);
        delete t;
        return cuda_fail(e, "slot table blob");
      }
    }
    blob.has_done = false;
    memset(blob.h + o_cnt, 0, 256);
    auto put = [&](size_t o, const void* src, size_t n) { if (n) memcpy(blob.h + o, src, n); };
    put(o_seq, t->seq_off.data(), t->seq_off.size() * 4);
    put(o_sel, t->sel_off.data(), t->sel_off.size() * 4);
    put(o_base, t->sel_base.data(), t->sel_base.size() * 4);
    put(o_len, t->sel_len.data(), t->sel_len.size() * 4);
    put(o_slot, t->sel_slot.data(), t->sel_slot.size() * 4);
    put(o_ioff, t->inv_off.data(), t->inv_off.size() * 4);
    put(o_iseq, t->inv_seq.data(), t->inv_seq.size() * 4);
    put(o_kto, t->kv_tile_off.data(), t->kv_tile_off.size() * 4);
    put(o_kt, t->kv_tiles.data(), t->kv_tiles.size() * sizeof(KvTile));
    put(o_fw, t->fwd_items.data(), t->fwd_items.size() * sizeof(FwdItem));
    put(o_si, t->simt_items.data(), t->simt_items.size() * sizeof(FwdItem));
    put(o_bw, t->bwd_items.data(), t->bwd_items.size() * sizeof(BwdItem));
    put(o_us, t->used_slots.data(), t->used_slots.size() * 4);
    put(o_qt, t->qtile_off.data(), t->qtile_off.size() * 4);
    put(o_pt, t->ptiles.data(), t->ptiles.size() * sizeof(PackedTile));
    put(o_sb, t->simt_bwd_items.data(), t->simt_bwd_items.size() * sizeof(BwdItem));
    cudaError_t e = cudaMemcpyAsync(blob.d, blob.h, off, cudaMemcpyHostToDevice, p->st_upload);
    if (e == cudaSuccess) e = cudaEventRecord(blob.ready, p->st_upload);
    if (e != cudaSuccess) { p->tab_free.push_back(blob); delete t; return cuda_fail(e, "slot table upload"); }
    t->blob = blob;
    t->d_blob = blob.d;
    char* d = t->d_blob;
    t->d_seq_off = (int32_t*)(d + o_seq);
    t->d_sel_off = (int32_t*)(d + o_sel);
    t->d_sel_base = (int32_t*)(d + o_base);
    t->d_sel_len = (int32_t*)(d + o_len);
    t->d_sel_slot = (int32_t*)(d + o_slot);
    t->d_inv_off = (int32_t*)(d + o_ioff);
    t->d_inv_seq = (int32_t*)(d + o_iseq);
    t->d_kv_tile_off = (int32_t*)(d + o_kto);
    t->d_kv_tiles = (KvTile*)(d + o_kt);
    t->d_fwd_items = (FwdItem*)(d + o_fw);
    t->d_simt_items = (FwdItem*)(d + o_si);
    t->d_bwd_items = (BwdItem*)(d + o_bw);
    t->d_used_slots = (int32_t*)(d + o_us);
    t->d_qtile_off = (int32_t*)(d + o_qt);
    t->d_ptiles = (PackedTile*)(d + o_pt);
    t->d_simt_bwd_items = (BwdItem*)(d + o_sb);
    t->d_counters = (int32_t*)(d + o_cnt);
  }
  *out = t;
  return CAS_OK;
}

int cas_slot_table_destroy(cas_slot_table* t) {
  if (!t) return CAS_OK;
  if (t->d_blob) {   // back to the pool; reusable once the last kernel that read it is done
    if (t->used && cudaEventRecord(t->blob.done, t->last_stream) == cudaSuccess) t->blob.has_done = true;
    else if (t->used) cudaDeviceSynchronize();
    t->pool->tab_free.push_back(t->blob);
  }
  if (t->d_dec_blob) {
    cudaDeviceSynchronize();
    cudaFree(t->d_dec_blob);
    cudaFreeHost(t->h_dec_blob);
  }
  if (t->dec_ready) cudaEventDestroy(t->dec_ready);
  delete t;
  return CAS_OK;
}

int cas_slot_table_info(const cas_slot_table* t, cas_table_info* o) {
  if (!t || !o) { set_error("null arg"); return CAS_ERR_INVALID_ARG; }
  o->B = t->B; o->T = t->T; o->nsel = t->nsel; o->n_kv_tiles = (int32_t)t->kv_tiles.size();
  o->pairs_per_head = t->pairs; o->prefix_tokens = t->prefix_tokens;
  o->unique_prefix_tokens = t->unique_prefix_tokens;
  return CAS_OK;
}

int cas_slot_table_export(const cas_slot_table* t, int32_t* sel_slot, int32_t* inv_off, int32_t* inv_seq,
                          int64_t* P) {
  if (!t) { set_error("null table"); return CAS_ERR_INVALID_ARG; }
  if (sel_slot && t->nsel) memcpy(sel_slot, t->sel_slot.data(), t->nsel * 4);
  if (inv_off) memcpy(inv_off, t->inv_off.data(), t->inv_off.size() * 4);
  if (inv_seq && t->nsel) memcpy(inv_seq, t->inv_seq.data(), t->nsel * 4);
  if (P) memcpy(P, t->P.data(), t->B * 8);
  return CAS_OK;
}

int cas_slot_table_fwd_split(const cas_slot_table* t, int32_t* n_tail, int32_t* n_parts) {
  if (!t || !n_tail || !n_parts) { set_error("null arg"); return CAS_ERR_INVALID_ARG; }
  *n_tail = t->fwd_plan_key < 0 ? 0 : t->fwd_n_tail;
  *n_parts = t->fwd_plan_key < 0 ? 1 : t->fwd_n_parts;
  return CAS_OK;
}

int cas_position_offsets(const cas_pool* p, const cas_slot_table* t, int64_t* total_resident, int64_t* P) {
  if (!p) { set_error("null pool"); return CAS_ERR_INVALID_ARG; }
  if (total_resident) {
    int64_t tot = 0;
    for (int c = 0; c < p->desc.n_carts; ++c) if (p->slot_of[c] >= 0) tot += p->cart_len[c];
    *total_resident = tot;
  }
  if (P) {
    if (!t) { set_error("null table"); return CAS_ERR_INVALID_ARG; }
    memcpy(P, t->P.data(), t->B * 8);
  }
  return CAS_OK;
}

// ---------------------------------------------------------------------------------------------
// attention dispatch
// ---------------------------------------------------------------------------------------------
static int check_attn(const cas_pool* p, const cas_slot_table* t, int Hq, const void* Ks, const void* Vs, float scale) {
  int rc = need_data(p);
  if (rc) return rc;
  // the kernels take the row maximum on the raw scores and multiply by scale afterwards: correct for scale > 0 only
  if (!(scale > 0.f) || !std::isfinite(scale)) { set_error("scale must be positive and finite"); return CAS_ERR_INVALID_ARG; }
  if (!t || t->pool != p) { set_error("table does not belong to this pool"); return CAS_ERR_INVALID_ARG; }
  if (Hq < 1 || Hq % p->desc.Hkv) { set_error("Hq must be a positive multiple of Hkv"); return CAS_ERR_SHAPE; }
  if ((Ks == nullptr) != (Vs == nullptr)) { set_error("K_self and V_self must both be given or both NULL"); return CAS_ERR_INVALID_ARG; }
  if (!Ks)
    for (int b = 0; b < t->B; ++b)
      if (t->sel_off[b + 1] == t->sel_off[b]) { set_error("sequence %d sees no key at all", b); return CAS_ERR_SHAPE; }
  for (int k = 0; k < t->nsel; ++k) {   // the table is a snapshot: its slots must still hold those cartridges
    const int c = t->sel_cart[k];
    if (p->slot_of[c] != t->sel_slot[k] || p->in_transit[c]) { set_error("stale slot table (cartridge %d moved)", c); return CAS_ERR_NOT_RESIDENT; }
  }
  return CAS_OK;
}

// The table's device blob is uploaded asynchronously: every stream that reads it first waits for the
// upload, and the table remembers the stream so that the blob is recycled only after its last reader.
static int table_on_stream(const cas_slot_table* t, void* stream) {
  if (!t->d_blob) return CAS_OK;
  CAS_CUDA(cudaStreamWaitEvent((cudaStream_t)stream, t->blob.ready, 0));
  if (t->used && t->last_stream != (cudaStream_t)stream) {   // keep one "last reader": chain the streams
    CAS_CUDA(cudaEventRecord(t->blob.done, t->last_stream));
    CAS_CUDA(cudaStreamWaitEvent((cudaStream_t)stream, t->blob.done, 0));
  }
  t->last_stream = (cudaStream_t)stream;
  t->used = true;
  return CAS_OK;
}

static bool use_tc(const cas_pool* p, const cas_slot_table* t, int Hq, int* rc) {
  *rc = CAS_OK;
  if (g_impl == CAS_IMPL_SIMT) return false;
  const bool ok = tc_supported(p, t, Hq);
  if (g_impl == CAS_IMPL_TC && !ok) { set_error("tensor-core path needs bf16, D=128"); *rc = CAS_ERR_SHAPE; }
  return ok;
}

static int check_rope(const cas_pool* p, const cas_slot_table* t, int Hq, const cas_rope* rope) {
  if (!rope->cs) { set_error("rope: null cos/sin table"); return CAS_ERR_INVALID_ARG; }
  if (rope->layout != 0 && rope->layout != 1) { set_error("rope: layout must be 0 or 1"); return CAS_ERR_INVALID_ARG; }
  int rc = CAS_OK;
  if (!use_tc(p, t, Hq, &rc) || rc || tc_decode_supported(p, t, Hq)) {
    if (rc) return rc;
    set_error("fused RoPE runs on the tensor-core training kernels (bf16, D = 128, not decode-shaped): use cas_rope_apply");
    return CAS_ERR_SHAPE;
  }
  return CAS_OK;
}

static int attn_fwd_impl(cas_pool* p, const cas_slot_table* t, int32_t layer, int32_t Hq, const void* Q,
                         const void* Ks, const void* Vs, float scale, void* O, float* LSE, void* stream,
                         const cas_rope* rope, void* Q_rot, void* Ks_rot) {
  int rc = check_attn(p, t, Hq, Ks, Vs, scale);
  if (rc) return rc;
  if (layer < 0 || layer >= p->n_layers) { set_error("layer %d out of range", layer); return CAS_ERR_INVALID_ARG; }
  rc = table_on_stream(t, stream);
  if (rc) return rc;
  if (!Q || !O || !LSE) { set_error("null Q/O/LSE"); return CAS_ERR_INVALID_ARG; }
  AttnArgs a{};
  a.pool = p; a.tab = t; a.Hq = Hq; a.Hkv = p->desc.Hkv; a.D = p->desc.D; a.dtype = p->desc.dtype;
  a.Q = Q; a.Ks = Ks; a.Vs = Vs; a.O_out = O; a.LSE_out = LSE; a.scale = scale;
  a.stream = (cudaStream_t)stream;
  a.layer = layer; a.L = &p->layers[layer];
  if (rope) {
    rc = check_rope(p, t, Hq, rope);
    if (rc) return rc;
    if (!Q_rot || (Ks && !Ks_rot)) { set_error("rope: Q_rot / K_self_rot outputs missing"); return CAS_ERR_INVALID_ARG; }
    if (Ks) {   // K_self (1/G of the query bytes) is rotated by its own small pass; Q inside the forward kernel
      rc = rope_table_rotate(Ks, Ks_rot, rope->cs, t->T, p->desc.Hkv, rope->layout, 0, (cudaStream_t)stream);
      if (rc) return rc;
      a.Ks = Ks_rot;
    }
    a.rope_cs = rope->cs; a.rope_layout = rope->layout; a.Q_rot = Q_rot;
    return tc_attn_fwd(a);
  }
  const bool tc = use_tc(p, t, Hq, &rc);
  if (rc) return rc;
  if (tc && tc_decode_supported(p, t, Hq)) {
    // one query token per sequence whose only self key is itself: the decode kernel with a 1-token "cache"
    const std::vector<int32_t> ones(t->B, 1);
    return tc_decode_fwd(a, Ks, Vs, 1, ones.data());
  }
  return tc ? tc_attn_fwd(a) : simt_attn_fwd(a);
}

int cas_prefix_attn_fwd_layer(cas_pool* p, const cas_slot_table* t, int32_t layer, int32_t Hq, const void* Q,
                              const void* Ks, const void* Vs, float scale, void* O, float* LSE, void* stream) {
  return attn_fwd_impl(p, t, layer, Hq, Q, Ks, Vs, scale, O, LSE, stream, nullptr, nullptr, nullptr);
}

int cas_prefix_attn_fwd_noalloc(cas_pool* p, const cas_slot_table* t, int32_t layer, int32_t Hq, const void* Q,
                                const void* Ks, const void* Vs, float scale, void* O, float* LSE, void* stream) {
  int rc = check_attn(p, t, Hq, Ks, Vs, scale);
  if (rc) return rc;
  if (layer < 0 || layer >= p->n_layers) { set_error("layer %d out of range", layer); return CAS_ERR_INVALID_ARG; }
  if (!Q || !O || !LSE) { set_error("null Q/O/LSE"); return CAS_ERR_INVALID_ARG; }
  // only the tensor-core training kernel: the decode kernel allocates its work list and scratch at a table's first
  // call, and the CUDA-core path has no scratch to place
  if (!use_tc(p, t, Hq, &rc) || rc || tc_decode_supported(p, t, Hq)) {
    if (rc) return rc;
    set_error("cas_prefix_attn_fwd_noalloc runs the tensor-core forward kernel (bf16, D = 128, not decode-shaped)");
    return CAS_ERR_SHAPE;
  }
  rc = table_on_stream(t, stream);
  if (rc) return rc;
  AttnArgs a{};
  a.pool = p; a.tab = t; a.Hq = Hq; a.Hkv = p->desc.Hkv; a.D = p->desc.D; a.dtype = p->desc.dtype;
  a.Q = Q; a.Ks = Ks; a.Vs = Vs; a.O_out = O; a.LSE_out = LSE; a.scale = scale;
  a.stream = (cudaStream_t)stream;
  a.layer = layer; a.L = &p->layers[layer];
  a.static_scratch = true;
  return tc_attn_fwd(a);
}

int cas_prefix_attn_fwd_rope(cas_pool* p, const cas_slot_table* t, int32_t layer, int32_t Hq, const void* Q,
                             const void* Ks, const void* Vs, const cas_rope* rope, void* Q_rot, void* Ks_rot,
                             float scale, void* O, float* LSE, void* stream) {
  if (!rope) { set_error("null rope"); return CAS_ERR_INVALID_ARG; }
  return attn_fwd_impl(p, t, layer, Hq, Q, Ks, Vs, scale, O, LSE, stream, rope, Q_rot, Ks_rot);
}

int cas_prefix_attn_fwd(cas_pool* p, const cas_slot_table* t, int32_t Hq, const void* Q, const void* Ks,
                        const void* Vs, float scale, void* O, float* LSE, void* stream) {
  return cas_prefix_attn_fwd_layer(p, t, 0, Hq, Q, Ks, Vs, scale, O, LSE, stream);
}

int cas_decode_attn_layer(cas_pool* p, const cas_slot_table* t, int32_t layer, int32_t Hq, const void* Q,
                          const void* K_cache, const void* V_cache, int32_t cache_cap, const int32_t* self_len,
                          float scale, void* O, float* LSE, void* stream) {
  int rc = need_data(p);
  if (rc) return rc;
  if (layer < 0 || layer >= p->n_layers) { set_error("layer %d out of range", layer); return CAS_ERR_INVALID_ARG; }
  if (!t || t->pool != p) { set_error("table does not belong to this pool"); return CAS_ERR_INVALID_ARG; }
  if (Hq < 1 || Hq % p->desc.Hkv) { set_error("Hq must be a positive multiple of Hkv"); return CAS_ERR_SHAPE; }
  if (!(scale > 0.f) || !std::isfinite(scale)) { set_error("scale must be positive and finite"); return CAS_ERR_INVALID_ARG; }
  if (!Q || !O || !LSE) { set_error("null Q/O/LSE"); return CAS_ERR_INVALID_ARG; }
  if ((K_cache == nullptr) != (V_cache == nullptr)) { set_error("K_cache and V_cache: both or none"); return CAS_ERR_INVALID_ARG; }
  if (K_cache && (!self_len || cache_cap < 1)) { set_error("a self cache needs self_len and cache_cap >= 1"); return CAS_ERR_INVALID_ARG; }
  if (t->max_lq != 1) { set_error("cas_decode_attn needs one query token per sequence"); return CAS_ERR_SHAPE; }
  for (int k = 0; k < t->nsel; ++k) {
    const int c = t->sel_cart[k];
    if (p->slot_of[c] != t->sel_slot[k] || p->in_transit[c]) { set_error("stale slot table (cartridge %d moved)", c); return CAS_ERR_NOT_RESIDENT; }
  }
  if (!tc_decode_supported(p, t, Hq)) { set_error("cas_decode_attn needs a bf16 pool with D = 128"); return CAS_ERR_SHAPE; }
  rc = table_on_stream(t, stream);
  if (rc) return rc;
  AttnArgs a{};
  a.pool = p; a.tab = t; a.Hq = Hq; a.Hkv = p->desc.Hkv; a.D = p->desc.D; a.dtype = p->desc.dtype;
  a.Q = Q; a.O_out = O; a.LSE_out = LSE; a.scale = scale;
  a.stream = (cudaStream_t)stream;
  a.layer = layer; a.L = &p->layers[layer];
  return tc_decode_fwd(a, K_cache, V_cache, cache_cap, self_len);
}

int cas_decode_attn(cas_pool* p, const cas_slot_table* t, int32_t Hq, const void* Q, const void* K_cache,
                    const void* V_cache, int32_t cache_cap, const int32_t* self_len, float scale, void* O, float* LSE,
                    void* stream) {
  return cas_decode_attn_layer(p, t, 0, Hq, Q, K_cache, V_cache, cache_cap, self_len, scale, O, LSE, stream);
}

// PAPER.md:142 (sec. 3 Retrieval): "we map each retrieved chunk to a document id, which in turn is associated with a
// cartridge.  The final list contains the unique cartridge ids in the order of their retrieval."
int cas_select_retrieved(const int32_t* chunk_ids, int32_t k, const int32_t* chunk_to_cart, int32_t n_chunks,
                         int32_t max_carts, int32_t* out_carts, int32_t* n_out) {
  if (k < 0 || (k && !chunk_ids) || !chunk_to_cart || n_chunks < 0 || !out_carts || !n_out || max_carts < 0) { set_error("bad args"); return CAS_ERR_INVALID_ARG; }
  int n = 0;
  for (int i = 0; i < k && n < max_carts; ++i) {
    if (chunk_ids[i] < 0 || chunk_ids[i] >= n_chunks) { set_error("chunk id %d out of range", chunk_ids[i]); return CAS_ERR_INVALID_ARG; }
    const int32_t c = chunk_to_cart[chunk_ids[i]];
    bool seen = false;
    for (int j = 0; j < n; ++j) seen |= out_carts[j] == c;
    if (!seen) out_carts[n++] = c;
  }
  *n_out = n;
  return CAS_OK;
}

int cas_prefix_attn_bwd_workspace_bytes(const cas_pool* p, const cas_slot_table* t, int32_t Hq, size_t* bytes) {
  if (!p || !t || !bytes || Hq < 1) { set_error("null arg"); return CAS_ERR_INVALID_ARG; }
  *bytes = std::max(simt_bwd_workspace(t, Hq), tc_bwd_workspace(t, Hq, p->desc.D));
  return CAS_OK;
}

static int attn_bwd_impl(cas_pool* p, const cas_slot_table* t, int32_t layer, int32_t Hq, const void* Q,
                         const void* Ks, const void* Vs, const void* O, const float* LSE, const void* dO,
                         float scale, void* dQ, void* dKs, void* dVs, void* workspace, size_t workspace_bytes,
                         void* stream, const cas_rope* rope) {
  int rc = check_attn(p, t, Hq, Ks, Vs, scale);
  if (rc) return rc;
  if (rope) {
    rc = check_rope(p, t, Hq, rope);
    if (rc) return rc;
  }
  if (layer < 0 || layer >= p->n_layers) { set_error("layer %d out of range", layer); return CAS_ERR_INVALID_ARG; }
  int32_t* dirty = p->grad_dirty.data() + (size_t)layer * p->desc.n_slots;
  rc = table_on_stream(t, stream);
  if (rc) return rc;
  if (!Q || !O || !LSE || !dO || !dQ) { set_error("null Q/O/LSE/dO/dQ"); return CAS_ERR_INVALID_ARG; }
  if ((dKs == nullptr) != (dVs == nullptr) || (dKs && !Ks)) { set_error("dK_self/dV_self: both or none, and only with K_self"); return CAS_ERR_INVALID_ARG; }
  size_t need = 0;
  cas_prefix_attn_bwd_workspace_bytes(p, t, Hq, &need);
  if (!workspace || workspace_bytes < need) { set_error("workspace too small: need %zu bytes", need); return CAS_ERR_CAPACITY; }
  AttnArgs a{};
  a.pool = p; a.tab = t; a.Hq = Hq; a.Hkv = p->desc.Hkv; a.D = p->desc.D; a.dtype = p->desc.dtype;
  a.Q = Q; a.Ks = Ks; a.Vs = Vs; a.O = O; a.LSE_in = LSE; a.dO = dO; a.dQ = dQ; a.dKs = dKs; a.dVs = dVs;
  a.scale = scale; a.workspace = workspace; a.workspace_bytes = workspace_bytes;
  a.stream = (cudaStream_t)stream;
  a.layer = layer; a.L = &p->layers[layer];
  const bool tc = use_tc(p, t, Hq, &rc);
  if (rc) return rc;
  if (!tc || p->pack) {
    // the CUDA-core path accumulates read-modify-write, and so do the per-sequence packed tiles of a paged pool
    // (several CTAs add to one cartridge's rows): give the clean slots about to be touched real zeros
    std::vector<ZeroDesc> zs;
    for (int sl : t->used_slots)
      if (!dirty[sl]) {
        const int64_t o = (int64_t)p->slot_base[sl] * p->row_elems;
        zs.push_back({a.L->grad_K + o, a.L->grad_V + o, (int64_t)p->slot_cap[sl] * p->row_elems});
      }
    if (!zs.empty()) {
      rc = launch_zero_slots(zs.data(), (int)zs.size(), (cudaStream_t)stream);
      if (rc) return rc;
    }
  }
  if (rope) { a.rope_cs = rope->cs; a.rope_layout = rope->layout; }      // dq_convert_kernel applies R^T to dQ
  rc = tc ? tc_attn_bwd(a) : simt_attn_bwd(a);
  if (rc) return rc;
  for (int s2 : t->used_slots) dirty[s2] = 1;
  if (rope && dKs)   // dK_self back through the rotation (in place)
    return rope_table_rotate(dKs, dKs, rope->cs, t->T, p->desc.Hkv, rope->layout, 1, (cudaStream_t)stream);
  return CAS_OK;
}

int cas_prefix_attn_bwd_layer(cas_pool* p, const cas_slot_table* t, int32_t layer, int32_t Hq, const void* Q,
                              const void* Ks, const void* Vs, const void* O, const float* LSE, const void* dO,
                              float scale, void* dQ, void* dKs, void* dVs, void* workspace, size_t workspace_bytes,
                              void* stream) {
  return attn_bwd_impl(p, t, layer, Hq, Q, Ks, Vs, O, LSE, dO, scale, dQ, dKs, dVs, workspace, workspace_bytes, stream,
                       nullptr);
}

int cas_prefix_attn_bwd_rope(cas_pool* p, const cas_slot_table* t, int32_t layer, int32_t Hq, const void* Q_rot,
                             const void* Ks_rot, const void* Vs, const void* O, const float* LSE, const void* dO,
                             const cas_rope* rope, float scale, void* dQ, void* dKs, void* dVs, void* workspace,
                             size_t workspace_bytes, void* stream) {
  if (!rope) { set_error("null rope"); return CAS_ERR_INVALID_ARG; }
  return attn_bwd_impl(p, t, layer, Hq, Q_rot, Ks_rot, Vs, O, LSE, dO, scale, dQ, dKs, dVs, workspace, workspace_bytes,
                       stream, rope);
}

int cas_prefix_attn_bwd(cas_pool* p, const cas_slot_table* t, int32_t Hq, const void* Q, const void* Ks,
                        const void* Vs, const void* O, const float* LSE, const void* dO, float scale,
                        void* dQ, void* dKs, void* dVs, void* workspace, size_t workspace_bytes, void* stream) {
  return cas_prefix_attn_bwd_layer(p, t, 0, Hq, Q, Ks, Vs, O, LSE, dO, scale, dQ, dKs, dVs, workspace, workspace_bytes,
                                   stream);
}

// ---------------------------------------------------------------------------------------------
// Adam
// ---------------------------------------------------------------------------------------------
int cas_adam_step(cas_pool* p, const cas_adam_cfg* cfg, const int32_t* slots, int32_t n,
                  const float* lr_scale, void* stream) {
  if (!p || !cfg) { set_error("null arg"); return CAS_ERR_INVALID_ARG; }
  if (cfg->n_frozen < 0 || !(cfg->beta1 >= 0 && cfg->beta1 < 1) || !(cfg->beta2 >= 0 && cfg->beta2 < 1)) {
    set_error("bad Adam config");
    return CAS_ERR_INVALID_ARG;
  }
  std::vector<int32_t> list;
  if (slots) {
    if (n < 0) { set_error("n < 0"); return CAS_ERR_INVALID_ARG; }
    list.assign(slots, slots + n);
  } else {
    for (int s = 0; s < p->desc.n_slots; ++s)
      if (p->cart_in[s] >= 0 && !p->in_transit[p->cart_in[s]]) list.push_back(s);
  }
  std::set<int32_t> seen;
  for (int s : list) {
    if (s < 0 || s >= p->desc.n_slots || !seen.insert(s).second) { set_error("bad / duplicate slot %d", s); return CAS_ERR_INVALID_ARG; }
    if (p->cart_in[s] < 0) { set_error("slot %d is empty", s); return CAS_ERR_NOT_RESIDENT; }
    if (p->in_transit[p->cart_in[s]]) { set_error("slot %d in transit", s); return CAS_ERR_BUSY; }
  }
  const int cnt = (int)list.size(), S = p->desc.n_slots;
  if (p->dev && cnt) {
    // every layer of every listed slot in one go (PAPER.md:42: a cartridge is Z in R^{L x p x d x 2}; :85 one step count
    // and one lr scale per cartridge, not per layer)
    std::vector<AdamSlotDesc> h((size_t)cnt * p->n_layers);
    for (int l = 0; l < p->n_layers; ++l) {
      const PoolLayer& L = p->layers[l];
      for (int i = 0; i < cnt; ++i) {
        const int s = list[i], c = p->cart_in[s];
        const int64_t o = (int64_t)p->slot_base[s] * p->row_elems;
        const double t = (double)(p->opt_steps[c] + 1);
        AdamSlotDesc& d = h[(size_t)l * cnt + i];
        d.state = p->slot_state(l, s, 0);
        d.wK = (char*)L.pool_K + o * p->elem_bytes;
        d.wV = (char*)L.pool_V + o * p->elem_bytes;
        d.gK = L.grad_K + o;
        d.gV = L.grad_V + o;
        d.cap_elems = (int64_t)p->slot_cap[s] * p->row_elems;
        d.n_elems = (int64_t)p->cart_len[c] * p->row_elems;
        d.frozen_elems = std::min<int64_t>(cfg->n_frozen, p->cart_len[c]) * p->row_elems;
        d.step_size_scale = lr_scale ? lr_scale[i] : 1.0f;
        d.bc1 = (float)(1.0 - pow((double)cfg->beta1, t));
        d.bc2 = (float)(1.0 - pow((double)cfg->beta2, t));
        d.has_grad = p->grad_dirty[(size_t)l * S + s] ? 1 : 0;
      }
    }
    int rc = launch_adam(h.data(), (int)h.size(), *cfg, p->desc.dtype, (cudaStream_t)stream);
    if (rc) return rc;
  }
  for (int s : list) {
    p->opt_steps[p->cart_in[s]] += 1;
    if (cfg->zero_grad)
      for (int l = 0; l < p->n_layers; ++l) p->grad_dirty[(size_t)l * S + s] = 0;
  }
  return CAS_OK;
}

int cas_grad_zero(cas_pool* p, const int32_t* slots, int32_t n, void* stream) {
  int rc = need_data(p);
  if (rc) return rc;
  std::vector<int32_t> list;
  if (slots) list.assign(slots, slots + std::max(n, 0));
  else for (int s = 0; s < p->desc.n_slots; ++s) list.push_back(s);
  for (int s : list) {
    if (s < 0 || s >= p->desc.n_slots) { set_error("bad slot"); return CAS_ERR_INVALID_ARG; }
    for (int l = 0; l < p->n_layers; ++l) p->grad_dirty[(size_t)l * p->desc.n_slots + s] = 0;   // clean = zero gradient
  }
  return CAS_OK;
}

// ---------------------------------------------------------------------------------------------
// rotation (K3) and swap engine (K2, K4)
// ---------------------------------------------------------------------------------------------
int cas_plan_rotation(const cas_pool* p, int64_t step, int32_t n_in, int32_t n_out, const int32_t* protect,
                      int32_t n_protect, uint64_t seed, cas_manifest_entry* entries, int32_t capacity,
                      int32_t* n_entries) {
  if (!p || !entries || !n_entries || n_protect < 0 || (n_protect && !protect)) { set_error("null arg"); return CAS_ERR_INVALID_ARG; }
  const int N = p->desc.n_carts, S = p->desc.n_slots;
  std::vector<char> prot(N, 0);
  for (int i = 0; i < n_protect; ++i) {
    if (protect[i] < 0 || protect[i] >= N) { set_error("bad protected id"); return CAS_ERR_INVALID_ARG; }
    prot[protect[i]] = 1;
  }
  std::vector<int32_t> evictable, waiting;
  for (int c = 0; c < N; ++c) {
    if (p->in_transit[c]) continue;
    if (p->slot_of[c] >= 0) { if (!prot[c]) evictable.push_back(c); }
    else waiting.push_back(c);
  }
  std::sort(evictable.begin(), evictable.end(), [&](int a, int b) {
    return p->last_used[a] != p->last_used[b] ? p->last_used[a] < p->last_used[b] : a < b;
  });
  if ((int)evictable.size() > std::max(n_out, 0)) evictable.resize(std::max(n_out, 0));
  std::vector<uint64_t> hsh(N, 0);
  for (int c : waiting) hsh[c] = mix64(seed, (uint64_t)step, (uint64_t)c);
  std::sort(waiting.begin(), waiting.end(), [&](int a, int b) {
    if (p->opt_steps[a] != p->opt_steps[b]) return p->opt_steps[a] < p->opt_steps[b];
    if (hsh[a] != hsh[b]) return hsh[a] < hsh[b];
    return a < b;
  });
  std::vector<int32_t> freeslots;
  for (int s = 0; s < S; ++s) if (p->cart_in[s] < 0) freeslots.push_back(s);
  for (int c : evictable) freeslots.push_back(p->slot_of[c]);
  std::sort(freeslots.begin(), freeslots.end());
  std::vector<char> used(freeslots.size(), 0);
  struct Arrival { int32_t cart, slot, base_tok; };
  std::vector<Arrival> arrivals;
  if (p->paged) {
    // the lowest unused slot handle + the first-fit run of pages that are free now, or freed by this round's evictees,
    // and that no earlier arrival of this plan has taken; a cartridge that fits nowhere is skipped
    std::vector<char> leaving(N, 0), taken(p->n_pages, 0);
    for (int c : evictable) leaving[c] = 1;
    size_t next_handle = 0;
    for (int c : waiting) {
      if ((int)arrivals.size() >= std::max(n_in, 0) || next_handle >= freeslots.size()) break;
      const int32_t n = p->pages_for(c);
      const int32_t b = first_fit(p->n_pages, n, [&](int32_t q) {
        const int32_t o = p->page_owner[q];
        return (o < 0 || leaving[o]) && p->page_claim[q] < 0 && !taken[q];
      });
      if (b < 0) continue;
      for (int32_t q = b; q < b + n; ++q) taken[q] = 1;
      arrivals.push_back({c, freeslots[next_handle++], b * p->tile});
    }
  } else {
    for (int c : waiting) {
      if ((int)arrivals.size() >= std::max(n_in, 0)) break;
      for (size_t i = 0; i < freeslots.size(); ++i)
        if (!used[i] && p->slot_cap[freeslots[i]] >= p->cart_len[c]) {
          used[i] = 1;
          arrivals.push_back({c, freeslots[i], p->slot_base[freeslots[i]]});
          break;
        }
    }
  }
  std::vector<std::pair<int32_t, int32_t>> outs;       // (slot, cart)
  for (int c : evictable) outs.push_back({p->slot_of[c], c});
  std::sort(outs.begin(), outs.end());
  const int total = (int)(outs.size() + arrivals.size());
  if (total > capacity) { set_error("manifest needs %d entries", total); return CAS_ERR_CAPACITY; }
  int k = 0;
  for (auto& o : outs) entries[k++] = {o.second, o.first, CAS_DIR_OUT, p->slot_base[o.first], p->home_off[o.second], p->home_bytes(o.second)};
  for (auto& a : arrivals) entries[k++] = {a.cart, a.slot, CAS_DIR_IN, a.base_tok, p->home_off[a.cart], p->home_bytes(a.cart)};
  *n_entries = k;
  return CAS_OK;
}

static int copy_cart(cas_pool* p, int c, int s, bool to_host, cudaStream_t st) {
  const int64_t n = (int64_t)p->cart_len[c] * p->row_elems;
  const cudaMemcpyKind kind = to_host ? cudaMemcpyDeviceToHost : cudaMemcpyHostToDevice;
  for (int l = 0; l < p->n_layers; ++l) {
    if (p->cart_len[c] == p->slot_cap[s]) {   // the six tensors of a layer are contiguous on both sides
      void* d = p->slot_state(l, s, 0);
      void* h = p->home(c, l, 0);
      CAS_CUDA(cudaMemcpyAsync(to_host ? h : d, to_host ? d : h, 6 * n * 4, kind, st));
    } else {
      for (int w = 0; w < 6; ++w) {
        void* d = p->slot_state(l, s, w);
        void* h = p->home(c, l, w);
        CAS_CUDA(cudaMemcpyAsync(to_host ? h : d, to_host ? d : h, n * 4, kind, st));
      }
    }
  }
  return CAS_OK;
}

int cas_swap_out(cas_pool* p, const cas_manifest_entry* e, int32_t n, int64_t step, void* after_stream) {
  if (!p || (n && !e) || n < 0) { set_error("null arg"); return CAS_ERR_INVALID_ARG; }
  for (int i = 0; i < n; ++i) {
    if (e[i].dir != CAS_DIR_OUT) continue;
    const int c = e[i].cart, s = e[i].slot;
    if (c < 0 || c >= p->desc.n_carts || s < 0 || s >= p->desc.n_slots) { set_error("bad manifest entry"); return CAS_ERR_INVALID_ARG; }
    if (p->slot_of[c] != s) { set_error("cartridge %d is not in slot %d", c, s); return CAS_ERR_NOT_RESIDENT; }
    if (p->in_transit[c]) { set_error("cartridge %d already in transit", c); return CAS_ERR_BUSY; }
    if (p->any_dirty(s)) { set_error("slot %d has un-consumed gradients", s); return CAS_ERR_BUSY; }
    if (e[i].host_off != p->home_off[c] || e[i].nbytes != p->home_bytes(c)) { set_error("manifest bytes mismatch"); return CAS_ERR_INVALID_ARG; }
  }
  if (p->dev) {
    if (!p->pinned) { set_error("no pinned arena"); return CAS_ERR_INVALID_ARG; }
    if (after_stream != (void*)p->side) {
      CAS_CUDA(cudaEventRecord(p->ev_main, (cudaStream_t)after_stream));
      CAS_CUDA(cudaStreamWaitEvent(p->side, p->ev_main, 0));
    }
  }
  for (int i = 0; i < n; ++i) {
    if (e[i].dir != CAS_DIR_OUT) continue;
    if (p->dev) {
      int rc = copy_cart(p, e[i].cart, e[i].slot, true, p->side);
      if (rc) return rc;
      CAS_CUDA(cudaEventRecord(p->ev_slot[e[i].slot], p->side));   // the slot is free once this copy is done
      // ... and so is the cartridge's pinned home complete: a later arrival of the SAME cartridge (into any slot)
      // must not read its home before this copy has landed
      if (!p->ev_cart[e[i].cart]) CAS_CUDA(cudaEventCreateWithFlags(&p->ev_cart[e[i].cart], cudaEventDisableTiming));
      CAS_CUDA(cudaEventRecord(p->ev_cart[e[i].cart], p->side));
      if (p->paged) CAS_CUDA(cudaEventRecord(p->ev_out_last, p->side));
    }
    p->in_transit[e[i].cart] = 1;
    p->pending.push_back({e[i], step});
  }
  return CAS_OK;
}

int cas_swap_in(cas_pool* p, const cas_manifest_entry* e, int32_t n, int64_t step) {
  if (!p || (n && !e) || n < 0) { set_error("null arg"); return CAS_ERR_INVALID_ARG; }
  std::set<int32_t> leaving, taken;
  std::vector<int32_t> claim = p->page_claim;   // paged pool: pages claimed by arrivals in flight (+ this call's)
  for (auto& q : p->pending) {
    if (q.e.dir == CAS_DIR_OUT) leaving.insert(q.e.slot);
    else taken.insert(q.e.slot);
  }
  for (int i = 0; i < n; ++i) {
    if (e[i].dir != CAS_DIR_IN) continue;
    const int c = e[i].cart, s = e[i].slot;
    if (c < 0 || c >= p->desc.n_carts || s < 0 || s >= p->desc.n_slots) { set_error("bad manifest entry"); return CAS_ERR_INVALID_ARG; }
    if (p->slot_of[c] >= 0 || p->in_transit[c]) { set_error("cartridge %d already resident / in transit", c); return CAS_ERR_BUSY; }
    if (!(p->cart_in[s] < 0 || leaving.count(s)) || !taken.insert(s).second) { set_error("slot %d occupied", s); return CAS_ERR_BUSY; }
    if (!p->paged && p->slot_cap[s] < p->cart_len[c]) { set_error("slot %d too small", s); return CAS_ERR_CAPACITY; }
    if (e[i].host_off != p->home_off[c] || e[i].nbytes != p->home_bytes(c)) { set_error("manifest bytes mismatch"); return CAS_ERR_INVALID_ARG; }
    if (p->paged) {
      const int32_t np_ = p->pages_for(c), b = e[i].base_tok / p->tile;
      if (e[i].base_tok % p->tile || b < 0 || b + np_ > p->n_pages) { set_error("bad extent for cartridge %d", c); return CAS_ERR_INVALID_ARG; }
      for (int32_t q = b; q < b + np_; ++q) {
        const int32_t o = p->page_owner[q];
        if (claim[q] >= 0 || (o >= 0 && p->in_transit[o] != 1)) { set_error("page %d is occupied", q); return CAS_ERR_BUSY; }
      }
      for (int32_t q = b; q < b + np_; ++q) claim[q] = c;
    }
  }
  if (p->paged) p->page_claim = claim;   // every entry is valid: the claims stand
  if (p->dev && !p->pinned) { set_error("no pinned arena"); return CAS_ERR_INVALID_ARG; }
  if (p->paged) {
    // the slot handles take their arrivals' extents now: the copies below are addressed through them
    for (int i = 0; i < n; ++i) {
      if (e[i].dir != CAS_DIR_IN) continue;
      p->slot_base[e[i].slot] = e[i].base_tok;
      p->slot_cap[e[i].slot] = p->pages_for(e[i].cart) * p->tile;
    }
    // pages freed by ANY earlier eviction (this round's or an older one whose copy may still be in flight)
    if (p->dev) CAS_CUDA(cudaStreamWaitEvent(p->side_in, p->ev_out_last, 0));
  }
  // all copies first, then the refresh kernels: a kernel between two copies would hold the next copy
  // back until the kernel finds a free SM under the attention kernels of the main stream
  for (int i = 0; i < n && p->dev; ++i) {
    if (e[i].dir != CAS_DIR_IN) continue;
    const int c = e[i].cart, s = e[i].slot;
    // after the eviction that freed this slot -- in this round or in an EARLIER, already committed one (its D2H copy
    // may still be running, and it is also what carries the wait on the main-stream work that last used the slot).
    // ev_slot[s] holds the record of the slot's last eviction copy; waiting on a never-recorded event is a no-op.
    CAS_CUDA(cudaStreamWaitEvent(p->side_in, p->ev_slot[s], 0));
    if (p->ev_cart[c]) CAS_CUDA(cudaStreamWaitEvent(p->side_in, p->ev_cart[c], 0));   // its own last eviction copy
    int rc = copy_cart(p, c, s, false, p->side_in);
    if (rc) return rc;
  }
  for (int i = 0; i < n; ++i) {
    if (e[i].dir != CAS_DIR_IN) continue;
    const int c = e[i].cart, s = e[i].slot;
    if (p->dev) {
      const int64_t o = (int64_t)p->slot_base[s] * p->row_elems, nel = (int64_t)p->cart_len[c] * p->row_elems;
      for (int l = 0; l < p->n_layers; ++l) {
        const PoolLayer& L = p->layers[l];
        int rc = launch_refresh(p->slot_state(l, s, 0), p->slot_state(l, s, 1), (char*)L.pool_K + o * p->elem_bytes,
                                (char*)L.pool_V + o * p->elem_bytes, L.grad_K + o, L.grad_V + o, nel, p->desc.dtype,
                                p->side_in);
        if (rc) return rc;
      }
    }
    p->in_transit[c] = 2;
    p->pending.push_back({e[i], step});
  }
  return CAS_OK;
}

int cas_swap_commit(cas_pool* p, void* main_stream) {
  if (!p) { set_error("null pool"); return CAS_ERR_INVALID_ARG; }
  if (p->dev && !p->pending.empty()) {
    CAS_CUDA(cudaEventRecord(p->ev_side, p->side));
    CAS_CUDA(cudaStreamWaitEvent((cudaStream_t)main_stream, p->ev_side, 0));
    CAS_CUDA(cudaEventRecord(p->ev_side_in, p->side_in));
    CAS_CUDA(cudaStreamWaitEvent((cudaStream_t)main_stream, p->ev_side_in, 0));
  }
  for (auto& q : p->pending)
    if (q.e.dir == CAS_DIR_OUT) {
      p->slot_of[q.e.cart] = -1;
      p->in_transit[q.e.cart] = 0;
      if (p->cart_in[q.e.slot] == q.e.cart) p->cart_in[q.e.slot] = -1;
      if (p->paged)
        for (int32_t& o : p->page_owner) if (o == q.e.cart) o = -1;
    }
  for (auto& q : p->pending)
    if (q.e.dir == CAS_DIR_IN) {
      p->slot_of[q.e.cart] = q.e.slot;
      p->cart_in[q.e.slot] = q.e.cart;
      p->in_transit[q.e.cart] = 0;
      p->last_used[q.e.cart] = q.step;
      if (p->paged)
        for (int32_t pg = 0; pg < p->n_pages; ++pg)
          if (p->page_claim[pg] == q.e.cart) { p->page_owner[pg] = q.e.cart; p->page_claim[pg] = -1; }
    }
  p->pending.clear();
  return CAS_OK;
}

// ---------------------------------------------------------------------------------------------
// end-to-end step from host buffers
// ---------------------------------------------------------------------------------------------
static StepScratch step_scratch(const cas_pool* p, const cas_slot_table* t, int Hq) {
  StepScratch s{};
  const size_t eb = p->elem_bytes, T = t->T, D = p->desc.D, Hkv = p->desc.Hkv;
  size_t o = 0;
  auto add = [&](size_t bytes) { size_t r = o; o = (size_t)round_up((int64_t)(o + bytes), 1024); return r; };
  s.oQ = add(T * Hq * D * eb);   s.oKs = add(T * Hkv * D * eb); s.oVs = add(T * Hkv * D * eb);
  s.odO = add(T * Hq * D * eb);  s.oO = add(T * Hq * D * eb);   s.oLSE = add(T * Hq * 4);
  s.odQ = add(T * Hq * D * eb);  s.odKs = add(T * Hkv * D * eb); s.odVs = add(T * Hkv * D * eb);
  s.set_bytes = o;
  cas_prefix_attn_bwd_workspace_bytes(p, t, Hq, &s.ws_bytes);
  s.oWs = 2 * s.set_bytes;
  s.total = s.oWs + s.ws_bytes;
  return s;
}

int cas_train_step_host_scratch_bytes(const cas_pool* p, const cas_slot_table* t, int32_t Hq, size_t* bytes) {
  if (!p || !t || !bytes || Hq < 1) { set_error("null arg"); return CAS_ERR_INVALID_ARG; }
  *bytes = step_scratch(p, t, Hq).total;
  return CAS_OK;
}

int cas_train_step_host_wait(cas_pool* p, void* stream) {
  if (!p) { set_error("null arg"); return CAS_ERR_INVALID_ARG; }
  // an event that was never recorded counts as complete
  for (int k = 0; k < 2; ++k) CAS_CUDA(cudaStreamWaitEvent((cudaStream_t)stream, p->ev_step[5 + 5 * k], 0));
  return CAS_OK;
}

// One step.  Streams: the caller's (kernels), st_h2d (inputs), st_d2h (results).  Consecutive steps alternate between
// two device buffer sets, so the inputs of step i+1 cross the host link while step i computes and the results of
// step i leave while step i+1 computes: in steady state a step costs max(kernels, H2D bytes, D2H bytes), not their
// sum.  Hazards, all expressed as events: set k's inputs are overwritten only after the backward pass of step i-2
// (their last reader), set k's results only after the read-back of step i-2; the backward workspace is shared and
// ordered by the caller's stream.
static int train_step_host(cas_pool* p, const cas_slot_table* t, int32_t Hq, const void* hQ, const void* hKs,
                           const void* hVs, const void* hdO, float scale, const cas_adam_cfg* cfg, void* hO,
                           float* hLSE, void* hdQ, void* hdKs, void* hdVs, void* scratch, size_t scratch_bytes,
                           void* stream, bool wait_readback) {
  int rc = need_data(p);
  if (rc) return rc;
  if (!t || !hQ || !hKs || !hVs || !hdO || !cfg || !hO || !hLSE || !hdQ || !scratch) { set_error("null arg"); return CAS_ERR_INVALID_ARG; }
  if (p->n_layers != 1) { set_error("cas_train_step_host drives single-layer pools; use cas_train_step_layers"); return CAS_ERR_SHAPE; }
  if ((hdKs == nullptr) != (hdVs == nullptr)) { set_error("hdK_self / hdV_self: both or none"); return CAS_ERR_INVALID_ARG; }
  const StepScratch s = step_scratch(p, t, Hq);
  if (scratch_bytes < s.total) { set_error("scratch too small: need %zu", s.total); return CAS_ERR_CAPACITY; }
  cudaStream_t st = (cudaStream_t)stream;
  const size_t eb = p->elem_bytes, T = t->T, D = p->desc.D, Hkv = p->desc.Hkv;
  cudaEvent_t* ev = p->ev_step;
  const bool same_layout = p->step_prev_scratch == scratch && p->step_prev_stream == st &&
                           memcmp(&p->step_prev_layout, &s, sizeof(StepScratch)) == 0;
  if (!same_layout) {
    // first call, or the regions moved (ragged batches: T changes per step; another scratch or stream): everything
    // still in flight on the old layout has to finish first
    rc = cas_train_step_host_wait(p, stream);
    if (rc) return rc;
    p->step_count = 0;
  }
  const int k = (int)(p->step_count & 1);
  ++p->step_count;
  p->step_prev_scratch = scratch;
  p->step_prev_stream = st;
  p->step_prev_layout = s;
  char* d = (char*)scratch + (size_t)k * s.set_bytes;
  char* ws = (char*)scratch + s.oWs;
  cudaEvent_t eIn1 = ev[1 + 5 * k], eIn2 = ev[2 + 5 * k], eFwd = ev[3 + 5 * k], eBwd = ev[4 + 5 * k], eOut = ev[5 + 5 * k];
  if (same_layout) {
    // step i-2 has read this set's inputs.  NOT ordered after the caller's stream: that would put these copies behind
    // the previous step's Adam -- the host inputs must hold their data when the call is made.
    CAS_CUDA(cudaStreamWaitEvent(p->st_h2d, eBwd, 0));
  } else {
    CAS_CUDA(cudaEventRecord(ev[0], st));
    CAS_CUDA(cudaStreamWaitEvent(p->st_h2d, ev[0], 0));
    CAS_CUDA(cudaStreamWaitEvent(p->st_d2h, ev[0], 0));
  }
  CAS_CUDA(cudaMemcpyAsync(d + s.oQ, hQ, T * Hq * D * eb, cudaMemcpyHostToDevice, p->st_h2d));
  CAS_CUDA(cudaMemcpyAsync(d + s.oKs, hKs, T * Hkv * D * eb, cudaMemcpyHostToDevice, p->st_h2d));
  CAS_CUDA(cudaMemcpyAsync(d + s.oVs, hVs, T * Hkv * D * eb, cudaMemcpyHostToDevice, p->st_h2d));
  CAS_CUDA(cudaEventRecord(eIn1, p->st_h2d));
  CAS_CUDA(cudaMemcpyAsync(d + s.odO, hdO, T * Hq * D * eb, cudaMemcpyHostToDevice, p->st_h2d));
  CAS_CUDA(cudaEventRecord(eIn2, p->st_h2d));
  CAS_CUDA(cudaStreamWaitEvent(st, eIn1, 0));
  if (same_layout) { CAS_CUDA(cudaStreamWaitEvent(st, eOut, 0)); }       // step i-2's results have left this set
  rc = cas_prefix_attn_fwd(p, t, Hq, d + s.oQ, d + s.oKs, d + s.oVs, scale, d + s.oO, (float*)(d + s.oLSE), stream);
  if (rc) return rc;
  CAS_CUDA(cudaEventRecord(eFwd, st));
  CAS_CUDA(cudaStreamWaitEvent(p->st_d2h, eFwd, 0));
  CAS_CUDA(cudaMemcpyAsync(hO, d + s.oO, T * Hq * D * eb, cudaMemcpyDeviceToHost, p->st_d2h));
  CAS_CUDA(cudaMemcpyAsync(hLSE, d + s.oLSE, T * Hq * 4, cudaMemcpyDeviceToHost, p->st_d2h));
  CAS_CUDA(cudaStreamWaitEvent(st, eIn2, 0));
  rc = cas_prefix_attn_bwd(p, t, Hq, d + s.oQ, d + s.oKs, d + s.oVs, d + s.oO, (float*)(d + s.oLSE), d + s.odO,
                           scale, d + s.odQ, d + s.odKs, d + s.odVs, ws, s.ws_bytes, stream);
  if (rc) return rc;
  CAS_CUDA(cudaEventRecord(eBwd, st));
  CAS_CUDA(cudaStreamWaitEvent(p->st_d2h, eBwd, 0));
  CAS_CUDA(cudaMemcpyAsync(hdQ, d + s.odQ, T * Hq * D * eb, cudaMemcpyDeviceToHost, p->st_d2h));
  if (hdKs) {
    CAS_CUDA(cudaMemcpyAsync(hdKs, d + s.odKs, T * Hkv * D * eb, cudaMemcpyDeviceToHost, p->st_d2h));
    CAS_CUDA(cudaMemcpyAsync(hdVs, d + s.odVs, T * Hkv * D * eb, cudaMemcpyDeviceToHost, p->st_d2h));
  }
  CAS_CUDA(cudaEventRecord(eOut, p->st_d2h));
  rc = cas_adam_step(p, cfg, nullptr, 0, nullptr, stream);
  if (rc) return rc;
  if (wait_readback) CAS_CUDA(cudaStreamWaitEvent(st, eOut, 0));
  return CAS_OK;
}

int cas_train_step_host(cas_pool* p, const cas_slot_table* t, int32_t Hq, const void* hQ, const void* hKs,
                        const void* hVs, const void* hdO, float scale, const cas_adam_cfg* cfg, void* hO,
                        float* hLSE, void* hdQ, void* hdKs, void* hdVs, void* scratch, size_t scratch_bytes,
                        void* stream) {
  return train_step_host(p, t, Hq, hQ, hKs, hVs, hdO, scale, cfg, hO, hLSE, hdQ, hdKs, hdVs, scratch, scratch_bytes,
                         stream, true);
}

int cas_train_step_host_async(cas_pool* p, const cas_slot_table* t, int32_t Hq, const void* hQ, const void* hKs,
                              const void* hVs, const void* hdO, float scale, const cas_adam_cfg* cfg, void* hO,
                              float* hLSE, void* hdQ, void* hdKs, void* hdVs, void* scratch, size_t scratch_bytes,
                              void* stream) {
  return train_step_host(p, t, Hq, hQ, hKs, hVs, hdO, scale, cfg, hO, hLSE, hdQ, hdKs, hdVs, scratch, scratch_bytes,
                         stream, false);
}

// ---------------------------------------------------------------------------------------------
// one optimizer step over all layers and several micro-batches (device buffers)
// ---------------------------------------------------------------------------------------------
int cas_train_step_layers_workspace_bytes(const cas_pool* p, const cas_slot_table* const* tables, int32_t n_micro,
                                          int32_t Hq, size_t* bytes) {
  if (!p || !tables || n_micro < 1 || !bytes) { set_error("null arg"); return CAS_ERR_INVALID_ARG; }
  size_t mx = 0;
  for (int m = 0; m < n_micro; ++m) {
    size_t b = 0;
    int rc = cas_prefix_attn_bwd_workspace_bytes(p, tables[m], Hq, &b);
    if (rc) return rc;
    mx = std::max(mx, b);
  }
  *bytes = mx;
  return CAS_OK;
}

int cas_train_step_layers(cas_pool* p, const cas_slot_table* const* tables, int32_t n_micro, int32_t Hq,
                          const cas_layer_io* io, float scale, const cas_adam_cfg* cfg, const float* lr_scale,
                          void* workspace, size_t workspace_bytes, void* stream) {
  int rc = need_data(p);
  if (rc) return rc;
  if (!tables || n_micro < 1 || !io || !cfg) { set_error("null arg"); return CAS_ERR_INVALID_ARG; }
  const int L = p->n_layers;
  for (int m = 0; m < n_micro; ++m) {
    const cas_slot_table* t = tables[m];
    // forward through the layer stack, then backward in reverse order: the order a model visits its layers in
    for (int l = 0; l < L; ++l) {
      const cas_layer_io& x = io[(size_t)m * L + l];
      rc = attn_fwd_impl(p, t, l, Hq, x.Q, x.K_self, x.V_self, scale, x.O, x.LSE, stream, x.rope, x.Q_rot, x.K_self_rot);
      if (rc) return rc;
    }
    for (int l = L - 1; l >= 0; --l) {
      const cas_layer_io& x = io[(size_t)m * L + l];
      rc = attn_bwd_impl(p, t, l, Hq, x.rope ? x.Q_rot : x.Q, x.rope && x.K_self ? x.K_self_rot : x.K_self, x.V_self, x.O,
                         x.LSE, x.dO, scale, x.dQ, x.dK_self, x.dV_self, workspace, workspace_bytes, stream, x.rope);
      if (rc) return rc;
    }
  }
  // ONE Adam step consumes the gradients every micro-batch has accumulated into the slots of every layer
  return cas_adam_step(p, cfg, nullptr, 0, lr_scale, stream);
}

}  // extern "C"
