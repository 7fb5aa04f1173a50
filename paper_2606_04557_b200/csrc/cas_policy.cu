// Budget-manager policy helpers on the host: the Eq. 1 mixture sampler
// (PAPER.md:64-66), the global learning-rate schedule (Table 5 :366-373) and the bucketed
// per-cartridge warmup.  Pure integer / scalar logic, no device work.  The integer results are
// bit-exact against oracle/bookkeeping.py, which implements the same documented rules independently
// (R29-R31).
#include <algorithm>
#include <vector>

#include "cas_internal.h"

namespace cas {

// DESIGN.md R15: SplitMix64 finaliser over seed + gamma*(step+1) + 0xD1B54A32D192ED03*(cart+1).
static inline uint64_t mix3(uint64_t seed, uint64_t a, uint64_t b) {
  uint64_t z = seed + 0x9E3779B97F4A7C15ull * (a + 1) + 0xD1B54A32D192ED03ull * (b + 1);
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}
// R31: d-th draw of example b at step `step`
static inline uint64_t draw(uint64_t seed, uint64_t step, uint64_t b, uint64_t d) {
  return mix3(mix3(seed, step, b), d, 0);
}
static inline uint64_t below(uint64_t x, uint64_t n) { return ((x >> 32) * n) >> 32; }   // integer in [0, n)

}  // namespace cas

extern "C" {

int cas_sample_selection(const cas_pool* p, int32_t B, const int32_t* targets, double p_iso, int32_t k_min,
                         int32_t k_max, uint64_t seed, int64_t step, int32_t* sel_off, int32_t* sel_cart,
                         int32_t capacity) {
  using namespace cas;
  if (!p || !targets || !sel_off || !sel_cart || B < 1) { set_error("null / empty args"); return CAS_ERR_INVALID_ARG; }
  if (!(p_iso >= 0.0 && p_iso <= 1.0) || k_min < 0 || k_max < k_min) { set_error("bad P_iso / k range"); return CAS_ERR_INVALID_ARG; }
  std::vector<int32_t> stable;
  for (int c = 0; c < p->desc.n_carts; ++c)
    if (p->slot_of[c] >= 0 && !p->in_transit[c]) stable.push_back(c);
  const uint64_t thr = (uint64_t)(p_iso * 9007199254740992.0);   // floor(P_iso * 2^53)
  int32_t n_out = 0;
  sel_off[0] = 0;
  std::vector<int32_t> cand;
  for (int b = 0; b < B; ++b) {
    const int tgt = targets[b];
    if (tgt < 0 || tgt >= p->desc.n_carts) { set_error("target %d out of range", tgt); return CAS_ERR_INVALID_ARG; }
    if (p->slot_of[tgt] < 0 || p->in_transit[tgt]) { set_error("target cartridge %d not resident", tgt); return CAS_ERR_NOT_RESIDENT; }
    if (n_out >= capacity) { set_error("selection capacity"); return CAS_ERR_CAPACITY; }
    sel_cart[n_out++] = tgt;
    if ((draw(seed, (uint64_t)step, (uint64_t)b, 0) >> 11) >= thr) {
      cand.clear();
      for (int c : stable) if (c != tgt) cand.push_back(c);
      int64_t k = k_min + (int64_t)below(draw(seed, (uint64_t)step, (uint64_t)b, 1), (uint64_t)(k_max - k_min + 1));
      k = std::min<int64_t>(k, (int64_t)cand.size());
      if (n_out + k > capacity) { set_error("selection capacity"); return CAS_ERR_CAPACITY; }
      for (int64_t j = 0; j < k; ++j) {
        const size_t r = (size_t)j + (size_t)below(draw(seed, (uint64_t)step, (uint64_t)b, 2 + (uint64_t)j), cand.size() - (size_t)j);
        std::swap(cand[(size_t)j], cand[r]);
        sel_cart[n_out++] = cand[(size_t)j];
      }
    }
    sel_off[b + 1] = n_out;
  }
  return CAS_OK;
}

int cas_lr_schedule(const cas_lr_cfg* c, int64_t t, double* eta) {
  using namespace cas;
  if (!c || !eta || t < 0) { set_error("null arg / negative step"); return CAS_ERR_INVALID_ARG; }
  if (c->warmup_steps < 0 || c->total_steps < c->warmup_steps || !(c->alpha_f >= 0.0)) { set_error("bad schedule"); return CAS_ERR_INVALID_ARG; }
  if (t < c->warmup_steps) {
    *eta = c->warmup_min_lr + (c->eta0 - c->warmup_min_lr) * ((double)t / (double)c->warmup_steps);
  } else if (t >= c->total_steps) {
    *eta = c->alpha_f * c->eta0;
  } else {
    *eta = c->eta0 * (1.0 - (1.0 - c->alpha_f) * ((double)(t - c->warmup_steps) / (double)(c->total_steps - c->warmup_steps)));
  }
  return CAS_OK;
}

int cas_warmup_scales(const cas_pool* p, const int32_t* slots, int32_t n, int32_t w_c, int32_t n_b, float* scale) {
  using namespace cas;
  if (!p || !scale || n < 0 || (n && !slots) || w_c < 1 || n_b < 1) { set_error("bad args"); return CAS_ERR_INVALID_ARG; }
  for (int i = 0; i < n; ++i) {
    const int s = slots[i];
    if (s < 0 || s >= p->desc.n_slots) { set_error("bad slot %d", s); return CAS_ERR_INVALID_ARG; }
    const int c = p->cart_in[s];
    if (c < 0) { set_error("slot %d is empty", s); return CAS_ERR_NOT_RESIDENT; }
    const int64_t num = std::min<int64_t>(p->opt_steps[c] + 1, w_c) * n_b;
    const int64_t level = (num + w_c - 1) / w_c;
    scale[i] = (float)((double)level / (double)n_b);
  }
  return CAS_OK;
}

}  // extern "C"
