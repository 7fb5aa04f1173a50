"""Seeded input generators (numpy PCG64).  Recipe: DESIGN.md "Input recipe"; SURVEY.md 8(d).

Everything here is *input drawing*: shapes, value distributions, the per-sequence cartridge draws
BASELINE.json's configs fix ("target + k seeded distractors", "probability proportional to
cartridge length", "top-8 of a seeded random ranking").  No attention / Adam / rotation arithmetic.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Optional, Sequence

import numpy as np

from .configs import CasConfig

BASE_SEED = 260604


def round_to_dtype(a: np.ndarray, dtype: str) -> np.ndarray:
    """Round fp32 values once (RNE) to the storage dtype and return them as fp32 again, so that
    the oracle and the CUDA path consume bit-identical inputs (SURVEY.md 8(c) precision contract)."""
    a = np.ascontiguousarray(a, dtype=np.float32)
    if dtype == "f32":
        return a
    if dtype == "bf16":
        import torch

        return torch.from_numpy(a).to(torch.bfloat16).to(torch.float32).numpy()
    raise ValueError(dtype)


@dataclass
class Workload:
    cfg: CasConfig
    seed: int
    cart_len: np.ndarray            # int32 [n_carts]
    cart_off: np.ndarray            # int64 [n_carts+1] token offsets into cart_K/cart_V
    cart_K: np.ndarray              # f32 [sum(len), Hkv, D] (values already rounded to cfg.dtype)
    cart_V: np.ndarray
    seq_off: np.ndarray             # int32 [B+1]
    sel_off: np.ndarray             # int32 [B+1]
    sel_cart: np.ndarray            # int32 [nsel] cartridge ids, target first then distractors
    Q: np.ndarray                   # f32 [T, Hq, D]
    K_self: np.ndarray              # f32 [T, Hkv, D]
    V_self: np.ndarray
    dO: Optional[np.ndarray]        # f32 [T, Hq, D] or None (forward-only configs)
    resident: np.ndarray            # int32 [n_slots] cartridge id initially in slot s
    extra: dict = field(default_factory=dict)

    @property
    def T(self) -> int:
        return int(self.seq_off[-1])

    def cart_kv(self, c: int):
        a, b = int(self.cart_off[c]), int(self.cart_off[c + 1])
        return self.cart_K[a:b], self.cart_V[a:b]

    def pairs_per_head(self) -> int:
        """Visible (query,key) pairs per query head: sum_b Lq_b*P_b + Lq_b(Lq_b+1)/2."""
        tot = 0
        for b in range(len(self.seq_off) - 1):
            lq = int(self.seq_off[b + 1] - self.seq_off[b])
            sel = self.sel_cart[self.sel_off[b]:self.sel_off[b + 1]]
            pb = int(self.cart_len[sel].sum())
            tot += lq * pb + lq * (lq + 1) // 2
        return tot


def _normal(rng: np.random.Generator, shape, std: float, dtype: str) -> np.ndarray:
    a = rng.standard_normal(size=shape, dtype=np.float32)
    if std != 1.0:
        a *= np.float32(std)
    return round_to_dtype(a, dtype)


def draw_cart_lengths(cfg: CasConfig, rng: np.random.Generator) -> np.ndarray:
    if cfg.cart_len > 0:
        return np.full(cfg.n_carts, cfg.cart_len, dtype=np.int32)
    if cfg.len_pages_max > 0:        # whole 16-token pages, 1..len_pages_max of them
        return (16 * rng.integers(1, cfg.len_pages_max + 1, size=cfg.n_carts)).astype(np.int32)
    # config 4: round(lognormal(mu, sigma)) clamped to [len_min, len_max]
    raw = np.exp(rng.normal(cfg.len_mu, cfg.len_sigma, size=cfg.n_carts))
    return np.clip(np.rint(raw), cfg.len_min, cfg.len_max).astype(np.int32)


def draw_selection(rng: np.random.Generator, candidates: Sequence[int], n_dist: int,
                   cart_len: np.ndarray, mode: str) -> List[int]:
    """One sequence's cartridge list: target first, then ``n_dist`` distinct distractors in draw
    order.  ``mode``: "uniform" (configs 1-3), "prop_len" (config 4: target and distractors with
    probability proportional to cartridge length, without replacement, by exact integer
    cumulative sums), "all" (config 5-i), "topk" (config 5-ii: first 1+n_dist of a seeded random
    ranking of the candidates)."""
    cand = [int(c) for c in candidates]
    if mode == "all":
        return cand
    if mode == "topk":
        perm = rng.permutation(len(cand))
        return [cand[i] for i in perm[: 1 + n_dist]]
    k = min(1 + n_dist, len(cand))
    if mode == "uniform":
        idx = rng.choice(len(cand), size=k, replace=False)
        return [cand[i] for i in idx]
    if mode == "prop_len":
        out = []
        pool = list(cand)
        for _ in range(k):
            w = np.asarray([int(cart_len[c]) for c in pool], dtype=np.int64)
            cum = np.cumsum(w)
            r = int(rng.integers(0, int(cum[-1])))
            j = int(np.searchsorted(cum, r, side="right"))
            out.append(pool.pop(j))
        return out
    raise ValueError(mode)


def draw_batch_selection(cfg: CasConfig, rng: np.random.Generator, candidates: Sequence[int],
                         cart_len: np.ndarray):
    """sel_off / sel_cart for one batch of cfg.B sequences."""
    sel_off = [0]
    sel = []
    for _ in range(cfg.B):
        if cfg.n_dist == -1:
            nd = int(rng.integers(0, cfg.n_dist_max + 1))
        elif cfg.n_dist == -2:
            nd = len(candidates) - 1
        else:
            nd = cfg.n_dist
        s = draw_selection(rng, candidates, nd, cart_len, cfg.selection)
        sel.extend(s)
        sel_off.append(len(sel))
    return np.asarray(sel_off, dtype=np.int32), np.asarray(sel, dtype=np.int32)


def draw_batch_selection_uniform(cfg: CasConfig, rng: np.random.Generator, candidates: np.ndarray):
    """The "uniform" recipe of draw_batch_selection for a whole batch in a few array operations (same
    distribution: per sequence a target and n_dist distinct distractors, uniform without replacement, in draw
    order; another random stream).  For drivers that draw a fresh batch every step among the currently resident
    cartridges (bench.py's rotation configs), where 32 calls of Generator.choice cost more host time than the step
    costs on the GPU.  Holds no method arithmetic."""
    assert cfg.selection == "uniform" and cfg.n_dist != -2
    cand = np.asarray(candidates, dtype=np.int32)
    n = len(cand)
    if cfg.n_dist == -1:
        nd = rng.integers(0, cfg.n_dist_max + 1, size=cfg.B)
    else:
        nd = np.full(cfg.B, cfg.n_dist, dtype=np.int64)
    k = np.minimum(1 + nd, n).astype(np.int64)
    kmax = int(k.max())
    # the first kmax entries of a uniform random permutation of the candidates, per sequence: smallest random keys
    keys = rng.random((cfg.B, n))
    first = np.argpartition(keys, kmax - 1, axis=1)[:, :kmax] if kmax < n else np.argsort(keys, axis=1)
    order = np.take_along_axis(keys, first, axis=1).argsort(axis=1)
    first = np.take_along_axis(first, order, axis=1)                  # draw order = ascending key
    sel_off = np.zeros(cfg.B + 1, dtype=np.int32)
    np.cumsum(k, out=sel_off[1:])
    mask = np.arange(kmax)[None, :] < k[:, None]
    return sel_off, cand[first[mask]].astype(np.int32)


def draw_query_block(cfg: CasConfig, rng: np.random.Generator, seq_off: np.ndarray,
                     with_dO: bool = True):
    """Q ~ N(0,1); self K/V ~ N(0, kv_std); dO ~ N(0,1)."""
    T = int(seq_off[-1])
    Q = _normal(rng, (T, cfg.Hq, cfg.D), 1.0, cfg.dtype)
    Ks = _normal(rng, (T, cfg.Hkv, cfg.D), cfg.kv_std, cfg.dtype)
    Vs = _normal(rng, (T, cfg.Hkv, cfg.D), cfg.kv_std, cfg.dtype)
    dO = _normal(rng, (T, cfg.Hq, cfg.D), 1.0, cfg.dtype) if with_dO else None
    return Q, Ks, Vs, dO


def make_workload(cfg: CasConfig, seed: Optional[int] = None) -> Workload:
    seed = BASE_SEED if seed is None else seed
    rng = np.random.Generator(np.random.PCG64(seed))
    cart_len = draw_cart_lengths(cfg, rng)
    cart_off = np.zeros(cfg.n_carts + 1, dtype=np.int64)
    np.cumsum(cart_len, out=cart_off[1:])
    tot = int(cart_off[-1])
    cart_K = _normal(rng, (tot, cfg.Hkv, cfg.D), cfg.kv_std, cfg.dtype)
    cart_V = _normal(rng, (tot, cfg.Hkv, cfg.D), cfg.kv_std, cfg.dtype)

    if cfg.Lq > 0:
        lq = np.full(cfg.B, cfg.Lq, dtype=np.int64)
    else:
        lq = rng.integers(cfg.lq_min, cfg.lq_max + 1, size=cfg.B)
    seq_off = np.zeros(cfg.B + 1, dtype=np.int32)
    seq_off[1:] = np.cumsum(lq)

    resident = np.arange(cfg.n_slots, dtype=np.int32)      # cartridges 0..n_slots-1 start on GPU
    sel_off, sel_cart = draw_batch_selection(cfg, rng, resident.tolist(), cart_len)
    Q, Ks, Vs, dO = draw_query_block(cfg, rng, seq_off, with_dO=cfg.backward)
    return Workload(cfg=cfg, seed=seed, cart_len=cart_len, cart_off=cart_off, cart_K=cart_K,
                    cart_V=cart_V, seq_off=seq_off, sel_off=sel_off, sel_cart=sel_cart, Q=Q,
                    K_self=Ks, V_self=Vs, dO=dO, resident=resident)
