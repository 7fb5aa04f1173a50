"""CAS hot-path ORACLE (floating-point part) -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Plain, slow, obviously-correct CPU implementation (numpy, float64) of what the hot path computes:
masked prefix attention forward (F1-F4), its exact gradient (B1-B6), textbook Adam with a bf16
working copy (A1-A4).  It is the plain definition written out: the visible keys of a sequence are
materialised by concatenation and the causal mask is a dense boolean matrix.  ``numpy.matmul`` is the
only library primitive used.  No blocking, no online softmax, no fusion.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline / ``--impl reference``
legs may import this module.  It shares no code with ``paper_2606_04557_b200`` and imports nothing
from it.

Passages followed (PAPER.md = /root/reference/PAPER.md at build time; SURVEY.md 8(c) restates them):
  * PAPER.md:42  (sec. 2 Background)  a cartridge Z in R^{L x p x d x 2} is a trainable KV prefix
    "injected into the model's attention layers"; PAPER.md:111 (sec. 2.5) selected cartridges are
    "sequentially concatenated" and prepended; PAPER.md:71 (sec. 2.1) "each packed sample sees a
    different subset via an attention mask"  -> visible-key set F1.
  * PAPER.md:44  "only the key-value vectors in Z receive gradients" -> gradients B5 go to the
    selected blocks only; PAPER.md:75 evicted (here: unselected) cartridges receive no gradients;
    PAPER.md:176 all active cartridges are back-propagated simultaneously -> sums over sequences.
  * PAPER.md:81 (sec. 2.2) "Adam (Kingma and Ba, 2014) with fp32 precision, while we keep the weights
    in bfloat16"; PAPER.md:85 per-cartridge LR scale; PAPER.md:390 (Table 5) frozen first token.
Readings of silent points (scale, head grouping, eps placement ...) are DESIGN.md R1-R12.

Pins (tests/test_oracle_pins.py): brute-force python loops, finite differences, closed forms (K=0 ->
uniform softmax, LSE = ln(count)), conservation laws, torch SDPA float64 + autograd on the explicit
concat/mask, torch.optim.Adam, torch bf16 cast, Adam closed forms, the paper's MiB figures.
"""
from __future__ import annotations

from typing import Dict, List, Optional, Sequence, Tuple

import numpy as np

F64 = np.float64


def _visible_kv(blocks_K, blocks_V, sel_b: Sequence[int], K_self, V_self, t0: int, t1: int, g: int):
    """F1: keys/values visible to sequence b for KV head g: all tokens of the selected blocks, in
    table order, followed by the sequence's own tokens (masked causally by the caller)."""
    ks = [np.asarray(blocks_K[s][:, g, :], dtype=F64) for s in sel_b]
    vs = [np.asarray(blocks_V[s][:, g, :], dtype=F64) for s in sel_b]
    n_prefix = int(sum(k.shape[0] for k in ks))
    if K_self is not None:
        ks.append(np.asarray(K_self[t0:t1, g, :], dtype=F64))
        vs.append(np.asarray(V_self[t0:t1, g, :], dtype=F64))
    D = (K_self.shape[-1] if K_self is not None else blocks_K[sel_b[0]].shape[-1])
    if not ks:
        return np.zeros((0, D), F64), np.zeros((0, D), F64), 0
    return np.concatenate(ks, 0), np.concatenate(vs, 0), n_prefix


def _mask(Lq: int, n_prefix: int, n_self: int) -> np.ndarray:
    """F1: True where key j is visible to query row i: every prefix key; self key t' <= i."""
    m = np.ones((Lq, n_prefix + n_self), dtype=bool)
    if n_self:
        m[:, n_prefix:] = np.tril(np.ones((Lq, n_self), dtype=bool))
    return m


def attn_fwd(Q, blocks_K, blocks_V, sel: Sequence[Sequence[int]], seq_off, K_self, V_self,
             scale: float, Hkv: int, kv_heads: Optional[Sequence[int]] = None):
    """F1-F4.  Q [T,Hq,D]; blocks_K[s]/blocks_V[s] [len_s,Hkv,D]; sel[b] = ordered distinct block
    ids of sequence b; K_self/V_self [T,Hkv,D] or None (prefix only).  Returns O [T,Hq,D] and
    LSE [T,Hq] (natural log), float64.  Query head h uses KV head g = h // (Hq//Hkv).
    ``kv_heads`` restricts the computation to those KV heads (other heads are left NaN)."""
    T, Hq, D = Q.shape
    G = Hq // Hkv
    assert G * Hkv == Hq
    O = np.full((T, Hq, D), np.nan, F64)
    LSE = np.full((T, Hq), np.nan, F64)
    gs = range(Hkv) if kv_heads is None else kv_heads
    for b in range(len(seq_off) - 1):
        t0, t1 = int(seq_off[b]), int(seq_off[b + 1])
        Lq = t1 - t0
        for g in gs:
            Kc, Vc, n_prefix = _visible_kv(blocks_K, blocks_V, sel[b], K_self, V_self, t0, t1, g)
            mask = _mask(Lq, n_prefix, Kc.shape[0] - n_prefix)
            for h in range(g * G, (g + 1) * G):
                q = np.asarray(Q[t0:t1, h, :], dtype=F64)
                s = scale * (q @ Kc.T)                       # F2
                s = np.where(mask, s, -np.inf)
                m = s.max(axis=1, keepdims=True)             # F3
                e = np.exp(s - m)
                l = e.sum(axis=1, keepdims=True)
                LSE[t0:t1, h] = (m + np.log(l))[:, 0]
                p = e / l
                O[t0:t1, h, :] = p @ Vc                      # F4
    return O, LSE


def attn_bwd(Q, blocks_K, blocks_V, sel: Sequence[Sequence[int]], seq_off, K_self, V_self,
             dO, scale: float, Hkv: int, kv_heads: Optional[Sequence[int]] = None,
             grad_K: Optional[Dict[int, np.ndarray]] = None,
             grad_V: Optional[Dict[int, np.ndarray]] = None):
    """B1-B6, recomputing P from the definition.  Returns dQ [T,Hq,D], grad_K, grad_V (dicts
    block id -> [len_s,Hkv,D], only for blocks selected by some sequence; accumulated onto the
    passed-in dicts when given, "+=" semantics), dK_self, dV_self [T,Hkv,D] (overwrite semantics;
    None if K_self is None)."""
    T, Hq, D = Q.shape
    G = Hq // Hkv
    dQ = np.full((T, Hq, D), np.nan, F64)
    grad_K = {} if grad_K is None else grad_K
    grad_V = {} if grad_V is None else grad_V
    gs = list(range(Hkv)) if kv_heads is None else list(kv_heads)
    dKs = dVs = None
    if K_self is not None:
        dKs = np.full(K_self.shape, np.nan, F64)
        dVs = np.full(V_self.shape, np.nan, F64)
        dKs[:, gs, :] = 0.0
        dVs[:, gs, :] = 0.0
    for b in range(len(seq_off) - 1):
        t0, t1 = int(seq_off[b]), int(seq_off[b + 1])
        Lq = t1 - t0
        for s_id in sel[b]:
            if s_id not in grad_K:
                grad_K[s_id] = np.zeros(blocks_K[s_id].shape, F64)
                grad_V[s_id] = np.zeros(blocks_V[s_id].shape, F64)
        for g in gs:
            Kc, Vc, n_prefix = _visible_kv(blocks_K, blocks_V, sel[b], K_self, V_self, t0, t1, g)
            mask = _mask(Lq, n_prefix, Kc.shape[0] - n_prefix)
            dKc = np.zeros_like(Kc)
            dVc = np.zeros_like(Vc)
            for h in range(g * G, (g + 1) * G):
                q = np.asarray(Q[t0:t1, h, :], dtype=F64)
                do = np.asarray(dO[t0:t1, h, :], dtype=F64)
                s = np.where(mask, scale * (q @ Kc.T), -np.inf)
                m = s.max(axis=1, keepdims=True)
                e = np.exp(s - m)
                p = e / e.sum(axis=1, keepdims=True)
                o = p @ Vc
                delta = (do * o).sum(axis=1, keepdims=True)   # B1
                dp = do @ Vc.T                                # B2
                ds = p * (dp - delta)                         # B3 (p = 0 on masked keys)
                dQ[t0:t1, h, :] = scale * (ds @ Kc)           # B4
                dKc += scale * (ds.T @ q)                     # B5/B6 summed over the G heads
                dVc += p.T @ do
            pos = 0
            for s_id in sel[b]:                               # B5: scatter into the block grads
                n = blocks_K[s_id].shape[0]
                grad_K[s_id][:, g, :] += dKc[pos:pos + n]
                grad_V[s_id][:, g, :] += dVc[pos:pos + n]
                pos += n
            if K_self is not None:                            # B6
                dKs[t0:t1, g, :] = dKc[n_prefix:]
                dVs[t0:t1, g, :] = dVc[n_prefix:]
    return dQ, grad_K, grad_V, dKs, dVs


# ----------------------------------------------------------------------------------------------
# bf16 round-to-nearest-even (the cast of the fp32 master copy to the bf16 working copy)
# ----------------------------------------------------------------------------------------------
def bf16_rne_bits(x32: np.ndarray) -> np.ndarray:
    """fp32 -> bf16 bit patterns (uint16), round to nearest even; NaN stays NaN (quiet)."""
    x32 = np.ascontiguousarray(x32, dtype=np.float32)
    u = x32.view(np.uint32).astype(np.uint64)
    lsb = (u >> 16) & 1
    r = ((u + 0x7FFF + lsb) >> 16).astype(np.uint32)
    nan = np.isnan(x32)
    r = np.where(nan, (u >> 16).astype(np.uint32) | 0x40, r)
    return r.astype(np.uint16)


def bf16_rne(x32: np.ndarray) -> np.ndarray:
    """fp32 -> nearest-even bf16 value, returned as fp32."""
    bits = bf16_rne_bits(x32).astype(np.uint32) << 16
    return bits.view(np.float32).reshape(np.shape(x32))


# ----------------------------------------------------------------------------------------------
# Adam (Kingma & Ba 2014, Algorithm 1), per cartridge
# ----------------------------------------------------------------------------------------------
def adam_step(p, m, v, g, t: int, lr: float, beta1: float, beta2: float, eps: float,
              lr_scale: float = 1.0, n_frozen: int = 0):
    """One Adam step on one cartridge tensor ([len,Hkv,D]; K and V are updated separately with
    the same t).  ``t`` is the step count AFTER the increment (t >= 1).  The first ``n_frozen``
    tokens are left untouched (params and moments).  float64 arithmetic on the given values;
    returns (p, m, v) float64.  eps is added outside the square root; no weight decay."""
    p = np.array(p, dtype=F64)
    m = np.array(m, dtype=F64)
    v = np.array(v, dtype=F64)
    g = np.asarray(g, dtype=F64)
    a = slice(n_frozen, None)
    m[a] = beta1 * m[a] + (1.0 - beta1) * g[a]
    v[a] = beta2 * v[a] + (1.0 - beta2) * g[a] * g[a]
    mhat = m[a] / (1.0 - beta1 ** t)
    vhat = v[a] / (1.0 - beta2 ** t)
    p[a] = p[a] - (lr * lr_scale) * mhat / (np.sqrt(vhat) + eps)
    return p, m, v


def cartridge_bytes(n_layers: int, tokens: int, Hkv: int, D: int, bytes_per_el: int = 2) -> int:
    """Exact byte size of a cartridge Z in R^{L x p x d x 2}, d = Hkv*D."""
    return n_layers * tokens * Hkv * D * 2 * bytes_per_el


# ---------------------------------------------------------------------------------------------
# NEXT-1: RoPE with the cartridge position offset
# ---------------------------------------------------------------------------------------------
def rope(X, seq_off, pos_off, base: float, layout: int = 0, inverse: bool = False):
    """Rotary position embedding of the packed tokens X [T, H, D] (RoFormer, Su et al. 2024, cited at
    PAPER.md:77 and :320), with the paper's offset: "query token position IDs must be offset by the total
    number of active cartridge KV tokens, which occupy the prefix of the sequence".

    Token i of sequence b has position id m = pos_off[b] + i (R7: the caller passes either the
    sum of resident cartridge lengths or the visible prefix P_b from cas_position_offsets).  RoFormer
    Eq. 13/34: dimension pair k (k = 0..D/2-1) is rotated by the angle m * theta_k, theta_k = base^(-2k/D):
        [x_a']   [cos  -sin] [x_a]
        [x_b'] = [sin   cos] [x_b]
    layout 0: the pair is (x[2k], x[2k+1]) (RoFormer's interleaved form); layout 1: (x[k], x[k+D/2]) (the
    "rotate-half" storage convention of the Qwen3 checkpoints the paper trains on -- a fixed permutation of
    the dimensions).  inverse=True rotates by -m*theta_k: the transpose, i.e. the backward pass of the map.
    Plain float64 loops over the pairs; no tables, no fusion."""
    X = np.asarray(X, dtype=F64)
    T, H, D = X.shape
    assert D % 2 == 0
    out = np.empty_like(X)
    B = len(seq_off) - 1
    for b in range(B):
        for t in range(int(seq_off[b]), int(seq_off[b + 1])):
            m = float(int(pos_off[b]) + (t - int(seq_off[b])))
            for k in range(D // 2):
                ang = m * (float(base) ** (-2.0 * k / D))
                if inverse:
                    ang = -ang
                c, s = np.cos(ang), np.sin(ang)
                ia, ib = (2 * k, 2 * k + 1) if layout == 0 else (k, k + D // 2)
                xa, xb = X[t, :, ia], X[t, :, ib]
                out[t, :, ia] = xa * c - xb * s
                out[t, :, ib] = xa * s + xb * c
    return out
