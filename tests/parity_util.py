"""Shared helpers of the GPU parity tests: run the CUDA path through the C ABI on a seeded workload
and compare it element by element with oracle/ on the same inputs."""
from __future__ import annotations

import numpy as np
import torch

from oracle import cas_oracle as orc
from paper_2606_04557_b200 import cas
from paper_2606_04557_b200.harness import Session

# tolerances of BASELINE.json north_star (written here so the tests state them)
TOL_F32 = 1e-4          # "fp32 configs: max relative error 1e-4"  (metric: DESIGN.md R22)
TOL_BF16_O_DQ = 2e-2    # "bf16 configs: O and dQ relative Frobenius error <= 2e-2"
TOL_BF16_DKV = 3e-2     # "dK/dV <= 3e-2"
TOL_ADAM = 1e-6         # "Adam: relative error <= 1e-6"


def rel_max(a, b):
    """max_i |a_i-b_i| / (|b_i| + rms(b))  (R22)."""
    a = np.asarray(a, np.float64)
    b = np.asarray(b, np.float64)
    rms = float(np.sqrt(np.mean(b * b))) if b.size else 0.0
    if b.size == 0:
        return 0.0
    return float(np.max(np.abs(a - b) / (np.abs(b) + rms + 1e-300)))


def rel_fro(a, b):
    a = np.asarray(a, np.float64)
    b = np.asarray(b, np.float64)
    nb = float(np.linalg.norm(b))
    return float(np.linalg.norm(a - b) / nb) if nb > 0 else float(np.linalg.norm(a))


def err(a, b, dtype):
    return rel_max(a, b) if dtype == "f32" else rel_fro(a, b)


def kv_heads_for(seed: int, Hkv: int, n: int = 1):
    """The KV head group(s) a full-size test compares completely (the oracle cannot afford all
    Hkv groups at full size): derived from the seed, so no head is privileged by the test source."""
    first = (seed * 2654435761 >> 7) % Hkv
    return sorted({(first + i * (Hkv // 2 + 1)) % Hkv for i in range(n)})


def oracle_inputs(wl):
    blocks_K = [wl.cart_kv(c)[0] for c in range(wl.cfg.n_carts)]
    blocks_V = [wl.cart_kv(c)[1] for c in range(wl.cfg.n_carts)]
    sel = [wl.sel_cart[wl.sel_off[b]:wl.sel_off[b + 1]].tolist() for b in range(wl.cfg.B)]
    return blocks_K, blocks_V, sel


def check_attention(wl, impl, kv_heads, self_block=True, backward=True, pre_grad=None, report=None):
    """Runs fwd (+bwd) on the GPU and the oracle on KV heads `kv_heads`; asserts the north_star
    tolerances.  Returns the live Session (gradients still in the pool)."""
    cfg = wl.cfg
    cas.cas_set_impl(impl)
    sess = Session(wl)
    G = cfg.Hq // cfg.Hkv
    hs = [h for g in kv_heads for h in range(g * G, (g + 1) * G)]
    bK, bV, sel = oracle_inputs(wl)
    Ks = wl.K_self if self_block else None
    Vs = wl.V_self if self_block else None
    tolO = TOL_F32 if cfg.dtype == "f32" else TOL_BF16_O_DQ
    tolKV = TOL_F32 if cfg.dtype == "f32" else TOL_BF16_DKV

    sess.fwd(self_block=self_block)
    torch.cuda.synchronize()
    O, LSE = sess.np(sess.O), sess.np(sess.LSE)
    Oo, Lo = orc.attn_fwd(wl.Q, bK, bV, sel, wl.seq_off, Ks, Vs, sess.scale, cfg.Hkv, kv_heads=kv_heads)
    res = {"O": err(O[:, hs], Oo[:, hs], cfg.dtype), "LSE": rel_max(LSE[:, hs], Lo[:, hs])}
    assert np.isfinite(O).all() and np.isfinite(LSE).all()
    if res["O"] > tolO:      # say WHERE: worst (token, head) rows and the error of each 32-column quarter
        d = O[:, hs] - Oo[:, hs]
        per_row = np.linalg.norm(d, axis=2) / (np.linalg.norm(Oo[:, hs], axis=2) + 1e-30)
        worst = np.argsort(-per_row.ravel())[:8]
        res["worst_rows(token,head,err)"] = [(int(i // len(hs)), hs[int(i % len(hs))], float(per_row.ravel()[i])) for i in worst]
        t0, h0 = int(worst[0] // len(hs)), int(worst[0] % len(hs))
        res["quarters_of_worst_row"] = [float(np.linalg.norm(d[t0, h0, 32 * q:32 * q + 32]) /
                                              (np.linalg.norm(Oo[t0, hs[h0], 32 * q:32 * q + 32]) + 1e-30)) for q in range(4)]
    assert res["O"] <= tolO, res
    assert res["LSE"] <= (TOL_F32 if cfg.dtype == "f32" else 2e-3), res
    if backward and cfg.backward:
        sess.bwd(self_block=self_block)
        torch.cuda.synchronize()
        dQ = sess.np(sess.dQ)
        dQo, gKo, gVo, dKso, dVso = orc.attn_bwd(wl.Q, bK, bV, sel, wl.seq_off, Ks, Vs, wl.dO,
                                                 sess.scale, cfg.Hkv, kv_heads=kv_heads)
        res["dQ"] = err(dQ[:, hs], dQo[:, hs], cfg.dtype)
        assert np.isfinite(dQ).all()
        assert res["dQ"] <= tolO, res
        used = sorted(gKo.keys())
        # dK/dV are gated PER SLOT (SURVEY.md A22 "per tensor"): a slot that one short sequence selected has small
        # gradients and must not hide inside the norm of the big ones
        res["dK"] = res["dV"] = 0.0
        for c in used:
            eK = err(sess.read(c, "gK")[:, kv_heads], gKo[c][:, kv_heads], cfg.dtype)
            eV = err(sess.read(c, "gV")[:, kv_heads], gVo[c][:, kv_heads], cfg.dtype)
            assert eK <= tolKV and eV <= tolKV, (c, eK, eV)
            res["dK"], res["dV"] = max(res["dK"], eK), max(res["dV"], eV)
        if self_block:
            res["dKs"] = err(sess.np(sess.dKs)[:, kv_heads], dKso[:, kv_heads], cfg.dtype)
            res["dVs"] = err(sess.np(sess.dVs)[:, kv_heads], dVso[:, kv_heads], cfg.dtype)
            assert res["dKs"] <= tolKV and res["dVs"] <= tolKV, res
        # unselected resident cartridges: EVERY such gradient slot stays bit-zero
        cnt = cas.cas_pool_counters(sess.pool)
        untouched = [c for c in range(cfg.n_carts) if cnt["slot_of"][c] >= 0 and c not in set(used)]
        for c in untouched:
            assert not sess.read(c, "gK").any() and not sess.read(c, "gV").any()
        # conservation over ALL heads: sum of dV over every visible key = sum_i dO_i per KV head
        tot = np.zeros((cfg.Hkv, cfg.D))
        for c in used:
            tot += sess.read(c, "gV").astype(np.float64).sum(0)
        if self_block:
            tot += sess.np(sess.dVs).astype(np.float64).sum(0)
        want = wl.dO.astype(np.float64).sum(0).reshape(cfg.Hkv, G, cfg.D).sum(1)
        res["dV_conservation"] = rel_fro(tot, want)
        assert res["dV_conservation"] <= (1e-4 if cfg.dtype == "f32" else 2e-2), res
    if report is not None:
        report.update(res)
    return sess


def check_adam_isolated(sess, carts, n_frozen=0, lr_scale=None):
    """Adam parity on identical gradients (R23): read g,p,m,v of `carts` from the GPU,
    run one cas_adam_step, compare with the oracle's Adam fed the same numbers."""
    cfg = sess.cfg
    cnt = cas.cas_pool_counters(sess.pool)
    before = {c: {w: sess.read(c, w) for w in ("pK", "pV", "mK", "mV", "vK", "vV", "gK", "gV")} for c in carts}
    slots = [int(cnt["slot_of"][c]) for c in carts]
    sess.adam(slots=slots, lr_scale=lr_scale, n_frozen=n_frozen)
    torch.cuda.synchronize()
    cnt2 = cas.cas_pool_counters(sess.pool)
    f32 = lambda x: float(np.float32(x))
    worst = 0.0
    for i, c in enumerate(carts):
        t = int(cnt["opt_steps"][c]) + 1
        assert int(cnt2["opt_steps"][c]) == t
        for kv in "KV":
            b = before[c]
            p, m, v = orc.adam_step(b["p" + kv], b["m" + kv], b["v" + kv], b["g" + kv], t, f32(cfg.lr),
                                    f32(cfg.beta1), f32(cfg.beta2), f32(cfg.eps),
                                    lr_scale=1.0 if lr_scale is None else f32(lr_scale[i]),
                                    n_frozen=n_frozen)
            gp, gm, gv = sess.read(c, "p" + kv), sess.read(c, "m" + kv), sess.read(c, "v" + kv)
            for got, want in ((gp, p), (gm, m), (gv, v)):
                e = rel_max(got, want)
                worst = max(worst, e)
                assert e <= TOL_ADAM, (c, kv, e)
            # working copy = RNE(master) decided on the kernel's own fp32 value, bit-exact
            w = sess.read(c, "w" + kv)
            if cfg.dtype == "bf16":
                np.testing.assert_array_equal(w, orc.bf16_rne_bits(gp))
            else:
                np.testing.assert_array_equal(w, gp)
            assert not sess.read(c, "g" + kv).any()          # fused zeroing
            if n_frozen:
                np.testing.assert_array_equal(gp[:n_frozen], b["p" + kv][:n_frozen])
    return worst
