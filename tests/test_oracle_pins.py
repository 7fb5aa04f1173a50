"""Pins for oracle/cas_oracle.py (CPU only).  Each test checks the oracle against something that
is NOT the oracle: python-loop brute force, finite differences, closed forms, conservation laws,
torch SDPA/autograd in float64, torch.optim.Adam, torch's bf16 cast, the paper's printed MiB.
SURVEY.md 8(c) P1-P9."""
import math
import os

import numpy as np
import pytest
import torch

from oracle import cas_oracle as orc

HERE = os.path.dirname(os.path.abspath(__file__))


def tiny_problem(seed=0, Hq=4, Hkv=2, D=8, lens=(5, 3, 7, 4), Lqs=(6, 4), sel=((2, 0), (0, 3, 1)),
                 kv_std=0.7, with_self=True):
    rng = np.random.default_rng(seed)
    bK = [rng.normal(0, kv_std, (l, Hkv, D)) for l in lens]
    bV = [rng.normal(0, kv_std, (l, Hkv, D)) for l in lens]
    seq_off = np.concatenate([[0], np.cumsum(Lqs)]).astype(np.int32)
    T = int(seq_off[-1])
    Q = rng.normal(0, 1, (T, Hq, D))
    Ks = rng.normal(0, kv_std, (T, Hkv, D)) if with_self else None
    Vs = rng.normal(0, kv_std, (T, Hkv, D)) if with_self else None
    dO = rng.normal(0, 1, (T, Hq, D))
    return dict(Q=Q, bK=bK, bV=bV, sel=[list(s) for s in sel], seq_off=seq_off, Ks=Ks, Vs=Vs,
                dO=dO, scale=1.0 / math.sqrt(D), Hkv=Hkv)


def run_fwd(p, **kw):
    return orc.attn_fwd(p["Q"], p["bK"], p["bV"], p["sel"], p["seq_off"], p["Ks"], p["Vs"],
                        p["scale"], p["Hkv"], **kw)


def run_bwd(p, **kw):
    return orc.attn_bwd(p["Q"], p["bK"], p["bV"], p["sel"], p["seq_off"], p["Ks"], p["Vs"],
                        p["dO"], p["scale"], p["Hkv"], **kw)


# ---------------------------------------------------------------- P1: brute force, python loops
def brute_force_fwd(p):
    Q = p["Q"]
    T, Hq, D = Q.shape
    G = Hq // p["Hkv"]
    O = np.zeros((T, Hq, D))
    LSE = np.zeros((T, Hq))
    for b in range(len(p["seq_off"]) - 1):
        t0, t1 = int(p["seq_off"][b]), int(p["seq_off"][b + 1])
        for t in range(t0, t1):
            for h in range(Hq):
                g = h // G
                keys, vals = [], []
                for s in p["sel"][b]:
                    for j in range(p["bK"][s].shape[0]):
                        keys.append(p["bK"][s][j, g])
                        vals.append(p["bV"][s][j, g])
                if p["Ks"] is not None:
                    for t2 in range(t0, t + 1):
                        keys.append(p["Ks"][t2, g])
                        vals.append(p["Vs"][t2, g])
                sc = [p["scale"] * sum(Q[t, h, d] * k[d] for d in range(D)) for k in keys]
                mx = max(sc)
                z = sum(math.exp(x - mx) for x in sc)
                LSE[t, h] = mx + math.log(z)
                for j, v in enumerate(vals):
                    w = math.exp(sc[j] - LSE[t, h])
                    for d in range(D):
                        O[t, h, d] += w * v[d]
    return O, LSE


def test_p1_forward_brute_force():
    p = tiny_problem()
    O, LSE = run_fwd(p)
    Ob, Lb = brute_force_fwd(p)
    np.testing.assert_allclose(O, Ob, rtol=1e-12, atol=1e-13)
    np.testing.assert_allclose(LSE, Lb, rtol=1e-12, atol=1e-13)


def test_p1_forward_brute_force_prefix_only_and_empty_selection():
    p = tiny_problem(seed=3, with_self=False)
    O, LSE = run_fwd(p)
    Ob, Lb = brute_force_fwd(p)
    np.testing.assert_allclose(O, Ob, rtol=1e-12, atol=1e-13)
    p = tiny_problem(seed=4, sel=((), (1,)))          # sequence 0 = plain causal attention
    O, LSE = run_fwd(p)
    Ob, Lb = brute_force_fwd(p)
    np.testing.assert_allclose(O, Ob, rtol=1e-12, atol=1e-13)
    np.testing.assert_allclose(LSE, Lb, rtol=1e-12, atol=1e-13)


# ---------------------------------------------------------------- P2: finite differences
def loss(p):
    O, _ = run_fwd(p)
    return float((O * p["dO"]).sum())


def test_p2_backward_finite_differences():
    p = tiny_problem(seed=1)
    dQ, gK, gV, dKs, dVs = run_bwd(p)
    rng = np.random.default_rng(7)
    h = 1e-5

    def fd(arr, idx):
        old = arr[idx]
        arr[idx] = old + h
        lp = loss(p)
        arr[idx] = old - h
        lm = loss(p)
        arr[idx] = old
        return (lp - lm) / (2 * h)

    for _ in range(12):
        idx = tuple(rng.integers(0, n) for n in p["Q"].shape)
        assert abs(fd(p["Q"], idx) - dQ[idx]) < 1e-7
        idx = tuple(rng.integers(0, n) for n in p["Ks"].shape)
        assert abs(fd(p["Ks"], idx) - dKs[idx]) < 1e-7
        assert abs(fd(p["Vs"], idx) - dVs[idx]) < 1e-7
    for s in range(len(p["bK"])):
        for _ in range(6):
            idx = tuple(rng.integers(0, n) for n in p["bK"][s].shape)
            assert abs(fd(p["bK"][s], idx) - gK[s][idx]) < 1e-7      # block 0 is shared by 2 seqs
            assert abs(fd(p["bV"][s], idx) - gV[s][idx]) < 1e-7


# ---------------------------------------------------------------- P3: invariants of north_star
def test_p3_order_invariance():
    p = tiny_problem(seed=2)
    O1, L1 = run_fwd(p)
    p2 = dict(p)
    p2["sel"] = [list(reversed(s)) for s in p["sel"]]
    O2, L2 = run_fwd(p2)
    np.testing.assert_allclose(O1, O2, rtol=1e-12, atol=1e-14)
    np.testing.assert_allclose(L1, L2, rtol=1e-12, atol=1e-14)


def test_p3_unselected_blocks_get_no_gradient():
    p = tiny_problem(seed=5, sel=((2,), (2, 3)))
    _, gK, gV, _, _ = run_bwd(p)
    assert set(gK.keys()) == {2, 3} and set(gV.keys()) == {2, 3}
    pre = {s: np.zeros_like(p["bK"][s]) for s in range(4)}
    prev = {s: np.zeros_like(p["bV"][s]) for s in range(4)}
    _, gK2, gV2, _, _ = run_bwd(p, grad_K=pre, grad_V=prev)
    for s in (0, 1):
        assert not gK2[s].any() and not gV2[s].any()      # exact zero


def test_p3_shared_block_gradient_is_sum_of_per_sequence_gradients():
    p = tiny_problem(seed=6)                                # block 0 selected by both sequences
    _, gK, gV, _, _ = run_bwd(p)
    tot_K = np.zeros_like(gK[0])
    tot_V = np.zeros_like(gV[0])
    for b in range(2):
        t0, t1 = int(p["seq_off"][b]), int(p["seq_off"][b + 1])
        q = dict(p)
        q["Q"], q["dO"] = p["Q"][t0:t1], p["dO"][t0:t1]
        q["Ks"], q["Vs"] = p["Ks"][t0:t1], p["Vs"][t0:t1]
        q["sel"] = [p["sel"][b]]
        q["seq_off"] = np.array([0, t1 - t0])
        _, gk, gv, _, _ = run_bwd(q)
        tot_K += gk[0]
        tot_V += gv[0]
    np.testing.assert_allclose(gK[0], tot_K, rtol=1e-12, atol=1e-14)
    np.testing.assert_allclose(gV[0], tot_V, rtol=1e-12, atol=1e-14)


def test_p3_accumulate_semantics():
    p = tiny_problem(seed=8)
    _, gK, gV, _, _ = run_bwd(p)
    pre = {s: np.full(p["bK"][s].shape, 0.25) for s in range(4)}
    prev = {s: np.full(p["bV"][s].shape, -0.5) for s in range(4)}
    _, gK2, gV2, _, _ = run_bwd(p, grad_K=pre, grad_V=prev)
    for s in gK:
        np.testing.assert_allclose(gK2[s], gK[s] + 0.25, rtol=1e-13)
        np.testing.assert_allclose(gV2[s], gV[s] - 0.5, rtol=1e-13)


# ---------------------------------------------------------------- P4: torch SDPA + autograd, fp64
def sdpa_reference(p):
    """Explicit concat + boolean mask per sequence, torch SDPA float64 with autograd; dK/dV are
    scattered back to the blocks by hand."""
    Hkv = p["Hkv"]
    Q = torch.tensor(p["Q"], dtype=torch.float64, requires_grad=True)
    bK = [torch.tensor(x, dtype=torch.float64, requires_grad=True) for x in p["bK"]]
    bV = [torch.tensor(x, dtype=torch.float64, requires_grad=True) for x in p["bV"]]
    Ks = torch.tensor(p["Ks"], dtype=torch.float64, requires_grad=True)
    Vs = torch.tensor(p["Vs"], dtype=torch.float64, requires_grad=True)
    T, Hq, D = Q.shape
    G = Hq // Hkv
    outs = []
    for b in range(len(p["seq_off"]) - 1):
        t0, t1 = int(p["seq_off"][b]), int(p["seq_off"][b + 1])
        Lq = t1 - t0
        Kc = torch.cat([bK[s] for s in p["sel"][b]] + [Ks[t0:t1]], 0)     # [Nk,Hkv,D]
        Vc = torch.cat([bV[s] for s in p["sel"][b]] + [Vs[t0:t1]], 0)
        npre = Kc.shape[0] - Lq
        mask = torch.ones(Lq, Kc.shape[0], dtype=torch.bool)
        mask[:, npre:] = torch.tril(torch.ones(Lq, Lq, dtype=torch.bool))
        q = Q[t0:t1].permute(1, 0, 2)[None]                               # [1,Hq,Lq,D]
        k = Kc.permute(1, 0, 2).repeat_interleave(G, 0)[None]
        v = Vc.permute(1, 0, 2).repeat_interleave(G, 0)[None]
        o = torch.nn.functional.scaled_dot_product_attention(q, k, v, attn_mask=mask,
                                                             scale=p["scale"])
        outs.append(o[0].permute(1, 0, 2))
    O = torch.cat(outs, 0)
    (O * torch.tensor(p["dO"], dtype=torch.float64)).sum().backward()
    z = lambda t: np.zeros(t.shape) if t.grad is None else t.grad.numpy()
    return O.detach().numpy(), Q.grad.numpy(), [z(x) for x in bK], [z(x) for x in bV], \
        Ks.grad.numpy(), Vs.grad.numpy()


@pytest.mark.parametrize("seed,Hq,Hkv,D", [(11, 6, 2, 16), (12, 4, 4, 8), (13, 8, 1, 32)])
def test_p4_matches_torch_sdpa_autograd(seed, Hq, Hkv, D):
    p = tiny_problem(seed=seed, Hq=Hq, Hkv=Hkv, D=D, lens=(9, 17, 5, 12, 8), Lqs=(13, 7, 21),
                     sel=((4, 0, 2), (1,), (2, 3, 0, 1)))
    O, _ = run_fwd(p)
    dQ, gK, gV, dKs, dVs = run_bwd(p)
    Or, dQr, gKr, gVr, dKsr, dVsr = sdpa_reference(p)
    np.testing.assert_allclose(O, Or, rtol=1e-10, atol=1e-12)
    np.testing.assert_allclose(dQ, dQr, rtol=1e-9, atol=1e-11)
    np.testing.assert_allclose(dKs, dKsr, rtol=1e-9, atol=1e-11)
    np.testing.assert_allclose(dVs, dVsr, rtol=1e-9, atol=1e-11)
    for s in range(5):
        np.testing.assert_allclose(gK[s], gKr[s], rtol=1e-9, atol=1e-11)
        np.testing.assert_allclose(gV[s], gVr[s], rtol=1e-9, atol=1e-11)


# ---------------------------------------------------------------- P5: closed forms
def test_p5_zero_keys_uniform_softmax():
    p = tiny_problem(seed=20)
    for k in p["bK"]:
        k[:] = 0
    p["Ks"][:] = 0
    O, LSE = run_fwd(p)
    dQ, *_ = run_bwd(p)
    G = p["Q"].shape[1] // p["Hkv"]
    for b in range(2):
        t0, t1 = int(p["seq_off"][b]), int(p["seq_off"][b + 1])
        Pb = sum(p["bK"][s].shape[0] for s in p["sel"][b])
        for i in range(t1 - t0):
            n = Pb + i + 1
            np.testing.assert_allclose(LSE[t0 + i], math.log(n), rtol=1e-13)
            for h in range(p["Q"].shape[1]):
                g = h // G
                vis = np.concatenate([p["bV"][s][:, g] for s in p["sel"][b]] +
                                     [p["Vs"][t0:t0 + i + 1, g]], 0)
                np.testing.assert_allclose(O[t0 + i, h], vis.mean(0), rtol=1e-12, atol=1e-14)
    np.testing.assert_allclose(dQ, 0, atol=1e-15)


def test_p5_constant_values_kill_dq_dk():
    p = tiny_problem(seed=21)
    c = np.linspace(-1, 1, p["Q"].shape[2])
    for v in p["bV"]:
        v[:] = c
    p["Vs"][:] = c
    dQ, gK, gV, dKs, dVs = run_bwd(p)
    np.testing.assert_allclose(dQ, 0, atol=1e-13)
    np.testing.assert_allclose(dKs, 0, atol=1e-13)
    for s in gK:
        np.testing.assert_allclose(gK[s], 0, atol=1e-13)


# ---------------------------------------------------------------- P6: conservation
def test_p6_dv_conservation_and_row_sums():
    p = tiny_problem(seed=22)
    dQ, gK, gV, dKs, dVs = run_bwd(p)
    Hq = p["Q"].shape[1]
    G = Hq // p["Hkv"]
    # rows of P sum to 1  =>  sum over all visible keys of dV  =  sum_i dO_i  (per kv head group)
    tot_dV = sum(g.sum(0) for g in gV.values()) + dVs.sum(0)               # [Hkv, D]
    tot_dO = p["dO"].sum(0).reshape(p["Hkv"], G, -1).sum(1)
    np.testing.assert_allclose(tot_dV, tot_dO, rtol=1e-12, atol=1e-13)
    # sum_j ds_j = 0 per row  =>  with all keys equal to one vector u, dQ = scale*(sum_j ds_j) u = 0
    u = np.random.default_rng(0).normal(size=p["Q"].shape[2])
    for k in p["bK"]:
        k[:] = u
    p["Ks"][:] = u
    dQ2, *_ = run_bwd(p)
    np.testing.assert_allclose(dQ2, 0, atol=1e-13)


def test_single_block_reduces_to_plain_prefix_attention():
    """One selected cartridge == ordinary attention over [prefix ; causal self] (north_star)."""
    p = tiny_problem(seed=23, sel=((1,), (1,)), Lqs=(5, 5))
    O, _ = run_fwd(p)
    Q = torch.tensor(p["Q"])
    G = Q.shape[1] // p["Hkv"]
    for b in range(2):
        t0 = 5 * b
        K = torch.cat([torch.tensor(p["bK"][1]), torch.tensor(p["Ks"][t0:t0 + 5])], 0)
        V = torch.cat([torch.tensor(p["bV"][1]), torch.tensor(p["Vs"][t0:t0 + 5])], 0)
        n = p["bK"][1].shape[0]
        for h in range(Q.shape[1]):
            s = p["scale"] * Q[t0:t0 + 5, h] @ K[:, h // G].T
            s[:, n:] = s[:, n:].masked_fill(~torch.tril(torch.ones(5, 5, dtype=torch.bool)),
                                            float("-inf"))
            o = torch.softmax(s, -1) @ V[:, h // G]
            np.testing.assert_allclose(O[t0:t0 + 5, h], o.numpy(), rtol=1e-12, atol=1e-14)


def test_kv_head_subset_matches_full():
    p = tiny_problem(seed=24)
    O, LSE = run_fwd(p)
    O1, L1 = run_fwd(p, kv_heads=[1])
    np.testing.assert_array_equal(O1[:, 2:], O[:, 2:])
    assert np.isnan(O1[:, :2]).all()
    dQ, gK, gV, dKs, dVs = run_bwd(p)
    dQ1, gK1, gV1, dKs1, dVs1 = run_bwd(p, kv_heads=[1])
    np.testing.assert_array_equal(dQ1[:, 2:], dQ[:, 2:])
    for s in gK:
        np.testing.assert_array_equal(gK1[s][:, 1], gK[s][:, 1])
        assert not gK1[s][:, 0].any()


# ---------------------------------------------------------------- P7: Adam
def test_p7_adam_first_step_closed_form():
    rng = np.random.default_rng(0)
    g = rng.normal(size=(6, 2, 4))
    p0 = rng.normal(size=(6, 2, 4))
    lr, eps = 1e-3, 1e-8
    p, m, v = orc.adam_step(p0, np.zeros_like(p0), np.zeros_like(p0), g, 1, lr, 0.9, 0.999, eps)
    np.testing.assert_allclose(p, p0 - lr * g / (np.abs(g) + eps), rtol=1e-12)
    np.testing.assert_allclose(m, 0.1 * g, rtol=1e-12)
    np.testing.assert_allclose(v, 0.001 * g * g, rtol=1e-12)


def test_p7_adam_constant_gradient_closed_form():
    g = np.array([[[0.3, -2.0, 1e-3]]])
    p = np.zeros_like(g)
    m = np.zeros_like(g)
    v = np.zeros_like(g)
    lr, eps = 1e-2, 1e-8
    for t in range(1, 8):
        p, m, v = orc.adam_step(p, m, v, g, t, lr, 0.9, 0.999, eps)
        np.testing.assert_allclose(p, -t * lr * g / (np.abs(g) + eps), rtol=1e-10)


def test_p7_adam_zero_state_zero_grad_is_noop_and_frozen_tokens():
    rng = np.random.default_rng(1)
    p0 = rng.normal(size=(5, 1, 3))
    z = np.zeros_like(p0)
    p, m, v = orc.adam_step(p0, z, z, z, 1, 1e-3, 0.9, 0.999, 1e-8)
    assert np.array_equal(p, p0) and not m.any() and not v.any()
    g = rng.normal(size=p0.shape)
    p, m, v = orc.adam_step(p0, z, z, g, 1, 1e-3, 0.9, 0.999, 1e-8, n_frozen=2)
    assert np.array_equal(p[:2], p0[:2]) and not m[:2].any() and not v[:2].any()
    assert (p[2:] != p0[2:]).all()


def test_p7_adam_matches_torch_optim():
    rng = np.random.default_rng(2)
    p0 = rng.normal(size=(7, 2, 5))
    w = torch.tensor(p0, dtype=torch.float64, requires_grad=True)
    opt = torch.optim.Adam([w], lr=3e-3, betas=(0.9, 0.999), eps=1e-8, foreach=False)
    p, m, v = p0, np.zeros_like(p0), np.zeros_like(p0)
    for t in range(1, 6):
        g = rng.normal(size=p0.shape)
        w.grad = torch.tensor(g)
        opt.step()
        p, m, v = orc.adam_step(p, m, v, g, t, 3e-3, 0.9, 0.999, 1e-8)
        np.testing.assert_allclose(p, w.detach().numpy(), rtol=1e-11, atol=1e-13)
    # lr_scale multiplies the learning rate (PAPER.md:85 eta_eff = eta_t * min(1, s/W_c))
    pa, _, _ = orc.adam_step(p0, m, v, g, 3, 1e-3, 0.9, 0.999, 1e-8, lr_scale=0.25)
    pb, _, _ = orc.adam_step(p0, m, v, g, 3, 0.25e-3, 0.9, 0.999, 1e-8)
    np.testing.assert_allclose(pa, pb, rtol=1e-14)


# ---------------------------------------------------------------- P8: bf16 RNE vs torch
def test_p8_bf16_rne_matches_torch():
    rng = np.random.default_rng(3)
    x = np.concatenate([
        rng.normal(size=100000).astype(np.float32),
        (rng.normal(size=10000) * 1e-30).astype(np.float32),
        (rng.normal(size=10000) * 1e30).astype(np.float32),
        np.array([0.0, -0.0, 1.0, 1.00390625, 1.001953125, 1.005859375, np.inf, -np.inf,
                  3.3895314e38, 1e-45], dtype=np.float32),      # ties, overflow to inf, denormal
    ])
    want = torch.from_numpy(x).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
    got = orc.bf16_rne_bits(x)
    np.testing.assert_array_equal(got, want)
    np.testing.assert_array_equal(orc.bf16_rne(x),
                                  torch.from_numpy(x).to(torch.bfloat16).float().numpy())


# ---------------------------------------------------------------- P9: paper's printed sizes
def test_p9_cartridge_bytes_vs_paper():
    rows = [l.split() for l in open(os.path.join(HERE, "golden", "paper_kv_footprint.txt"))
            if l.strip() and not l.startswith("#")]
    assert len(rows) == 3
    for name, L, Hkv, D, tok, mib in rows:
        got = orc.cartridge_bytes(int(L), int(tok), int(Hkv), int(D)) / 2 ** 20
        assert abs(got - float(mib)) < 1.0, (name, got)          # paper prints "~" integers
    # "x4 with gradients and Adam moments": ~551 MiB printed, exact 562.5 (2% off)
    four = 4 * orc.cartridge_bytes(36, 1000, 8, 128) / 2 ** 20
    assert abs(four - 551) / 551 < 0.03


# ---------------------------------------------------------------------------------------------
# NEXT-1: RoPE with the cartridge offset (oracle.rope) -- pinned by an independent complex-number
# formulation, the closed form at D = 2, and the properties RoFormer proves
# ---------------------------------------------------------------------------------------------
def _rope_inputs(seed=5, T=11, H=3, D=8):
    rng = np.random.default_rng(seed)
    return rng.standard_normal((T, H, D)), np.array([0, 4, 11]), np.array([7, 130])


@pytest.mark.parametrize("layout", [0, 1])
def test_rope_equals_complex_multiplication(layout):
    # RoFormer Eq. 12: f(x, m) = x * e^{i m theta} on the complexified pairs -- a different formulation
    X, so, po = _rope_inputs()
    T, H, D = X.shape
    base = 10000.0
    got = orc.rope(X, so, po, base, layout)
    k = np.arange(D // 2)
    theta = base ** (-2.0 * k / D)
    pos = np.concatenate([po[b] + np.arange(so[b + 1] - so[b]) for b in range(2)]).astype(np.float64)
    z = (X[:, :, 0::2] + 1j * X[:, :, 1::2]) if layout == 0 else (X[:, :, :D // 2] + 1j * X[:, :, D // 2:])
    w = z * np.exp(1j * pos[:, None, None] * theta[None, None, :])
    want = np.empty_like(X)
    if layout == 0:
        want[:, :, 0::2], want[:, :, 1::2] = w.real, w.imag
    else:
        want[:, :, :D // 2], want[:, :, D // 2:] = w.real, w.imag
    np.testing.assert_allclose(got, want, rtol=0, atol=1e-12)


def test_rope_closed_form_d2_and_offset():
    # D = 2: theta_0 = 1, so token i of a sequence with offset P is rotated by exactly (P + i) radians
    X = np.array([[[1.0, 0.0]], [[0.0, 2.0]]])
    got = orc.rope(X, np.array([0, 2]), np.array([3]), 10000.0, 0)
    np.testing.assert_allclose(got[0, 0], [np.cos(3.0), np.sin(3.0)], atol=1e-15)
    np.testing.assert_allclose(got[1, 0], [-2 * np.sin(4.0), 2 * np.cos(4.0)], atol=1e-15)


@pytest.mark.parametrize("layout", [0, 1])
def test_rope_properties(layout):
    X, so, po = _rope_inputs(seed=6)
    base = 1.0e6
    Y = orc.rope(X, so, po, base, layout)
    # rotation: norms of every (token, head) row are preserved; position 0 is the identity
    np.testing.assert_allclose(np.linalg.norm(Y, axis=-1), np.linalg.norm(X, axis=-1), rtol=1e-13)
    np.testing.assert_allclose(orc.rope(X[:1], np.array([0, 1]), np.array([0]), base, layout), X[:1], atol=0)
    # inverse = transpose: undoes the map, and <rope(x), y> = <x, rope^T(y)>
    np.testing.assert_allclose(orc.rope(Y, so, po, base, layout, inverse=True), X, atol=1e-12)
    Z = np.random.default_rng(9).standard_normal(X.shape)
    np.testing.assert_allclose(np.sum(Y * Z), np.sum(X * orc.rope(Z, so, po, base, layout, inverse=True)), rtol=1e-12)
    # relative-position property (RoFormer Eq. 11): <f(q,m), f(k,n)> depends on m - n only, so shifting
    # every offset by the same number of cartridge tokens leaves all q.k scores of a sequence unchanged
    Y2 = orc.rope(X, so, po + 512, base, layout)
    s1 = np.einsum("thd,uhd->htu", Y[:4], Y[:4])
    s2 = np.einsum("thd,uhd->htu", Y2[:4], Y2[:4])
    np.testing.assert_allclose(s1, s2, atol=1e-9)
    # the two layouts are the same map up to the fixed permutation of dimensions
    D = X.shape[-1]
    perm = np.concatenate([np.arange(0, D, 2), np.arange(1, D, 2)])      # interleaved -> half-split
    np.testing.assert_allclose(orc.rope(X, so, po, base, 0)[:, :, perm], orc.rope(X[:, :, perm], so, po, base, 1),
                               atol=1e-12)
