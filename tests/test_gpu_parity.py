"""GPU parity: the CUDA path (through the C ABI) against oracle/ on the same seeded inputs.
Small cases compare every output element; full-size configs compare every output element of one KV
head group (the oracle computes that group completely) plus properties over all heads."""
import numpy as np
import pytest
import torch

from paper_2606_04557_b200 import _build, cas
from paper_2606_04557_b200.harness import Session
from workloads import CONFIGS, make_workload

from oracle import cas_oracle as orc
from parity_util import (TOL_BF16_DKV, TOL_BF16_O_DQ, check_adam_isolated, check_attention, kv_heads_for,
                         rel_fro)

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def built():
    _build.build()
    yield
    cas.cas_set_impl(cas.CAS_IMPL_AUTO)


def small_ragged(dtype="bf16", D=128, seed=5):
    """config-4-shaped (lognormal lengths, proportional draws, ragged Lq) at oracle-friendly size:
    lengths span 1..6 KV tiles with ragged tails, query lengths span 1..4 Q tiles."""
    return CONFIGS["c4"].scaled(name="c4_small", dtype=dtype, Hq=8, Hkv=2, D=D, n_carts=12, n_slots=12,
                                B=5, len_mu=5.3, len_sigma=0.8, len_min=17, len_max=700, lq_min=3,
                                lq_max=450, n_dist_max=6), seed


# ------------------------------------------------------------------ config 1 (tiny fp32), complete
def test_c1_tiny_fp32_full_parity_and_adam():
    wl = make_workload(CONFIGS["c1"])
    rep = {}
    sess = check_attention(wl, cas.CAS_IMPL_AUTO, kv_heads=[0], report=rep)
    used = sorted(set(wl.sel_cart.tolist()))
    worst = check_adam_isolated(sess, used)
    print("c1", rep, "adam", worst)
    sess.close()


def test_c1_prefix_only_and_accumulate():
    wl = make_workload(CONFIGS["c1"], seed=11)
    sess = check_attention(wl, cas.CAS_IMPL_AUTO, kv_heads=[0], self_block=False)
    # second backward accumulates (+=): gradients double
    c = int(wl.sel_cart[0])
    g1 = sess.read(c, "gK").copy()
    sess.bwd(self_block=False)
    torch.cuda.synchronize()
    np.testing.assert_allclose(sess.read(c, "gK"), 2 * g1, rtol=1e-6, atol=1e-9)
    sess.close()


def test_sequence_without_cartridges_is_plain_causal_attention():
    wl = make_workload(CONFIGS["c1"], seed=12)
    n0 = int(wl.sel_off[1])
    wl.sel_cart = wl.sel_cart[n0:].copy()
    wl.sel_off = np.array([0, 0, len(wl.sel_cart)], dtype=np.int32)
    check_attention(wl, cas.CAS_IMPL_AUTO, kv_heads=[0]).close()


def test_adam_frozen_tokens_lr_scale_and_second_step():
    wl = make_workload(CONFIGS["c1"], seed=13)
    sess = check_attention(wl, cas.CAS_IMPL_AUTO, kv_heads=[0])
    used = sorted(set(wl.sel_cart.tolist()))
    check_adam_isolated(sess, used, n_frozen=1, lr_scale=[0.25 * (i + 1) for i in range(len(used))])
    sess.bwd()                                  # new gradients, t = 2 (bias correction changes)
    torch.cuda.synchronize()
    check_adam_isolated(sess, used)
    # a resident cartridge nobody selected: g = 0, m = v = 0  ->  exact no-op (R10)
    rest = [c for c in range(4) if c not in used]
    for c in rest:
        p0 = sess.read(c, "pK").copy()
        check_adam_isolated(sess, [c])
        np.testing.assert_array_equal(sess.read(c, "pK"), p0)
    sess.close()


# ------------------------------------------------------------------ small ragged cases, complete
@pytest.mark.parametrize("impl", [cas.CAS_IMPL_SIMT, cas.CAS_IMPL_AUTO])
@pytest.mark.parametrize("dtype,D", [("bf16", 128), ("f32", 64), ("bf16", 64)])
def test_small_ragged_all_heads(impl, dtype, D):
    cfg, seed = small_ragged(dtype, D)
    wl = make_workload(cfg, seed)
    rep = {}
    sess = check_attention(wl, impl, kv_heads=[0, 1], report=rep)
    print(dtype, D, impl, rep)
    check_adam_isolated(sess, sorted(set(wl.sel_cart.tolist()))[:3])
    sess.close()


@pytest.mark.parametrize("impl", [cas.CAS_IMPL_SIMT, cas.CAS_IMPL_AUTO])
def test_small_c2_shape(impl):
    cfg = CONFIGS["c2"].scaled(name="c2_small", n_carts=12, n_slots=12, cart_len=320, B=3, Lq=384, n_dist=3)
    wl = make_workload(cfg, 21)
    rep = {}
    check_attention(wl, impl, kv_heads=[0, 5], report=rep).close()
    print(rep)


@pytest.mark.parametrize("impl", [cas.CAS_IMPL_SIMT, cas.CAS_IMPL_AUTO])
def test_small_decode_shape(impl):
    cfg = CONFIGS["c5_top8"].scaled(name="c5_small", n_carts=20, n_slots=20, cart_len=200, B=9, n_dist=4)
    wl = make_workload(cfg, 22)
    check_attention(wl, impl, kv_heads=[0, 3, 7]).close()
    cfg = CONFIGS["c5_all"].scaled(name="c5_small_all", n_carts=6, n_slots=6, cart_len=130, B=3)
    check_attention(make_workload(cfg, 23), impl, kv_heads=[1]).close()
    # more sequences than one 128-row block (128/G = 32 sequences), several KV chunks per group (split-KV
    # partials + combine), a ragged last tile, and the prefix-only call (no self key)
    cfg = CONFIGS["c5_all"].scaled(name="c5_small_rows", n_carts=5, n_slots=5, cart_len=300, B=40)
    check_attention(make_workload(cfg, 24), impl, kv_heads=[0, 6]).close()
    check_attention(make_workload(cfg, 25), impl, kv_heads=[2], self_block=False).close()


# ------------------------------------------------------------------ full-size configs
# Reading: at full size the oracle computes complete KV head GROUPS (every output element of the
# G query heads of the group, every slot gradient row of that KV head); the groups are derived from the workload
# seed (kv_heads_for), the remaining groups are covered by the all-head properties in check_attention (finite
# outputs, dV conservation over all heads, untouched slots bit-zero).
def test_c2_full_size_two_kv_head_groups():
    wl = make_workload(CONFIGS["c2"])
    rep = {}
    heads = kv_heads_for(wl.seed, wl.cfg.Hkv, 2)
    sess = check_attention(wl, cas.CAS_IMPL_AUTO, kv_heads=heads, report=rep)
    print("c2", heads, rep)
    used = sorted(set(wl.sel_cart.tolist()))
    check_adam_isolated(sess, used[:2])
    sess.close()


def test_c4_full_size_one_kv_head_group():
    wl = make_workload(CONFIGS["c4"])
    rep = {}
    heads = kv_heads_for(wl.seed + 4, wl.cfg.Hkv, 1)
    check_attention(wl, cas.CAS_IMPL_AUTO, kv_heads=heads, report=rep).close()
    print("c4", heads, rep)


def test_c5_full_size_decode():
    for i, name in enumerate(("c5_all", "c5_top8")):
        wl = make_workload(CONFIGS[name])
        rep = {}
        heads = kv_heads_for(wl.seed + 5 + i, wl.cfg.Hkv, 1)
        check_attention(wl, cas.CAS_IMPL_AUTO, kv_heads=heads, report=rep).close()
        print(name, heads, rep)


def _host_step_buffers(sess, wl):
    tdt = sess.tdt
    cfg = wl.cfg
    pin = lambda a: torch.from_numpy(a).to(tdt).pin_memory()
    h = dict(Q=pin(wl.Q), Ks=pin(wl.K_self), Vs=pin(wl.V_self), dO=pin(wl.dO))
    h["O"], h["dQ"] = torch.empty_like(h["Q"]).pin_memory(), torch.empty_like(h["Q"]).pin_memory()
    h["dKs"], h["dVs"] = torch.empty_like(h["Ks"]).pin_memory(), torch.empty_like(h["Ks"]).pin_memory()
    h["LSE"] = torch.empty((sess.tab.T, cfg.Hq), dtype=torch.float32).pin_memory()
    return h


def _host_step(sess, tab, h, scratch):
    cas.cas_train_step_host(sess.pool, tab, sess.cfg.Hq, h["Q"], h["Ks"], h["Vs"], h["dO"], sess.scale,
                            sess.adam_cfg(), h["O"], h["LSE"], h["dQ"], h["dKs"], h["dVs"], scratch)


def test_train_step_host_matches_the_separate_calls():
    """cas_train_step_host (pinned HOST buffers, copies overlapped on the library's copy streams) gives the
    same O / LSE / dQ / dK_self / dV_self bits as fwd + bwd called one by one, leaves the same gradients consumed
    by the same Adam step, and can be called back to back on the same scratch."""
    cfg = CONFIGS["c2"].scaled(name="c2_host", n_carts=8, n_slots=8, cart_len=300, B=3, Lq=333, n_dist=2)
    wl = make_workload(cfg, 41)
    cas.cas_set_impl(cas.CAS_IMPL_AUTO)
    ref = Session(wl)
    ref.fwd()
    ref.bwd()
    ref.adam()
    torch.cuda.synchronize()
    sess = Session(wl)
    h = _host_step_buffers(sess, wl)
    scratch = torch.empty(cas.cas_train_step_host_scratch_bytes(sess.pool, sess.tab, cfg.Hq), dtype=torch.uint8,
                          device="cuda")
    _host_step(sess, sess.tab, h, scratch)
    torch.cuda.synchronize()
    assert torch.equal(h["O"], ref.O.cpu()) and torch.equal(h["LSE"], ref.LSE.cpu())
    assert torch.equal(h["dKs"], ref.dKs.cpu()) and torch.equal(h["dVs"], ref.dVs.cpu())   # deterministic (cas.h)
    # dQ goes through fp32 L2 reductions whose order is not fixed: compare within bf16 rounding
    assert rel_fro(h["dQ"].float().numpy(), ref.dQ.float().cpu().numpy()) < 1e-2
    for c in sorted(set(wl.sel_cart.tolist()))[:3]:
        for what in ("pK", "mV", "vK"):
            a, b = sess.read(c, what), ref.read(c, what)
            assert rel_fro(a, b) < 1e-5, (c, what)
    O1 = h["O"].clone()
    for _ in range(2):      # back to back on the same scratch; parameters moved, so O changes but stays finite
        _host_step(sess, sess.tab, h, scratch)
    torch.cuda.synchronize()
    assert torch.isfinite(h["O"].float()).all() and not torch.equal(h["O"], O1)
    ref.close()
    sess.close()


def test_train_step_host_back_to_back_with_changing_layout():
    """Ragged training: T changes from step to step, so the regions of the shared scratch MOVE between two
    back-to-back calls: the inputs of step n+1 must not land on the outputs step n is still copying
    to the host.  Two different batches alternate on one scratch without any synchronisation in between; every
    step's host results must equal those of the same step run alone (same pool state: lr = 0 keeps the
    parameters fixed, so each batch has one right answer)."""
    base = CONFIGS["c2"].scaled(name="c2_hostA", n_carts=8, n_slots=8, cart_len=300, B=3, Lq=900, n_dist=2, lr=0.0)
    wlA = make_workload(base, 43)
    wlB = make_workload(base.scaled(name="c2_hostB", B=2, Lq=150), 43)      # same seed: same cartridges
    np.testing.assert_array_equal(wlA.cart_K, wlB.cart_K)
    cas.cas_set_impl(cas.CAS_IMPL_AUTO)
    sess = Session(wlA)
    tabA = sess.tab
    tabB = cas.cas_slot_table_build(sess.pool, wlB.seq_off, wlB.sel_off, wlB.sel_cart, 0)
    sess.cfg = wlA.cfg
    hA, hB = _host_step_buffers(sess, wlA), None
    sess.tab = tabB
    hB = _host_step_buffers(sess, wlB)
    sess.tab = tabA
    nb = max(cas.cas_train_step_host_scratch_bytes(sess.pool, t, base.Hq) for t in (tabA, tabB))
    scratch = torch.empty(nb, dtype=torch.uint8, device="cuda")
    want = {}
    for name, tab, h in (("A", tabA, hA), ("B", tabB, hB)):                 # each batch alone, fully synchronised
        _host_step(sess, tab, h, scratch)
        torch.cuda.synchronize()
        want[name] = {k: h[k].clone() for k in ("O", "LSE", "dKs", "dVs", "dQ")}
        for k in ("O", "LSE", "dKs", "dVs", "dQ"):
            h[k].zero_()
    for rep in range(3):                                                     # A B A B A B, no sync in between
        _host_step(sess, tabA, hA, scratch)
        _host_step(sess, tabB, hB, scratch)
    torch.cuda.synchronize()
    for name, h in (("A", hA), ("B", hB)):
        for k in ("O", "LSE", "dKs", "dVs"):
            assert torch.equal(h[k], want[name][k]), (name, k)
        assert rel_fro(h["dQ"].float().numpy(), want[name]["dQ"].float().numpy()) < 1e-2, name
    tabB.close()
    sess.close()


def test_train_step_host_async_pipelines_steps_over_two_buffer_sets():
    """cas_train_step_host_async: six steps with DIFFERENT inputs are issued back to back without any
    synchronisation (step i+1's inputs are copied into the other buffer set while step i computes, step i's dQ is
    still leaving while step i+1 runs); after cas_train_step_host_wait every step's host results equal those of
    the same step run alone with the per-call-complete variant (lr = 0: the parameters stay fixed, so each input
    has one right answer).  Catches a buffer set overwritten before its last reader, results read back from the
    wrong set, and a wait that does not cover both sets."""
    base = CONFIGS["c2"].scaled(name="c2_async", n_carts=8, n_slots=8, cart_len=300, B=3, Lq=700, n_dist=2, lr=0.0)
    wls = [make_workload(base, 43)]
    cas.cas_set_impl(cas.CAS_IMPL_AUTO)
    sess = Session(wls[0])
    rng = np.random.Generator(np.random.PCG64(44))
    from workloads import round_to_dtype
    hs = []
    for i in range(6):                              # same table (same layout), fresh Q / K_self / V_self / dO per step
        h = _host_step_buffers(sess, wls[0])
        if i:
            for k in ("Q", "Ks", "Vs", "dO"):
                a = round_to_dtype(rng.standard_normal(tuple(h[k].shape), dtype=np.float32) * (0.5 + 0.3 * i), "bf16")
                h[k].copy_(torch.from_numpy(a).to(sess.tdt))
        hs.append(h)
    scratch = torch.empty(cas.cas_train_step_host_scratch_bytes(sess.pool, sess.tab, base.Hq), dtype=torch.uint8,
                          device="cuda")
    want = []
    for h in hs:                                    # each step alone, fully synchronised
        _host_step(sess, sess.tab, h, scratch)
        torch.cuda.synchronize()
        want.append({k: h[k].clone() for k in ("O", "LSE", "dKs", "dVs", "dQ")})
        for k in ("O", "LSE", "dKs", "dVs", "dQ"):
            h[k].fill_(7.0)
    assert not torch.equal(want[0]["O"], want[1]["O"])
    for h in hs:
        cas.cas_train_step_host_async(sess.pool, sess.tab, base.Hq, h["Q"], h["Ks"], h["Vs"], h["dO"], sess.scale,
                                      sess.adam_cfg(), h["O"], h["LSE"], h["dQ"], h["dKs"], h["dVs"], scratch)
    cas.cas_train_step_host_wait(sess.pool)
    torch.cuda.current_stream().synchronize()       # the CALLER's stream only: the wait made it cover the copies
    for i, h in enumerate(hs):
        for k in ("O", "LSE", "dKs", "dVs"):
            assert torch.equal(h[k], want[i][k]), (i, k)
        assert rel_fro(h["dQ"].float().numpy(), want[i]["dQ"].float().numpy()) < 1e-2, i
    sess.close()


@pytest.mark.parametrize("self_block", [True, False])
def test_forward_tail_split_matches_whole_blocks_and_the_oracle(self_block):
    """tc_fwd_kernel's tail split (cas.h cas_slot_table_fwd_split): 25 row blocks x 8 heads = 200 CTAs on 148 SMs,
    the 52 that would run alone in the last wave are cut along the KV axis and merged by fwd_combine_kernel.  The
    split rows live in the LAST KV head group: that group is compared with the oracle (a wrong tile range or merge
    weight fails 2e-2 there), and every row of O / LSE is compared with the same launch run unsplit (row by row: a
    single wrong tail row cannot hide in a Frobenius norm over the batch).  Ragged lengths: partly filled last
    row blocks, 128-row blocks (one Q tile) and prefix tiles with a ragged end."""
    import os
    cfg = CONFIGS["c2"].scaled(name="c2_tail", Hq=8, Hkv=2, n_carts=9, n_slots=9, cart_len=0, len_mu=6.0,
                               len_sigma=0.5, len_min=200, len_max=900, B=5, Lq=0, lq_min=1050, lq_max=1270, n_dist=2)
    wl = make_workload(cfg, 47)
    assert sum((int(l) + 255) // 256 for l in np.diff(wl.seq_off)) * cfg.Hq > 148
    cas.cas_set_impl(cas.CAS_IMPL_AUTO)
    sess = check_attention(wl, cas.CAS_IMPL_AUTO, kv_heads=[cfg.Hkv - 1], self_block=self_block, backward=False)
    n_tail, n_parts = cas.cas_slot_table_fwd_split(sess.tab)
    assert n_tail > 0 and n_parts >= 2, (n_tail, n_parts)
    O1, L1 = sess.O.clone(), sess.LSE.clone()
    os.environ["CAS_FWD_NO_SPLIT"] = "1"
    try:
        tab2 = cas.cas_slot_table_build(sess.pool, wl.seq_off, wl.sel_off, wl.sel_cart, 0)
        old, sess.tab = sess.tab, tab2
        sess.O.zero_()
        sess.fwd(self_block=self_block)
        torch.cuda.synchronize()
        assert cas.cas_slot_table_fwd_split(tab2) == (0, 1)
    finally:
        del os.environ["CAS_FWD_NO_SPLIT"]
    a, b = O1.float().cpu().numpy(), sess.O.float().cpu().numpy()
    per_row = np.linalg.norm(a - b, axis=2) / (np.linalg.norm(b, axis=2) + 1e-30)
    assert per_row.max() <= 1e-2, per_row.max()                  # bf16 rounding of a differently ordered sum
    assert (per_row > 0).sum() <= n_tail * 256                   # only the split rows may differ at all
    np.testing.assert_allclose(L1.cpu().numpy(), sess.LSE.cpu().numpy(), rtol=1e-5, atol=1e-5)
    sess.tab = old
    tab2.close()
    sess.close()
    print("tail split", n_tail, n_parts)


def test_cta_pair_mma_selftest():
    """tcgen05.mma.cta_group::2 on a 2-CTA cluster (the primitives kept in cas_sm100.cuh for the next kernels):
    exact against an integer-valued reference."""
    g = torch.Generator().manual_seed(3)
    A = (torch.randint(-8, 9, (256, 64), generator=g).float() / 8).to(torch.bfloat16).cuda()
    B = (torch.randint(-6, 7, (128, 64), generator=g).float() / 4).to(torch.bfloat16).cuda()
    D = torch.zeros((256, 128), dtype=torch.float32, device="cuda")
    cas.cas_selftest_cta_pair_mma(A, B, D)
    torch.cuda.synchronize()
    want = A.double().cpu() @ B.double().cpu().T
    assert torch.equal(D.double().cpu(), want)


def test_gradient_slots_accumulate_then_overwrite_after_adam():
    """Gradient-slot life cycle on the tensor-core path (R32), every stage against the ORACLE: a second
    backward pass accumulates (+=: the oracle is handed its own first result to add to), Adam consumes the gradients
    (the slot becomes clean = zero gradient, its buffer is NOT zeroed), and the next backward pass OVERWRITES the
    stale buffer: its result must equal the oracle's backward pass on the UPDATED bf16 working copies -- stale bytes
    leaking into it (2*g_old + g_new instead of g_new) fail the 3e-2 gate.  An untouched slot reads as exactly zero
    throughout and, updated by Adam from m = v = 0 with g = 0, does not move."""
    cfg = CONFIGS["c2"].scaled(name="c2_life", n_carts=6, n_slots=6, cart_len=200, B=2, Lq=260, n_dist=1)
    wl = make_workload(cfg, 51)
    cas.cas_set_impl(cas.CAS_IMPL_AUTO)
    sess = Session(wl)
    used = sorted(set(wl.sel_cart.tolist()))
    unused = [c for c in range(cfg.n_carts) if c not in used]
    assert unused
    heads = list(range(cfg.Hkv))
    sel = [wl.sel_cart[wl.sel_off[b]:wl.sel_off[b + 1]].tolist() for b in range(cfg.B)]

    def working_copies():
        bK = {c: (sess.read(c, "wK").astype(np.uint32) << 16).view(np.float32) for c in used}
        bV = {c: (sess.read(c, "wV").astype(np.uint32) << 16).view(np.float32) for c in used}
        return bK, bV

    def oracle_bwd(bK, bV, gK=None, gV=None):
        return orc.attn_bwd(wl.Q, bK, bV, sel, wl.seq_off, wl.K_self, wl.V_self, wl.dO, sess.scale, cfg.Hkv,
                            kv_heads=heads, grad_K=gK, grad_V=gV)

    def check(gKo, gVo, dQo):
        for c in used:
            assert rel_fro(sess.read(c, "gK"), gKo[c]) <= TOL_BF16_DKV, c
            assert rel_fro(sess.read(c, "gV"), gVo[c]) <= TOL_BF16_DKV, c
        assert rel_fro(sess.np(sess.dQ), dQo) <= TOL_BF16_O_DQ
        for c in unused:
            assert not sess.read(c, "gK").any() and not sess.read(c, "gV").any()

    bK0, bV0 = working_copies()
    sess.fwd()
    sess.bwd()
    torch.cuda.synchronize()
    dQo, gKo, gVo, _, _ = oracle_bwd(bK0, bV0)
    check(gKo, gVo, dQo)
    sess.bwd()                                   # accumulate: the oracle adds a second pass onto its first result
    torch.cuda.synchronize()
    dQo, gKo, gVo, _, _ = oracle_bwd(bK0, bV0, gKo, gVo)
    check(gKo, gVo, dQo)
    g_stale = {c: sess.read(c, "gK").copy() for c in used}
    p_unused = sess.read(unused[0], "pK").copy()
    sess.adam()                                  # consumes the gradients; clean slots are updated with g = 0
    torch.cuda.synchronize()
    for c in used:
        assert not sess.read(c, "gK").any()      # clean slot reads as zero although its buffer still holds 2*g
    np.testing.assert_array_equal(sess.read(unused[0], "pK"), p_unused)   # g = 0 from m = v = 0: exact no-op
    assert np.abs(sess.read(unused[0], "mK")).max() == 0
    bK1, bV1 = working_copies()
    assert any(not np.array_equal(bK1[c], bK0[c]) for c in used)          # the step moved the working copies
    sess.fwd()
    sess.bwd()                                   # first touch after Adam: overwrite, not stale + g
    torch.cuda.synchronize()
    dQo, gKo, gVo, _, _ = oracle_bwd(bK1, bV1)
    check(gKo, gVo, dQo)
    for c in used:                               # and the stale bytes were really there to leak
        assert rel_fro(sess.read(c, "gK") + g_stale[c], gKo[c]) > 0.5
    sess.close()
