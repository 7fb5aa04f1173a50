"""GPU parity: the CUDA path (through the C ABI) against oracle/ on the same seeded inputs.
Small cases compare every output element; full-size configs compare every output element of one KV
head group (the oracle computes that group completely) plus properties over all heads."""
import numpy as np
import pytest
import torch

from paper_2606_04557_b200 import _build, cas
from paper_2606_04557_b200.harness import Session
from workloads import CONFIGS, make_workload

from parity_util import check_adam_isolated, check_attention, rel_fro

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


# ------------------------------------------------------------------ full-size configs, one KV head
def test_c2_full_size_one_kv_head():
    wl = make_workload(CONFIGS["c2"])
    rep = {}
    sess = check_attention(wl, cas.CAS_IMPL_AUTO, kv_heads=[3], report=rep)
    print("c2", rep)
    used = sorted(set(wl.sel_cart.tolist()))
    check_adam_isolated(sess, used[:2])
    sess.close()


def test_c4_full_size_one_kv_head():
    wl = make_workload(CONFIGS["c4"])
    rep = {}
    check_attention(wl, cas.CAS_IMPL_AUTO, kv_heads=[6], report=rep).close()
    print("c4", rep)


def test_c5_full_size_decode():
    for name, g in (("c5_all", 2), ("c5_top8", 5)):
        wl = make_workload(CONFIGS[name])
        rep = {}
        check_attention(wl, cas.CAS_IMPL_AUTO, kv_heads=[g], report=rep).close()
        print(name, rep)


def test_train_step_host_matches_the_separate_calls():
    """cas_train_step_host (pinned HOST buffers, copies overlapped on the library's copy streams) gives the
    same O / LSE / dQ bits as fwd + bwd called one by one, leaves the same gradients consumed by the same
    Adam step, and can be called back to back on the same scratch."""
    cfg = CONFIGS["c2"].scaled(name="c2_host", n_carts=8, n_slots=8, cart_len=300, B=3, Lq=333, n_dist=2)
    wl = make_workload(cfg, 41)
    cas.cas_set_impl(cas.CAS_IMPL_AUTO)
    ref = Session(wl)
    ref.fwd()
    ref.bwd()
    ref.adam()
    torch.cuda.synchronize()
    sess = Session(wl)
    tdt = sess.tdt
    pin = lambda a: torch.from_numpy(a).to(tdt).pin_memory()
    hQ, hKs, hVs, hdO = pin(wl.Q), pin(wl.K_self), pin(wl.V_self), pin(wl.dO)
    hO, hdQ = torch.empty_like(hQ).pin_memory(), torch.empty_like(hQ).pin_memory()
    hLSE = torch.empty((sess.tab.T, cfg.Hq), dtype=torch.float32).pin_memory()
    scratch = torch.empty(cas.cas_train_step_host_scratch_bytes(sess.pool, sess.tab, cfg.Hq), dtype=torch.uint8,
                          device="cuda")
    cas.cas_train_step_host(sess.pool, sess.tab, cfg.Hq, hQ, hKs, hVs, hdO, sess.scale, sess.adam_cfg(), hO, hLSE,
                            hdQ, scratch)
    torch.cuda.synchronize()
    assert torch.equal(hO, ref.O.cpu()) and torch.equal(hLSE, ref.LSE.cpu())
    # dQ goes through fp32 L2 reductions whose order is not fixed: compare within bf16 rounding
    assert rel_fro(hdQ.float().numpy(), ref.dQ.float().cpu().numpy()) < 1e-2
    for c in sorted(set(wl.sel_cart.tolist()))[:3]:
        for what in ("pK", "mV", "vK"):
            a, b = sess.read(c, what), ref.read(c, what)
            assert rel_fro(a, b) < 1e-5, (c, what)
    O1 = hO.clone()
    for _ in range(2):      # back to back on the same scratch; parameters moved, so O changes but stays finite
        cas.cas_train_step_host(sess.pool, sess.tab, cfg.Hq, hQ, hKs, hVs, hdO, sess.scale, sess.adam_cfg(), hO,
                                hLSE, hdQ, scratch)
    torch.cuda.synchronize()
    assert torch.isfinite(hO.float()).all() and not torch.equal(hO, O1)
    ref.close()
    sess.close()


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


def test_forward_cta_pair_kernel_parity():
    """The opt-in CTA-pair forward kernel (CAS_FWD_PAIRS=1, cas_tc_fwd2.cu) against the oracle: ragged lengths,
    512-row blocks with 257..512 rows, leftover blocks on the single-CTA kernel, prefix-only call.  Runs in a
    subprocess because the switch is read once per process."""
    import os
    import subprocess
    import sys
    code = (
        "import sys; sys.path.insert(0, 'tests')\n"
        "from parity_util import check_attention\n"
        "from paper_2606_04557_b200 import cas\n"
        "from workloads import CONFIGS, make_workload\n"
        "cfg = CONFIGS['c4'].scaled(name='c4_pairs', n_carts=10, n_slots=10, B=5, len_mu=5.5, len_min=40, len_max=500,\n"
        "                           lq_min=200, lq_max=1300, n_dist_max=4)\n"
        "check_attention(make_workload(cfg, 61), cas.CAS_IMPL_AUTO, kv_heads=[1, 6], backward=False).close()\n"
        "check_attention(make_workload(cfg, 62), cas.CAS_IMPL_AUTO, kv_heads=[3], backward=False, self_block=False).close()\n"
        "cfg = CONFIGS['c2'].scaled(name='c2_pairs', n_carts=6, n_slots=6, cart_len=384, B=2, Lq=1024, n_dist=2)\n"
        "check_attention(make_workload(cfg, 63), cas.CAS_IMPL_AUTO, kv_heads=[0, 7], backward=False).close()\n"
        "print('pairs ok')\n")
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    r = subprocess.run([sys.executable, "-c", code], cwd=root, env=dict(os.environ, CAS_FWD_PAIRS="1"),
                       capture_output=True, text=True, timeout=600)
    assert r.returncode == 0 and "pairs ok" in r.stdout, r.stdout[-2000:] + r.stderr[-2000:]


def test_gradient_slots_accumulate_then_overwrite_after_adam():
    """Gradient-slot life cycle on the tensor-core path: a second backward pass accumulates (+=), Adam consumes
    the gradients (the slot becomes clean = zero gradient, its buffer is NOT zeroed), the next backward pass
    overwrites the stale buffer, an untouched slot reads as exactly zero throughout, and a clean slot updated by
    Adam behaves as g = 0."""
    cfg = CONFIGS["c2"].scaled(name="c2_life", n_carts=6, n_slots=6, cart_len=200, B=2, Lq=260, n_dist=1)
    wl = make_workload(cfg, 51)
    cas.cas_set_impl(cas.CAS_IMPL_AUTO)
    sess = Session(wl)
    used = sorted(set(wl.sel_cart.tolist()))
    unused = [c for c in range(cfg.n_carts) if c not in used]
    assert unused
    sess.fwd()
    sess.bwd()
    torch.cuda.synchronize()
    g1 = {c: (sess.read(c, "gK").copy(), sess.read(c, "gV").copy()) for c in used}
    assert all(np.abs(g1[c][0]).max() > 0 for c in used)
    sess.bwd()                                   # accumulate: exactly twice (same summands, fp32 adds of equal values)
    torch.cuda.synchronize()
    for c in used:
        np.testing.assert_allclose(sess.read(c, "gK"), 2 * g1[c][0], rtol=1e-6, atol=1e-12)
        np.testing.assert_allclose(sess.read(c, "gV"), 2 * g1[c][1], rtol=1e-6, atol=1e-12)
    for c in unused:
        assert not sess.read(c, "gK").any() and not sess.read(c, "gV").any()
    p_unused = sess.read(unused[0], "pK").copy()
    sess.adam()                                  # consumes the gradients; clean slots are updated with g = 0
    torch.cuda.synchronize()
    for c in used:
        assert not sess.read(c, "gK").any()      # clean slot reads as zero although its buffer still holds 2*g1
    np.testing.assert_array_equal(sess.read(unused[0], "pK"), p_unused)   # g = 0 from m = v = 0: exact no-op
    assert np.abs(sess.read(unused[0], "mK")).max() == 0
    sess.fwd()
    sess.bwd()                                   # first touch after Adam: overwrite, not 2*g1 + g
    torch.cuda.synchronize()
    for c in used:
        g = sess.read(c, "gK")
        assert rel_fro(g, g1[c][0]) < 0.5        # same order as one backward pass (parameters moved by one step)
        assert rel_fro(g, 3 * g1[c][0]) > 0.5
    sess.close()
