"""GPU parity of cas_decode_attn: decode with a GROWING self cache ("2048
maximum completion tokens") over retrieval-selected cartridges, against the oracle at every step of
a generation loop.

Oracle: the plain definition oracle.cas_oracle.attn_fwd.  A decode step of sequence b with n tokens in its cache is
the last row of that sequence's attention: the n-1 earlier tokens are keys that precede the query exactly like a
prefix block, so they are handed to attn_fwd as one more (per-sequence) block in front of the 1-token causal self
block -- no new oracle arithmetic."""
import numpy as np
import pytest
import torch

from oracle import cas_oracle as orc
from oracle.bookkeeping import select_retrieved
from paper_2606_04557_b200 import _build, cas
from workloads import CONFIGS, make_workload, round_to_dtype

from parity_util import TOL_BF16_O_DQ, kv_heads_for, rel_fro, rel_max

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def built():
    _build.build()
    cas.cas_set_impl(cas.CAS_IMPL_AUTO)


def bf16_dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).to("cuda").to(torch.bfloat16)


def oracle_decode(wl, sel, q, Kc, Vc, lens, scale, kv_heads):
    """q [B,Hq,D]; Kc/Vc [B,cap,Hkv,D] (fp32 holding bf16 values); keys of b = its cartridges + cache[b][:lens[b]]."""
    cfg = wl.cfg
    B = len(sel)
    bK = {c: wl.cart_kv(c)[0] for s in sel for c in s}
    bV = {c: wl.cart_kv(c)[1] for s in sel for c in s}
    sel2, Ks, Vs = [], np.zeros((B, cfg.Hkv, cfg.D), np.float32), np.zeros((B, cfg.Hkv, cfg.D), np.float32)
    for b in range(B):
        n = int(lens[b])
        s = list(sel[b])
        if n > 1:                                   # earlier tokens of the sequence: one more block before the query
            bK[("cache", b)], bV[("cache", b)] = Kc[b, :n - 1], Vc[b, :n - 1]
            s.append(("cache", b))
        Ks[b], Vs[b] = Kc[b, n - 1], Vc[b, n - 1]  # the current token's own key/value (causal diagonal)
        sel2.append(s)
    return orc.attn_fwd(q, bK, bV, sel2, np.arange(B + 1), Ks, Vs, scale, cfg.Hkv, kv_heads=kv_heads)


def run_loop(cfg, seed, sel, start_len, steps, cap, kv_heads):
    wl = make_workload(cfg, seed)
    B = len(sel)
    pool = cas.Pool(cas.CAS_BF16, cfg.Hkv, cfg.D, wl.cart_len, cfg.n_slots)
    for c in range(cfg.n_carts):
        cas.cas_pool_load(pool, c, *wl.cart_kv(c))
    sel_off = np.concatenate([[0], np.cumsum([len(s) for s in sel])]).astype(np.int32)
    sel_cart = np.array([c for s in sel for c in s], dtype=np.int32)
    tab = cas.cas_slot_table_build(pool, np.arange(B + 1, dtype=np.int32), sel_off, sel_cart, 0)
    rng = np.random.Generator(np.random.PCG64(seed + 77))
    G = cfg.Hq // cfg.Hkv
    hs = [h for g in kv_heads for h in range(g * G, (g + 1) * G)]
    # the whole token stream of every sequence, drawn up front (values already rounded to bf16)
    # key scale alternates per sequence: cartridge-sized keys (the prefix matters) / large keys (peaked softmax, the
    # running max moves and the lazy rescale of O triggers)
    kstd = np.where(np.arange(B) % 2 == 0, 0.05, 3.0).astype(np.float32)[:, None, None, None]
    Kall = round_to_dtype(rng.standard_normal((B, cap, cfg.Hkv, cfg.D), dtype=np.float32) * kstd, "bf16")
    Vall = round_to_dtype(rng.standard_normal((B, cap, cfg.Hkv, cfg.D), dtype=np.float32), "bf16")
    Kc = torch.zeros((B, cap, cfg.Hkv, cfg.D), dtype=torch.bfloat16, device="cuda")    # finite beyond self_len (cas.h)
    Vc = torch.zeros_like(Kc)
    lens = np.array(start_len, dtype=np.int32)
    for b in range(B):                               # prompt tokens already in the cache
        Kc[b, :lens[b]] = bf16_dev(Kall[b, :lens[b]])
        Vc[b, :lens[b]] = bf16_dev(Vall[b, :lens[b]])
    O = torch.empty((B, cfg.Hq, cfg.D), dtype=torch.bfloat16, device="cuda")
    LSE = torch.empty((B, cfg.Hq), dtype=torch.float32, device="cuda")
    scale = 1.0 / float(np.sqrt(cfg.D))
    worst = 0.0
    for step in range(steps):
        q = round_to_dtype(rng.standard_normal((B, cfg.Hq, cfg.D), dtype=np.float32), "bf16")
        for b in range(B):                           # append the current token, then attend (it sees itself)
            Kc[b, lens[b]] = bf16_dev(Kall[b, lens[b]])
            Vc[b, lens[b]] = bf16_dev(Vall[b, lens[b]])
        lens += 1
        cas.cas_decode_attn(pool, tab, cfg.Hq, bf16_dev(q), Kc, Vc, cap, lens, scale, O, LSE)
        torch.cuda.synchronize()
        Oo, Lo = oracle_decode(wl, sel, q, Kall, Vall, lens, scale, kv_heads)
        got = O.float().cpu().numpy()
        assert np.isfinite(got).all()
        e = rel_fro(got[:, hs], Oo[:, hs])
        # per sequence too: a short self-only row must not hide behind the long-prefix rows
        for b in range(B):
            assert rel_fro(got[b][hs], Oo[b][hs]) <= TOL_BF16_O_DQ, (step, b, lens[b])
        assert rel_max(LSE.cpu().numpy()[:, hs], Lo[:, hs]) <= 2e-3, step
        worst = max(worst, e)
    tab.close()
    pool.close()
    return worst


def test_generation_loop_64_steps_small():
    """64 decode steps; the caches start at 0, 3, 4, 0, 250 and 127 tokens, so the run crosses the inline-self
    threshold (4 -> 5 keys), the first tile boundary (128 -> 129) and the second (256 -> 257); sequence 3 selects
    no cartridge at all (self cache only, from its very first token), sequences 0 and 1 share their whole selection
    (one row block), the selections come from retrieval-ordered de-duplication."""
    cfg = CONFIGS["c5_top8"].scaled(name="c5_gen", Hq=8, Hkv=2, n_carts=9, n_slots=9, cart_len=200, B=6)
    chunk_to_cart = [0, 0, 1, 2, 2, 3, 4, 5, 5, 6, 7, 8]
    ranked = [[4, 3, 0, 11, 1], [4, 3, 0, 11, 1], [9, 9, 2], [], [5, 6, 7, 8, 10, 3], [1]]
    sel = [cas.cas_select_retrieved(r, chunk_to_cart, 4).tolist() for r in ranked]
    assert sel == [select_retrieved(r, chunk_to_cart, 4) for r in ranked]
    assert sel[0] == [2, 0, 8] and sel[3] == []
    worst = run_loop(cfg, 71, sel, start_len=[0, 3, 4, 0, 250, 127], steps=64, cap=320, kv_heads=[0, 1])
    print("generation loop worst rel. Frobenius error", worst)


def test_decode_many_sequences_long_caches_ragged_cartridges():
    """More sequences than one row block (G = 4: 32 sequences per block), ragged cartridge lengths, caches of up to
    ~700 tokens (6 tiles) with very different lengths per sequence (the ticket queue balances them), 3 steps."""
    cfg = CONFIGS["c4"].scaled(name="c4_dec", Hq=16, Hkv=4, n_carts=14, n_slots=14, B=40, Lq=1, n_dist=1,
                               selection="uniform", len_mu=5.5, len_min=17, len_max=600, backward=False)
    rng = np.random.default_rng(5)
    sel = [rng.choice(14, size=int(rng.integers(0, 5)), replace=False).tolist() for _ in range(40)]
    sel[7] = list(range(14))
    start = rng.integers(0, 700, size=40).tolist()
    start[0], start[1] = 0, 699
    worst = run_loop(cfg, 72, sel, start_len=start, steps=3, cap=704, kv_heads=[1, 2])
    print("worst", worst)


def test_c5_full_size_with_2048_token_caches():
    """BASELINE.json configs[4] (500 x 512-token cartridges, 64 sequences, top-8 selection) with the paper's decode
    budget: every sequence has between 1 and 2048 cached tokens.  One KV head group against the oracle,
    finite outputs on all."""
    cfg = CONFIGS["c5_top8"]
    rng = np.random.default_rng(11)
    wl = make_workload(cfg)
    sel = [wl.sel_cart[wl.sel_off[b]:wl.sel_off[b + 1]].tolist() for b in range(cfg.B)]
    start = rng.integers(0, 2047, size=cfg.B).tolist()
    start[0], start[1], start[2] = 2046, 0, 4
    worst = run_loop(cfg, wl.seed, sel, start_len=start, steps=2, cap=2048,
                     kv_heads=kv_heads_for(wl.seed + 9, cfg.Hkv, 1))
    print("c5 with caches", worst)


def test_decode_argument_errors():
    cfg = CONFIGS["c5_top8"].scaled(name="c5_err", Hq=8, Hkv=2, n_carts=3, n_slots=3, cart_len=64, B=2)
    wl = make_workload(cfg, 3)
    pool = cas.Pool(cas.CAS_BF16, cfg.Hkv, cfg.D, wl.cart_len, cfg.n_slots)
    tab = cas.cas_slot_table_build(pool, [0, 1, 2], [0, 1, 1], [2], 0)
    q = torch.zeros((2, 8, 128), dtype=torch.bfloat16, device="cuda")
    Kc = torch.zeros((2, 16, 2, 128), dtype=torch.bfloat16, device="cuda")
    O, LSE = torch.empty_like(q), torch.empty((2, 8), dtype=torch.float32, device="cuda")
    for lens, name in (([1, 0], "CAS_ERR_SHAPE"), ([17, 1], "CAS_ERR_INVALID_ARG")):   # no key at all / beyond cap
        with pytest.raises(cas.CasError) as e:
            cas.cas_decode_attn(pool, tab, 8, q, Kc, Kc, 16, lens, 0.1, O, LSE)
        assert e.value.name == name
    with pytest.raises(cas.CasError) as e:
        cas.cas_decode_attn(pool, tab, 8, q, Kc, Kc, 16, [1, 1], -1.0, O, LSE)
    assert e.value.name == "CAS_ERR_INVALID_ARG"
    tab.close()
    tab = cas.cas_slot_table_build(pool, [0, 2, 3], [0, 1, 1], [2], 0)                # two query tokens in a sequence
    with pytest.raises(cas.CasError) as e:
        cas.cas_decode_attn(pool, tab, 8, q, Kc, Kc, 16, [1, 1], 0.1, O, LSE)
    assert e.value.name == "CAS_ERR_SHAPE"
    tab.close()
    pool.close()


def test_decode_is_bitwise_repeatable_under_stale_scratch():
    """The decode kernel's split-KV partials, row counters and ticket live in library scratch that is reused from
    launch to launch; its result must not depend on what the scratch held or on CTA timing: 200 launches on the
    full-size top-8 config give bit-identical O and LSE (the merge order of a row's partials is fixed)."""
    from paper_2606_04557_b200.harness import Session
    wl = make_workload(CONFIGS["c5_top8"])
    junk = torch.full((100_000_000,), 3.0e30, device="cuda")      # leave non-zero bytes in the allocator's free blocks
    del junk
    sess = Session(wl)
    sess.fwd()
    torch.cuda.synchronize()
    O0, L0 = sess.O.clone(), sess.LSE.clone()
    for it in range(200):
        sess.O.fill_(9.0)
        sess.fwd()
        assert torch.equal(sess.O, O0) and torch.equal(sess.LSE, L0), it
    sess.close()
