"""GPU parity of the layer axis and micro-batch accumulation: PAPER.md:42 a cartridge is
Z in R^{L x p x d x 2}; PAPER.md:375-376 several packed micro-batches per optimizer step.  cas_train_step_layers =
for every micro-batch: forward through the layers, backward in reverse order (gradients ACCUMULATE in the slots),
then ONE Adam -- compared with the same loop written with the oracle."""
import numpy as np
import pytest
import torch

from oracle import cas_oracle as orc
from paper_2606_04557_b200 import _build, cas
from workloads import CONFIGS, make_workload, round_to_dtype
from workloads.generate import draw_batch_selection, draw_query_block

from parity_util import TOL_ADAM, TOL_BF16_DKV, TOL_BF16_O_DQ, rel_fro, rel_max

pytestmark = pytest.mark.gpu
STATE = ("pK", "pV", "mK", "mV", "vK", "vV")


@pytest.fixture(scope="module", autouse=True)
def built():
    _build.build()
    cas.cas_set_impl(cas.CAS_IMPL_AUTO)


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).to("cuda").to(torch.bfloat16)


def make_pool(cfg, L, seed, n_slots=None):
    """A pool with L layers; layer l of cartridge c holds its own seeded K/V (values rounded to bf16)."""
    wl = make_workload(cfg, seed)
    rng = np.random.Generator(np.random.PCG64(seed + 500))
    pool = cas.Pool(cas.CAS_BF16, cfg.Hkv, cfg.D, wl.cart_len, n_slots or cfg.n_slots, n_layers=L)
    KV = {}
    for l in range(L):
        for c in range(cfg.n_carts):
            n = int(wl.cart_len[c])
            K = round_to_dtype(rng.standard_normal((n, cfg.Hkv, cfg.D), dtype=np.float32) * cfg.kv_std, "bf16")
            V = round_to_dtype(rng.standard_normal((n, cfg.Hkv, cfg.D), dtype=np.float32) * cfg.kv_std, "bf16")
            KV[(l, c)] = (K, V)
            cas.cas_pool_load(pool, c, K, V, layer=l)
    return wl, pool, KV


def test_train_step_layers_L4_four_micro_batches():
    L, n_micro = 4, 4
    cfg = CONFIGS["c2"].scaled(name="c2_layers", Hq=8, Hkv=2, n_carts=7, n_slots=7, cart_len=200, B=2, Lq=260,
                               n_dist=2)
    wl, pool, KV = make_pool(cfg, L, 81)
    rng = np.random.Generator(np.random.PCG64(82))
    heads = list(range(cfg.Hkv))
    scale = 1.0 / float(np.sqrt(cfg.D))
    tabs, batches, io = [], [], []
    for m in range(n_micro):
        lq = [[260, 131], [77, 300], [129, 128], [1, 257]][m]      # different packing per micro-batch
        seq_off = np.concatenate([[0], np.cumsum(lq)]).astype(np.int32)
        sel_off, sel_cart = draw_batch_selection(cfg, rng, list(range(cfg.n_carts)), wl.cart_len)
        tabs.append(cas.cas_slot_table_build(pool, seq_off, sel_off, sel_cart, m))
        per_layer, io_m = [], []
        for l in range(L):
            Q, Ks, Vs, dO = draw_query_block(cfg, rng, seq_off)
            per_layer.append((Q, Ks, Vs, dO))
            T = int(seq_off[-1])
            t = dict(Q=dev(Q), K_self=dev(Ks), V_self=dev(Vs), dO=dev(dO),
                     O=torch.empty((T, cfg.Hq, cfg.D), dtype=torch.bfloat16, device="cuda"),
                     LSE=torch.empty((T, cfg.Hq), dtype=torch.float32, device="cuda"))
            t["dQ"] = torch.empty_like(t["O"])
            t["dK_self"], t["dV_self"] = torch.empty_like(t["K_self"]), torch.empty_like(t["K_self"])
            io_m.append(t)
        batches.append((seq_off, sel_off, sel_cart, per_layer))
        io.append(io_m)
    ws = torch.empty(cas.cas_train_step_layers_workspace_bytes(pool, tabs, cfg.Hq), dtype=torch.uint8, device="cuda")
    before = {(l, c): {w: cas.cas_pool_read(pool, c, w, layer=l) for w in STATE} for l in range(L)
              for c in range(cfg.n_carts)}
    acfg = cas.AdamCfg(cfg.lr, cfg.beta1, cfg.beta2, cfg.eps, 1, 0)     # zero_grad = 0: gradients stay readable
    cas.cas_train_step_layers(pool, tabs, cfg.Hq, io, scale, acfg, workspace=ws)
    torch.cuda.synchronize()
    # ---- the oracle loop
    f32 = lambda x: float(np.float32(x))
    for l in range(L):
        bK = {c: KV[(l, c)][0] for c in range(cfg.n_carts)}
        bV = {c: KV[(l, c)][1] for c in range(cfg.n_carts)}
        gK, gV = {}, {}
        for m in range(n_micro):
            seq_off, sel_off, sel_cart, per_layer = batches[m]
            Q, Ks, Vs, dO = per_layer[l]
            sel = [sel_cart[sel_off[b]:sel_off[b + 1]].tolist() for b in range(cfg.B)]
            Oo, Lo = orc.attn_fwd(Q, bK, bV, sel, seq_off, Ks, Vs, scale, cfg.Hkv, kv_heads=heads)
            dQo, gK, gV, dKso, dVso = orc.attn_bwd(Q, bK, bV, sel, seq_off, Ks, Vs, dO, scale, cfg.Hkv,
                                                   kv_heads=heads, grad_K=gK, grad_V=gV)   # "+=" across micro-batches
            t = io[m][l]
            assert rel_fro(t["O"].float().cpu().numpy(), Oo) <= TOL_BF16_O_DQ, (m, l)
            assert rel_max(t["LSE"].cpu().numpy(), Lo) <= 2e-3
            assert rel_fro(t["dQ"].float().cpu().numpy(), dQo) <= TOL_BF16_O_DQ, (m, l)
            assert rel_fro(t["dK_self"].float().cpu().numpy(), dKso) <= TOL_BF16_DKV
            assert rel_fro(t["dV_self"].float().cpu().numpy(), dVso) <= TOL_BF16_DKV
        for c in range(cfg.n_carts):
            g_gpu = {kv: cas.cas_pool_read(pool, c, "g" + kv, layer=l) for kv in "KV"}
            if c in gK:                                              # accumulated over all micro-batches, per slot
                assert rel_fro(g_gpu["K"], gK[c]) <= TOL_BF16_DKV, (l, c)
                assert rel_fro(g_gpu["V"], gV[c]) <= TOL_BF16_DKV, (l, c)
            else:
                assert not g_gpu["K"].any() and not g_gpu["V"].any()
            # ONE Adam step (t = 1) on exactly these gradients, first token frozen
            b = before[(l, c)]
            for kv in "KV":
                p, mm, vv = orc.adam_step(b["p" + kv], b["m" + kv], b["v" + kv], g_gpu[kv], 1, f32(cfg.lr),
                                          f32(cfg.beta1), f32(cfg.beta2), f32(cfg.eps), n_frozen=1)
                gp = cas.cas_pool_read(pool, c, "p" + kv, layer=l)
                assert rel_max(gp, p) <= TOL_ADAM and rel_max(cas.cas_pool_read(pool, c, "m" + kv, layer=l), mm) <= TOL_ADAM
                assert rel_max(cas.cas_pool_read(pool, c, "v" + kv, layer=l), vv) <= TOL_ADAM
                np.testing.assert_array_equal(cas.cas_pool_read(pool, c, "w" + kv, layer=l), orc.bf16_rne_bits(gp))
    cnt = cas.cas_pool_counters(pool)
    assert cnt["opt_steps"].tolist() == [1] * cfg.n_carts           # one optimizer step per cartridge, not per layer
    for t in tabs:
        t.close()
    pool.close()


def test_swap_moves_every_layer():
    """Rotation with a layer axis: evicting and re-loading a cartridge moves the parameters and moments of ALL its
    layers, byte-exact, and re-derives every layer's working copy."""
    L = 2
    cfg = CONFIGS["c3"].scaled(name="c3_layers", Hq=8, Hkv=2, n_carts=6, n_slots=3, cart_len=256, B=1, Lq=64, n_dist=0,
                               rotate_in=2, rotate_out=2)
    wl, pool, KV = make_pool(cfg, L, 83, n_slots=3)
    main = torch.cuda.current_stream()
    state0 = {(l, c): [cas.cas_pool_read(pool, c, w, layer=l).copy() for w in STATE] for l in range(L) for c in range(6)}
    for l in range(L):
        for c in range(6):
            np.testing.assert_array_equal(state0[(l, c)][0], KV[(l, c)][0])
    for step in range(3):
        man, n = cas.cas_plan_rotation(pool, step, 2, 2, [], 11)
        assert man[0].nbytes == L * 6 * 256 * cfg.Hkv * cfg.D * 4
        cas.cas_swap_out(pool, man, n, step, after_stream=main)
        cas.cas_swap_in(pool, man, n, step)
        cas.cas_swap_commit(pool, main)
    torch.cuda.synchronize()
    cnt = cas.cas_pool_counters(pool)
    for l in range(L):
        for c in range(6):
            for w, old in zip(STATE, state0[(l, c)]):
                np.testing.assert_array_equal(cas.cas_pool_read(pool, c, w, layer=l), old)
            if cnt["slot_of"][c] >= 0:
                np.testing.assert_array_equal(cas.cas_pool_read(pool, c, "wK", layer=l),
                                              orc.bf16_rne_bits(state0[(l, c)][0]))
    pool.close()
