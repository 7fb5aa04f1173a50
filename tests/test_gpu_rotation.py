"""GPU tests of the budget manager: swap out/in through pinned host memory on the side stream
(PAPER.md:73-75), byte-exact round trips, manifests and counters bit-exact against the Python
bookkeeping oracle, attention parity after rotation (the slot table follows the moved cartridges)."""
import numpy as np
import pytest
import torch

from oracle import cas_oracle as orc
from oracle.bookkeeping import PoolBook
from paper_2606_04557_b200 import _build, cas
from paper_2606_04557_b200.harness import Session
from workloads import CONFIGS, make_workload
from workloads.generate import draw_batch_selection

from parity_util import TOL_BF16_DKV, TOL_BF16_O_DQ, rel_fro

pytestmark = pytest.mark.gpu
STATE = ("pK", "pV", "mK", "mV", "vK", "vV")


@pytest.fixture(scope="module", autouse=True)
def built():
    _build.build()


def counters_equal(pool, bk):
    c = cas.cas_pool_counters(pool)
    assert c["slot_of"].tolist() == bk.slot_of and c["cart_in"].tolist() == bk.cart_in
    assert c["opt_steps"].tolist() == bk.opt_steps and c["last_used"].tolist() == bk.last_used
    assert c["in_transit"].tolist() == bk.in_transit and c["grad_dirty"].tolist() == bk.grad_dirty


def run_rotation(cfg, steps, seed, check_attn_every=1):
    wl = make_workload(cfg, seed)
    sess = Session(wl)
    bk = PoolBook(wl.cart_len.tolist(), cfg.n_slots, cfg.Hkv, cfg.D, tile_tokens=cfg.tile_tokens or 128,
                  budget_tokens=cfg.budget_tokens)
    bk.slot_table(wl.seq_off.tolist(), wl.sel_off.tolist(), wl.sel_cart.tolist(), 0)   # Session's own table
    rng = np.random.Generator(np.random.PCG64(seed + 1))
    main = torch.cuda.current_stream()
    G = cfg.Hq // cfg.Hkv
    # host mirror of every cartridge's fp32 master params (to feed the oracle after Adam updates)
    for step in range(steps):
        stable = bk.stable_resident()
        sel_off, sel_cart = draw_batch_selection(cfg, rng, stable, wl.cart_len)
        sess.set_batch(wl.seq_off, sel_off, sel_cart, wl.Q, wl.K_self, wl.V_self, wl.dO, step)
        want = bk.slot_table(wl.seq_off.tolist(), sel_off.tolist(), sel_cart.tolist(), step)
        got = cas.cas_slot_table_export(sess.tab)
        assert got["sel_slot"].tolist() == want[0] and got["inv_off"].tolist() == want[1]
        assert got["inv_seq"].tolist() == want[2] and got["P"].tolist() == want[3]
        prot = sorted(set(sel_cart.tolist()))
        man, n = cas.cas_plan_rotation(sess.pool, step, cfg.rotate_in, cfg.rotate_out, prot, 260604)
        wman = bk.plan_rotation(step, cfg.rotate_in, cfg.rotate_out, prot, 260604)
        assert [man[i].as_tuple() for i in range(n)] == [e.as_tuple() for e in wman]
        outs = [e for e in wman if e.dir == 0]
        ins = [e for e in wman if e.dir == 1]
        before_out = {e.cart: [sess.read(e.cart, w).copy() for w in STATE] for e in outs}
        before_in = {e.cart: [sess.read(e.cart, w).copy() for w in STATE] for e in ins}
        cas.cas_swap_out(sess.pool, man, n, step, after_stream=main)
        cas.cas_swap_in(sess.pool, man, n, step)
        bk.swap_out(wman, step)
        bk.swap_in(wman, step)
        assert sess.pool.slot_base.tolist() == bk.slot_base and sess.pool.slot_cap.tolist() == bk.slot_cap
        # compute overlaps with the copies in flight on the side stream
        sess.fwd()
        sess.bwd()
        bk.mark_grads(want[0])
        if step % check_attn_every == 0:
            torch.cuda.synchronize()
            g = step % cfg.Hkv
            hs = list(range(g * G, (g + 1) * G))
            # oracle inputs: the CURRENT working copies of the selected cartridges (bf16 -> fp32)
            blocks_K, blocks_V = {}, {}
            for c in prot:
                blocks_K[c] = (sess.read(c, "wK").astype(np.uint32) << 16).view(np.float32)
                blocks_V[c] = (sess.read(c, "wV").astype(np.uint32) << 16).view(np.float32)
            sel = [sel_cart[sel_off[b]:sel_off[b + 1]].tolist() for b in range(cfg.B)]
            Oo, _ = orc.attn_fwd(wl.Q, blocks_K, blocks_V, sel, wl.seq_off, wl.K_self, wl.V_self,
                                 sess.scale, cfg.Hkv, kv_heads=[g])
            assert rel_fro(sess.np(sess.O)[:, hs], Oo[:, hs]) <= TOL_BF16_O_DQ
            dQo, gKo, gVo, dKso, dVso = orc.attn_bwd(wl.Q, blocks_K, blocks_V, sel, wl.seq_off, wl.K_self,
                                                     wl.V_self, wl.dO, sess.scale, cfg.Hkv, kv_heads=[g])
            # every output of the backward pass (north_star: "O, dQ, dK/dV"), dK/dV per slot
            assert rel_fro(sess.np(sess.dQ)[:, hs], dQo[:, hs]) <= TOL_BF16_O_DQ
            for c in prot:
                assert rel_fro(sess.read(c, "gK")[:, g], gKo[c][:, g]) <= TOL_BF16_DKV, (step, c)
                assert rel_fro(sess.read(c, "gV")[:, g], gVo[c][:, g]) <= TOL_BF16_DKV, (step, c)
            assert rel_fro(sess.np(sess.dKs)[:, g], dKso[:, g]) <= TOL_BF16_DKV
            assert rel_fro(sess.np(sess.dVs)[:, g], dVso[:, g]) <= TOL_BF16_DKV
        sess.adam()
        bk.adam_slots()
        cas.cas_swap_commit(sess.pool, main)
        bk.commit()
        counters_equal(sess.pool, bk)
        torch.cuda.synchronize()
        for e in outs:      # K2: bytes in the pinned home == bytes that were in the slot
            for w, old in zip(STATE, before_out[e.cart]):
                np.testing.assert_array_equal(sess.read(e.cart, w), old)
        for e in ins:       # arrival: state bytes identical, working copy = RNE(master), grads zero
            for w, old in zip(STATE, before_in[e.cart]):
                np.testing.assert_array_equal(sess.read(e.cart, w), old)
            np.testing.assert_array_equal(sess.read(e.cart, "wK"), orc.bf16_rne_bits(before_in[e.cart][0]))
            np.testing.assert_array_equal(sess.read(e.cart, "wV"), orc.bf16_rne_bits(before_in[e.cart][1]))
            assert not sess.read(e.cart, "gK").any() and not sess.read(e.cart, "gV").any()
    # least-trained-first: after enough rotations every cartridge has been trained
    sess.close()
    return bk


def test_rotation_small_many_steps():
    cfg = CONFIGS["c3"].scaled(name="c3_small", Hq=8, Hkv=2, n_carts=24, n_slots=12, cart_len=256, B=2,
                               Lq=200, n_dist=3, rotate_in=4, rotate_out=4)
    bk = run_rotation(cfg, steps=8, seed=31)
    assert min(bk.opt_steps) >= 1


def test_rotation_ragged_lengths_uniform_slots():
    cfg = CONFIGS["c4"].scaled(name="c4_rot", Hq=4, Hkv=2, n_carts=14, n_slots=6, B=2, len_mu=5.0,
                               len_min=20, len_max=400, lq_min=50, lq_max=300, n_dist=2, n_dist_max=2,
                               selection="uniform", rotate_in=2, rotate_out=2)
    run_rotation(cfg, steps=6, seed=32)


def test_c3_full_size_two_steps():
    """Full c3 (32 heads, 2048-token cartridges, 128 slots, 16 in / 16 out per step): O, dQ, dK/dV per slot and
    dK_self/dV_self against the oracle at BOTH steps -- step 1 runs on working copies the step-0 Adam has moved and
    on a rotated pool (KV head group = step % Hkv)."""
    run_rotation(CONFIGS["c3"], steps=2, seed=260604, check_attn_every=1)


def test_arrival_into_a_slot_freed_in_an_earlier_round():
    """n_out > n_in leaves slots free after the round is committed; an arrival planned in a LATER round
    into such a slot must still be ordered after that slot's eviction copy (which may be in flight: nothing
    synchronises between the rounds here) -- the evictee's home must hold the bytes the slot held, the arrival's
    slot the bytes of its home, and the attention that follows must see the arrival."""
    cfg = CONFIGS["c3"].scaled(name="c3_late", Hq=8, Hkv=2, n_carts=12, n_slots=8, cart_len=2048, B=2, Lq=130,
                               n_dist=1, rotate_in=0, rotate_out=3)
    wl = make_workload(cfg, 33)
    sess = Session(wl)
    bk = PoolBook(wl.cart_len.tolist(), cfg.n_slots, cfg.Hkv, cfg.D)
    bk.slot_table(wl.seq_off.tolist(), wl.sel_off.tolist(), wl.sel_cart.tolist(), 0)
    main = torch.cuda.current_stream()
    prot = sorted(set(wl.sel_cart.tolist()))
    state0 = {c: [sess.read(c, w).copy() for w in STATE] for c in range(cfg.n_carts)}
    # round 0: three evictions, no arrival
    man, n = cas.cas_plan_rotation(sess.pool, 0, 0, 3, prot, 7)
    wman = bk.plan_rotation(0, 0, 3, prot, 7)
    assert [man[i].as_tuple() for i in range(n)] == [e.as_tuple() for e in wman] and n == 3
    cas.cas_swap_out(sess.pool, man, n, 0, after_stream=main)
    bk.swap_out(wman, 0)
    cas.cas_swap_commit(sess.pool, main)
    bk.commit()
    # round 1, immediately: two arrivals into slots freed by round 0
    man1, n1 = cas.cas_plan_rotation(sess.pool, 1, 2, 0, prot, 7)
    wman1 = bk.plan_rotation(1, 2, 0, prot, 7)
    assert [man1[i].as_tuple() for i in range(n1)] == [e.as_tuple() for e in wman1] and n1 == 2
    freed = {e.slot for e in wman}
    assert all(e.slot in freed for e in wman1)
    cas.cas_swap_in(sess.pool, man1, n1, 1)
    bk.swap_in(wman1, 1)
    cas.cas_swap_commit(sess.pool, main)
    bk.commit()
    counters_equal(sess.pool, bk)
    torch.cuda.synchronize()
    for e in wman:          # evictees: the pinned home holds exactly what the slot held
        for w, old in zip(STATE, state0[e.cart]):
            np.testing.assert_array_equal(sess.read(e.cart, w), old)
    for e in wman1:         # arrivals: the slot holds exactly what the home held
        for w, old in zip(STATE, state0[e.cart]):
            np.testing.assert_array_equal(sess.read(e.cart, w), old)
        np.testing.assert_array_equal(sess.read(e.cart, "wK"), orc.bf16_rne_bits(state0[e.cart][0]))
    sess.close()
