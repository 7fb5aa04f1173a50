"""GPU parity of RoPE FUSED into the attention calls ("query token position IDs
must be offset by the total number of active cartridge KV tokens"): cas_rope_table + cas_prefix_attn_fwd_rope /
_bwd_rope against the oracle's own composition -- oracle.rope on Q and K_self, oracle.attn_fwd / attn_bwd on the
rotated tensors, oracle.rope(inverse) on dQ and dK_self.  No new oracle arithmetic: the chain rule through a rotation
is its transpose (pinned in tests/test_oracle_pins.py).

The rotated queries are a defined bf16 OUTPUT of the forward call (Q_rot, consumed by the backward call), so the
oracle's attention runs on oracle.rope(Q) rounded to bf16 -- the rounding is the storage format of that output, the
same one the stand-alone cas_rope_apply test allows (4e-3)."""
import numpy as np
import pytest
import torch

from oracle import cas_oracle as orc
from paper_2606_04557_b200 import _build, cas
from paper_2606_04557_b200.harness import Session
from workloads import CONFIGS, make_workload, round_to_dtype

from parity_util import TOL_BF16_DKV, TOL_BF16_O_DQ, oracle_inputs, rel_fro, rel_max

pytestmark = pytest.mark.gpu
BASE = 1.0e6


@pytest.fixture(scope="module", autouse=True)
def built():
    _build.build()
    cas.cas_set_impl(cas.CAS_IMPL_AUTO)


def run_fused(wl, layout, kv_heads, pos_off, self_block=True):
    cfg = wl.cfg
    sess = Session(wl)
    G = cfg.Hq // cfg.Hkv
    hs = [h for g in kv_heads for h in range(g * G, (g + 1) * G)]
    cs = torch.empty((wl.T, cfg.D // 2, 2), dtype=torch.float32, device="cuda")
    cas.cas_rope_table(wl.seq_off, pos_off, cfg.D, BASE, cs)
    rope = cas.Rope(cs, layout)
    Q_rot, Ks_rot = torch.zeros_like(sess.Q), torch.zeros_like(sess.Ks)
    Q0, Ks0 = sess.Q.clone(), sess.Ks.clone()
    Ks, Vs = (sess.Ks, sess.Vs) if self_block else (None, None)
    cas.cas_prefix_attn_fwd_rope(sess.pool, sess.tab, cfg.Hq, sess.Q, Ks, Vs, rope, Q_rot, Ks_rot if self_block else None,
                                 sess.scale, sess.O, sess.LSE)
    cas.cas_prefix_attn_bwd_rope(sess.pool, sess.tab, cfg.Hq, Q_rot, Ks_rot if self_block else None, Vs, sess.O,
                                 sess.LSE, sess.dO, rope, sess.scale, sess.dQ, sess.dKs if self_block else None,
                                 sess.dVs if self_block else None, sess.ws)
    torch.cuda.synchronize()
    assert torch.equal(sess.Q, Q0) and torch.equal(sess.Ks, Ks0)          # the inputs are const
    # ---- the oracle's composition
    bK, bV, sel = oracle_inputs(wl)
    Qr = round_to_dtype(orc.rope(wl.Q, wl.seq_off, pos_off, BASE, layout).astype(np.float32), "bf16")
    Kr = round_to_dtype(orc.rope(wl.K_self, wl.seq_off, pos_off, BASE, layout).astype(np.float32), "bf16")
    got_Qr = Q_rot.float().cpu().numpy()
    assert rel_fro(got_Qr, Qr) <= 4e-3                                     # every head: the rotation itself
    assert np.abs(got_Qr - Qr).max() <= 2.0 ** -7 * np.abs(Qr).max()       # no element off by more than an ulp or two
    if self_block:
        assert rel_fro(Ks_rot.float().cpu().numpy(), Kr) <= 4e-3
    Ko, Vo = (Kr, wl.V_self) if self_block else (None, None)
    Oo, Lo = orc.attn_fwd(Qr, bK, bV, sel, wl.seq_off, Ko, Vo, sess.scale, cfg.Hkv, kv_heads=kv_heads)
    O, LSE = sess.np(sess.O), sess.np(sess.LSE)
    assert rel_fro(O[:, hs], Oo[:, hs]) <= TOL_BF16_O_DQ
    assert rel_max(LSE[:, hs], Lo[:, hs]) <= 2e-3
    dQo, gKo, gVo, dKso, dVso = orc.attn_bwd(Qr, bK, bV, sel, wl.seq_off, Ko, Vo, wl.dO, sess.scale, cfg.Hkv,
                                             kv_heads=kv_heads)
    dQ_want = orc.rope(dQo, wl.seq_off, pos_off, BASE, layout, inverse=True)
    assert rel_fro(sess.np(sess.dQ)[:, hs], dQ_want[:, hs]) <= TOL_BF16_O_DQ
    for c in sorted(gKo.keys()):
        assert rel_fro(sess.read(c, "gK")[:, kv_heads], gKo[c][:, kv_heads]) <= TOL_BF16_DKV, c
        assert rel_fro(sess.read(c, "gV")[:, kv_heads], gVo[c][:, kv_heads]) <= TOL_BF16_DKV, c
    if self_block:
        dKs_want = orc.rope(dKso, wl.seq_off, pos_off, BASE, layout, inverse=True)
        assert rel_fro(sess.np(sess.dKs)[:, kv_heads], dKs_want[:, kv_heads]) <= TOL_BF16_DKV
        assert rel_fro(sess.np(sess.dVs)[:, kv_heads], dVso[:, kv_heads]) <= TOL_BF16_DKV
    # the fused result must differ from the un-rotated attention: with kv_std = 1 the scores have unit spread, so
    # attention computed on un-rotated queries (a rotation lost between shared memory and the MMA) is far off
    sess.fwd(self_block=self_block)
    torch.cuda.synchronize()
    assert rel_fro(sess.np(sess.O)[:, hs], Oo[:, hs]) > 10 * TOL_BF16_O_DQ
    return sess


@pytest.mark.parametrize("layout", [0, 1])
def test_fused_rope_small_ragged(layout):
    """Ragged sequences (one Q tile, two Q tiles, a partly filled last tile), ragged cartridges, the paper's offset =
    visible prefix tokens per sequence (cas_position_offsets), both pair layouts, all KV head groups.  K/V ~ N(0, 1)
    instead of the workloads' 0.02: the softmax must be peaked enough for O to depend on the rotation."""
    cfg = CONFIGS["c2"].scaled(name="c2_rope", Hq=8, Hkv=2, n_carts=7, n_slots=7, cart_len=0, len_mu=5.5, len_sigma=0.6,
                               len_min=40, len_max=500, B=4, Lq=0, lq_min=60, lq_max=420, n_dist=2, kv_std=1.0)
    wl = make_workload(cfg, 61 + layout)
    sess0 = Session(wl)
    _, P = cas.cas_position_offsets(sess0.pool, sess0.tab)
    sess0.close()
    run_fused(wl, layout, [0, 1], np.asarray(P, dtype=np.int64)).close()


def test_fused_rope_prefix_only_and_large_offsets():
    """Prefix-only call (no self block: only Q is rotated) with position offsets of a 256,000-token prefix, where a
    float angle would be off by 1e-2 rad."""
    cfg = CONFIGS["c2"].scaled(name="c2_rope_p", Hq=8, Hkv=2, n_carts=5, n_slots=5, cart_len=300, B=3, Lq=200, n_dist=1, kv_std=1.0)
    wl = make_workload(cfg, 63)
    run_fused(wl, 1, [1], np.array([256000, 0, 99999], dtype=np.int64), self_block=False).close()


def test_fused_rope_with_the_forward_tail_split():
    """More blocks than SMs with a part-filled last wave: the split blocks' parts all rotate their own copy of the Q
    tile in shared memory, part 0 writes Q_rot."""
    cfg = CONFIGS["c2"].scaled(name="c2_rope_tail", Hq=8, Hkv=2, n_carts=9, n_slots=9, cart_len=0, len_mu=6.0,
                               len_sigma=0.5, len_min=200, len_max=900, B=5, Lq=0, lq_min=1050, lq_max=1270, n_dist=2, kv_std=1.0)
    wl = make_workload(cfg, 47)
    sess = run_fused(wl, 1, [cfg.Hkv - 1], np.full(cfg.B, 4096, dtype=np.int64))
    assert cas.cas_slot_table_fwd_split(sess.tab)[0] > 0
    sess.close()


def test_fused_rope_in_the_layered_step_equals_the_separate_calls():
    """cas_train_step_layers with io[].rope: same O / dQ bits as cas_prefix_attn_fwd_rope + _bwd_rope called by hand
    (L = 2, one micro-batch); and the argument errors of the fused calls."""
    L = 2
    cfg = CONFIGS["c2"].scaled(name="c2_rope_l", Hq=8, Hkv=2, n_carts=5, n_slots=5, cart_len=200, B=2, Lq=260, n_dist=1)
    wl = make_workload(cfg, 65)
    pool = cas.Pool(cas.CAS_BF16, cfg.Hkv, cfg.D, wl.cart_len, cfg.n_slots, n_layers=L)
    for l in range(L):
        for c in range(cfg.n_carts):
            cas.cas_pool_load(pool, c, *wl.cart_kv(c), layer=l)
    tab = cas.cas_slot_table_build(pool, wl.seq_off, wl.sel_off, wl.sel_cart, 0)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to("cuda").to(torch.bfloat16)
    cs = torch.empty((wl.T, cfg.D // 2, 2), dtype=torch.float32, device="cuda")
    cas.cas_rope_table(wl.seq_off, np.array([1000, 2000], dtype=np.int64), cfg.D, BASE, cs)
    rope = cas.Rope(cs, 1)
    scale = 1.0 / float(np.sqrt(cfg.D))

    def bufs():
        t = dict(Q=dev(wl.Q), K_self=dev(wl.K_self), V_self=dev(wl.V_self), dO=dev(wl.dO))
        t["O"], t["dQ"], t["Q_rot"] = torch.empty_like(t["Q"]), torch.empty_like(t["Q"]), torch.empty_like(t["Q"])
        t["dK_self"], t["dV_self"], t["K_self_rot"] = (torch.empty_like(t["K_self"]) for _ in range(3))
        t["LSE"] = torch.empty((wl.T, cfg.Hq), dtype=torch.float32, device="cuda")
        t["rope"] = rope
        return t

    io = [[bufs() for _ in range(L)]]
    ws = torch.empty(cas.cas_train_step_layers_workspace_bytes(pool, [tab], cfg.Hq), dtype=torch.uint8, device="cuda")
    acfg = cas.AdamCfg(0.0, cfg.beta1, cfg.beta2, cfg.eps, 1, 0)             # lr = 0: the pool does not move
    cas.cas_train_step_layers(pool, [tab], cfg.Hq, io, scale, acfg, workspace=ws)
    torch.cuda.synchronize()
    for l in range(L):
        t = bufs()
        cas.cas_prefix_attn_fwd_rope(pool, tab, cfg.Hq, t["Q"], t["K_self"], t["V_self"], rope, t["Q_rot"], t["K_self_rot"],
                                     scale, t["O"], t["LSE"], layer=l)
        torch.cuda.synchronize()
        assert torch.equal(t["O"], io[0][l]["O"]) and torch.equal(t["Q_rot"], io[0][l]["Q_rot"])
        assert torch.equal(t["LSE"], io[0][l]["LSE"])
    with pytest.raises(cas.CasError) as e:                                   # missing outputs
        cas.cas_prefix_attn_fwd_rope(pool, tab, cfg.Hq, t["Q"], t["K_self"], t["V_self"], rope, None, None, scale, t["O"],
                                     t["LSE"])
    assert e.value.name == "CAS_ERR_INVALID_ARG"
    with pytest.raises(cas.CasError) as e:                                   # bad layout
        cas.cas_prefix_attn_fwd_rope(pool, tab, cfg.Hq, t["Q"], t["K_self"], t["V_self"], cas.Rope(cs, 2), t["Q_rot"],
                                     t["K_self_rot"], scale, t["O"], t["LSE"])
    assert e.value.name == "CAS_ERR_INVALID_ARG"
    tab.close()
    pool.close()
