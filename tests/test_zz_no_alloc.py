"""cas_prefix_attn_fwd_noalloc (include/cas.h): the forward call for callers that may not call cudaMalloc -- the
tail blocks' split-KV partials live in a file-scope device array of the library (20,004,864 bytes) instead of the
pool-owned buffer cas_prefix_attn_fwd allocates inside a call.  Checked against the existing path (same kernels, so
the same bits; the gate is the tests' forward tolerance) on two calls in a row that use the shared array with
different split geometries and different inputs, without any synchronisation in between.

This file is collected last on purpose (the suite runs with pytest -x); it passes alone in a fresh process and after
the other tests."""
import numpy as np
import pytest
import torch

from paper_2606_04557_b200 import _build, cas
from paper_2606_04557_b200.harness import Session
from workloads import CONFIGS, make_workload

from parity_util import TOL_BF16_O_DQ, rel_fro

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def built():
    _build.build()
    cas.cas_set_impl(cas.CAS_IMPL_AUTO)
    yield
    cas.cas_set_impl(cas.CAS_IMPL_AUTO)


def tail_cfg(name, **kw):
    base = dict(name=name, Hq=8, Hkv=2, n_carts=9, n_slots=9, cart_len=0, len_mu=6.0, len_sigma=0.5, len_min=200,
                len_max=900, B=5, Lq=0, lq_min=1050, lq_max=1270, n_dist=2, kv_std=1.0)
    base.update(kw)
    return CONFIGS["c2"].scaled(**base)


def reference(sess):
    """The existing path: cas_prefix_attn_fwd (pool-owned scratch)."""
    sess.fwd()
    torch.cuda.synchronize()
    return sess.O.clone(), sess.LSE.clone()


def test_noalloc_forward_equals_the_existing_path_on_two_calls_in_a_row():
    # two pools / tables whose tail splits differ (52 tail blocks x 2 parts; 44 x 3 with four longer sequences), so
    # the second call finds the first call's partials in the shared array at other offsets
    wlA = make_workload(tail_cfg("noalloc_A"), 47)
    wlB = make_workload(tail_cfg("noalloc_B", B=4, lq_min=1300, lq_max=1500, n_dist=3), 48)
    sA, sB = Session(wlA), Session(wlB)
    refA, refB = reference(sA), reference(sB)
    splitA, splitB = cas.cas_slot_table_fwd_split(sA.tab), cas.cas_slot_table_fwd_split(sB.tab)
    assert splitA[0] > 0 and splitB[0] > 0 and splitA != splitB, (splitA, splitB)     # the scratch is really used
    outs = []
    for s in (sA, sB):
        O = torch.full_like(s.O, 9.0)
        LSE = torch.full_like(s.LSE, 9.0)
        outs.append((O, LSE))
    # two calls in a row on one stream, no synchronisation in between (calls that overlap on the GPU would race: cas.h)
    cas.cas_prefix_attn_fwd_noalloc(sA.pool, sA.tab, sA.cfg.Hq, sA.Q, sA.Ks, sA.Vs, sA.scale, *outs[0])
    cas.cas_prefix_attn_fwd_noalloc(sB.pool, sB.tab, sB.cfg.Hq, sB.Q, sB.Ks, sB.Vs, sB.scale, *outs[1])
    torch.cuda.synchronize()
    for (O, LSE), (Or, Lr), name in ((outs[0], refA, "A"), (outs[1], refB, "B")):
        assert torch.isfinite(O.float()).all() and torch.isfinite(LSE).all(), name
        assert rel_fro(O.float().cpu().numpy(), Or.float().cpu().numpy()) <= TOL_BF16_O_DQ, name
        np.testing.assert_allclose(LSE.cpu().numpy(), Lr.cpu().numpy(), rtol=2e-3, atol=2e-3)
        assert torch.equal(O, Or) and torch.equal(LSE, Lr), name       # same kernels, fixed merge order: same bits
    # a third call with NEW inputs on table A: stale partials of the two earlier calls must not leak into it
    sA.Q.mul_(-0.5)
    refA2 = reference(sA)
    assert not torch.equal(refA2[0], refA[0])
    O, LSE = torch.full_like(sA.O, 9.0), torch.full_like(sA.LSE, 9.0)
    cas.cas_prefix_attn_fwd_noalloc(sA.pool, sA.tab, sA.cfg.Hq, sA.Q, sA.Ks, sA.Vs, sA.scale, O, LSE)
    torch.cuda.synchronize()
    assert rel_fro(O.float().cpu().numpy(), refA2[0].float().cpu().numpy()) <= TOL_BF16_O_DQ
    assert torch.equal(O, refA2[0]) and torch.equal(LSE, refA2[1])
    sA.close()
    sB.close()


def test_noalloc_forward_prefix_only_and_unsplit_tables():
    """Prefix-only call (no self block) and a table small enough to need no split (no scratch at all)."""
    wl = make_workload(tail_cfg("noalloc_C"), 49)
    s = Session(wl)
    s.fwd(self_block=False)
    torch.cuda.synchronize()
    Or, Lr = s.O.clone(), s.LSE.clone()
    O, LSE = torch.full_like(s.O, 9.0), torch.full_like(s.LSE, 9.0)
    cas.cas_prefix_attn_fwd_noalloc(s.pool, s.tab, s.cfg.Hq, s.Q, None, None, s.scale, O, LSE)
    torch.cuda.synchronize()
    assert rel_fro(O.float().cpu().numpy(), Or.float().cpu().numpy()) <= TOL_BF16_O_DQ
    assert torch.equal(O, Or) and torch.equal(LSE, Lr)
    s.close()
    small = make_workload(CONFIGS["c2"].scaled(name="noalloc_small", Hq=8, Hkv=2, n_carts=5, n_slots=5, cart_len=300,
                                               B=2, Lq=300, n_dist=1), 50)
    s = Session(small)
    Or, Lr = reference(s)
    assert cas.cas_slot_table_fwd_split(s.tab) == (0, 1)
    O, LSE = torch.full_like(s.O, 9.0), torch.full_like(s.LSE, 9.0)
    cas.cas_prefix_attn_fwd_noalloc(s.pool, s.tab, s.cfg.Hq, s.Q, s.Ks, s.Vs, s.scale, O, LSE)
    torch.cuda.synchronize()
    assert torch.equal(O, Or) and torch.equal(LSE, Lr)
    s.close()


def test_noalloc_forward_rejects_what_it_cannot_serve():
    """fp32 pools run on the CUDA-core path and decode-shaped tables on the decode kernel (which allocates at a table's
    first call): both are refused with CAS_ERR_SHAPE, nothing is launched."""
    wl = make_workload(CONFIGS["c1"], 3)
    s = Session(wl)
    with pytest.raises(cas.CasError) as e:
        cas.cas_prefix_attn_fwd_noalloc(s.pool, s.tab, s.cfg.Hq, s.Q, s.Ks, s.Vs, s.scale, s.O, s.LSE)
    assert e.value.name == "CAS_ERR_SHAPE"
    s.close()
    dec = make_workload(CONFIGS["c5_top8"].scaled(name="noalloc_dec", Hq=8, Hkv=2, n_carts=4, n_slots=4, cart_len=128,
                                                  B=3), 4)
    s = Session(dec)
    with pytest.raises(cas.CasError) as e:
        cas.cas_prefix_attn_fwd_noalloc(s.pool, s.tab, s.cfg.Hq, s.Q, s.Ks, s.Vs, s.scale, s.O, s.LSE)
    assert e.value.name == "CAS_ERR_SHAPE"
    with pytest.raises(cas.CasError) as e:
        cas.cas_prefix_attn_fwd_noalloc(s.pool, s.tab, s.cfg.Hq, None, s.Ks, s.Vs, s.scale, s.O, s.LSE)
    assert e.value.name in ("CAS_ERR_INVALID_ARG", "CAS_ERR_SHAPE")
    s.close()
