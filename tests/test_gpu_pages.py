"""GPU parity of the paged pool: PAPER.md:442-446 -- cartridge sizes are whole 16-token pages
("fixed-size pages of 16 tokens ... minimum cartridge size of 16 tokens"), Table 8 16-64-token
cartridges at 50-100x compression.  With tile_tokens = 16 the pool is allocated in pages, a sequence's small
cartridges (and the ragged ends of its big ones) are PACKED into shared 128-key MMA tiles, their gradients are
scattered back per key, and rotation moves contiguous page runs chosen first-fit."""
import numpy as np
import pytest
import torch

from paper_2606_04557_b200 import _build, cas
from workloads import CONFIGS, make_workload

from parity_util import check_adam_isolated, check_attention
from test_gpu_rotation import run_rotation

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def built():
    _build.build()
    yield
    cas.cas_set_impl(cas.CAS_IMPL_AUTO)


def pages_cfg(**kw):
    base = dict(name="c_pages_small", Hq=8, Hkv=2, n_carts=24, n_slots=24, B=5, Lq=150, n_dist_max=6, rotate_in=0,
                rotate_out=0, budget_tokens=0)
    base.update(kw)
    return CONFIGS["c_pages"].scaled(**base)


@pytest.mark.parametrize("impl", [cas.CAS_IMPL_AUTO, cas.CAS_IMPL_SIMT])
def test_tiny_cartridges_packed_into_shared_tiles(impl):
    """16-64-token cartridges, all resident: every sequence's whole prefix (1-7 cartridges) fits ONE or TWO packed
    tiles; forward, backward (dK/dV per slot, several sequences adding to one cartridge), Adam, untouched slots."""
    cfg = pages_cfg()
    wl = make_workload(cfg, 91)
    assert set(wl.cart_len.tolist()) <= {16, 32, 48, 64}
    rep = {}
    sess = check_attention(wl, impl, kv_heads=[0, 1], report=rep)
    lay_tokens = sess.pool.pool_tokens
    assert lay_tokens == int(wl.cart_len.sum())                       # whole pages: not a token wasted
    check_adam_isolated(sess, sorted(set(wl.sel_cart.tolist()))[:4])
    sess.close()
    print(impl, rep)


def test_ragged_lengths_full_tiles_plus_packed_remainders():
    """Arbitrary lengths (1..700) in a 16-token-page pool: whole 128-key tiles are read in place and shared by all
    selecting sequences, the ragged ends (with a partly filled last page) go to the per-sequence packed tiles; also
    the prefix-only call."""
    cfg = pages_cfg(name="c_pages_ragged", cart_len=0, len_pages_max=0, len_mu=5.0, len_sigma=1.0, len_min=1,
                    len_max=700, Lq=0, lq_min=3, lq_max=300, n_carts=16, n_slots=16, selection="prop_len")
    wl = make_workload(cfg, 92)
    assert any(l % 16 for l in wl.cart_len.tolist()) and max(wl.cart_len) > 128
    rep = {}
    sess = check_attention(wl, cas.CAS_IMPL_AUTO, kv_heads=[0, 1], report=rep)
    assert sess.pool.pool_tokens <= int(sum((l + 15) // 16 * 16 for l in wl.cart_len))
    sess.close()
    check_attention(make_workload(cfg, 93), cas.CAS_IMPL_AUTO, kv_heads=[1], self_block=False).close()
    print(rep)


def test_decode_over_packed_pages():
    cfg = pages_cfg(name="c_pages_dec", B=9, Lq=1, backward=False, n_dist_max=5)
    check_attention(make_workload(cfg, 94), cas.CAS_IMPL_AUTO, kv_heads=[0, 1]).close()
    cfg = pages_cfg(name="c_pages_dec2", B=40, Lq=1, backward=False, n_dist=-2, selection="all", n_carts=9, n_slots=9)
    check_attention(make_workload(cfg, 95), cas.CAS_IMPL_AUTO, kv_heads=[1]).close()


def test_rotation_in_a_paged_pool():
    """Rotation with first-fit page runs: manifests (with extents), slot handles and counters bit-exact against the
    bookkeeping oracle, byte-exact swaps, attention parity on the rotated pool at every step; the pool holds its
    cartridges within 10 % of the sum of their lengths."""
    cfg = pages_cfg(name="c_pages_rot", n_carts=40, n_slots=16, B=3, Lq=200, n_dist_max=4, rotate_in=4, rotate_out=4,
                    budget_tokens=16 * 48)
    bk = run_rotation(cfg, steps=8, seed=96)
    resident = [c for c in range(40) if bk.slot_of[c] >= 0]
    assert sum(bk.cart_len[c] for c in resident) >= 0.6 * cfg.budget_tokens
    assert min(bk.opt_steps) >= 0


def test_c_pages_full_size_one_step():
    """The full-size c_pages workload (400 cartridges of 16-64 tokens, 200 resident in an 8,960-token pool -- within
    10 % of the 8,304 tokens they hold -- 32 samples x 256 tokens, 20 in / 20 out): two rotation steps with
    attention parity on one KV head group each."""
    cfg = CONFIGS["c_pages"]
    wl = make_workload(cfg)
    assert cfg.budget_tokens <= 1.10 * int(wl.cart_len[:cfg.n_slots].sum())
    run_rotation(cfg, steps=2, seed=260604)
