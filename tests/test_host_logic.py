"""CPU-only tests of libcas' host logic through the C ABI: the library loads, exports every symbol
declared in include/cas.h, and its integer bookkeeping (slot tables, inverted tables, rotation
plans, manifests, counters) is bit-exact against the independent pure-Python oracle.  Uses
bookkeeping-only pools (dev_arena == NULL), so no CUDA call is made."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from oracle.bookkeeping import BookError, PoolBook, position_offsets
from paper_2606_04557_b200 import _build, cas

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module", autouse=True)
def built():
    _build.build()


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "cas.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    names = set(re.findall(r"\b(cas_[a-z_0-9]+)\s*\(", hdr))
    assert len(names) >= 25
    lib = cas.lib()
    for n in sorted(names):
        assert hasattr(lib, n), n
    assert "libcas" in cas.cas_version()


def host_pool(cart_len, n_slots, Hkv=2, D=32, tile=0):
    return cas.Pool(cas.CAS_BF16, Hkv, D, cart_len, n_slots, tile_tokens=tile, device=None)


def manifest_tuples(arr, n):
    return [arr[i].as_tuple() for i in range(n)]


def counters_equal(pool, bk):
    c = cas.cas_pool_counters(pool)
    assert c["slot_of"].tolist() == bk.slot_of
    assert c["cart_in"].tolist() == bk.cart_in
    assert c["opt_steps"].tolist() == bk.opt_steps
    assert c["last_used"].tolist() == bk.last_used
    assert c["in_transit"].tolist() == bk.in_transit
    assert c["grad_dirty"].tolist() == bk.grad_dirty


def test_layer_axis_layout_and_manifest_bytes():
    """a cartridge has a layer axis; its pinned home (and a manifest entry's nbytes) covers all L layers,
    the device arena holds L carvings."""
    lens = [48, 16, 80, 32, 64]
    one = cas.Pool(cas.CAS_BF16, 2, 32, lens, 3, tile_tokens=16, device=None)
    pool = cas.Pool(cas.CAS_BF16, 2, 32, lens, 3, tile_tokens=16, device=None, n_layers=4)
    bk = PoolBook(lens, 3, 2, 32, tile_tokens=16, n_layers=4)
    assert pool.dev_bytes == 4 * one.dev_bytes and pool.host_bytes == 4 * one.host_bytes
    assert pool.host_bytes == sum(bk.home_bytes(c) for c in range(5))
    man, n = cas.cas_plan_rotation(pool, 0, 2, 2, [0], 5)
    assert manifest_tuples(man, n) == [e.as_tuple() for e in bk.plan_rotation(0, 2, 2, [0], 5)]
    assert man[0].nbytes == 4 * 6 * lens[man[0].cart] * 64 * 4


def test_layout_matches_oracle():
    rng = np.random.default_rng(0)
    lens = rng.integers(1, 700, size=17).tolist()
    for n_slots, tile in ((17, 0), (5, 0), (17, 16), (4, 64)):
        pool = host_pool(lens, n_slots, tile=tile)
        bk = PoolBook(lens, n_slots, 2, 32, tile_tokens=tile or 128)
        assert pool.slot_base.tolist() == bk.slot_base
        assert pool.slot_cap.tolist() == bk.slot_cap
        assert pool.pool_tokens == bk.pool_tokens
        assert pool.host_bytes == sum(bk.home_bytes(c) for c in range(17))
        counters_equal(pool, bk)


def run_protocol(N, S, steps, n_in, n_out, seed, rng, lens=None, B=3, nsel=4, tile=0, budget=0):
    """K4 step protocol driven identically through the library and the oracle."""
    lens = lens or [256] * N
    pool = cas.Pool(cas.CAS_BF16, 2, 32, lens, S, tile_tokens=tile, device=None, budget_tokens=budget)
    bk = PoolBook(lens, S, 2, 32, tile_tokens=tile or 128, budget_tokens=budget)
    assert pool.slot_base.tolist() == bk.slot_base and pool.slot_cap.tolist() == bk.slot_cap
    acfg = cas.AdamCfg(1e-3, 0.9, 0.999, 1e-8, 0, 1)
    for step in range(steps):
        stable = bk.stable_resident()
        sel, sel_off = [], [0]
        for b in range(B):
            k = int(rng.integers(0, min(nsel, len(stable)) + 1))
            sel += rng.choice(stable, size=k, replace=False).tolist()
            sel_off.append(len(sel))
        seq_off = np.concatenate([[0], np.cumsum(rng.integers(1, 300, size=B))])
        tab = cas.cas_slot_table_build(pool, seq_off, sel_off, sel, step)
        want = bk.slot_table(seq_off.tolist(), sel_off, sel, step)
        got = cas.cas_slot_table_export(tab)
        assert got["sel_slot"].tolist() == want[0]
        assert got["inv_off"].tolist() == want[1]
        assert got["inv_seq"].tolist() == want[2]
        assert got["P"].tolist() == want[3]
        lq = np.diff(seq_off)
        assert tab.info.pairs_per_head == int(sum(l * p + l * (l + 1) // 2 for l, p in zip(lq, want[3])))
        tot, P = cas.cas_position_offsets(pool, tab)
        assert (tot, P.tolist()) == position_offsets(bk, want[3])
        man, n = cas.cas_plan_rotation(pool, step, n_in, n_out, sorted(set(sel)), seed)
        wman = bk.plan_rotation(step, n_in, n_out, sorted(set(sel)), seed)
        assert manifest_tuples(man, n) == [e.as_tuple() for e in wman]
        cas.cas_swap_out(pool, man, n, step, host_only=True)
        cas.cas_swap_in(pool, man, n, step)
        bk.swap_out(wman, step)
        bk.swap_in(wman, step)
        counters_equal(pool, bk)
        assert pool.slot_base.tolist() == bk.slot_base and pool.slot_cap.tolist() == bk.slot_cap
        cas.cas_adam_step(pool, acfg, host_only=True)
        bk.adam_slots()
        cas.cas_swap_commit(pool, host_only=True)
        bk.commit()
        counters_equal(pool, bk)
        tab.close()
    return pool, bk


def test_protocol_bit_exact_uniform():
    rng = np.random.default_rng(1)
    run_protocol(N=40, S=12, steps=50, n_in=3, n_out=3, seed=0xDEADBEEFCAFE, rng=rng)


def test_protocol_bit_exact_config3_shape():
    rng = np.random.default_rng(2)
    pool, bk = run_protocol(N=256, S=128, steps=24, n_in=16, n_out=16, seed=260604, rng=rng, B=4, nsel=16)
    assert sum(1 for c in range(256) if bk.slot_of[c] >= 0) == 128


def test_protocol_bit_exact_ragged_lengths_and_uneven_in_out():
    rng = np.random.default_rng(3)
    lens = rng.integers(16, 900, size=30).tolist()
    run_protocol(N=30, S=9, steps=40, n_in=4, n_out=2, seed=7, rng=rng, lens=lens)
    run_protocol(N=30, S=9, steps=40, n_in=1, n_out=5, seed=8, rng=rng, lens=lens)


def test_protocol_bit_exact_paged_pool():
    """16-token pages, first-fit extents, Table 8's 50-100x size range (16-64 tokens) and a
    wider one (fragmentation: some arrivals are skipped); manifests (with their extents), slot handles and counters
    bit-exact against the oracle over many rotations."""
    rng = np.random.default_rng(4)
    lens = (16 * rng.integers(1, 5, size=60)).tolist()                      # 16..64 tokens
    run_protocol(N=60, S=20, steps=60, n_in=5, n_out=5, seed=9, rng=rng, lens=lens, tile=16, budget=16 * 64)
    lens = rng.integers(1, 400, size=40).tolist()                           # ragged, not multiples of the page
    run_protocol(N=40, S=12, steps=60, n_in=4, n_out=3, seed=10, rng=rng, lens=lens, tile=16, budget=16 * 240)
    with pytest.raises(cas.CasError) as e:                                  # the initial cartridges must fit
        cas.Pool(cas.CAS_BF16, 2, 32, [64] * 8, 4, tile_tokens=16, device=None, budget_tokens=16 * 15)
    assert e.value.name == "CAS_ERR_CAPACITY"


def test_hand_worked_trace_through_the_library():
    NB = 6 * 16 * 4 * 4
    pool = cas.Pool(cas.CAS_F32, 1, 32, [16] * 6, 3, tile_tokens=16, device=None)
    NB = 6 * 16 * 32 * 4
    for c, s in enumerate([0, 0, 0, 5, 2, 9]):
        cas.cas_pool_set_counters(pool, c, s, -1)
    tab = cas.cas_slot_table_build(pool, [0, 4, 9], [0, 2, 3], [1, 0, 1], 0)
    e = cas.cas_slot_table_export(tab)
    assert e["sel_slot"].tolist() == [1, 0, 1] and e["inv_off"].tolist() == [0, 1, 3, 3]
    assert e["inv_seq"].tolist() == [0, 0, 1] and e["P"].tolist() == [32, 16]
    man, n = cas.cas_plan_rotation(pool, 0, 1, 1, [0, 1], 1)
    assert manifest_tuples(man, n) == [(2, 2, 0, 32, 2 * NB, NB), (4, 2, 1, 32, 4 * NB, NB)]


@pytest.mark.parametrize("args,code", [
    (([0, 4], [0, 2], [1, 1]), "CAS_ERR_INVALID_ARG"),     # duplicate
    (([0, 4], [0, 1], [5]), "CAS_ERR_NOT_RESIDENT"),
    (([0, 0], [0, 1], [1]), "CAS_ERR_SHAPE"),              # empty sequence
    (([0, 4], [0, 1], [99]), "CAS_ERR_INVALID_ARG"),
])
def test_error_codes(args, code):
    pool = host_pool([64] * 6, 3)
    with pytest.raises(cas.CasError) as ei:
        cas.cas_slot_table_build(pool, *args, 0)
    assert ei.value.name == code


def test_busy_and_data_errors():
    pool = host_pool([64] * 6, 3)
    man, n = cas.cas_plan_rotation(pool, 0, 1, 1, [], 1)
    cas.cas_swap_out(pool, man, n, 0, host_only=True)
    with pytest.raises(cas.CasError) as ei:
        cas.cas_slot_table_build(pool, [0, 4], [0, 1], [man[0].cart], 0)
    assert ei.value.name == "CAS_ERR_BUSY"
    with pytest.raises(cas.CasError) as ei:
        cas.cas_swap_out(pool, man, n, 0, host_only=True)
    assert ei.value.name == "CAS_ERR_BUSY"
    with pytest.raises(cas.CasError) as ei:                  # no data in a bookkeeping-only pool
        cas.cas_pool_load(pool, 0, np.zeros((64, 2, 32), np.float32), np.zeros((64, 2, 32), np.float32))
    assert ei.value.name == "CAS_ERR_INVALID_ARG"
    with pytest.raises(cas.CasError):
        cas.Pool(cas.CAS_BF16, 2, 48, [64], 1, device=None)  # D not a multiple of 32


# ---------------------------------------------------------------------------------------------
# NEXT-3: Eq. 1 sampler, LR schedule, per-cartridge warmup -- the library against the oracle, bit-exact
# ---------------------------------------------------------------------------------------------
def test_sampler_bit_exact_against_oracle():
    from oracle.bookkeeping import PoolBook, sample_selection
    cart_len = [64] * 30
    pool = host_pool(cart_len, 20)                         # cartridges 0..19 resident
    bk = PoolBook(cart_len, 20, 2, 32)
    rng = np.random.default_rng(5)
    for step, (p_iso, kmin, kmax) in enumerate([(0.75, 1, 10), (0.0, 3, 3), (1.0, 1, 5), (0.3, 0, 25), (0.5, 19, 40)]):
        targets = rng.integers(0, 20, size=257).tolist()
        so, sc = cas.cas_sample_selection(pool, targets, p_iso, kmin, kmax, 260604 + step, step)
        wo, wc = sample_selection(bk, targets, p_iso, kmin, kmax, 260604 + step, step)
        assert so.tolist() == wo and sc.tolist() == wc
        tab = cas.cas_slot_table_build(pool, np.arange(258, dtype=np.int32), so, sc, step)   # a valid selection
        tab.close()
    with pytest.raises(cas.CasError) as e:
        cas.cas_sample_selection(pool, [25], 0.5, 1, 2, 1, 0)                                # not resident
    assert e.value.name == "CAS_ERR_NOT_RESIDENT"
    pool.close()


def test_lr_schedule_and_warmup_scales_against_oracle():
    from oracle.bookkeeping import lr_global, warmup_scale
    cfg = cas.LrCfg(0.1, 200, 0.002, 0.02, 14200)
    for t in [0, 1, 57, 199, 200, 201, 5000, 14199, 14200, 99999]:
        assert cas.cas_lr_schedule(cfg, t) == lr_global(t, 0.1, 200, 0.002, 0.02, 14200)
    pool = host_pool([32] * 8, 8)
    for c, s in enumerate([0, 1, 4, 5, 9, 14, 19, 400]):
        cas.cas_pool_set_counters(pool, c, s, 0)
    got = cas.cas_warmup_scales(pool, list(range(8)), 20, 4)
    want = [warmup_scale(s, 20, 4) for s in [0, 1, 4, 5, 9, 14, 19, 400]]
    assert got.tolist() == [np.float32(w) for w in want]
    assert cas.cas_warmup_scales(pool, [3, 0], 7, 3).tolist() == [np.float32(warmup_scale(5, 7, 3)),
                                                                  np.float32(warmup_scale(0, 7, 3))]
    pool.close()


def test_select_retrieved_bit_exact_against_oracle():
    from oracle.bookkeeping import select_retrieved
    rng = np.random.default_rng(17)
    for _ in range(300):
        n_chunks = int(rng.integers(1, 60))
        mp = rng.integers(0, 15, size=n_chunks).tolist()
        k = int(rng.integers(0, 12))
        ranked = rng.integers(0, n_chunks, size=k).tolist()          # repeats allowed: a chunk may be returned twice
        cap = int(rng.integers(0, 9))
        assert cas.cas_select_retrieved(ranked, mp, cap).tolist() == select_retrieved(ranked, mp, cap)
    with pytest.raises(cas.CasError) as e:
        cas.cas_select_retrieved([3], [0, 1], 2)
    assert e.value.name == "CAS_ERR_INVALID_ARG"


def test_batch_sampler_for_the_bench_keeps_the_uniform_recipe():
    """workloads.generate.draw_batch_selection_uniform (bench.py's rotation configs draw a fresh batch every step):
    same recipe as draw_batch_selection("uniform") -- per sequence a target and n_dist DISTINCT distractors among the
    candidates, every candidate equally likely at every position, n_dist ~ U{0..n_dist_max} -- checked as properties
    and by frequencies over many draws."""
    from workloads import CONFIGS
    from workloads.generate import draw_batch_selection_uniform
    cfg = CONFIGS["c_pages"]
    rng = np.random.Generator(np.random.PCG64(7))
    cand = np.arange(40, 240, dtype=np.int32)[::2]                  # 100 candidates, not 0..n-1
    counts = np.zeros(cfg.n_dist_max + 2, np.int64)
    first = np.zeros(400, np.int64)
    for _ in range(300):
        sel_off, sel_cart = draw_batch_selection_uniform(cfg, rng, cand)
        assert sel_off[0] == 0 and len(sel_off) == cfg.B + 1 and sel_off[-1] == len(sel_cart)
        assert np.isin(sel_cart, cand).all()
        for b in range(cfg.B):
            s = sel_cart[sel_off[b]:sel_off[b + 1]]
            assert 1 <= len(s) <= cfg.n_dist_max + 1 and len(set(s.tolist())) == len(s)
            counts[len(s)] += 1
            first[s[0]] += 1
    n = 300 * cfg.B
    # list lengths 1..11 equally likely (binomial 5-sigma band), targets uniform over the candidates
    exp = n / (cfg.n_dist_max + 1)
    assert counts[0] == 0 and np.all(np.abs(counts[1:] - exp) < 5 * np.sqrt(exp))
    f = first[cand]
    assert first.sum() == f.sum() and np.all(np.abs(f - n / len(cand)) < 5 * np.sqrt(n / len(cand)))
    # a fixed n_dist (config 3: target + 15 distractors of 64)
    c3 = CONFIGS["c3"]
    sel_off, sel_cart = draw_batch_selection_uniform(c3, rng, np.arange(64))
    assert np.diff(sel_off).tolist() == [1 + c3.n_dist] * c3.B
