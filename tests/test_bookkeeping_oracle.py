"""Pins for oracle/bookkeeping.py: a rotation trace worked by hand in this file,
published SplitMix64 test vectors for the priority hash, and structural properties."""
import numpy as np
import pytest

from oracle.bookkeeping import DIR_IN, DIR_OUT, BookError, PoolBook, mix64, position_offsets

NB = 6 * 16 * 4 * 4          # bytes of one 16-token cartridge home: 6 tensors x 16 x (Hkv*D=4) x 4 B
# manifest tuples: (cart, slot, dir, base_tok, host_off, nbytes); base_tok = first pool token of the slot (16 per slot)


def make_book():
    bk = PoolBook([16] * 6, n_slots=3, Hkv=1, D=4, tile_tokens=16)
    bk.opt_steps = [0, 0, 0, 5, 2, 9]
    return bk


def test_splitmix64_vectors():
    """SplitMix64 seeded with 0 emits 0xE220A8397B1DCDAF, 0x6E789E6AA1B965F4, 0x06C45D188009454F
    (widely published reference outputs).  With seed = -0xD1B54A32D192ED03 (mod 2^64) and cart 0
    our pre-mix state is exactly gamma*(step+1), i.e. the generator's state sequence."""
    seed = (-0xD1B54A32D192ED03) % (1 << 64)
    assert mix64(seed, 0, 0) == 0xE220A8397B1DCDAF
    assert mix64(seed, 1, 0) == 0x6E789E6AA1B965F4
    assert mix64(seed, 2, 0) == 0x06C45D188009454F


def test_hand_worked_rotation_trace():
    bk = make_book()
    assert bk.slot_base == [0, 16, 32] and bk.pool_tokens == 48
    assert bk.home_off == [NB * c for c in range(6)]
    # ---- step 0
    sel_slot, inv_off, inv_seq, P = bk.slot_table([0, 4, 9], [0, 2, 3], [1, 0, 1], step=0)
    assert sel_slot == [1, 0, 1]
    assert inv_off == [0, 1, 3, 3] and inv_seq == [0, 0, 1]
    assert P == [32, 16]
    assert position_offsets(bk, P) == (48, [32, 16])          # 3 resident cartridges x 16 tokens
    assert bk.last_used == [0, 0, -1, -1, -1, -1]
    man = bk.plan_rotation(0, n_in=1, n_out=1, protect=[0, 1], seed=1)
    assert [e.as_tuple() for e in man] == [(2, 2, DIR_OUT, 32, 2 * NB, NB), (4, 2, DIR_IN, 32, 4 * NB, NB)]
    bk.swap_out(man, 0)
    bk.swap_in(man, 0)
    assert bk.stable_resident() == [0, 1]
    assert bk.adam_slots() == [0, 1]
    bk.commit()
    assert bk.slot_of == [0, 1, -1, -1, 2, -1] and bk.cart_in == [0, 1, 4]
    assert bk.opt_steps == [1, 1, 0, 5, 2, 9]
    assert bk.last_used == [0, 0, -1, -1, 0, -1]
    # ---- step 1
    sel_slot, inv_off, inv_seq, P = bk.slot_table([0, 3, 5], [0, 1, 3], [4, 0, 4], step=1)
    assert sel_slot == [2, 0, 2]
    assert inv_off == [0, 1, 1, 3] and inv_seq == [1, 0, 1]
    man = bk.plan_rotation(1, n_in=2, n_out=2, protect=[0, 4], seed=1)
    assert [e.as_tuple() for e in man] == [(1, 1, DIR_OUT, 16, NB, NB), (2, 1, DIR_IN, 16, 2 * NB, NB)]
    bk.swap_out(man, 1)
    bk.swap_in(man, 1)
    assert bk.adam_slots() == [0, 2]
    bk.commit()
    assert bk.opt_steps == [2, 1, 0, 5, 3, 9]
    assert bk.slot_of == [0, -1, 1, -1, 2, -1]
    assert bk.last_used == [1, 0, 1, -1, 1, -1]
    # ---- step 2: LRU ties -> smaller cartridge id; arrivals fill freed slots ascending
    man = bk.plan_rotation(2, n_in=1, n_out=2, protect=[], seed=1)
    assert [e.as_tuple() for e in man] == [(0, 0, DIR_OUT, 0, 0, NB), (2, 1, DIR_OUT, 16, 2 * NB, NB),
                                           (1, 0, DIR_IN, 0, NB, NB)]


def test_position_offsets_hand_worked_ragged():
    """PAPER.md:77 "offset by the total number of active cartridge KV tokens": lengths 16, 48, 32, 80, 64 with
    the first three resident -> 96 active tokens; a sample that sees cartridges 2 and 0 has a 48-token visible
    prefix (R7 returns both readings).  After cartridge 1 (48) is swapped for cartridge 4 (64) the
    active total is 16 + 32 + 64 = 112."""
    bk = PoolBook([16, 48, 32, 80, 64], n_slots=3, Hkv=1, D=4, tile_tokens=16)
    _, _, _, P = bk.slot_table([0, 3, 8], [0, 2, 3], [2, 0, 1], step=0)
    assert position_offsets(bk, P) == (96, [48, 48])
    bk.adam_slots()
    man = bk.plan_rotation(1, n_in=1, n_out=1, protect=[0, 2], seed=3)
    assert [(e.cart, e.dir) for e in man][0] == (1, DIR_OUT)
    bk.swap_out(man, 1)
    arrival = [e.cart for e in man if e.dir == DIR_IN]
    bk.swap_in(man, 1)
    assert position_offsets(bk, [])[0] == 96                  # residency flips at commit, not before
    bk.commit()
    assert position_offsets(bk, [])[0] == 96 - 48 + bk.cart_len[arrival[0]]


def test_validation_errors():
    bk = make_book()
    with pytest.raises(BookError, match="duplicate"):
        bk.slot_table([0, 4], [0, 2], [1, 1], 0)
    with pytest.raises(BookError, match="NOT_RESIDENT"):
        bk.slot_table([0, 4], [0, 1], [5], 0)
    with pytest.raises(BookError, match="SHAPE"):
        bk.slot_table([0, 0], [0, 1], [1], 0)
    man = bk.plan_rotation(0, 1, 1, [], 1)
    bk.swap_out(man, 0)
    with pytest.raises(BookError, match="BUSY"):
        bk.slot_table([0, 4], [0, 1], [man[0].cart], 0)       # evictee is in transit
    bk2 = make_book()
    bk2.mark_grads([0])
    man = bk2.plan_rotation(0, 1, 1, [], 1)                   # evicts cartridge 0 in slot 0
    assert man[0].slot == 0
    with pytest.raises(BookError, match="BUSY"):
        bk2.swap_out(man, 0)                                  # un-consumed grads


def test_rotation_properties_random():
    rng = np.random.default_rng(0)
    N, S = 40, 12
    bk = PoolBook([128] * N, S, Hkv=2, D=8)
    for step in range(60):
        stable = bk.stable_resident()
        sel = list(rng.choice(stable, size=4, replace=False))
        sel_slot, inv_off, inv_seq, P = bk.slot_table([0, 5], [0, 4], sel, step)
        man = bk.plan_rotation(step, 3, 3, sel, seed=99)
        outs = [e for e in man if e.dir == DIR_OUT]
        ins = [e for e in man if e.dir == DIR_IN]
        assert not ({e.cart for e in outs} & set(int(c) for c in sel))
        assert [e.slot for e in outs] == sorted(e.slot for e in outs)
        # evictees are the least recently used unprotected residents
        lu_out = max(bk.last_used[e.cart] for e in outs)
        rest = [c for c in stable if c not in sel and c not in {e.cart for e in outs}]
        assert all(bk.last_used[c] >= lu_out for c in rest)
        # arrivals have minimal opt_steps among the waiting cartridges, hash-ordered inside ties
        waiting = [c for c in range(N) if bk.slot_of[c] < 0]
        worst_in = max(bk.opt_steps[e.cart] for e in ins)
        assert all(bk.opt_steps[c] >= worst_in for c in waiting if c not in {e.cart for e in ins})
        keys = [(bk.opt_steps[e.cart], mix64(99, step, e.cart), e.cart) for e in ins]
        assert keys == sorted(keys)
        bk.swap_out(man, step)
        bk.swap_in(man, step)
        bk.mark_grads(sel_slot)
        bk.adam_slots()
        bk.commit()
        # every resident cartridge sits in exactly one slot and vice versa
        res = [c for c in range(N) if bk.slot_of[c] >= 0]
        assert len(res) == S and sorted(bk.slot_of[c] for c in res) == list(range(S))
        assert all(bk.cart_in[bk.slot_of[c]] == c for c in res)
    # least-trained-first gives near-uniform coverage ("ensuring uniform coverage")
    assert max(bk.opt_steps) - min(bk.opt_steps) <= 12


# ---------------------------------------------------------------------------------------------
# NEXT-3 pins: Eq. 1 sampler and schedules
# ---------------------------------------------------------------------------------------------
def _book(n=12, slots=12):
    from oracle.bookkeeping import PoolBook
    return PoolBook([64] * n, slots, 2, 32)


def test_sampler_structure_and_distribution():
    from oracle.bookkeeping import sample_selection
    bk = _book()
    n_ex = 6000
    targets = [i % 12 for i in range(n_ex)]
    so, sc = sample_selection(bk, targets, 0.75, 1, 10, 260604, 3)
    sizes = np.diff(so)
    iso = 0
    kcount = np.zeros(11)
    dist_hits = np.zeros(12)
    for b in range(n_ex):
        sel = sc[so[b]:so[b + 1]]
        assert sel[0] == targets[b] and len(set(sel)) == len(sel)          # target first, a SET (Eq. 1)
        if len(sel) == 1:
            iso += 1
        else:
            kcount[len(sel) - 1] += 1
            for c in sel[1:]:
                dist_hits[c] += 1
    # Eq. 1: isolation w.p. P_iso = 0.75 (binomial std 0.0056); k uniform on {1..10}; distractors uniform
    assert abs(iso / n_ex - 0.75) < 0.02
    mixed = n_ex - iso
    assert kcount[0] == 0 and np.all(np.abs(kcount[1:] / mixed - 0.1) < 0.03)
    assert np.all(np.abs(dist_hits / dist_hits.sum() - 1 / 12) < 0.01)
    assert sizes.max() <= 11


def test_sampler_edge_cases_and_determinism():
    from oracle.bookkeeping import sample_selection, BookError
    bk = _book(n=4, slots=4)
    so, sc = sample_selection(bk, [0, 1, 2, 3] * 50, 0.0, 5, 9, 7, 0)       # k > card(Z_dist) = 3 -> clamp (A6)
    assert all(sorted(sc[so[b]:so[b + 1]]) == [0, 1, 2, 3] for b in range(200))
    assert sample_selection(bk, [2], 1.0, 1, 3, 7, 0) == ([0, 1], [2])        # P_iso = 1: target only
    a = sample_selection(bk, [0, 1], 0.5, 1, 3, 11, 5)
    assert a == sample_selection(bk, [0, 1], 0.5, 1, 3, 11, 5)                # same counters, same draw
    bk2 = _book(n=6, slots=3)                                                 # cartridges 3..5 are not resident
    with pytest.raises(BookError):
        sample_selection(bk2, [4], 0.5, 1, 2, 1, 0)
    so, sc = sample_selection(bk2, [0] * 300, 0.0, 2, 2, 1, 0)
    assert set(sc) == {0, 1, 2}                                               # distractors only among residents


def test_lr_schedule_table5_values():
    from oracle.bookkeeping import lr_global, warmup_scale
    # Table 5: eta0 = 0.1, W = 200, warmup minimum 0.002, alpha_f = 0.02; 14,200 steps (:338)
    args = (0.1, 200, 0.002, 0.02, 14200)
    assert lr_global(0, *args) == 0.002
    assert abs(lr_global(100, *args) - 0.051) < 1e-15                         # halfway up the warmup
    assert lr_global(200, *args) == 0.1
    assert abs(lr_global(7200, *args) - 0.1 * (1 - 0.98 * 0.5)) < 1e-15       # halfway down: 0.051
    assert abs(lr_global(14200, *args) - 0.002) < 1e-15 and lr_global(10 ** 6, *args) == lr_global(14200, *args)
    ts = np.arange(200, 14201, 500)
    assert np.all(np.diff([lr_global(int(t), *args) for t in ts]) < 0)        # strictly decreasing after warmup
    # PAPER.md:85 with W_c = 20, N_b = 4: levels 1/4, 1/2, 3/4, 1; never zero; >= the unbucketed min(1,(s+1)/W_c)
    got = [warmup_scale(s, 20, 4) for s in range(25)]
    assert got[:5] == [0.25] * 5 and got[5:10] == [0.5] * 5 and got[10:15] == [0.75] * 5 and got[15:] == [1.0] * 10
    assert all(warmup_scale(s, 20, 4) >= min(1.0, (s + 1) / 20) for s in range(60))
    assert len({warmup_scale(s, 20, 4) for s in range(100)}) == 4             # "at most N_b param groups"
    assert warmup_scale(0, 1, 4) == 1.0


def test_select_retrieved_hand_worked_and_order_preserving():
    """chunk -> document -> cartridge, unique ids in retrieval order.  Hand-worked: the ranked chunks
    7, 2, 9, 3, 2 belong to documents 3, 1, 3, 0, 1 -> cartridges [3, 1, 0]; with room for two -> [3, 1]."""
    from oracle.bookkeeping import select_retrieved
    chunk_to_cart = [5, 5, 1, 0, 4, 4, 2, 3, 2, 3]
    assert select_retrieved([7, 2, 9, 3, 2], chunk_to_cart, 10) == [3, 1, 0]
    assert select_retrieved([7, 2, 9, 3, 2], chunk_to_cart, 2) == [3, 1]
    assert select_retrieved([], chunk_to_cart, 4) == []
    # against Python's own order-preserving de-duplication on random rankings (Table 9's setting: 10 chunks)
    rng = np.random.default_rng(9)
    for _ in range(200):
        mp = rng.integers(0, 12, size=40).tolist()
        ranked = rng.permutation(40)[:10].tolist()
        assert select_retrieved(ranked, mp, 99) == list(dict.fromkeys(mp[c] for c in ranked))
    with pytest.raises(BookError):
        select_retrieved([40], [0] * 40, 3)


def test_paged_pool_first_fit_hand_worked():
    """16-token pages, a cartridge owns ceil(len/16) contiguous pages chosen
    first-fit.  Budget 10 pages; cartridges of 3, 2, 4, 1, 2, 5 pages; three slot handles.  By hand:
      creation:  c0 -> pages 0-2, c1 -> 3-4, c2 -> 5-8            (page 9 free)
      round 0 (evict 2 LRU = c0, c1; arrivals by least steps = c3 (1 page), c4 (2 pages), c5 (5 pages)):
                 c3 -> page 0 (first fit), c4 -> pages 1-2, c5 needs 5: pages 3,4 (freed) + 9 are not contiguous with
                 anything long enough -> skipped; handles: c3 -> slot 0, c4 -> slot 1
      after commit: pages [c3, c4, c4, -, -, c2, c2, c2, c2, -]
      round 1 (evict c2; arrival c5, 5 pages): first fit over free + freed = pages 3..9 -> base 3."""
    lens = [48, 32, 64, 16, 32, 80]
    bk = PoolBook(lens, n_slots=3, Hkv=1, D=4, tile_tokens=16, budget_tokens=160)
    assert bk.slot_base == [0, 48, 80] and bk.slot_cap == [48, 32, 64]
    assert bk.page_owner == [0, 0, 0, 1, 1, 2, 2, 2, 2, -1]
    bk.opt_steps = [0, 0, 0, 1, 2, 3]                       # arrival priority: c3, then c4, then c5
    bk.slot_table([0, 2], [0, 1], [2], step=0)              # c2 is used at step 0 -> c0, c1 are the LRU pair
    man = bk.plan_rotation(0, n_in=3, n_out=2, protect=[2], seed=1)
    assert [(e.cart, e.slot, e.dir, e.base_tok) for e in man] == [(0, 0, DIR_OUT, 0), (1, 1, DIR_OUT, 48),
                                                                   (3, 0, DIR_IN, 0), (4, 1, DIR_IN, 16)]
    bk.swap_out(man, 0)
    bk.swap_in(man, 0)
    assert bk.slot_base[:2] == [0, 16] and bk.slot_cap[:2] == [16, 32]
    bk.adam_slots()
    bk.commit()
    assert bk.page_owner == [3, 4, 4, -1, -1, 2, 2, 2, 2, -1]
    bk.opt_steps[0] = bk.opt_steps[1] = 9                   # the 5-page cartridge c5 is now the least trained one waiting
    man = bk.plan_rotation(1, n_in=1, n_out=1, protect=[3, 4], seed=1)
    assert [(e.cart, e.slot, e.dir, e.base_tok) for e in man] == [(2, 2, DIR_OUT, 80), (5, 2, DIR_IN, 48)]
    # an extent that overlaps a page of a resident, stable cartridge is refused
    from oracle.bookkeeping import ManifestEntry
    bad = ManifestEntry(5, 2, DIR_IN, bk.home_off[5], bk.home_bytes(5), 0)
    with pytest.raises(BookError, match="BUSY"):
        bk.swap_in([bad], 1)
