"""CAS hot-path ORACLE (integer bookkeeping) -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Pure-Python (arbitrary-precision ints, lists, sorts) restatement of the budget manager's integer
state machine: slot tables (K1), swap round-trip accounting (K2), the rotation plan (K3) and the
per-step protocol (K4) of DESIGN.md "Bookkeeping".  The CUDA library implements the same rules
independently in C++ (``csrc/cas_host.cu``); the two share no code and are compared bit-exactly.

Passages followed:
  * PAPER.md:73 (sec. 2.1 Budget Manager): "maintains a fixed GPU pool of B <= N cartridges, keeping
    the remaining N-B cartridges offloaded to CPU memory"; samples only from active cartridges.
  * PAPER.md:75 (Pool rotation): "a fraction phi of the pool is evicted and replaced with new
    cartridges from persistent storage ... preferentially swaps in cartridges that have received
    the fewest optimizer steps"; Table 5 "Prioritize least trained: Yes".
  * BASELINE.json configs[2]: "swap in 16 priority-drawn cartridges and evict 16 LRU".
  * per-sample cartridge subsets -> per-sequence slot lists.
Tie-breaks the paper does not give are DESIGN.md readings R13-R16.
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import List, Optional, Sequence, Tuple

MASK64 = (1 << 64) - 1

DIR_OUT = 0
DIR_IN = 1


def mix64(seed: int, step: int, cart: int) -> int:
    """DESIGN.md R15: priority hash = SplitMix64 finaliser of
    seed + 0x9E3779B97F4A7C15*(step+1) + 0xD1B54A32D192ED03*(cart+1)  (mod 2^64)."""
    z = (seed + 0x9E3779B97F4A7C15 * (step + 1) + 0xD1B54A32D192ED03 * (cart + 1)) & MASK64
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & MASK64
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & MASK64
    return z ^ (z >> 31)


class BookError(Exception):
    def __init__(self, code: str, msg: str = ""):
        super().__init__(f"{code}: {msg}")
        self.code = code


@dataclass
class ManifestEntry:
    cart: int
    slot: int
    dir: int
    host_off: int
    nbytes: int
    base_tok: int = 0        # first pool token of the cartridge's extent (OUT: where it sits, IN: where it goes)

    def as_tuple(self):
        return (self.cart, self.slot, self.dir, self.base_tok, self.host_off, self.nbytes)


class PoolBook:
    """Integer state of the cartridge pool."""

    def __init__(self, cart_len: Sequence[int], n_slots: int, Hkv: int, D: int,
                 tile_tokens: int = 128, n_layers: int = 1, budget_tokens: int = 0):
        self.n_layers = int(n_layers)               # Z in R^{L x p x d x 2}; a home holds all L layers
        self.cart_len = [int(x) for x in cart_len]
        self.n_carts = len(self.cart_len)
        self.n_slots = int(n_slots)
        self.row_elems = Hkv * D
        self.tile = tile_tokens
        up = lambda x: (x + tile_tokens - 1) // tile_tokens * tile_tokens
        # PAGED pool (budget_tokens > 0; cartridge sizes are multiples of the 16-token page of the
        # paged KV cache, "enabling efficient memory allocation and deallocation during ... pool rotation"): the pool
        # is budget_tokens/tile pages; a resident cartridge owns a contiguous run of ceil(len/tile) pages chosen
        # first-fit (lowest base); slots are mere handles whose base/capacity change with their occupant.
        self.budget = int(budget_tokens)
        self.paged = self.budget > 0
        if self.paged:
            assert self.budget % tile_tokens == 0
            self.n_pages = self.budget // tile_tokens
            self.page_owner = [-1] * self.n_pages       # committed owner (cartridge id) of every page
            self.page_claim = [-1] * self.n_pages       # arrival in flight that will own the page at commit
            self.slot_cap = [0] * self.n_slots
            self.slot_base = [0] * self.n_slots
            for c in range(min(self.n_slots, self.n_carts)):
                n = up(self.cart_len[c]) // tile_tokens
                base = self._first_fit(n, lambda o, cl: o < 0 and cl < 0)
                if base < 0:
                    raise BookError("CAPACITY", "initial cartridges do not fit the page budget")
                for q in range(base, base + n):
                    self.page_owner[q] = c
                self.slot_base[c], self.slot_cap[c] = base * tile_tokens, n * tile_tokens
            self.pool_tokens = self.budget
        else:
            # slot capacities: everything resident -> slot s is sized for cartridge s;
            # otherwise uniform slots sized for the longest cartridge.
            if self.n_slots == self.n_carts:
                self.slot_cap = [up(l) for l in self.cart_len]
            else:
                cap = up(max(self.cart_len))
                self.slot_cap = [cap] * self.n_slots
            self.slot_base = [0] * self.n_slots
            for s in range(1, self.n_slots):
                self.slot_base[s] = self.slot_base[s - 1] + self.slot_cap[s - 1]
            self.pool_tokens = self.slot_base[-1] + self.slot_cap[-1] if self.n_slots else 0
        # pinned homes: 6 fp32 tensors (pK,pV,mK,mV,vK,vV) of len*Hkv*D per cartridge, packed
        self.home_off = [0] * self.n_carts
        for c in range(1, self.n_carts):
            self.home_off[c] = self.home_off[c - 1] + self.home_bytes(c - 1)
        # state: the first n_slots cartridges start resident, slot s <- cartridge s
        self.slot_of = [-1] * self.n_carts
        self.cart_in = [-1] * self.n_slots
        for s in range(min(self.n_slots, self.n_carts)):
            self.slot_of[s] = s
            self.cart_in[s] = s
        self.opt_steps = [0] * self.n_carts
        self.last_used = [-1] * self.n_carts
        self.in_transit = [0] * self.n_carts        # 0 stable, 1 leaving, 2 arriving
        self.grad_dirty = [0] * self.n_slots
        self.pending: List[Tuple[ManifestEntry, int]] = []   # (entry, plan step)

    def _first_fit(self, n: int, free) -> int:
        """Lowest base page of a run of n pages that are all free(owner, claim); -1 if there is none."""
        run = 0
        for q in range(self.n_pages):
            run = run + 1 if free(self.page_owner[q], self.page_claim[q]) else 0
            if run == n:
                return q - n + 1
        return -1

    def pages_of(self, c: int) -> List[int]:
        return [q for q in range(self.n_pages) if self.page_owner[q] == c]

    def home_bytes(self, c: int) -> int:
        return self.n_layers * 6 * self.cart_len[c] * self.row_elems * 4

    # ---- K1 ---------------------------------------------------------------------------------
    def slot_table(self, seq_off: Sequence[int], sel_off: Sequence[int], sel_cart: Sequence[int],
                   step: int):
        B = len(seq_off) - 1
        if B < 1 or len(sel_off) != B + 1 or seq_off[0] != 0 or sel_off[0] != 0:
            raise BookError("INVALID_ARG", "offsets")
        for b in range(B):
            if seq_off[b + 1] <= seq_off[b]:
                raise BookError("SHAPE", "Lq_b >= 1 required")
            if sel_off[b + 1] < sel_off[b]:
                raise BookError("INVALID_ARG", "sel_off not monotone")
        if sel_off[B] != len(sel_cart):
            raise BookError("INVALID_ARG", "sel_off[B] != nsel")
        sel_slot = []
        P = []
        for b in range(B):
            seen = set()
            pb = 0
            for k in range(sel_off[b], sel_off[b + 1]):
                c = int(sel_cart[k])
                if c < 0 or c >= self.n_carts:
                    raise BookError("INVALID_ARG", "cartridge id")
                if c in seen:
                    raise BookError("INVALID_ARG", "duplicate cartridge in one sequence")
                seen.add(c)
                if self.slot_of[c] < 0:
                    raise BookError("NOT_RESIDENT", str(c))
                if self.in_transit[c]:
                    raise BookError("BUSY", str(c))
                sel_slot.append(self.slot_of[c])
                pb += self.cart_len[c]
            P.append(pb)
        for c in set(int(x) for x in sel_cart):
            self.last_used[c] = step
        # inverted CSR: entries sorted by (slot asc, sequence asc)
        pairs = sorted((sel_slot[k], b) for b in range(B) for k in range(sel_off[b], sel_off[b + 1]))
        inv_off = [0] * (self.n_slots + 1)
        for s, _ in pairs:
            inv_off[s + 1] += 1
        for s in range(self.n_slots):
            inv_off[s + 1] += inv_off[s]
        inv_seq = [b for _, b in pairs]
        return sel_slot, inv_off, inv_seq, P

    # ---- K3 ---------------------------------------------------------------------------------
    def plan_rotation(self, step: int, n_in: int, n_out: int, protect: Sequence[int], seed: int
                      ) -> List[ManifestEntry]:
        prot = set(int(c) for c in protect)
        evictable = [c for c in range(self.n_carts)
                     if self.slot_of[c] >= 0 and not self.in_transit[c] and c not in prot]
        evictable.sort(key=lambda c: (self.last_used[c], c))
        evictees = evictable[:max(0, n_out)]
        waiting = [c for c in range(self.n_carts) if self.slot_of[c] < 0 and not self.in_transit[c]]
        waiting.sort(key=lambda c: (self.opt_steps[c], mix64(seed, step, c), c))
        free = [s for s in range(self.n_slots) if self.cart_in[s] < 0]
        free += [self.slot_of[c] for c in evictees]
        free.sort()
        arrivals = []
        used = set()
        if self.paged:
            # the lowest unused slot handle + the first-fit run of pages that are free now, or are freed by this round's
            # evictees, and that no earlier arrival of this plan has taken; a cartridge that fits nowhere is skipped
            ev = set(evictees)
            taken = [False] * self.n_pages
            for c in waiting:
                if len(arrivals) >= max(0, n_in):
                    break
                hs = [s for s in free if s not in used]
                if not hs:
                    break
                n = -(-self.cart_len[c] // self.tile)
                run, base = 0, -1
                for q in range(self.n_pages):
                    ok = (self.page_owner[q] < 0 or self.page_owner[q] in ev) and self.page_claim[q] < 0 and not taken[q]
                    run = run + 1 if ok else 0
                    if run == n:
                        base = q - n + 1
                        break
                if base < 0:
                    continue
                for q in range(base, base + n):
                    taken[q] = True
                used.add(hs[0])
                arrivals.append((c, hs[0], base * self.tile))
        else:
            for c in waiting:
                if len(arrivals) >= max(0, n_in):
                    break
                # first free slot (ascending) that is large enough and not yet paired
                for s in free:
                    if s not in used and self.slot_cap[s] >= self.cart_len[c]:
                        used.add(s)
                        arrivals.append((c, s, self.slot_base[s]))
                        break
        outs = sorted(((self.slot_of[c], c) for c in evictees))
        man = [ManifestEntry(c, s, DIR_OUT, self.home_off[c], self.home_bytes(c), self.slot_base[s]) for s, c in outs]
        man += [ManifestEntry(c, s, DIR_IN, self.home_off[c], self.home_bytes(c), bt)
                for c, s, bt in arrivals]
        return man

    # ---- K4 (state transitions of swap_out / swap_in / commit / adam) -------------------------
    def swap_out(self, man: Sequence[ManifestEntry], step: int):
        for e in man:
            if e.dir != DIR_OUT:
                continue
            if self.slot_of[e.cart] != e.slot or self.in_transit[e.cart]:
                raise BookError("NOT_RESIDENT" if self.slot_of[e.cart] != e.slot else "BUSY")
            if self.grad_dirty[e.slot]:
                raise BookError("BUSY", "un-consumed grads")
        for e in man:
            if e.dir == DIR_OUT:
                self.in_transit[e.cart] = 1
                self.pending.append((e, step))

    def swap_in(self, man: Sequence[ManifestEntry], step: int):
        leaving = {e.slot for e, _ in self.pending if e.dir == DIR_OUT}
        for e in man:
            if e.dir != DIR_IN:
                continue
            if self.slot_of[e.cart] >= 0 or self.in_transit[e.cart]:
                raise BookError("BUSY", "arrival already resident / in transit")
            if not (self.cart_in[e.slot] < 0 or e.slot in leaving):
                raise BookError("BUSY", "slot occupied")
            if not self.paged and self.slot_cap[e.slot] < self.cart_len[e.cart]:
                raise BookError("CAPACITY")
            if self.paged:
                n = -(-self.cart_len[e.cart] // self.tile)
                b = e.base_tok // self.tile
                if e.base_tok % self.tile or b < 0 or b + n > self.n_pages:
                    raise BookError("INVALID_ARG", "extent")
                for q in range(b, b + n):
                    o = self.page_owner[q]
                    if self.page_claim[q] >= 0 or (o >= 0 and self.in_transit[o] != 1):
                        raise BookError("BUSY", "page occupied")
        for e in man:
            if e.dir == DIR_IN:
                self.in_transit[e.cart] = 2
                self.pending.append((e, step))
                if self.paged:
                    n = -(-self.cart_len[e.cart] // self.tile)
                    b = e.base_tok // self.tile
                    for q in range(b, b + n):
                        self.page_claim[q] = e.cart
                    self.slot_base[e.slot], self.slot_cap[e.slot] = e.base_tok, n * self.tile

    def commit(self):
        for e, step in self.pending:
            if e.dir == DIR_OUT:
                self.slot_of[e.cart] = -1
                self.in_transit[e.cart] = 0
                if self.cart_in[e.slot] == e.cart:
                    self.cart_in[e.slot] = -1
                if self.paged:
                    for q in range(self.n_pages):
                        if self.page_owner[q] == e.cart:
                            self.page_owner[q] = -1
        for e, step in self.pending:
            if e.dir == DIR_IN:
                self.slot_of[e.cart] = e.slot
                self.cart_in[e.slot] = e.cart
                self.in_transit[e.cart] = 0
                self.last_used[e.cart] = step
                if self.paged:
                    for q in range(self.n_pages):
                        if self.page_claim[q] == e.cart:
                            self.page_owner[q], self.page_claim[q] = e.cart, -1
        self.pending = []

    def mark_grads(self, sel_slot: Sequence[int]):
        for s in set(sel_slot):
            self.grad_dirty[s] = 1

    def adam_slots(self, slots: Optional[Sequence[int]] = None) -> List[int]:
        """Slots an adam_step covers: the given list, or every resident, not-in-transit slot
        (ascending).  Increments opt_steps of their cartridges, clears grad_dirty."""
        if slots is None:
            slots = [s for s in range(self.n_slots)
                     if self.cart_in[s] >= 0 and not self.in_transit[self.cart_in[s]]]
        for s in slots:
            c = self.cart_in[s]
            if c < 0:
                raise BookError("NOT_RESIDENT")
            if self.in_transit[c]:
                raise BookError("BUSY")
        for s in slots:
            self.opt_steps[self.cart_in[s]] += 1
            self.grad_dirty[s] = 0
        return list(slots)

    def stable_resident(self) -> List[int]:
        return [c for c in range(self.n_carts) if self.slot_of[c] >= 0 and not self.in_transit[c]]


def position_offsets(book: PoolBook, P: Sequence[int]):
    """query position ids are offset by the number of active cartridge KV tokens.
    Returns (sum of resident cartridge lengths  [the packed layout of PAPER.md:71, every active
    cartridge sits in the prompt], per-sequence visible prefix lengths P_b)  -- DESIGN.md R7."""
    tot = sum(book.cart_len[c] for c in range(book.n_carts) if book.slot_of[c] >= 0)
    return tot, list(P)


# ---------------------------------------------------------------------------------------------
# NEXT-3: Eq. 1 mixture sampler and the learning-rate schedules
# ---------------------------------------------------------------------------------------------
def _draw(seed: int, step: int, b: int, d: int) -> int:
    """d-th 64-bit draw of example b at step `step`: mix64(mix64(seed, step, b), d, 0)  (R31)."""
    return mix64(mix64(seed, step, b), d, 0)


def sample_selection(book: PoolBook, targets: Sequence[int], p_iso: float, k_min: int, k_max: int, seed: int,
                     step: int):
    """PAPER.md:64-66, Eq. 1: with probability P_iso the example sees only its target cartridge Z*; otherwise
    Z* plus S ~ U(Z_dist, k), k ~ U(k_min, k_max), Z_dist = pool \\ Z*.  Readings (R31):
    the pool is the set of resident, stable cartridges; k's endpoints are inclusive integers; k is clamped to
    card(Z_dist); S is drawn without replacement by a partial Fisher-Yates shuffle of Z_dist in ascending id
    order; the target comes first, distractors in draw order.  All randomness comes from the counter-based
    generator above: draw 0 decides isolation (top 53 bits < floor(P_iso * 2^53)), draw 1 gives k, draw 2+j
    the j-th swap; an integer in [0, n) is ((x >> 32) * n) >> 32.  Returns (sel_off, sel_cart)."""
    stable = book.stable_resident()
    sel_off, sel_cart = [0], []
    thr = int(p_iso * (1 << 53))
    for b, tgt in enumerate(targets):
        if book.slot_of[tgt] < 0 or book.in_transit[tgt]:
            raise BookError("NOT_RESIDENT", f"target {tgt}")
        sel_cart.append(tgt)
        if (_draw(seed, step, b, 0) >> 11) >= thr:
            cand = [c for c in stable if c != tgt]
            k = k_min + (((_draw(seed, step, b, 1) >> 32) * (k_max - k_min + 1)) >> 32)
            k = min(k, len(cand))
            for j in range(k):
                r = j + (((_draw(seed, step, b, 2 + j) >> 32) * (len(cand) - j)) >> 32)
                cand[j], cand[r] = cand[r], cand[j]
                sel_cart.append(cand[j])
        sel_off.append(len(sel_cart))
    return sel_off, sel_cart


def lr_global(t: int, eta0: float, warmup_steps: int, warmup_min_lr: float, alpha_f: float, total_steps: int) -> float:
    """PAPER.md:83 "slow linear decay schedule" with Table 5 (:368-372): global warmup over W steps, final LR
    multiplier alpha_f, "Warmup minimum LR".  Reading DESIGN.md R29: eta rises linearly from warmup_min_lr at
    t = 0 to eta0 at t = W, then falls linearly to alpha_f * eta0 at t = total_steps and stays there."""
    if t < warmup_steps:
        return warmup_min_lr + (eta0 - warmup_min_lr) * (t / warmup_steps)
    if t >= total_steps:
        return alpha_f * eta0
    return eta0 * (1.0 - (1.0 - alpha_f) * ((t - warmup_steps) / (total_steps - warmup_steps)))


def warmup_scale(s: int, w_c: int, n_b: int) -> float:
    """eta_eff = eta_t * min(1, s / W_c) for a cartridge with s optimizer steps, bucketed into N_b
    levels.  Reading SURVEY.md A12 / DESIGN.md R30: the step being taken counts (s + 1), so a fresh cartridge does
    not get a zero learning rate, and the scale is rounded UP to the next of the N_b levels 1/N_b .. 1:
    ceil(min(1, (s+1)/W_c) * N_b) / N_b, in exact integer arithmetic."""
    num = min(s + 1, w_c) * n_b                      # min(1,(s+1)/W_c) * N_b = num / w_c
    level = -(-num // w_c)                           # ceil
    return level / n_b


# ---------------------------------------------------------------------------------------------
# NEXT-4: retrieval-ordered cartridge selection
# ---------------------------------------------------------------------------------------------
def select_retrieved(chunk_ids: Sequence[int], chunk_to_cart: Sequence[int], max_carts: int) -> List[int]:
    """PAPER.md:142 (sec. 3, Retrieval): "we map each retrieved chunk to a document id, which in turn is associated
    with a cartridge.  The final list contains the unique cartridge ids in the order of their retrieval."
    chunk_ids are ranked best first; at most max_carts cartridges are kept (the k of "top-k cartridges")."""
    out: List[int] = []
    for ch in chunk_ids:
        if len(out) >= max_carts:
            break
        if ch < 0 or ch >= len(chunk_to_cart):
            raise BookError("INVALID_ARG", "chunk id")
        c = int(chunk_to_cart[ch])
        if c not in out:
            out.append(c)
    return out
