"""Thin ctypes binding of libcas (include/cas.h).  Argument marshalling only: every step of the hot
path runs inside the library's CUDA kernels.  There is NO fallback: if libcas.so is missing or a
call fails, a CasError is raised.

Function names mirror the C ABI (``cas_prefix_attn_fwd`` ...); ``Pool`` / ``SlotTable`` only hold
the opaque handles and the torch tensors that back the caller-owned arenas.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libcas.so")

CAS_F32, CAS_BF16 = 0, 1
CAS_DIR_OUT, CAS_DIR_IN = 0, 1
CAS_IMPL_AUTO, CAS_IMPL_SIMT, CAS_IMPL_TC = 0, 1, 2
ERR_NAMES = {0: "CAS_OK", -1: "CAS_ERR_INVALID_ARG", -2: "CAS_ERR_SHAPE", -3: "CAS_ERR_NOT_RESIDENT",
             -4: "CAS_ERR_BUSY", -5: "CAS_ERR_CAPACITY", -6: "CAS_ERR_CUDA"}


class CasError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"{ERR_NAMES.get(code, code)}: {msg}")
        self.code = code
        self.name = ERR_NAMES.get(code, str(code))


class PoolDesc(C.Structure):
    _fields_ = [("dtype", C.c_int32), ("Hkv", C.c_int32), ("D", C.c_int32), ("n_carts", C.c_int32),
                ("n_slots", C.c_int32), ("tile_tokens", C.c_int32), ("cart_len", C.POINTER(C.c_int32)),
                ("n_layers", C.c_int32), ("pool_tokens_budget", C.c_int64)]


class PoolLayout(C.Structure):
    _fields_ = [("pool_K", C.c_void_p), ("pool_V", C.c_void_p), ("grad_K", C.c_void_p),
                ("grad_V", C.c_void_p), ("state", C.c_void_p), ("slot_base", C.POINTER(C.c_int32)),
                ("slot_cap", C.POINTER(C.c_int32)), ("pool_tokens", C.c_int64)]


class ManifestEntry(C.Structure):
    _fields_ = [("cart", C.c_int32), ("slot", C.c_int32), ("dir", C.c_int32), ("base_tok", C.c_int32),
                ("host_off", C.c_int64), ("nbytes", C.c_int64)]

    def as_tuple(self):
        return (self.cart, self.slot, self.dir, self.base_tok, self.host_off, self.nbytes)


class AdamCfg(C.Structure):
    _fields_ = [("lr", C.c_float), ("beta1", C.c_float), ("beta2", C.c_float), ("eps", C.c_float),
                ("n_frozen", C.c_int32), ("zero_grad", C.c_int32)]


class TableInfo(C.Structure):
    _fields_ = [("B", C.c_int32), ("T", C.c_int32), ("nsel", C.c_int32), ("n_kv_tiles", C.c_int32),
                ("pairs_per_head", C.c_int64), ("prefix_tokens", C.c_int64),
                ("unique_prefix_tokens", C.c_int64)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise CasError(-6, f"{LIB_PATH} not built; run `python -m paper_2606_04557_b200._build` "
                               "(there is no CPU fallback)")
        _lib = C.CDLL(LIB_PATH)
        _lib.cas_version.restype = C.c_char_p
    return _lib


def _check(rc: int):
    if rc != 0:
        buf = C.create_string_buffer(512)
        lib().cas_last_error(buf, C.c_size_t(512))
        raise CasError(rc, buf.value.decode())


def _i32(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.int32)


def _p(a: Optional[np.ndarray], typ=C.c_int32):
    return None if a is None else a.ctypes.data_as(C.POINTER(typ))


def _dptr(t) -> C.c_void_p:
    """Device / pinned pointer of a torch tensor (or None)."""
    return C.c_void_p(None if t is None else t.data_ptr())


def _stream(s) -> C.c_void_p:
    if s is None:
        import torch

        s = torch.cuda.current_stream()
    return C.c_void_p(s.cuda_stream)


def cas_version() -> str:
    return lib().cas_version().decode()


def cas_set_impl(impl: int):
    _check(lib().cas_set_impl(C.c_int(impl)))


def cas_pool_query_bytes(desc: PoolDesc):
    d, h = C.c_size_t(0), C.c_size_t(0)
    _check(lib().cas_pool_query_bytes(C.byref(desc), C.byref(d), C.byref(h)))
    return d.value, h.value


class Pool:
    """Owns the torch tensors backing the arenas + the opaque cas_pool handle."""

    def __init__(self, dtype: int, Hkv: int, D: int, cart_len: Sequence[int], n_slots: int,
                 tile_tokens: int = 0, device: Optional[str] = "cuda:0", side_stream=None, n_layers: int = 1,
                 budget_tokens: int = 0):
        self._cart_len = _i32(cart_len)
        self.n_layers = n_layers
        self.desc = PoolDesc(dtype, Hkv, D, len(self._cart_len), n_slots, tile_tokens,
                             _p(self._cart_len), n_layers, budget_tokens)
        self.dtype, self.Hkv, self.D = dtype, Hkv, D
        self.n_carts, self.n_slots = len(self._cart_len), n_slots
        self.dev_bytes, self.host_bytes = cas_pool_query_bytes(self.desc)
        self.handle = C.c_void_p(None)
        self.dev_arena = self.pinned_arena = self.side_stream = None
        dev_ptr = pin_ptr = side = C.c_void_p(None)
        if device is not None:
            import torch

            self.dev_arena = torch.empty(self.dev_bytes, dtype=torch.uint8, device=device)
            dev_ptr = _dptr(self.dev_arena)
            if n_slots < self.n_carts:
                self.pinned_arena = torch.empty(self.host_bytes, dtype=torch.uint8, pin_memory=True)
                pin_ptr = _dptr(self.pinned_arena)
            self.side_stream = side_stream or torch.cuda.Stream(device=device)
            side = C.c_void_p(self.side_stream.cuda_stream)
        _check(lib().cas_pool_create(C.byref(self.desc), dev_ptr, pin_ptr, side, C.byref(self.handle)))
        lay = PoolLayout()
        _check(lib().cas_pool_layout_get(self.handle, C.byref(lay)))
        self.layout = lay
        self.pool_tokens = lay.pool_tokens

    @property
    def slot_base(self) -> np.ndarray:
        """First pool token of every slot (in a paged pool it changes with the slot's occupant: read it afresh)."""
        lay = PoolLayout()
        _check(lib().cas_pool_layout_get(self.handle, C.byref(lay)))
        return np.ctypeslib.as_array(lay.slot_base, (self.n_slots,)).copy()

    @property
    def slot_cap(self) -> np.ndarray:
        lay = PoolLayout()
        _check(lib().cas_pool_layout_get(self.handle, C.byref(lay)))
        return np.ctypeslib.as_array(lay.slot_cap, (self.n_slots,)).copy()

    def close(self):
        if self.handle:
            lib().cas_pool_destroy(self.handle)
            self.handle = C.c_void_p(None)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def cas_pool_load(pool: Pool, cart: int, K: np.ndarray, V: np.ndarray, layer: int = 0):
    K = np.ascontiguousarray(K, dtype=np.float32)
    V = np.ascontiguousarray(V, dtype=np.float32)
    _check(lib().cas_pool_load_layer(pool.handle, C.c_int32(layer), C.c_int32(cart), _p(K, C.c_float),
                                     _p(V, C.c_float)))


READ_NAMES = {"pK": 0, "pV": 1, "mK": 2, "mV": 3, "vK": 4, "vV": 5, "gK": 6, "gV": 7, "wK": 8, "wV": 9}


def cas_pool_read(pool: Pool, cart: int, what, layer: int = 0) -> np.ndarray:
    w = READ_NAMES[what] if isinstance(what, str) else int(what)
    n = int(pool._cart_len[cart])
    if w < 8 or pool.dtype == CAS_F32:
        out = np.empty((n, pool.Hkv, pool.D), dtype=np.float32)
    else:
        out = np.empty((n, pool.Hkv, pool.D), dtype=np.uint16)       # raw bf16 bits
    _check(lib().cas_pool_read_layer(pool.handle, C.c_int32(layer), C.c_int32(cart), C.c_int32(w),
                                     C.c_void_p(out.ctypes.data)))
    return out


def cas_pool_counters(pool: Pool) -> dict:
    N, S = pool.n_carts, pool.n_slots
    o = dict(slot_of=np.empty(N, np.int32), cart_in=np.empty(S, np.int32), opt_steps=np.empty(N, np.int64),
             last_used=np.empty(N, np.int64), in_transit=np.empty(N, np.int32),
             grad_dirty=np.empty(S, np.int32))
    _check(lib().cas_pool_counters(pool.handle, _p(o["slot_of"]), _p(o["cart_in"]),
                                   _p(o["opt_steps"], C.c_int64), _p(o["last_used"], C.c_int64),
                                   _p(o["in_transit"]), _p(o["grad_dirty"])))
    return o


def cas_pool_set_counters(pool: Pool, cart: int, opt_steps: int, last_used: int):
    _check(lib().cas_pool_set_counters(pool.handle, C.c_int32(cart), C.c_int64(opt_steps),
                                       C.c_int64(last_used)))


class SlotTable:
    def __init__(self, pool: Pool, handle, B: int):
        self.pool, self.handle, self.B = pool, handle, B
        info = TableInfo()
        _check(lib().cas_slot_table_info(handle, C.byref(info)))
        self.info = info
        self.T, self.nsel = info.T, info.nsel

    def close(self):
        if self.handle:
            lib().cas_slot_table_destroy(self.handle)
            self.handle = C.c_void_p(None)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def cas_slot_table_build(pool: Pool, seq_off, sel_off, sel_cart, step: int = 0) -> SlotTable:
    seq_off, sel_off, sel_cart = _i32(seq_off), _i32(sel_off), _i32(sel_cart)
    B = len(seq_off) - 1
    if len(sel_off) != B + 1 or (len(sel_off) and sel_off[-1] != len(sel_cart)):
        raise CasError(-1, "sel_off / sel_cart length mismatch")
    h = C.c_void_p(None)
    _check(lib().cas_slot_table_build(pool.handle, C.c_int32(B), _p(seq_off), _p(sel_off),
                                      _p(sel_cart), C.c_int64(step), C.byref(h)))
    return SlotTable(pool, h, B)


def cas_slot_table_export(tab: SlotTable) -> dict:
    S = tab.pool.n_slots
    o = dict(sel_slot=np.empty(tab.nsel, np.int32), inv_off=np.empty(S + 1, np.int32),
             inv_seq=np.empty(tab.nsel, np.int32), P=np.empty(tab.B, np.int64))
    _check(lib().cas_slot_table_export(tab.handle, _p(o["sel_slot"]), _p(o["inv_off"]),
                                       _p(o["inv_seq"]), _p(o["P"], C.c_int64)))
    return o


def cas_position_offsets(pool: Pool, tab: Optional[SlotTable]):
    tot = C.c_int64(0)
    P = np.empty(tab.B, np.int64) if tab is not None else None
    _check(lib().cas_position_offsets(pool.handle, tab.handle if tab else None, C.byref(tot),
                                      _p(P, C.c_int64)))
    return tot.value, P


def cas_rope_apply(dtype: int, seq_off, pos_off, H: int, D: int, base: float, layout: int, inverse: bool, X,
                   stream=None):
    so = _i32(seq_off)
    po = np.ascontiguousarray(np.asarray(pos_off, dtype=np.int64))
    _check(lib().cas_rope_apply(C.c_int32(dtype), C.c_int32(len(so) - 1), _p(so), _p(po, C.c_int64), C.c_int32(H),
                                C.c_int32(D), C.c_double(base), C.c_int32(layout), C.c_int32(1 if inverse else 0),
                                _dptr(X), _stream(stream)))


def cas_prefix_attn_fwd(pool: Pool, tab: SlotTable, Hq: int, Q, K_self, V_self, scale: float, O, LSE,
                        stream=None, layer: int = 0):
    _check(lib().cas_prefix_attn_fwd_layer(pool.handle, tab.handle, C.c_int32(layer), C.c_int32(Hq), _dptr(Q),
                                           _dptr(K_self), _dptr(V_self), C.c_float(scale), _dptr(O), _dptr(LSE),
                                           _stream(stream)))


def cas_decode_attn(pool: Pool, tab: SlotTable, Hq: int, Q, K_cache, V_cache, cache_cap: int, self_len, scale: float,
                    O, LSE, stream=None, layer: int = 0):
    sl = None if self_len is None else _i32(self_len)
    _check(lib().cas_decode_attn_layer(pool.handle, tab.handle, C.c_int32(layer), C.c_int32(Hq), _dptr(Q),
                                       _dptr(K_cache), _dptr(V_cache), C.c_int32(cache_cap), _p(sl), C.c_float(scale),
                                       _dptr(O), _dptr(LSE), _stream(stream)))


def cas_select_retrieved(chunk_ids, chunk_to_cart, max_carts: int) -> np.ndarray:
    ch, mp = _i32(chunk_ids), _i32(chunk_to_cart)
    out = np.empty(max(max_carts, 1), np.int32)
    n = C.c_int32(0)
    _check(lib().cas_select_retrieved(_p(ch), C.c_int32(len(ch)), _p(mp), C.c_int32(len(mp)), C.c_int32(max_carts),
                                      _p(out), C.byref(n)))
    return out[:n.value].copy()


def cas_prefix_attn_bwd_workspace_bytes(pool: Pool, tab: SlotTable, Hq: int) -> int:
    n = C.c_size_t(0)
    _check(lib().cas_prefix_attn_bwd_workspace_bytes(pool.handle, tab.handle, C.c_int32(Hq), C.byref(n)))
    return n.value


def cas_prefix_attn_bwd(pool: Pool, tab: SlotTable, Hq: int, Q, K_self, V_self, O, LSE, dO, scale: float,
                        dQ, dK_self, dV_self, workspace, stream=None, layer: int = 0):
    _check(lib().cas_prefix_attn_bwd_layer(pool.handle, tab.handle, C.c_int32(layer), C.c_int32(Hq), _dptr(Q),
                                           _dptr(K_self), _dptr(V_self), _dptr(O), _dptr(LSE), _dptr(dO),
                                           C.c_float(scale), _dptr(dQ), _dptr(dK_self), _dptr(dV_self),
                                           _dptr(workspace),
                                           C.c_size_t(workspace.numel() * workspace.element_size()),
                                           _stream(stream)))


class Rope(C.Structure):
    """cas_rope: the device cos/sin table of cas_rope_table (kept alive here) and the pair layout."""
    _fields_ = [("cs", C.c_void_p), ("layout", C.c_int32), ("reserved", C.c_int32)]

    def __init__(self, table, layout: int):
        super().__init__(table.data_ptr(), layout, 0)
        self.table = table


def cas_rope_table(seq_off, pos_off, D: int, base: float, cs, stream=None):
    so, po = _i32(seq_off), np.ascontiguousarray(pos_off, dtype=np.int64)
    _check(lib().cas_rope_table(C.c_int32(len(so) - 1), _p(so), _p(po, C.c_int64), C.c_int32(D), C.c_double(base),
                                _dptr(cs), _stream(stream)))


def cas_prefix_attn_fwd_rope(pool: Pool, tab: SlotTable, Hq: int, Q, Ks, Vs, rope: Rope, Q_rot, Ks_rot, scale: float,
                             O, LSE, stream=None, layer: int = 0):
    _check(lib().cas_prefix_attn_fwd_rope(pool.handle, tab.handle, C.c_int32(layer), C.c_int32(Hq), _dptr(Q), _dptr(Ks),
                                          _dptr(Vs), C.byref(rope), _dptr(Q_rot), _dptr(Ks_rot), C.c_float(scale),
                                          _dptr(O), _dptr(LSE), _stream(stream)))


def cas_prefix_attn_bwd_rope(pool: Pool, tab: SlotTable, Hq: int, Q_rot, Ks_rot, Vs, O, LSE, dO, rope: Rope,
                             scale: float, dQ, dKs, dVs, workspace, stream=None, layer: int = 0):
    _check(lib().cas_prefix_attn_bwd_rope(pool.handle, tab.handle, C.c_int32(layer), C.c_int32(Hq), _dptr(Q_rot),
                                          _dptr(Ks_rot), _dptr(Vs), _dptr(O), _dptr(LSE), _dptr(dO), C.byref(rope),
                                          C.c_float(scale), _dptr(dQ), _dptr(dKs), _dptr(dVs), _dptr(workspace),
                                          C.c_size_t(workspace.numel() * workspace.element_size()), _stream(stream)))


def cas_prefix_attn_fwd_noalloc(pool: Pool, tab: SlotTable, Hq: int, Q, Ks, Vs, scale: float, O, LSE, stream=None,
                                layer: int = 0):
    _check(lib().cas_prefix_attn_fwd_noalloc(pool.handle, tab.handle, C.c_int32(layer), C.c_int32(Hq), _dptr(Q),
                                             _dptr(Ks), _dptr(Vs), C.c_float(scale), _dptr(O), _dptr(LSE),
                                             _stream(stream)))


class LayerIO(C.Structure):
    _fields_ = [("Q", C.c_void_p), ("K_self", C.c_void_p), ("V_self", C.c_void_p), ("dO", C.c_void_p),
                ("O", C.c_void_p), ("LSE", C.c_void_p), ("dQ", C.c_void_p), ("dK_self", C.c_void_p),
                ("dV_self", C.c_void_p), ("rope", C.c_void_p), ("Q_rot", C.c_void_p), ("K_self_rot", C.c_void_p)]


def cas_train_step_layers(pool: Pool, tabs, Hq: int, io, scale: float, cfg: AdamCfg, lr_scale=None, workspace=None,
                          stream=None):
    """io[m][l]: dict of torch tensors Q, K_self, V_self, dO, O, LSE, dQ, dK_self, dV_self (micro-batch m, layer l);
    optional fused RoPE: "rope" (a Rope), "Q_rot", "K_self_rot"."""
    n_micro, L = len(tabs), pool.n_layers
    arr = (LayerIO * (n_micro * L))()
    for m in range(n_micro):
        for l in range(L):
            for k, _ in LayerIO._fields_:
                t = io[m][l].get(k)
                if k == "rope":         # a Rope structure (kept alive by the caller's dict), passed by address
                    setattr(arr[m * L + l], k, None if t is None else C.addressof(t))
                else:
                    setattr(arr[m * L + l], k, None if t is None else t.data_ptr())
    tp = (C.c_void_p * n_micro)(*[t.handle for t in tabs])
    ls = None if lr_scale is None else np.ascontiguousarray(lr_scale, dtype=np.float32)
    _check(lib().cas_train_step_layers(pool.handle, tp, C.c_int32(n_micro), C.c_int32(Hq), arr, C.c_float(scale),
                                       C.byref(cfg), _p(ls, C.c_float), _dptr(workspace),
                                       C.c_size_t(workspace.numel() * workspace.element_size()), _stream(stream)))


def cas_train_step_layers_workspace_bytes(pool: Pool, tabs, Hq: int) -> int:
    n = C.c_size_t(0)
    tp = (C.c_void_p * len(tabs))(*[t.handle for t in tabs])
    _check(lib().cas_train_step_layers_workspace_bytes(pool.handle, tp, C.c_int32(len(tabs)), C.c_int32(Hq),
                                                       C.byref(n)))
    return n.value


def cas_adam_step(pool: Pool, cfg: AdamCfg, slots=None, lr_scale=None, stream=None, host_only=False):
    s = None if slots is None else _i32(slots)
    ls = None if lr_scale is None else np.ascontiguousarray(lr_scale, dtype=np.float32)
    st = C.c_void_p(None) if host_only else _stream(stream)
    _check(lib().cas_adam_step(pool.handle, C.byref(cfg), _p(s), C.c_int32(0 if s is None else len(s)),
                               _p(ls, C.c_float), st))


def cas_grad_zero(pool: Pool, slots=None, stream=None):
    s = None if slots is None else _i32(slots)
    _check(lib().cas_grad_zero(pool.handle, _p(s), C.c_int32(0 if s is None else len(s)), _stream(stream)))


def cas_plan_rotation(pool: Pool, step: int, n_in: int, n_out: int, protect, seed: int):
    prot = _i32(protect)
    cap = n_in + n_out + 8
    arr = (ManifestEntry * cap)()
    n = C.c_int32(0)
    _check(lib().cas_plan_rotation(pool.handle, C.c_int64(step), C.c_int32(n_in), C.c_int32(n_out),
                                   _p(prot), C.c_int32(len(prot)), C.c_uint64(seed), arr, C.c_int32(cap),
                                   C.byref(n)))
    return arr, n.value


def cas_swap_out(pool: Pool, man, n: int, step: int, after_stream=None, host_only=False):
    st = C.c_void_p(None) if host_only else _stream(after_stream)
    _check(lib().cas_swap_out(pool.handle, man, C.c_int32(n), C.c_int64(step), st))


def cas_swap_in(pool: Pool, man, n: int, step: int):
    _check(lib().cas_swap_in(pool.handle, man, C.c_int32(n), C.c_int64(step)))


def cas_swap_commit(pool: Pool, main_stream=None, host_only=False):
    st = C.c_void_p(None) if host_only else _stream(main_stream)
    _check(lib().cas_swap_commit(pool.handle, st))


def cas_selftest_cta_pair_mma(A, B, D, stream=None):
    _check(lib().cas_selftest_cta_pair_mma(_dptr(A), _dptr(B), _dptr(D), _stream(stream)))


class LrCfg(C.Structure):
    _fields_ = [("eta0", C.c_double), ("warmup_steps", C.c_int64), ("warmup_min_lr", C.c_double),
                ("alpha_f", C.c_double), ("total_steps", C.c_int64)]


def cas_sample_selection(pool: Pool, targets, p_iso: float, k_min: int, k_max: int, seed: int, step: int):
    tg = _i32(targets)
    B = len(tg)
    cap = B * (1 + max(k_max, 0))
    sel_off = np.empty(B + 1, np.int32)
    sel_cart = np.empty(max(cap, 1), np.int32)
    _check(lib().cas_sample_selection(pool.handle, C.c_int32(B), _p(tg), C.c_double(p_iso), C.c_int32(k_min),
                                      C.c_int32(k_max), C.c_uint64(seed), C.c_int64(step), _p(sel_off),
                                      _p(sel_cart), C.c_int32(cap)))
    return sel_off, sel_cart[:sel_off[B]].copy()


def cas_lr_schedule(cfg: LrCfg, t: int) -> float:
    eta = C.c_double(0.0)
    _check(lib().cas_lr_schedule(C.byref(cfg), C.c_int64(t), C.byref(eta)))
    return eta.value


def cas_warmup_scales(pool: Pool, slots, w_c: int, n_b: int) -> np.ndarray:
    sl = _i32(slots)
    out = np.empty(len(sl), np.float32)
    _check(lib().cas_warmup_scales(pool.handle, _p(sl), C.c_int32(len(sl)), C.c_int32(w_c), C.c_int32(n_b),
                                   _p(out, C.c_float)))
    return out


def cas_slot_table_fwd_split(tab: SlotTable):
    a, b = C.c_int32(0), C.c_int32(0)
    _check(lib().cas_slot_table_fwd_split(tab.handle, C.byref(a), C.byref(b)))
    return a.value, b.value


def cas_train_step_host_scratch_bytes(pool: Pool, tab: SlotTable, Hq: int) -> int:
    n = C.c_size_t(0)
    _check(lib().cas_train_step_host_scratch_bytes(pool.handle, tab.handle, C.c_int32(Hq), C.byref(n)))
    return n.value


def _train_step_host(fn, pool, tab, Hq, hQ, hKs, hVs, hdO, scale, cfg, hO, hLSE, hdQ, hdKs, hdVs, scratch, stream):
    _check(fn(pool.handle, tab.handle, C.c_int32(Hq), _dptr(hQ), _dptr(hKs), _dptr(hVs), _dptr(hdO), C.c_float(scale),
              C.byref(cfg), _dptr(hO), _dptr(hLSE), _dptr(hdQ), _dptr(hdKs), _dptr(hdVs), _dptr(scratch),
              C.c_size_t(scratch.numel() * scratch.element_size()), _stream(stream)))


def cas_train_step_host(pool: Pool, tab: SlotTable, Hq: int, hQ, hKs, hVs, hdO, scale: float, cfg: AdamCfg,
                        hO, hLSE, hdQ, hdKs, hdVs, scratch, stream=None):
    _train_step_host(lib().cas_train_step_host, pool, tab, Hq, hQ, hKs, hVs, hdO, scale, cfg, hO, hLSE, hdQ, hdKs,
                     hdVs, scratch, stream)


def cas_train_step_host_async(pool: Pool, tab: SlotTable, Hq: int, hQ, hKs, hVs, hdO, scale: float, cfg: AdamCfg,
                              hO, hLSE, hdQ, hdKs, hdVs, scratch, stream=None):
    _train_step_host(lib().cas_train_step_host_async, pool, tab, Hq, hQ, hKs, hVs, hdO, scale, cfg, hO, hLSE, hdQ,
                     hdKs, hdVs, scratch, stream)


def cas_train_step_host_wait(pool: Pool, stream=None):
    _check(lib().cas_train_step_host_wait(pool.handle, _stream(stream)))
