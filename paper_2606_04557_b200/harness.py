"""Device-side session for one workload: allocates the caller-owned buffers with torch, uploads the
seeded inputs, and calls the C ABI through ``cas``.  Used by tests, bench.py and smoke().  Holds no
arithmetic of the method; never imports ``oracle``."""
from __future__ import annotations

from typing import Optional

import numpy as np
import torch

from . import cas


def torch_dtype(dtype: str):
    return torch.float32 if dtype == "f32" else torch.bfloat16


class Session:
    def __init__(self, wl, device: str = "cuda:0", load: bool = True):
        cfg = wl.cfg
        self.wl, self.cfg, self.device = wl, cfg, device
        self.tdt = torch_dtype(cfg.dtype)
        self.pool = cas.Pool(cas.CAS_F32 if cfg.dtype == "f32" else cas.CAS_BF16, cfg.Hkv, cfg.D,
                             wl.cart_len, cfg.n_slots, tile_tokens=getattr(cfg, "tile_tokens", 0), device=device,
                             budget_tokens=getattr(cfg, "budget_tokens", 0))
        if load:
            for c in range(cfg.n_carts):
                K, V = wl.cart_kv(c)
                cas.cas_pool_load(self.pool, c, K, V)
        self.scale = 1.0 / float(np.sqrt(cfg.D))
        self.tab: Optional[cas.SlotTable] = None
        self.set_batch(wl.seq_off, wl.sel_off, wl.sel_cart, wl.Q, wl.K_self, wl.V_self, wl.dO, step=0)
        self.stream = torch.cuda.current_stream()

    def _dev(self, a: Optional[np.ndarray]):
        if a is None:
            return None
        return torch.from_numpy(a).to(self.device).to(self.tdt)

    def set_batch(self, seq_off, sel_off, sel_cart, Q, Ks, Vs, dO, step: int):
        cfg = self.cfg
        if self.tab is not None:
            self.tab.close()
        self.tab = cas.cas_slot_table_build(self.pool, seq_off, sel_off, sel_cart, step)
        self.Q, self.Ks, self.Vs, self.dO = self._dev(Q), self._dev(Ks), self._dev(Vs), self._dev(dO)
        T = self.tab.T
        dev = self.device
        self.O = torch.empty((T, cfg.Hq, cfg.D), dtype=self.tdt, device=dev)
        self.LSE = torch.empty((T, cfg.Hq), dtype=torch.float32, device=dev)
        if dO is not None:
            self.dQ = torch.empty_like(self.O)
            self.dKs = torch.empty((T, cfg.Hkv, cfg.D), dtype=self.tdt, device=dev)
            self.dVs = torch.empty_like(self.dKs)
            nb = cas.cas_prefix_attn_bwd_workspace_bytes(self.pool, self.tab, cfg.Hq)
            self.ws = torch.empty(nb, dtype=torch.uint8, device=dev)

    def adam_cfg(self, zero_grad: int = 1, n_frozen: int = 0) -> cas.AdamCfg:
        c = self.cfg
        return cas.AdamCfg(c.lr, c.beta1, c.beta2, c.eps, n_frozen, zero_grad)

    def fwd(self, stream=None, self_block: bool = True):
        cas.cas_prefix_attn_fwd(self.pool, self.tab, self.cfg.Hq, self.Q,
                                self.Ks if self_block else None, self.Vs if self_block else None,
                                self.scale, self.O, self.LSE, stream)

    def bwd(self, stream=None, self_block: bool = True):
        cas.cas_prefix_attn_bwd(self.pool, self.tab, self.cfg.Hq, self.Q,
                                self.Ks if self_block else None, self.Vs if self_block else None,
                                self.O, self.LSE, self.dO, self.scale, self.dQ,
                                self.dKs if self_block else None, self.dVs if self_block else None,
                                self.ws, stream)

    def adam(self, stream=None, slots=None, lr_scale=None, zero_grad: int = 1, n_frozen: int = 0):
        cas.cas_adam_step(self.pool, self.adam_cfg(zero_grad, n_frozen), slots, lr_scale, stream)

    def np(self, t: torch.Tensor) -> np.ndarray:
        return t.float().cpu().numpy()

    def read(self, cart: int, what: str) -> np.ndarray:
        return cas.cas_pool_read(self.pool, cart, what)

    def close(self):
        if self.tab is not None:
            self.tab.close()
            self.tab = None
        self.pool.close()
