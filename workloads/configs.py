"""The five BASELINE.json configs as plain data (shapes and distributions only).

Citations: BASELINE.json ``configs[0..4]``; geometry 32/8/128 follows the paper's Qwen3-8B base model
(App. A); cartridge sizes of hundreds to a few thousand tokens follow Table 8
(PAPER.md:450-484); packed sequence lengths follow Table 5.
"""
from __future__ import annotations

from dataclasses import dataclass, replace


@dataclass(frozen=True)
class CasConfig:
    name: str
    dtype: str            # "f32" | "bf16"  storage dtype of Q/K/V/O/dO/dQ
    Hq: int
    Hkv: int
    D: int
    n_carts: int
    n_slots: int          # HBM-resident slots (== n_carts when everything is resident)
    cart_len: int         # fixed cartridge length, or 0 => ragged lognormal (config 4)
    B: int                # sequences in the batch
    Lq: int               # query tokens per sequence, or 0 => ragged U{256..4096}
    n_dist: int           # distractors per sequence; -1 => U{0..31}; -2 => all cartridges selected
    kv_std: float         # std of pool / self K,V
    selection: str        # "uniform" | "prop_len" | "all" | "topk"
    backward: bool = True
    rotate_in: int = 0    # cartridges swapped in per step (config 3)
    rotate_out: int = 0
    # ragged parameters (config 4)
    len_mu: float = 7.0
    len_sigma: float = 0.8
    len_min: int = 256
    len_max: int = 4096
    lq_min: int = 256
    lq_max: int = 4096
    n_dist_max: int = 31
    # paged pools: page size of the pool (0 = the 128-token default),
    # token budget of a paged pool with rotation (0 = static slots), cartridge lengths = 16 x U{1..len_pages_max}
    tile_tokens: int = 0
    budget_tokens: int = 0
    len_pages_max: int = 0
    # Adam (BASELINE.json config 1; Table 5 gives no eps/betas, Kingma & Ba defaults)
    lr: float = 1e-3
    beta1: float = 0.9
    beta2: float = 0.999
    eps: float = 1e-8

    def scaled(self, **kw) -> "CasConfig":
        """Same distributions, smaller counts (development / parity at oracle-friendly sizes)."""
        return replace(self, **kw)


CONFIGS = {
    # configs[0]: tiny fp32
    "c1": CasConfig("c1_tiny_fp32", "f32", Hq=2, Hkv=1, D=64, n_carts=4, n_slots=4, cart_len=32,
                    B=2, Lq=48, n_dist=2, kv_std=0.125, selection="uniform"),
    # configs[1]: bf16 3B-like layer
    "c2": CasConfig("c2_3b_like_bf16", "bf16", Hq=24, Hkv=8, D=128, n_carts=64, n_slots=64,
                    cart_len=1024, B=8, Lq=1024, n_dist=7, kv_std=0.02, selection="uniform"),
    # configs[2]: bf16 8B-like layer + rotation
    "c3": CasConfig("c3_8b_like_bf16_swap", "bf16", Hq=32, Hkv=8, D=128, n_carts=256, n_slots=128,
                    cart_len=2048, B=4, Lq=2048, n_dist=15, kv_std=0.02, selection="uniform",
                    rotate_in=16, rotate_out=16),
    # configs[3]: ragged bf16
    "c4": CasConfig("c4_ragged_bf16", "bf16", Hq=32, Hkv=8, D=128, n_carts=400, n_slots=400,
                    cart_len=0, B=16, Lq=0, n_dist=-1, kv_std=0.02, selection="prop_len"),
    # configs[4]: decode-style inference, forward only; (i) all loaded, (ii) top-8
    "c5_all": CasConfig("c5_decode_all_bf16", "bf16", Hq=32, Hkv=8, D=128, n_carts=500,
                        n_slots=500, cart_len=512, B=64, Lq=1, n_dist=-2, kv_std=0.02,
                        selection="all", backward=False),
    "c5_top8": CasConfig("c5_decode_top8_bf16", "bf16", Hq=32, Hkv=8, D=128, n_carts=500,
                         n_slots=500, cart_len=512, B=64, Lq=1, n_dist=7, kv_std=0.02,
                         selection="topk", backward=False),
    # NEXT-2, paper-true cartridge sizes at 50-100x compression (Table 8: FinQA / TechQA rows with
    # min 16, max 64-ish tokens; sizes are whole 16-token pages): 400 cartridges of 16..64 tokens, 200
    # resident in a paged pool, packed batch of 32 samples x 256 tokens (8,192 tokens, Table 5), each
    # sample sees its target + U{0..10} distractors, 20 in / 20 out per step.
    "c_pages": CasConfig("c_pages_16tok_bf16", "bf16", Hq=32, Hkv=8, D=128, n_carts=400, n_slots=200, cart_len=0,
                         B=32, Lq=256, n_dist=-1, n_dist_max=10, kv_std=0.02, selection="uniform", rotate_in=20,
                         rotate_out=20, tile_tokens=16, budget_tokens=16 * 560, len_pages_max=4),
}


def get_config(name: str) -> CasConfig:
    return CONFIGS[name]
