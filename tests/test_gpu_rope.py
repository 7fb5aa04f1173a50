"""GPU parity of cas_rope_apply against oracle.rope on the same seeded
inputs: both pair layouts, forward and transposed map, fp32 and bf16, ragged sequences, position offsets as
large as a 256,000-token prefix, and the full c2 query tensor (sampled rows)."""
import numpy as np
import pytest
import torch

from oracle import cas_oracle as orc
from paper_2606_04557_b200 import _build, cas
from workloads import CONFIGS, make_workload

from parity_util import rel_fro, rel_max

pytestmark = pytest.mark.gpu
TOL_F32 = 2e-6     # fp32 in/out, angles in double: two roundings of the fused multiply-adds
TOL_BF16 = 4e-3    # one RNE rounding of each output to bf16 (2^-9 per element)


@pytest.fixture(scope="module", autouse=True)
def built():
    _build.build()


def run(X, seq_off, pos_off, base, layout, inverse, dtype):
    tdt = torch.float32 if dtype == "f32" else torch.bfloat16
    d = torch.from_numpy(X).to("cuda").to(tdt)
    T, H, D = X.shape
    cas.cas_rope_apply(cas.CAS_F32 if dtype == "f32" else cas.CAS_BF16, seq_off, pos_off, H, D, base, layout, inverse, d)
    torch.cuda.synchronize()
    return d.float().cpu().numpy()


@pytest.mark.parametrize("dtype,D", [("f32", 64), ("bf16", 128), ("bf16", 64)])
@pytest.mark.parametrize("layout", [0, 1])
@pytest.mark.parametrize("inverse", [False, True])
def test_rope_small_ragged(dtype, D, layout, inverse):
    rng = np.random.default_rng(100 + D + layout)
    lens = [37, 1, 300, 129]
    seq_off = np.concatenate([[0], np.cumsum(lens)]).astype(np.int32)
    pos_off = np.array([0, 4096, 32768, 256000], dtype=np.int64)     # c3- and c5-sized prefixes
    X = rng.standard_normal((int(seq_off[-1]), 5, D)).astype(np.float32)
    if dtype == "bf16":
        X = torch.from_numpy(X).to(torch.bfloat16).float().numpy()   # both sides consume the rounded inputs
    got = run(X, seq_off, pos_off, 1.0e6, layout, inverse, dtype)
    want = orc.rope(X, seq_off, pos_off, 1.0e6, layout, inverse)
    if dtype == "f32":
        assert rel_max(got, want) <= TOL_F32
    else:
        assert rel_fro(got, want) <= TOL_BF16
    # round trip on the device: the transposed map undoes the map up to the output rounding
    back = run(got, seq_off, pos_off, 1.0e6, layout, not inverse, dtype)
    assert rel_fro(back, X) <= (1e-6 if dtype == "f32" else 2 * TOL_BF16)


def test_rope_c2_full_size_sampled():
    wl = make_workload(CONFIGS["c2"])
    P = np.array([int(wl.cart_len[wl.sel_cart[wl.sel_off[b]:wl.sel_off[b + 1]]].sum()) for b in range(wl.cfg.B)],
                 dtype=np.int64)                                      # visible prefix per sequence (8192)
    Xq = torch.from_numpy(wl.Q).to(torch.bfloat16).float().numpy()
    got = run(Xq, wl.seq_off, P, 1.0e6, 1, False, "bf16")
    rows = np.random.default_rng(3).choice(wl.T, 48, replace=False)
    rows = np.concatenate([rows, [0, wl.T - 1]])
    for t in rows:                                                    # the oracle on single tokens
        b = int(np.searchsorted(wl.seq_off, t, side="right") - 1)
        want = orc.rope(Xq[t:t + 1], np.array([0, 1]), np.array([P[b] + t - wl.seq_off[b]]), 1.0e6, 1)
        assert rel_fro(got[t:t + 1], want) <= TOL_BF16
    assert np.isfinite(got).all()


def test_rope_error_codes():
    x = torch.zeros((4, 2, 24), dtype=torch.bfloat16, device="cuda")
    with pytest.raises(cas.CasError):
        cas.cas_rope_apply(cas.CAS_BF16, [0, 4], [0], 2, 24, 1e4, 1, False, x)     # D/2 not a 16-byte multiple
    with pytest.raises(cas.CasError):
        cas.cas_rope_apply(cas.CAS_BF16, [0, 4], [-1], 2, 32, 1e4, 0, False, x)    # negative offset


def test_rope_many_sequences_multiple_launches():
    # more sequences than one launch's parameter table holds (128): decode-like batch of 1- to 3-token sequences
    rng = np.random.default_rng(77)
    lens = rng.integers(1, 4, size=300)
    seq_off = np.concatenate([[0], np.cumsum(lens)]).astype(np.int32)
    pos_off = rng.integers(0, 300000, size=300).astype(np.int64)
    X = rng.standard_normal((int(seq_off[-1]), 3, 32)).astype(np.float32)
    got = run(X, seq_off, pos_off, 1.0e4, 0, False, "f32")
    assert rel_max(got, orc.rope(X, seq_off, pos_off, 1.0e4, 0)) <= TOL_F32
