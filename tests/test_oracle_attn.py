"""Pins for the oracle's attention (O6, O8) — CPU only.

  P1  full coverage => Eq. 1 = library softmax(QK^T/sqrt d)V
  P2  softmax rows sum to 1 (V = 1 => out = 1)
  P12 token-level N x N masked softmax on tiny, mask from the hand-derived worked example
  P14 Q = 0, V = one-hot(frame): out[:, c] = [c in A(t)]/|A(t)|, lse = ln(|A(t)| P)
  P15 invariances of Eq. 2 (key permutation inside a frame; affine maps of V)
  P16 per-frame gathered dense attention = the paper's "LVSA via SDPA" backend
"""
import math

import numpy as np
import pytest
import torch

from conftest import read_golden_sets
from oracle import lvsa_oracle as orc
from paper_2605_31057_b200 import inputs


def rand_qkv(N, H, d, seed, dtype=np.float32):
    rng = np.random.default_rng(seed)
    return tuple(rng.standard_normal((N, H, d)).astype(dtype) for _ in range(3))


def sdpa_fp64(q, k, v):
    """Library routine: torch scaled_dot_product_attention on CPU in fp64. q,k,v: [n, H, d]."""
    tq, tk, tv = (torch.from_numpy(np.ascontiguousarray(x)).double().permute(1, 0, 2)[None] for x in (q, k, v))
    o = torch.nn.functional.scaled_dot_product_attention(tq, tk, tv)
    return o[0].permute(1, 0, 2).numpy()


# ---------------------------------------------------------------- P1
@pytest.mark.parametrize("T,P,W,a", [(6, 17, 1, orc.ALL_TILES), (5, 20, 2, 0), (7, 11, 0, 7), (4, 33, 5, 1)])
def test_full_coverage_reduces_to_dense_eq1(T, P, W, a):
    H, d = 3, 32
    q, k, v = rand_qkv(T * P, H, d, 1)
    p = orc.pattern(T, W, a, 3)
    rows = np.arange(T * P)
    out, lse = orc.attn_rows(q, k, v, T, P, p.A, rows)
    np.testing.assert_allclose(out, sdpa_fp64(q, k, v), rtol=0, atol=1e-12)
    s = np.einsum("nhd,mhd->hnm", q.astype(np.float64), k.astype(np.float64)) / math.sqrt(d)
    want_lse = torch.logsumexp(torch.from_numpy(s), dim=-1).numpy().T
    np.testing.assert_allclose(lse, want_lse, rtol=0, atol=1e-12)


# ---------------------------------------------------------------- P2
def test_rows_sum_to_one():
    T, P, H, d = 9, 23, 2, 16
    q, k, v = rand_qkv(T * P, H, d, 2)
    v = np.ones_like(v)
    for s in range(4):
        p = orc.pattern(T, 1, 2, s)
        out, _ = orc.attn_rows(q, k, v, T, P, p.A, np.arange(T * P))
        assert np.abs(out - 1.0).max() <= 1e-14


# ---------------------------------------------------------------- P12
def test_tiny_matches_token_level_masked_softmax_from_worked_example():
    """Mask built from tests/golden/worked_example (hand-derived A(t)), NOT from the oracle's
    pattern code; dense masked softmax written with numpy on the N x N matrix."""
    T, P, H, d = 8, 64, 2, 64
    golden = {}
    for (s, t), mem in read_golden_sets("worked_example_T8_W1_a2.txt"):
        golden.setdefault(s, np.zeros((T, T), bool))[t, sorted(mem)] = True
    w = inputs.WORKLOADS["tiny"]
    q, k, v = (inputs.to_oracle_array(x[0]) for x in inputs.make_qkv(w, "cpu", torch.bfloat16))
    f64 = lambda x: torch.from_numpy(x.view(np.int16)).view(torch.bfloat16).double().numpy()
    qd, kd, vd = f64(q), f64(k), f64(v)
    frame = np.arange(T * P) // P
    for s, Aset in golden.items():
        M = Aset[frame][:, frame]
        logits = np.einsum("nhd,mhd->hnm", qd, kd) / math.sqrt(d)
        logits = np.where(M[None], logits, -np.inf)
        mx = logits.max(-1, keepdims=True)
        e = np.exp(logits - mx)
        want = np.einsum("hnm,mhd->nhd", e / e.sum(-1, keepdims=True), vd)
        want_lse = (mx[..., 0] + np.log(e.sum(-1))).T
        p = orc.pattern(T, w.W, w.a, s)
        out, lse = orc.attn_rows(q, k, v, T, P, p.A, np.arange(T * P))
        np.testing.assert_allclose(out, want, rtol=0, atol=1e-12)
        np.testing.assert_allclose(lse, want_lse, rtol=0, atol=1e-12)


# ---------------------------------------------------------------- P14
@pytest.mark.parametrize("name", ["tiny", "tiny_straddle", "small128"])
def test_closed_form_probe(name):
    w = inputs.WORKLOADS[name]
    q, k, v = (inputs.to_oracle_array(x[0]) for x in inputs.probe_qkv(w, "cpu", torch.bfloat16))
    for s in w.steps[:5]:
        p = orc.pattern(w.T, w.W, w.a, s)
        rows = np.arange(0, w.N, 7)
        out, lse = orc.attn_rows(q, k, v, w.T, w.P, p.A, rows)
        for i, n in enumerate(rows):
            t = n // w.P
            cnt = int(p.A[t].sum())
            want = np.zeros(w.d)
            want[:w.T] = p.A[t] / cnt
            assert np.abs(out[i] - want[None]).max() <= 1e-14
            assert np.abs(lse[i] - math.log(cnt * w.P)).max() <= 1e-12


# ---------------------------------------------------------------- P15
def test_invariances():
    T, P, H, d = 7, 19, 2, 16
    N = T * P
    q, k, v = rand_qkv(N, H, d, 5)
    p = orc.pattern(T, 1, 2, 2)
    rows = np.arange(N)
    out, lse = orc.attn_rows(q, k, v, T, P, p.A, rows)
    # permute tokens inside every key frame (K and V together): nothing changes
    rng = np.random.default_rng(0)
    perm = np.concatenate([t * P + rng.permutation(P) for t in range(T)])
    out2, lse2 = orc.attn_rows(q, k[perm], v[perm], T, P, p.A, rows)
    np.testing.assert_allclose(out2, out, rtol=0, atol=1e-13)
    np.testing.assert_allclose(lse2, lse, rtol=0, atol=1e-13)
    # V <- 2 V + u: out <- 2 out + u, lse unchanged (weights sum to 1); exact in fp32 for these u
    u = rng.integers(-3, 4, size=(1, H, d)).astype(np.float32)
    out3, lse3 = orc.attn_rows(q, k, (2 * v + u).astype(np.float32), T, P, p.A, rows)
    v_exact = (2 * v + u).astype(np.float32).astype(np.float64)
    # use the exactly representable transformed V as ground truth for the map
    out3_want, _ = orc.attn_rows(q, k, v, T, P, p.A, rows)
    resid = v_exact - (2 * v.astype(np.float64) + u)           # fp32 rounding of 2v+u
    assert np.abs(out3 - (2 * out3_want + u)).max() <= np.abs(resid).max() + 1e-12
    np.testing.assert_allclose(lse3, lse, rtol=0, atol=1e-13)


# ---------------------------------------------------------------- P16
def test_per_frame_gathered_sdpa_equivalence():
    """LVSA = for each query frame, dense attention over the gathered K, V of
    the frames in A(t).  The frame sets come from the golden worked example where available and
    from the closed-form-checked pattern otherwise."""
    T, P, H, d = 8, 29, 2, 32
    q, k, v = rand_qkv(T * P, H, d, 7)
    golden = {}
    for (s, t), mem in read_golden_sets("worked_example_T8_W1_a2.txt"):
        golden[(s, t)] = sorted(mem)
    for s in (0, 1):
        p = orc.pattern(T, 1, 2, s)
        out, _ = orc.attn_rows(q, k, v, T, P, p.A, np.arange(T * P))
        for t in range(T):
            keys = np.concatenate([np.arange(f * P, (f + 1) * P) for f in golden[(s, t)]])
            want = sdpa_fp64(q[t * P:(t + 1) * P], k[keys], v[keys])
            np.testing.assert_allclose(out[t * P:(t + 1) * P], want, rtol=0, atol=1e-12)


def test_bf16_and_fp32_input_decoding_agree():
    w = inputs.WORKLOADS["tiny_straddle"]
    qb, kb, vb = inputs.make_qkv(w, "cpu", torch.bfloat16)
    p = orc.pattern(w.T, w.W, w.a, 1)
    rows = np.arange(0, w.N, 3)
    o1, l1 = orc.attn_rows(*(inputs.to_oracle_array(x[0]) for x in (qb, kb, vb)), w.T, w.P, p.A, rows)
    o2, l2 = orc.attn_rows(*(inputs.to_oracle_array(x[0].float()) for x in (qb, kb, vb)), w.T, w.P, p.A, rows)
    assert np.array_equal(o1, o2) and np.array_equal(l1, l2)


def test_scale_argument():
    T, P, H, d = 4, 10, 1, 8
    q, k, v = rand_qkv(T * P, H, d, 9)
    p = orc.pattern(T, 1, orc.ALL_TILES, 0)
    o_default, _ = orc.attn_rows(q, k, v, T, P, p.A, np.arange(T * P))
    o_explicit, _ = orc.attn_rows(q, k, v, T, P, p.A, np.arange(T * P), scale=1 / math.sqrt(d))
    assert np.array_equal(o_default, o_explicit)
