"""Pins for the oracle's extension rows — CPU only.

  f1  schedule: the pattern of step s depends on s only through s mod T_per (Eq. 3)
  f2  text tokens inside self-attention (reading R23): every query attends
      to the n_text tokens after the video tokens, and they attend to everything
Each pin restates the definition with numpy / a torch library routine, never with oracle code.
"""
import math

import numpy as np
import pytest
import torch

from conftest import read_golden_sets
from oracle import lvsa_oracle as orc


def rand_qkv(N, H, d, seed):
    rng = np.random.default_rng(seed)
    return tuple(rng.standard_normal((N, H, d)).astype(np.float32) for _ in range(3))


# ---------------------------------------------------------------- f1
def test_pattern_depends_on_step_only_through_its_phase():
    for T, W, a, k0 in [(8, 1, 2, 0), (21, 2, 16, 0), (121, 2, 16, 0), (65, 2, 28, 0), (13, 1, 3, 2)]:
        T_per = math.ceil(T / a)
        for s in range(2 * T_per + 3):
            p, q = orc.pattern(T, W, a, s, initial_anchors=k0), orc.pattern(T, W, a, s % T_per, initial_anchors=k0)
            assert np.array_equal(p.A, q.A) and np.array_equal(p.w_lo, q.w_lo) and np.array_equal(p.w_hi, q.w_hi)
        # T_per distinct phases really are distinct anchor sets (Fig. 2)
        sets = {tuple(orc.pattern(T, W, a, r).inG) for r in range(T_per)}
        assert len(sets) == T_per


# ---------------------------------------------------------------- f2
def token_mask_with_text(A, T, P, n_text):
    """N x N boolean mask straight from reading R23, A = the [T, T] video pattern."""
    N = T * P + n_text
    M = np.ones((N, N), bool)                       # text rows and text columns: everything
    f = np.arange(T * P) // P
    M[:T * P, :T * P] = A[f][:, f].astype(bool)
    return M


def masked_softmax_np(q, k, v, M):
    d = q.shape[-1]
    logits = np.einsum("nhd,mhd->hnm", q.astype(np.float64), k.astype(np.float64)) / math.sqrt(d)
    logits = np.where(M[None], logits, -np.inf)
    mx = logits.max(-1, keepdims=True)
    e = np.exp(logits - mx)
    out = np.einsum("hnm,mhd->nhd", e / e.sum(-1, keepdims=True), v.astype(np.float64))
    return out, (mx[..., 0] + np.log(e.sum(-1))).T


def test_with_text_shape_and_values():
    golden = np.zeros((8, 8), np.uint8)
    for (s, t), mem in read_golden_sets("worked_example_T8_W1_a2.txt"):
        if s == 0:
            golden[t, sorted(mem)] = 1
    Af = orc.with_text(golden)
    assert Af.shape == (9, 9) and Af[8].all() and Af[:, 8].all() and np.array_equal(Af[:8, :8], golden)


@pytest.mark.parametrize("T,P,n_text,W,a", [(5, 12, 7, 1, 2), (6, 10, 25, 1, 2), (4, 9, 1, 0, 0), (3, 16, 16, 1, 1)])
def test_text_tokens_match_token_level_masked_softmax(T, P, n_text, W, a):
    H, d = 2, 16
    N = T * P + n_text
    q, k, v = rand_qkv(N, H, d, 11)
    for s in (0, 1, 2):
        p = orc.pattern(T, W, a, s)
        want, want_lse = masked_softmax_np(q, k, v, token_mask_with_text(p.A, T, P, n_text))
        out, lse = orc.attn_rows(q, k, v, T, P, orc.with_text(p.A), np.arange(N), n_text=n_text)
        np.testing.assert_allclose(out, want, rtol=0, atol=1e-12)
        np.testing.assert_allclose(lse, want_lse, rtol=0, atol=1e-12)


def test_text_rows_are_dense_and_video_rows_are_gathered_sdpa():
    """Library routine (torch SDPA, fp64): a text query sees every token (Eq. 1); a video query of
    frame t sees the keys of frames A(t) plus the text keys (the paper's per-frame SDPA backend,
    PAPER.md:130, with the text strip appended)."""
    T, P, n_text, H, d = 6, 14, 9, 2, 32
    N = T * P + n_text
    q, k, v = rand_qkv(N, H, d, 5)
    p = orc.pattern(T, 1, 2, 1)
    out, _ = orc.attn_rows(q, k, v, T, P, orc.with_text(p.A), np.arange(N), n_text=n_text)

    def sdpa(qs, ks, vs):
        tq, tk, tv = (torch.from_numpy(np.ascontiguousarray(x)).double().permute(1, 0, 2)[None] for x in (qs, ks, vs))
        return torch.nn.functional.scaled_dot_product_attention(tq, tk, tv)[0].permute(1, 0, 2).numpy()

    np.testing.assert_allclose(out[T * P:], sdpa(q[T * P:], k, v), rtol=0, atol=1e-12)
    for t in range(T):
        keys = np.concatenate([np.arange(f * P, (f + 1) * P) for f in np.nonzero(p.A[t])[0]] + [np.arange(T * P, N)])
        rows = np.arange(t * P, (t + 1) * P)
        np.testing.assert_allclose(out[rows], sdpa(q[rows], k[keys], v[keys]), rtol=0, atol=1e-12)


def brute_force_tile_index_with_text(T, P, n_text, Bq, Bk, A):
    N = T * P + n_text
    M = token_mask_with_text(A, T, P, n_text)
    nq, nk = -(-N // Bq), -(-N // Bk)
    Mp = np.zeros((N, nk * Bk), bool)
    Mp[:, :N] = M
    indptr, indices, flags = [0], [], []
    for i in range(nq):
        rows = slice(i * Bq, min((i + 1) * Bq, N))
        for j in range(nk):
            blk = Mp[rows, j * Bk:(j + 1) * Bk]
            if blk.any():
                indices.append(j)
                flags.append(0 if blk.all() else 1)
        indptr.append(len(indices))
    return np.array(indptr, np.int32), np.array(indices, np.int32), np.array(flags, np.uint8)


@pytest.mark.parametrize("T,P,n_text,Bq,Bk,W,a", [
    (8, 64, 64, 64, 64, 1, 2), (8, 40, 30, 64, 64, 1, 2), (9, 200, 77, 128, 128, 1, 2),
    (7, 13, 5, 16, 32, 1, 2), (5, 100, 300, 128, 128, 0, 0), (10, 7, 3, 16, 16, 1, 3)])
def test_tile_index_with_text_equals_token_level_brute_force(T, P, n_text, Bq, Bk, W, a):
    for s in range(3):
        p = orc.pattern(T, W, a, s)
        Af = orc.with_text(p.A)
        got = orc.tile_index(T, P, Bq, Bk, Af, n_text=n_text)
        want = brute_force_tile_index_with_text(T, P, n_text, Bq, Bk, p.A)
        for g, w_ in zip(got, want):
            assert np.array_equal(g, w_), (s,)
        assert orc.csr_keyset_equal(T, P, Bq, Bk, Af, *got, np.arange(T * P + n_text), n_text=n_text)   # O9


def test_no_text_tokens_is_the_base_path():
    T, P, H, d = 5, 12, 2, 16
    q, k, v = rand_qkv(T * P, H, d, 3)
    p = orc.pattern(T, 1, 2, 0)
    a0 = orc.attn_rows(q, k, v, T, P, p.A, np.arange(T * P))
    a1 = orc.attn_rows(q, k, v, T, P, p.A, np.arange(T * P), n_text=0)
    assert np.array_equal(a0[0], a1[0]) and np.array_equal(a0[1], a1[1])
