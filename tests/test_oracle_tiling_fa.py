"""Pins for the oracle's SECOND tile definition: frame-aligned kv tiles (reading R25; the
paper is silent on how tokens map to blocks) -- CPU only.

The tiling changes cost, never the result, so what pins it is (a) the tiling itself against its
stated properties, (b) the tile index against a token-level N x N brute force written here in numpy
(not a retyping of the C loops: it slices a dense mask), (c) the key set a kernel would recover from
CSR + flags being exactly the token predicate, each key once, with negative tests, (d) the special
case that reduces to the already pinned definition (P a multiple of Bk: both tilings coincide), and
(e) the kept-column count against the exact Eq. 2 count.
"""
import math

import numpy as np
import pytest

from oracle import lvsa_oracle as orc

PAD = 32


def frame_ids(T, P, n_text):
    return np.concatenate([np.repeat(np.arange(T), P), np.full(n_text, T, dtype=np.int64)])


SHAPES = [(8, 40, 64, 1, 2, 0), (9, 200, 128, 1, 2, 0), (7, 13, 64, 1, 2, 0), (5, 300, 128, 2, 0, 0),
          (6, 128, 128, 1, 2, 0), (4, 1560, 128, 1, 1, 0), (9, 200, 128, 1, 2, 77), (8, 40, 64, 1, 2, 30),
          (3, 50, 64, 0, 1, 200), (12, 70, 64, 2, 3, 1)]


@pytest.mark.parametrize("T,P,Bk,W,a,n_text", SHAPES)
def test_tiles_partition_the_tokens_inside_frames(T, P, Bk, W, a, n_text):
    col0, width = orc.kv_tiles_frame_aligned(T, P, Bk, n_text)
    N = T * P + n_text
    fr = frame_ids(T, P, n_text)
    # closed form of the count: ceil(P/Bk) per video frame + ceil(n_text/Bk)
    assert len(col0) == T * math.ceil(P / Bk) + math.ceil(n_text / Bk)
    # contiguous, in order, covering [0, N) exactly
    assert col0[0] == 0 and np.array_equal(col0[1:], (col0 + width)[:-1]) and col0[-1] + width[-1] == N
    assert width.min() >= 1 and width.max() <= Bk
    for c, w in zip(col0, width):
        f = fr[c:c + w]
        assert (f == f[0]).all()                              # never crosses a frame boundary
        first_of_frame = c == 0 or fr[c - 1] != f[0]
        last_of_frame = c + w == N or fr[c + w] != f[0]
        assert w == Bk or last_of_frame                       # only a frame's last tile is narrow
        assert first_of_frame or (c - np.argmax(fr == f[0])) % Bk == 0


@pytest.mark.parametrize("T,P,Bk,W,a,n_text", SHAPES)
def test_tile_index_equals_token_level_brute_force(T, P, Bk, W, a, n_text):
    Bq = Bk
    for s in (0, 1, 3):
        p = orc.pattern(T, W, a, s)
        A = orc.with_text(p.A) if n_text else p.A
        indptr, indices, flags = orc.tile_index_fa(T, P, Bq, Bk, A, n_text=n_text, pad=PAD)
        col0, width = orc.kv_tiles_frame_aligned(T, P, Bk, n_text)
        N = T * P + n_text
        fr = frame_ids(T, P, n_text)
        M = A[fr][:, fr].astype(bool)                         # token-level N x N mask (Eq. 2 predicate)
        nq = math.ceil(N / Bq)
        want_ptr, want_idx, want_flag = [0], [], []
        for i in range(nq):
            rows = M[i * Bq:min((i + 1) * Bq, N)]
            for j, (c, w) in enumerate(zip(col0, width)):
                blk = rows[:, c:c + w]
                if blk.any():
                    want_idx.append(j)
                    want_flag.append(int((not blk.all()) or (w % PAD != 0)))
            want_ptr.append(len(want_idx))
        assert np.array_equal(indptr, want_ptr) and np.array_equal(indices, want_idx)
        assert np.array_equal(flags, want_flag)
        rows = np.arange(N)
        assert orc.csr_keyset_equal_tiles(T, P, Bq, A, col0, width, indptr, indices, flags, rows, n_text=n_text, pad=PAD)


def test_keyset_check_detects_wrong_flag_dropped_tile_and_overlap():
    T, P, B = 9, 200, 128
    p = orc.pattern(T, 1, 2, 1)
    indptr, indices, flags = orc.tile_index_fa(T, P, B, B, p.A, pad=PAD)
    col0, width = orc.kv_tiles_frame_aligned(T, P, B)
    rows = np.arange(T * P)
    ok = lambda **kw: orc.csr_keyset_equal_tiles(T, P, B, p.A, kw.get("col0", col0), kw.get("width", width), indptr,
                                                 kw.get("indices", indices), kw.get("flags", flags), rows, pad=PAD)
    assert ok()
    part = np.nonzero(flags)[0]
    assert len(part) > 0
    f2 = flags.copy(); f2[part[0]] = 0                         # a PARTIAL tile treated as FULL
    assert not ok(flags=f2)
    i2 = indices.copy(); i2[3] = i2[2]                          # a tile visited twice, one dropped
    assert not ok(indices=i2)
    c2 = col0.copy(); c2[5] -= 8                                # a tile that overlaps its neighbour
    assert not ok(col0=c2)
    w2 = width.copy(); w2[1] += 32                              # a narrow tile claimed wider than it is
    assert not ok(width=w2)


@pytest.mark.parametrize("T,P,B", [(6, 128, 128), (5, 256, 128), (7, 64, 64), (4, 192, 64)])
def test_reduces_to_the_token0_tiling_when_frames_are_tile_aligned(T, P, B):
    """P a multiple of Bk: frame boundaries are tile boundaries, so the two definitions coincide and
    the frame-aligned index must equal the (separately pinned) index of reading R14 bit for bit."""
    for s in (0, 1, 2):
        for W, a in ((1, 2), (0, 0), (2, 1)):
            p = orc.pattern(T, W, a, s)
            want = orc.tile_index(T, P, B, B, p.A)
            got = orc.tile_index_fa(T, P, B, B, p.A, pad=PAD)
            for x, y in zip(want, got):
                assert np.array_equal(x, y)
            col0, width = orc.kv_tiles_frame_aligned(T, P, B)
            assert np.array_equal(col0, np.arange(T * P // B) * B) and (width == B).all()


def test_kept_columns_closed_form_and_ratio_to_exact_work():
    """Wan 2.1 shapes (P = 1560 = 12 x 128 + 24): 13 tiles per frame, the last padded 24 -> 32.  A q tile
    inside frame t keeps exactly the 13 tiles of each of the |A(t)| = 21 frames, so its
    kept columns are 21 * (12 * 128 + 32); over the whole index the computed work is within 1.2 % of the
    exact Eq. 2 work (the token-0 tiling of R14: 5.5 % above)."""
    T, P, B = 121, 1560, 128
    p = orc.pattern(T, 2, 16, 0)
    indptr, indices, flags = orc.tile_index_fa(T, P, B, B, p.A, pad=PAD)
    col0, width = orc.kv_tiles_frame_aligned(T, P, B)
    assert len(col0) == 121 * 13 and sorted(set(width.tolist())) == [24, 128]
    wpad = ((width + PAD - 1) // PAD) * PAD
    for t in (0, 5, 60, 120):
        i = (t * P) // B + 1                                   # a q tile entirely inside frame t
        assert (i * B) // P == t and ((i + 1) * B - 1) // P == t
        kept = indices[indptr[i]:indptr[i + 1]]
        assert len(kept) == 21 * 13 and int(wpad[kept].sum()) == 21 * (12 * 128 + 32)
        assert int(flags[indptr[i]:indptr[i + 1]].sum()) == 21          # only the 21 narrow tiles
    computed = float(wpad[indices].sum()) * B                  # (row, column) pairs a kernel computes
    exact = float(p.A.sum()) * P * P                           # key pairs of Eq. 2
    r14 = orc.tile_index(T, P, B, B, p.A)
    assert 1.0 <= computed / exact <= 1.012, computed / exact
    assert len(r14[1]) * B * B / exact >= 1.05
