"""Pins for the oracle's pattern builder (O2-O5, O7) — CPU only.

Each test checks oracle/lvsa_oracle.c against something the paper or the mathematics fixes,
never against a retyping of the oracle's own formula:
  P3  |A(t)| = |G| + min(2W+1, T-|G|)
  P4  |G^s| = ceil(T/T_per)
  P5  anchors cover every frame in T_per steps
  P6  Fig. 2 anchor sets                          PAPER.md:108  (tests/golden)
  P7  C = (81-1)/4+1 = 21, T = 21..121
  P8  adaptive window: exactly 2W+1 frames
  P9  Algorithm 1 post-conditions
  P10 G empty -> textbook clamped sliding window
  P13 kept-tile closed form; token-level N x N brute force for the tile index
"""
import math

import numpy as np
import pytest

from conftest import read_golden_sets
from oracle import lvsa_oracle as orc


def members(row):
    return frozenset(int(x) for x in np.nonzero(row)[0])


# ---------------------------------------------------------------- P6 / P7: printed values
def test_fig2_anchor_sets_golden():
    for (T, a, s), want in read_golden_sets("fig2_anchor_sets.txt"):
        p = orc.pattern(T, 1, a, s)
        assert members(p.inG) == want, (T, a, s)
        assert p.T_per == math.ceil(T / a)


def test_worked_example_golden():
    for (s, t), want in read_golden_sets("worked_example_T8_W1_a2.txt"):
        p = orc.pattern(8, 1, 2, s)
        assert members(p.A[t]) == want, (s, t)
    # rotation period T_per = 4: step 4 repeats step 0
    assert np.array_equal(orc.pattern(8, 1, 2, 4).A, orc.pattern(8, 1, 2, 0).A)


def test_a_bits_packing_pinned_by_hand():
    """Pattern.a_bits() produces the expected value of bit-exact GPU comparisons, so its word / bit
    order is pinned here without a device: the golden worked example packed by hand (bit x of word
    x // 32 of row t set iff x in A(t), include/lvsa.h), and a T = 40 case that reaches the second
    word, whose rows follow from the paper alone (a = 0: G is empty and A(t) is the clamped sliding
    window of PAPER.md:68)."""
    # s = 0 rows of tests/golden/worked_example_T8_W1_a2.txt, written as literals:
    # {0,1,2,3,4} = 0x1f, {0,2,3,4,5} = 0x3d, {0,3,4,5,6} = 0x79, {0,4,5,6,7} = 0xf1
    want0 = np.array([[0x1f], [0x1f], [0x1f], [0x3d], [0x3d], [0x79], [0xf1], [0xf1]], np.uint32)
    got0 = orc.pattern(8, 1, 2, 0).a_bits()
    assert got0.dtype == np.uint32 and got0.shape == (8, 1) and np.array_equal(got0, want0)
    # and every row of the golden file, packed here with plain Python integers
    for (s, t), want in read_golden_sets("worked_example_T8_W1_a2.txt"):
        assert int(orc.pattern(8, 1, 2, s).a_bits()[t, 0]) == sum(1 << x for x in want), (s, t)
    # T = 40, W = 2, no anchors: A(t) = [clamp(t-2), clamp(t-2)+4]; frames 30..34 straddle the words
    p = orc.pattern(40, 2, 0, 0)
    bits = p.a_bits()
    assert bits.shape == (40, 2)
    for t in range(40):
        lo = max(0, min(t - 2, 40 - 5))
        full = sum(1 << x for x in range(lo, lo + 5))
        assert (int(bits[t, 0]), int(bits[t, 1])) == (full & 0xffffffff, full >> 32), t
    assert (int(bits[32, 0]), int(bits[32, 1])) == (0xc0000000, 0x7)      # {30,31} | {32,33,34}


def test_wan_budget_constants():
    # C = (81-1)/4 + 1 = 21 latent frames; :110: T from 21 (1x) to 121 (6x)
    C = (81 - 1) // 4 + 1
    assert C == 21
    assert [(f - 1) // 4 + 1 for f in (81, 161, 241, 321, 401, 481)] == [21, 41, 61, 81, 101, 121]
    W = 2
    p = orc.pattern(121, W, C - (2 * W + 1), 0)
    assert p.T_per == 8 and p.n_global == 16          # ceil(121/16) = 8, ceil(121/8) = 16
    assert int(p.A.sum(1).min()) == int(p.A.sum(1).max()) == 21   # |A(t)| = 16 + 5 = C


SWEEP = [(T, W, a) for T in (1, 2, 3, 5, 8, 9, 13, 21, 30, 47, 65) for W in (0, 1, 2, 3, 5)
         for a in (0, 1, 2, 3, 5, 8, 16, 40, 100)]


# ---------------------------------------------------------------- P3, P4, P9
@pytest.mark.parametrize("tie_hi", [0, 1])
def test_closed_form_budget_and_postconditions(tie_hi):
    for T, W, a in SWEEP:
        for s in range(0, 12):
            p = orc.pattern(T, W, a, s, tie_hi)
            nG = int(p.inG.sum())
            if a > 0:
                T_per = math.ceil(T / a)
                assert p.T_per == T_per and p.phase == s % T_per
                assert nG == math.ceil(T / T_per) == p.n_global          # P4
            else:
                assert nG == 0
            target = min(2 * W + 1, T - nG)
            for t in range(T):
                # P3: PAPER.md:66 / :91
                assert int(p.A[t].sum()) == nG + target, (T, W, a, s, t)
                lo, hi = int(p.w_lo[t]), int(p.w_hi[t])
                nong = sum(1 for x in range(lo, hi + 1) if not p.inG[x])
                # P9: Alg. 1 loop exit condition
                assert nong >= target or (lo == 0 and hi == T - 1)
                assert 0 <= lo <= t <= hi <= T - 1              # t in A(t): no empty softmax row
                # result contains the adaptive window of PAPER.md:68
                alo = max(0, min(t - W, T - 1 - 2 * W))
                ahi = min(T - 1, max(t + W, 2 * W))
                assert lo <= alo and hi >= ahi
                # the loop adds exactly one frame per iteration
                assert (hi - lo) - (ahi - alo) == int(p.iters[t])
                # A(t) is exactly G u [lo, hi] (Def. 2)
                assert members(p.A[t]) == members(p.inG) | frozenset(range(lo, hi + 1))


# ---------------------------------------------------------------- P5
def test_rotation_covers_every_frame():
    for T, W, a in SWEEP:
        if a == 0:
            continue
        T_per = math.ceil(T / a)
        for s0 in (0, 3, 17):
            seen = np.zeros(T, int)
            for s in range(s0, s0 + T_per):
                seen += orc.pattern(T, W, a, s).inG
            assert seen.min() >= 1, (T, a, s0)                 # PAPER.md:102 "at least once"
            if T % T_per == 0:
                assert seen.max() == 1, (T, a, s0)             # PAPER.md:108 "exactly once"
            else:
                assert seen.sum() - T <= T_per - 1             # "may revisit at most T_per-1 frames"


# ---------------------------------------------------------------- P8, P10
def test_adaptive_window_without_anchors_is_clamped_sliding_window():
    for T in (5, 8, 21, 64):
        for W in (0, 1, 2, 3):
            if 2 * W + 1 > T:
                continue
            p = orc.pattern(T, W, 0, 3)
            assert p.iters.max() == 0                          # Alg. 1 is a no-op when G is empty
            for t in range(T):
                got = members(p.A[t])
                assert len(got) == 2 * W + 1 and t in got      # PAPER.md:68 "exactly 2W+1"
                # textbook: window of width 2W+1 centred on t, shifted inside [0, T-1]
                c = min(max(t, W), T - 1 - W)
                assert got == frozenset(range(c - W, c + W + 1))


def test_full_coverage_cases_are_dense():
    # 2W+1 >= T, a >= T, or ALL_TILES => A(t) = all frames (Def. 1)
    for T, W, a in [(5, 2, 0), (5, 3, 1), (7, 1, 7), (7, 0, 50), (9, 1, orc.ALL_TILES)]:
        assert orc.pattern(T, W, a, 2).A.all(), (T, W, a)


def test_tie_break_reading_R5():
    # T = 9, W = 1, G = {4} u ... choose a = 1 -> T_per = 9, s = 4 -> G = {4}
    p_lo = orc.pattern(9, 1, 1, 4, 0)
    p_hi = orc.pattern(9, 1, 1, 4, 1)
    assert members(p_lo.inG) == {4}
    # t = 4: adaptive [3,5] holds 2 non-global < 3; rooms equal (3 and 3)
    assert (int(p_lo.w_lo[4]), int(p_lo.w_hi[4])) == (2, 5)
    assert (int(p_hi.w_lo[4]), int(p_hi.w_hi[4])) == (3, 6)
    # both satisfy the paper's closed form
    assert p_lo.A[4].sum() == p_hi.A[4].sum() == 1 + 3


# ---------------------------------------------------------------- O7: tile index
def brute_force_tile_index(T, P, Bq, Bk, A):
    """Token-level N x N restatement: mask M[nq, nk] = A[nq // P][nk // P]; a kv tile is kept
    iff any (valid row, valid col) is allowed; PARTIAL iff any (valid row, col of the padded
    tile) is not allowed (columns >= N count as not allowed)."""
    N = T * P
    f = np.arange(N) // P
    M = A[f][:, f].astype(bool)
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


@pytest.mark.parametrize("T,P,Bq,Bk,W,a", [
    (8, 64, 64, 64, 1, 2), (8, 40, 64, 64, 1, 2), (9, 200, 128, 128, 1, 2), (7, 13, 16, 32, 1, 2),
    (12, 50, 64, 32, 2, 3), (5, 100, 128, 128, 0, 0), (6, 21, 64, 64, 1, orc.ALL_TILES),
    (10, 7, 16, 16, 1, 3)])
def test_tile_index_equals_token_level_brute_force(T, P, Bq, Bk, W, a):
    for s in range(5):
        p = orc.pattern(T, W, a, s)
        got = orc.tile_index(T, P, Bq, Bk, p.A)
        want = brute_force_tile_index(T, P, Bq, Bk, p.A)
        for g, w_ in zip(got, want):
            assert np.array_equal(g, w_), (s,)
        rows = np.arange(T * P)
        assert orc.csr_keyset_equal(T, P, Bq, Bk, p.A, *got, rows)       # O9


def test_csr_keyset_check_detects_a_wrong_flag_and_a_dropped_tile():
    T, P, B = 8, 40, 64
    p = orc.pattern(T, 1, 2, 1)
    indptr, indices, flags = orc.tile_index(T, P, B, B, p.A)
    rows = np.arange(T * P)
    assert flags.any()
    bad = flags.copy()
    bad[np.nonzero(flags)[0][0]] = 0                                    # PARTIAL marked FULL
    assert not orc.csr_keyset_equal(T, P, B, B, p.A, indptr, indices, bad, rows)
    ind2 = indices.copy()
    ind2[0] = (ind2[0] + 3) % (-(-T * P // B))                          # wrong tile listed
    assert not orc.csr_keyset_equal(T, P, B, B, p.A, indptr, ind2, flags, rows)


def test_kept_tile_closed_form_P13():
    # tiny (BASELINE.json config 1): Bk | P, so every q tile keeps |A(t)| * P / Bk = 5 tiles,
    # none PARTIAL; nnz = 8 * 5 = 40.
    for s in range(10):
        p = orc.pattern(8, 1, 2, s)
        indptr, indices, flags = orc.tile_index(8, 64, 64, 64, p.A)
        assert np.array_equal(np.diff(indptr), np.full(8, 5)) and not flags.any()
        for t in range(8):
            assert frozenset(indices[indptr[t]:indptr[t + 1]].tolist()) == members(p.A[t])
    # general closed form for q tiles inside one frame, P >= Bk: sum over maximal runs [x, y] of
    # A(t) of ( min(nk, ceil((y+1)P/Bk)) - floor(xP/Bk) )
    T, P, B = 21, 1560, 128
    N = T * P
    nk = -(-N // B)
    p = orc.pattern(T, 2, 16, 25)
    indptr, indices, flags = orc.tile_index(T, P, B, B, p.A)
    checked = 0
    for i in range(-(-N // B)):
        r0, r1 = i * B, min((i + 1) * B, N) - 1
        if r0 // P != r1 // P:
            continue
        t = r0 // P
        fr = sorted(members(p.A[t]))
        runs, x = [], fr[0]
        for u, v in zip(fr, fr[1:] + [None]):
            if v != u + 1:
                runs.append((x, u))
                x = v
        want = sum(min(nk, -(-(y + 1) * P // B)) - (x0 * P) // B for x0, y in runs)
        assert indptr[i + 1] - indptr[i] == want, i
        checked += 1
    assert checked > 200


def test_survey_tile_counts_rederived():
    # SURVEY.md section 8(a) quotes survey-derived nnz; the oracle re-derives them.
    p = orc.pattern(21, 2, 16, 25)
    assert orc.tile_index(21, 1560, 128, 128, p.A)[0][-1] == 51075
    p = orc.pattern(121, 2, 16, 25)
    indptr, indices, flags = orc.tile_index(121, 1560, 128, 128, p.A)
    assert indptr[-1] == 396647 and len(indptr) == 1476
    per = np.diff(indptr)
    assert per.min() == 268 and 269 <= per.max() <= 282
    assert 0.09 <= flags.mean() <= 0.12
    p0 = orc.pattern(121, 2, 16, 0)
    assert orc.tile_index(121, 1560, 128, 128, p0.A)[0][-1] == 398161
    # Eq. 3 depends on the step only through s mod T_per: steps 25 and 49 share phase 1
    assert np.array_equal(orc.pattern(121, 2, 16, 49).A, p.A)


def test_alg1_loop_statistics_report_only():
    # PAPER.md:91 prints "at most 8 iterations per call (mean 1.21)"; with reading R1 (W = 2,
    # C = 21) over T in {21..121} x 40 steps the oracle gives mean 1.209 (max 6).  The mean is
    # evidence for R1, not a pin the paper fixes; asserted loosely so a changed Alg. 1 shows up.
    tot = calls = mx = 0
    for T in (21, 41, 61, 81, 101, 121):
        for s in range(40):
            it = orc.pattern(T, 2, 16, s).iters
            tot += int(it.sum()); calls += T; mx = max(mx, int(it.max()))
    assert abs(tot / calls - 1.21) < 0.01 and mx <= 8


# ---------------------------------------------------------------- dedicated initial anchors (R22)
def test_initial_anchor_golden():
    # hand-derived example, PAPER.md:54, :58 + Algorithm 1 with G' = G^s u {0..k0-1}
    for (s, t), want in read_golden_sets("initial_anchor_example_T8_W1_a2_k1.txt"):
        p = orc.pattern(8, 1, 2, s, initial_anchors=1)
        assert members(p.A[t]) == want, (s, t)


def test_initial_anchors_invariants():
    for T, W, a in SWEEP:
        for k0 in (0, 1, 2, 5, T, T + 3):
            for s in (0, 1, 7):
                p = orc.pattern(T, W, a, s, initial_anchors=k0)
                base = orc.pattern(T, W, a, s)
                if k0 == 0:
                    # the paper's pattern is the special case k0 = 0
                    assert np.array_equal(p.A, base.A) and p.n_global == base.n_global
                # G' = G^s u {0..k0-1}, with G^s restated here from Eq. 3
                G = set()
                if a > 0:
                    T_per = math.ceil(T / a)
                    G = {((s % T_per) + i * T_per) % T for i in range(math.ceil(T / T_per))}
                Gp = G | set(range(min(k0, T)))
                assert members(p.inG) == frozenset(Gp) and p.n_global == len(Gp)
                # every query frame attends to the dedicated anchors
                assert p.A[:, :min(k0, T)].all()
                # closed-form budget with |G'|
                want = len(Gp) + min(2 * W + 1, T - len(Gp))
                assert (p.A.sum(1) == want).all(), (T, W, a, k0, s)
                assert all(p.A[t, t] for t in range(T))
                if k0 >= T:
                    assert p.A.all()     # every frame an anchor: dense (Def. 1)
