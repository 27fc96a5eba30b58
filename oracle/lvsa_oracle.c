/*
 * lvsa_oracle.c — TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 / exact-integer CPU restatement of the LVSA hot path of
 * arxiv/paper_2605_31057 ("LVSA: Training-Free Sparse Attention for Long Video
 * Diffusion"), written from /root/reference/PAPER.md only.  It shares no code,
 * header, table or helper with the CUDA path under paper_2605_31057_b200/csrc.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may call it.
 *
 * What is restated, in the paper's order and notation:
 *   O2  T_per = ceil(T / (C-(2W+1)))                    PAPER.md:62  (section 2)
 *       G^s   = {(s mod T_per + i*T_per) mod T}          PAPER.md:97  (Eq. 3)
 *   O3  adaptive window w'_lo, w'_hi
 *   O4  Algorithm 1, expanded window bounds
 *   O5  A(t) = G u W(t)                                  PAPER.md:49  (Def. 2)
 *   O6  token predicate frame(nk) in A(frame(nq))        PAPER.md:31,42 (Eq. 2)
 *   O7  tile index = definition over token tiles         DESIGN.md reading R14 (paper silent)
 *   O8  Eq. 2 = softmax over the allowed keys, fp64
 *   O9  the same key set recovered through CSR + flags + element mask
 *   O7b a second, frame-aligned kv tiling and its tile index     DESIGN.md reading R25 (cost only)
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): Fig. 2 anchor sets, the closed
 * form |A(t)| = |G| + min(2W+1, T-|G|), |G^s| = ceil(T/T_per)
 * (PAPER.md:102), coverage over T_per steps, exactly 2W+1
 * adaptive-window frames, dense reduction to library
 * softmax(QK^T/sqrt d)V, per-frame gathered SDPA,
 * rows summing to 1, the Q=0 closed form, token-level N x N brute force on tiny
 * inputs; for the second tile definition (O7b, tests/test_oracle_tiling_fa.py): the
 * partition properties of the tiling, the same N x N brute force, key-set equality with
 * negative tests, the reduction to O7 when P is a multiple of Bk, and the kept-column
 * closed form at the Wan shapes.  Parity UNPINNED (fixed by DESIGN.md readings, not by the paper):
 * the default W (R1), HunyuanVideo's C (R2), the Algorithm-1 tie-break (R5), and the two
 * extension rules the paper names without specifying: dedicated initial anchors (R22,
 * lvsa_oracle_pattern_ex) and text tokens inside self-attention (R23, frame_of;
 * PAPER.md:132).  Their pins (tests/test_oracle_extensions.py, test_oracle_pattern.py) check that
 * the oracle computes exactly the stated rule: a hand-derived golden example, closed-form budgets,
 * a token-level N x N numpy mask and library SDPA on gathered keys.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <time.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define LVSA_ORACLE_ALL_TILES (-1)

/* ---- O2: T_per and the rotating anchor set G^s (Eq. 3 :97) ---------------- */
/* a = C-(2W+1) is the anchor target.  a == 0: G empty (reading R7).  a >= T: T_per = 1, every
 * frame an anchor.  meta = {T_per, s mod T_per, |G^s| (counted, not assumed)}. */
void lvsa_oracle_anchor_set(int T, int a, int s, uint8_t *inG, int32_t *meta)
{
    memset(inG, 0, (size_t)T);
    if (a <= 0) { meta[0] = 0; meta[1] = 0; meta[2] = 0; return; }
    int T_per = (T + a - 1) / a;                 /* ceil(T / a) */
    int m = (T + T_per - 1) / T_per;             /* ceil(T / T_per) members, Eq. 3 */
    int r = s % T_per;
    for (int i = 0; i < m; ++i) inG[(r + i * T_per) % T] = 1;
    int cnt = 0;
    for (int t = 0; t < T; ++t) cnt += inG[t];
    meta[0] = T_per; meta[1] = r; meta[2] = cnt;
}

/* ---- O3 + O4: adaptive window then Algorithm 1 ----------- */
static int imin(int x, int y) { return x < y ? x : y; }
static int imax(int x, int y) { return x > y ? x : y; }

/* tie_hi == 0: equal room extends the low side (reading R5, the default). */
void lvsa_oracle_window(int T, int W, const uint8_t *inG, int nG, int tie_hi, int t,
                        int32_t *lo, int32_t *hi, int32_t *iters)
{
    /* Alg. 1 line 1: (l,h) <- (w'_lo(t), w'_hi(t)) */
    int l = imax(0, imin(t - W, T - 1 - 2 * W));
    int h = imin(T - 1, imax(t + W, 2 * W));
    /* line 2 */
    int target = imin(2 * W + 1, T - nG);
    /* line 3 */
    int nonglobal = 0;
    for (int x = l; x <= h; ++x) nonglobal += !inG[x];
    int it = 0;
    /* line 4 */
    while (nonglobal < target && (l > 0 || h < T - 1)) {
        /* line 5: extend the side with the most room by 1 (room = frames left before the
         * boundary on that side, reading R5) */
        int room_lo = l, room_hi = T - 1 - h, nw;
        if (room_lo > room_hi || (room_lo == room_hi && !tie_hi)) { l -= 1; nw = l; }
        else                                                      { h += 1; nw = h; }
        if (!inG[nw]) nonglobal += 1;
        ++it;
    }
    /* line 7 */
    *lo = l; *hi = h; *iters = it;
}

/* ---- O5: A(t) = G^s u [w_lo(t), w_hi(t)] as a T x T 0/1 matrix, row t = query frame ------ */
/* a == LVSA_ORACLE_ALL_TILES: A(t) = all frames (Def. 1).
 * k0 = number of dedicated initial anchors ("frame 0 is always a global anchor",
 * :58 "an extension including more dedicated initial anchors is a straightforward
 * generalization"; reading R22): G' = G^s u {0, ..., min(k0,T)-1}.  Frames of G' are
 * the "global" frames of Algorithm 1 (its target and its non-global count use |G'|); T_per is
 * still derived from a alone.  k0 = 0 is the paper's pattern.  meta[2] = |G'| (counted). */
void lvsa_oracle_pattern_ex(int T, int W, int a, int s, int tie_hi, int k0,
                            uint8_t *A, int32_t *w_lo, int32_t *w_hi, uint8_t *inG,
                            int32_t *iters, int32_t *meta)
{
    if (a == LVSA_ORACLE_ALL_TILES) {
        memset(A, 1, (size_t)T * T);
        memset(inG, 0, (size_t)T);
        for (int t = 0; t < T; ++t) { w_lo[t] = 0; w_hi[t] = T - 1; iters[t] = 0; }
        meta[0] = 0; meta[1] = 0; meta[2] = 0;
        return;
    }
    lvsa_oracle_anchor_set(T, a, s, inG, meta);
    for (int f = 0; f < k0 && f < T; ++f) inG[f] = 1;
    int cnt = 0;
    for (int t = 0; t < T; ++t) cnt += inG[t];
    meta[2] = cnt;
    for (int t = 0; t < T; ++t) {
        lvsa_oracle_window(T, W, inG, meta[2], tie_hi, t, &w_lo[t], &w_hi[t], &iters[t]);
        for (int x = 0; x < T; ++x)
            A[(size_t)t * T + x] = (uint8_t)(inG[x] || (x >= w_lo[t] && x <= w_hi[t]));
    }
}

void lvsa_oracle_pattern(int T, int W, int a, int s, int tie_hi,
                         uint8_t *A, int32_t *w_lo, int32_t *w_hi, uint8_t *inG,
                         int32_t *iters, int32_t *meta)
{
    lvsa_oracle_pattern_ex(T, W, a, s, tie_hi, 0, A, w_lo, w_hi, inG, iters, meta);
}

/* ---- token -> frame (reading R12), with the text extension (reading R23) ------ */
/* Video token n = t*P + p belongs to frame t.  When n_text > 0 the n_text tokens after the T*P
 * video tokens (HunyuanVideo's text tokens inside self-attention) form one
 * pseudo-frame with index T; A then has T+1 rows/columns, row T and column T all ones. */
static inline int64_t frame_of(int64_t n, int T, int P)
{
    return n < (int64_t)T * P ? n / P : T;
}

/* ---- O7: tile index straight from the definition -------------------------------------- */
/* K(i) = sorted { j : exists valid row nq of tile i and valid column nk of tile j with
 *                     M(nq,nk) },  M(nq,nk) = A[frame(nq)][frame(nk)],  frame(n) = n / P (R12)
 * flag(i,j) = 1 (PARTIAL) iff exists valid row nq of tile i and column c in [j*Bk,(j+1)*Bk)
 *             with c >= N or not M(nq,c);  else 0 (FULL).
 * M depends on tokens only through their frames, so "exists a token pair" is evaluated as
 * "exists a pair of frames present in the two tiles"; the frame lists are found by walking
 * every token of the tile.  No interval arithmetic.
 * indices == NULL: count only.  Returns nnz, or -1 if cap is too small. */
int64_t lvsa_oracle_tile_index(int T, int P, int n_text, int Bq, int Bk, const uint8_t *A,
                               int32_t *indptr, int32_t *indices, uint8_t *flags, int64_t cap)
{
    /* A is Tf x Tf, Tf = T + (n_text > 0) */
    const int64_t N = (int64_t)T * P + n_text;
    const int Tv = T;
    T = T + (n_text > 0 ? 1 : 0);
    const int64_t nq = (N + Bq - 1) / Bq, nk = (N + Bk - 1) / Bk;
    uint8_t *fq = (uint8_t *)malloc((size_t)T), *fk = (uint8_t *)malloc((size_t)T);
    /* frames present among the valid columns of every kv tile, nk x T */
    uint8_t *kfr = (uint8_t *)calloc((size_t)nk * T, 1);
    for (int64_t j = 0; j < nk; ++j)
        for (int64_t c = j * Bk; c < (j + 1) * Bk && c < N; ++c) kfr[j * T + frame_of(c, Tv, P)] = 1;
    int64_t nnz = 0;
    for (int64_t i = 0; i < nq; ++i) {
        if (indptr) indptr[i] = (int32_t)nnz;
        memset(fq, 0, (size_t)T);
        for (int64_t r = i * Bq; r < (i + 1) * Bq && r < N; ++r) fq[frame_of(r, Tv, P)] = 1;
        for (int64_t j = 0; j < nk; ++j) {
            memcpy(fk, kfr + j * T, (size_t)T);
            int any_allowed = 0, any_disallowed = ((j + 1) * Bk > N);
            for (int tq = 0; tq < T; ++tq) {
                if (!fq[tq]) continue;
                for (int tk = 0; tk < T; ++tk) {
                    if (!fk[tk]) continue;
                    if (A[(size_t)tq * T + tk]) any_allowed = 1; else any_disallowed = 1;
                }
            }
            if (!any_allowed) continue;
            if (indices) {
                if (nnz >= cap) { free(fq); free(fk); free(kfr); return -1; }
                indices[nnz] = (int32_t)j;
                flags[nnz] = (uint8_t)any_disallowed;
            }
            ++nnz;
        }
    }
    if (indptr) indptr[nq] = (int32_t)nnz;
    free(fq); free(fk); free(kfr);
    return nnz;
}

/* ---- O7b: frame-aligned kv tiling (reading R25; the paper does not say how tokens map
 * to blocks, and names further performance work as open) ----------- */
/* Second tile definition, cost-only: the result of Eq. 2 does not depend on it.  The q tiles stay
 * Bq tokens from token 0.  The kv tiles RESTART AT EVERY FRAME BOUNDARY: frame tau (P tokens; the
 * text pseudo-frame has n_text) is cut into ceil(F/Bk) tiles, all Bk wide except the frame's last;
 * tiles are numbered in token order.  So every kv tile lies inside ONE frame, and for a query row
 * a tile is attended as a whole or not at all.
 * Found by walking the tokens: a new tile starts at the first token of a frame and every Bk tokens
 * after it.  col0[j] = first token of tile j, width[j] = its tokens.  Returns nk (cap: array size,
 * -1 if too small; col0 == NULL: count only). */
int64_t lvsa_oracle_kv_tiles_frame_aligned(int T, int P, int n_text, int Bk, int32_t *col0,
                                           int32_t *width, int64_t cap)
{
    const int64_t N = (int64_t)T * P + n_text;
    int64_t nk = 0, in_tile = 0, prev_frame = -1;
    for (int64_t n = 0; n < N; ++n) {
        const int64_t f = frame_of(n, T, P);
        if (f != prev_frame || in_tile == Bk) {          /* open a new tile */
            if (col0) { if (nk >= cap) return -1; col0[nk] = (int32_t)n; width[nk] = 0; }
            ++nk; in_tile = 0; prev_frame = f;
        }
        if (width) width[nk - 1] += 1;
        ++in_tile;
    }
    return nk;
}

/* Tile index over that tiling.  A kernel computes a kv tile over wpad = ceil(width/pad)*pad columns
 * (pad = its column granularity; the columns past `width` are padding and never allowed):
 *   K(i)      = sorted { j : exists valid row nq of q tile i with M(nq, col0[j]) }
 *   flag(i,j) = 1 (PARTIAL) iff exists valid row nq of q tile i and c in [col0[j], col0[j]+wpad)
 *               with c - col0[j] >= width[j] or not M(nq, c);  else 0 (FULL)
 * M(nq, c) = A[frame(nq)][frame(c)].  Every column of the tile is walked (no use is made of the
 * fact that they share a frame).  indices == NULL: count only.  Returns nnz or -1. */
int64_t lvsa_oracle_tile_index_fa(int T, int P, int n_text, int Bq, int Bk, int pad, const uint8_t *A,
                                  int32_t *indptr, int32_t *indices, uint8_t *flags, int64_t cap)
{
    const int64_t N = (int64_t)T * P + n_text;
    const int Tf = T + (n_text > 0 ? 1 : 0);
    const int64_t nq = (N + Bq - 1) / Bq;
    const int64_t nk = lvsa_oracle_kv_tiles_frame_aligned(T, P, n_text, Bk, NULL, NULL, 0);
    int32_t *col0 = (int32_t *)malloc(sizeof(int32_t) * (size_t)(nk + 1));
    int32_t *width = (int32_t *)malloc(sizeof(int32_t) * (size_t)(nk + 1));
    lvsa_oracle_kv_tiles_frame_aligned(T, P, n_text, Bk, col0, width, nk);
    uint8_t *fq = (uint8_t *)malloc((size_t)Tf);
    int *qf = (int *)malloc(sizeof(int) * (size_t)Tf);
    int64_t nnz = 0;
    for (int64_t i = 0; i < nq; ++i) {
        if (indptr) indptr[i] = (int32_t)nnz;
        /* the frames present among the valid rows of q tile i, as a list (found by walking the rows) */
        memset(fq, 0, (size_t)Tf);
        for (int64_t r = i * Bq; r < (i + 1) * Bq && r < N; ++r) fq[frame_of(r, T, P)] = 1;
        int nqf = 0;
        for (int tq = 0; tq < Tf; ++tq) if (fq[tq]) qf[nqf++] = tq;
        for (int64_t j = 0; j < nk; ++j) {
            const int64_t wpad = ((width[j] + pad - 1) / pad) * (int64_t)pad;
            int any_allowed = 0, any_disallowed = 0;
            for (int64_t c = col0[j]; c < col0[j] + wpad; ++c) {
                if (c - col0[j] >= width[j]) { any_disallowed = 1; continue; }   /* padding column */
                const int64_t fk = frame_of(c, T, P);
                for (int x = 0; x < nqf; ++x) {
                    if (A[(size_t)qf[x] * Tf + fk]) any_allowed = 1; else any_disallowed = 1;
                }
            }
            if (!any_allowed) continue;
            if (indices) {
                if (nnz >= cap) { free(col0); free(width); free(fq); free(qf); return -1; }
                indices[nnz] = (int32_t)j;
                flags[nnz] = (uint8_t)any_disallowed;
            }
            ++nnz;
        }
    }
    if (indptr) indptr[nq] = (int32_t)nnz;
    free(col0); free(width); free(fq); free(qf);
    return nnz;
}

/* ---- input decoding (not method arithmetic): element e of a tensor stored as fp32 or as
 * raw bf16 bit patterns, widened exactly to double ----------------------------------------- */
static inline double ld_elem(const void *base, int is_bf16, int64_t e)
{
    if (is_bf16) {
        uint32_t u = (uint32_t)((const uint16_t *)base)[e] << 16;
        float f; memcpy(&f, &u, 4); return (double)f;
    }
    return (double)((const float *)base)[e];
}

/* ---- O8: Eq. 2 for a list of query rows, all heads ------------------------- */
/* q,k,v: [N, H, d] (token-major, head, channel), fp32 or raw bf16.  rows: token ids.
 * out: [nrows, H, d] fp64, lse: [nrows, H] fp64 (natural log, reading R15).
 * The key set is taken from the token predicate M directly (not from the tile list).
 * scale <= 0 means 1/sqrt(d) (Eq. 1). */
void lvsa_oracle_attn_rows(const void *q, const void *k, const void *v, int is_bf16,
                           int T, int P, int n_text, int H, int d, const uint8_t *A,
                           const int64_t *rows, int64_t nrows, double scale,
                           double *out, double *lse, int nthreads)
{
    /* A is Tf x Tf, Tf = T + (n_text > 0); q,k,v hold N = T*P + n_text tokens */
    const int64_t N = (int64_t)T * P + n_text;
    const int Tf = T + (n_text > 0 ? 1 : 0);
    if (scale <= 0.0) scale = 1.0 / sqrt((double)d);
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
#pragma omp parallel
    {
        double *sc = (double *)malloc(sizeof(double) * (size_t)N);
        double *qd = (double *)malloc(sizeof(double) * (size_t)d);
        double *acc = (double *)malloc(sizeof(double) * (size_t)d);
#pragma omp for schedule(dynamic, 1) collapse(2)
        for (int64_t ri = 0; ri < nrows; ++ri) {
            for (int h = 0; h < H; ++h) {
                const int64_t nqi = rows[ri];
                const uint8_t *Arow = A + (size_t)frame_of(nqi, T, P) * Tf;
                for (int c = 0; c < d; ++c) qd[c] = ld_elem(q, is_bf16, (nqi * H + h) * d + c);
                /* logits s_j = q.k_j / sqrt(d) over allowed keys, and their max */
                double mx = -INFINITY;
                for (int64_t n = 0; n < N; ++n) {
                    if (!Arow[frame_of(n, T, P)]) continue;
                    const int64_t e = (n * H + h) * d;
                    double dot = 0.0;
#pragma omp simd reduction(+ : dot)
                    for (int c = 0; c < d; ++c) dot += qd[c] * ld_elem(k, is_bf16, e + c);
                    sc[n] = dot * scale;
                    if (sc[n] > mx) mx = sc[n];
                }
                /* p_j = exp(s_j - mx); L = sum p_j; out = sum p_j v_j / L */
                double L = 0.0;
                for (int c = 0; c < d; ++c) acc[c] = 0.0;
                for (int64_t n = 0; n < N; ++n) {
                    if (!Arow[frame_of(n, T, P)]) continue;
                    const double p = exp(sc[n] - mx);
                    const int64_t e = (n * H + h) * d;
                    L += p;
#pragma omp simd
                    for (int c = 0; c < d; ++c) acc[c] += p * ld_elem(v, is_bf16, e + c);
                }
                for (int c = 0; c < d; ++c) out[(ri * H + h) * d + c] = acc[c] / L;
                lse[ri * H + h] = mx + log(L);
            }
        }
        free(sc); free(qd); free(acc);
    }
}

/* ---- O9: the key set of a row, recovered through CSR + flags + element mask -------------- */
/* Returns 1 iff { keys contributed through the tile list } == { n : M(nq, n) } for every row
 * in rows.  FULL tiles contribute every column of the tile without consulting M (that is what
 * a kernel does); PARTIAL tiles contribute columns c < N with M(nq, c). */
int lvsa_oracle_csr_keyset_equal(int T, int P, int n_text, int Bq, int Bk, const uint8_t *A,
                                 const int32_t *indptr, const int32_t *indices,
                                 const uint8_t *flags, const int64_t *rows, int64_t nrows)
{
    const int64_t N = (int64_t)T * P + n_text;
    const int Tf = T + (n_text > 0 ? 1 : 0);
    uint8_t *via = (uint8_t *)malloc((size_t)N + (size_t)Bk);
    int ok = 1;
    for (int64_t ri = 0; ri < nrows && ok; ++ri) {
        const int64_t nqi = rows[ri];
        const uint8_t *Arow = A + (size_t)frame_of(nqi, T, P) * Tf;
        memset(via, 0, (size_t)N + (size_t)Bk);
        const int64_t i = nqi / Bq;
        for (int32_t e = indptr[i]; e < indptr[i + 1]; ++e) {
            const int64_t j = indices[e];
            for (int64_t c = j * Bk; c < (j + 1) * Bk; ++c) {
                if (flags[e]) { if (c < N && Arow[frame_of(c, T, P)]) via[c] += 1; }
                else          { via[c] += 1; }
            }
        }
        for (int64_t n = 0; n < N + Bk; ++n) {
            const int want = (n < N) ? Arow[frame_of(n, T, P)] : 0;
            if (via[n] != want) { ok = 0; break; }
        }
    }
    free(via);
    return ok;
}

/* O9 for an explicit kv tiling (col0, width per tile) and column granularity pad: FULL tiles
 * contribute every one of their wpad columns without consulting M, PARTIAL tiles the columns inside
 * `width` with M.  Returns 1 iff every key of every row in rows is contributed exactly once and
 * nothing else is (which also catches overlapping or missing tiles). */
int lvsa_oracle_csr_keyset_equal_tiles(int T, int P, int n_text, int Bq, int pad, const uint8_t *A,
                                       const int32_t *col0, const int32_t *width,
                                       const int32_t *indptr, const int32_t *indices,
                                       const uint8_t *flags, const int64_t *rows, int64_t nrows)
{
    const int64_t N = (int64_t)T * P + n_text;
    const int Tf = T + (n_text > 0 ? 1 : 0);
    const int64_t slack = 4096;
    uint8_t *via = (uint8_t *)malloc((size_t)(N + slack));
    int ok = 1;
    for (int64_t ri = 0; ri < nrows && ok; ++ri) {
        const int64_t nqi = rows[ri];
        const uint8_t *Arow = A + (size_t)frame_of(nqi, T, P) * Tf;
        memset(via, 0, (size_t)(N + slack));
        const int64_t i = nqi / Bq;
        for (int32_t e = indptr[i]; e < indptr[i + 1]; ++e) {
            const int64_t j = indices[e];
            const int64_t wpad = ((width[j] + pad - 1) / pad) * (int64_t)pad;
            if (wpad > slack) { ok = 0; break; }
            for (int64_t c = col0[j]; c < col0[j] + wpad; ++c) {
                if (flags[e]) { if (c - col0[j] < width[j] && c < N && Arow[frame_of(c, T, P)]) via[c] += 1; }
                else          { via[c] += 1; }
            }
        }
        for (int64_t n = 0; n < N + slack && ok; ++n) {
            const int want = (n < N) ? Arow[frame_of(n, T, P)] : 0;
            if (via[n] != want) ok = 0;
        }
    }
    free(via);
    return ok;
}

/* ---- report-only timing of the metadata rebuild ("1.4 us per call",
 * "< 200 us per rebuild") ------------------------------------------------------------------ */
/* Runs reps full pattern rebuilds for steps 0..S-1; returns seconds per rebuild and the
 * Alg. 1 loop statistics over all (step, frame) calls. */
double lvsa_oracle_time_rebuild(int T, int W, int a, int S, int reps,
                                int32_t *max_iters, double *mean_iters)
{
    uint8_t *A = (uint8_t *)malloc((size_t)T * T), *inG = (uint8_t *)malloc((size_t)T);
    int32_t *lo = (int32_t *)malloc(sizeof(int32_t) * T), *hi = (int32_t *)malloc(sizeof(int32_t) * T);
    int32_t *it = (int32_t *)malloc(sizeof(int32_t) * T), meta[3];
    int64_t tot = 0, calls = 0; int32_t mxi = 0;
    struct timespec t0, t1;
    clock_gettime(CLOCK_MONOTONIC, &t0);
    for (int r = 0; r < reps; ++r)
        for (int s = 0; s < S; ++s) {
            lvsa_oracle_pattern(T, W, a, s, 0, A, lo, hi, inG, it, meta);
            if (r == 0) for (int t = 0; t < T; ++t) { tot += it[t]; ++calls; if (it[t] > mxi) mxi = it[t]; }
        }
    clock_gettime(CLOCK_MONOTONIC, &t1);
    free(A); free(inG); free(lo); free(hi); free(it);
    *max_iters = mxi; *mean_iters = calls ? (double)tot / (double)calls : 0.0;
    return ((t1.tv_sec - t0.tv_sec) + 1e-9 * (t1.tv_nsec - t0.tv_nsec)) / ((double)reps * S);
}

int lvsa_oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
