// GPU index builder: steps a1-a5 of the hot path.
//   lvsa_frames_kernel : T_per, G^s (Eq. 3), adaptive window,
//                        Algorithm 1, A(t) bitsets (Def. 2)
//   lvsa_tiles_kernel  : frame -> token -> tile mapping per pair of adjacent q tiles, count then
//                        fill: the CSR (indices + FULL/PARTIAL flags per q tile) and the attention
//                        kernel's work items (union list of the pair, which shares K/V loads)
//   lvsa_scan_kernel   : exclusive scans of the per-q-tile and per-item counts (one launch)
// Integer arithmetic only.  Written from the paper; shares nothing with oracle/.
#include <limits.h>

#include "lvsa_internal.h"

namespace {

__device__ __forceinline__ bool bit_test(const uint32_t *bits, int x) {
    return (bits[x >> 5] >> (x & 31)) & 1u;
}

// One block.  g_bits lives in shared memory; every thread then owns frames t, t+blockDim, ...
__global__ void lvsa_frames_kernel(int T, int W, int a, int s, int tie_hi, int k0, int has_text, int words,
                                   int32_t *__restrict__ w_lo, int32_t *__restrict__ w_hi,
                                   uint32_t *__restrict__ a_bits, int32_t *__restrict__ meta) {
    extern __shared__ uint32_t g_bits[];
    __shared__ int n_global_s;
    const int tid = threadIdx.x;
    for (int w = tid; w < words; w += blockDim.x) g_bits[w] = 0u;
    __syncthreads();
    const bool all_tiles = (a == LVSA_ANCHORS_ALL_TILES);
    int T_per = 0, phase = 0;
    if (!all_tiles && a > 0) {
        T_per = (T + a - 1) / a;                  // ceil(T / (C-(2W+1)))
        const int m = (T + T_per - 1) / T_per;    // ceil(T / T_per) anchors, Eq. 3
        phase = s % T_per;
        for (int i = tid; i < m; i += blockDim.x) {
            const int f = (phase + i * T_per) % T;
            atomicOr(&g_bits[f >> 5], 1u << (f & 31));
        }
    }
    // dedicated initial anchors: frames 0..k0-1 are global at every step (R22)
    if (!all_tiles)
        for (int f = tid; f < min(k0, T); f += blockDim.x) atomicOr(&g_bits[f >> 5], 1u << (f & 31));
    __syncthreads();
    if (tid == 0) {
        int c = 0;
        for (int w = 0; w < words; ++w) c += __popc(g_bits[w]);
        n_global_s = c;
        meta[4] = T_per; meta[5] = phase; meta[6] = c;
    }
    __syncthreads();
    const int n_global = n_global_s;
    for (int t = tid; t < T; t += blockDim.x) {
        int l, h;
        if (all_tiles) {
            l = 0; h = T - 1;                     // Def. 1: A(t) = all frames
        } else {
            // adaptive window
            l = max(0, min(t - W, T - 1 - 2 * W));
            h = min(T - 1, max(t + W, 2 * W));
            // Algorithm 1
            const int target = min(2 * W + 1, T - n_global);
            int nonglobal = 0;
            for (int x = l; x <= h; ++x) nonglobal += !bit_test(g_bits, x);
            while (nonglobal < target && (l > 0 || h < T - 1)) {
                const int room_lo = l, room_hi = T - 1 - h;
                int nw;
                if (room_lo > room_hi || (room_lo == room_hi && !tie_hi)) { l -= 1; nw = l; }
                else                                                      { h += 1; nw = h; }
                nonglobal += !bit_test(g_bits, nw);
            }
        }
        w_lo[t] = l; w_hi[t] = h;
        for (int w = 0; w < words; ++w) {
            // bits of [l, h] that fall into word w
            const int b0 = max(l, 32 * w), b1 = min(h, 32 * w + 31);
            uint32_t rm = 0u;
            if (b0 <= b1) {
                const int n = b1 - b0 + 1;
                rm = (n == 32 ? 0xffffffffu : ((1u << n) - 1u)) << (b0 - 32 * w);
            }
            uint32_t bits = g_bits[w] | rm;
            // text pseudo-frame T (R23): every video query attends to the text tokens
            if (has_text && (T >> 5) == w) bits |= 1u << (T & 31);
            a_bits[(size_t)t * words + w] = bits;
        }
    }
    // ... and the text tokens attend to every frame, themselves included: row T = bits 0..T
    if (has_text)
        for (int w = tid; w < words; w += blockDim.x) {
            const int n = min(32, T + 1 - 32 * w);
            a_bits[(size_t)T * words + w] = n <= 0 ? 0u : (n == 32 ? 0xffffffffu : ((1u << n) - 1u));
        }
}

// One block per work item = group of two adjacent q tiles (the 256 query rows that share K/V
// loads in the attention kernel).  Threads stride over kv tiles in ascending chunks, so the fill
// pass writes in order.  For every kv tile the thread decides kept / PARTIAL for each of the two
// q tiles (frame -> token -> tile mapping, reading R14); the item's list is the union, each
// entry tagged with the per-q-tile state (skip / full / partial).
//   FILL = false: counts[i] per q tile, icounts[g] per item.
//   FILL = true : indices/flags at indptr[i] (the CSR), item_tiles at item_ptr[g].
//   ALIGNED = true: frame-aligned kv tiles (reading R25): tile j lies inside one frame, is PARTIAL
//   iff some row of the q tile does not attend to that frame or its width is not a multiple of
//   LVSA_KV_PAD; Tv = video frames (Tf minus the text pseudo-frame).
template <bool FILL, bool ALIGNED>
__global__ void lvsa_tiles_kernel(long long N, int P, int Tv, int Tf, int Bq, int Bk, int nq, int nk, int words,
                                  const uint32_t *__restrict__ a_bits,
                                  int32_t *__restrict__ indptr, int32_t *__restrict__ item_ptr,
                                  int32_t *__restrict__ counts, int32_t *__restrict__ icounts,
                                  int32_t *__restrict__ indices, uint8_t *__restrict__ flags,
                                  int32_t *__restrict__ item_tiles, int32_t *__restrict__ item_col0,
                                  int32_t *__restrict__ meta, unsigned long long *__restrict__ kept_cols) {
    __shared__ int warp_tot[3][32];
    const int g = blockIdx.x, tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int nwarps = blockDim.x >> 5;
    if (FILL && meta[7]) {
        // Allocation bound exceeded: nothing is filled.  The host reports it at lvsa_index_info /
        // copy_host; a kernel that is launched on this index anyway must not walk the unfilled lists, so
        // the list ends are poisoned (negative totals) and the attention kernels trap on them.
        if (g == 0 && tid == 0) { indptr[nq] = -1; item_ptr[gridDim.x] = -1; }
        return;
    }
    // rows and frames of the two q tiles; frame of a token: n / P, tokens past the video (text,
    // R23) belong to the last frame row Tf-1
    const int i0 = 2 * g, i1 = 2 * g + 1;
    const bool has1 = i1 < nq;
    int fa[2], fb[2];
#pragma unroll
    for (int w = 0; w < 2; ++w) {
        const long long r0 = (long long)(i0 + w) * Bq;
        const long long r1 = min(r0 + Bq, N) - 1;
        fa[w] = min((int)(r0 / P), Tf - 1);
        fb[w] = (w == 0 || has1) ? min((int)(r1 / P), Tf - 1) : fa[w] - 1;   // empty range: no q tile 1
    }
    int run[3] = {0, 0, 0}, n_part = 0;
    long long n_cols = 0;   // computed kv columns over the kept (q tile, kv tile) pairs of this thread
    int base[3] = {0, 0, 0};
    if (FILL) { base[0] = indptr[i0]; base[1] = has1 ? indptr[i1] : 0; base[2] = item_ptr[g]; }
    for (int j0 = 0; j0 < nk; j0 += blockDim.x) {
        const int j = j0 + tid;
        bool kept[2] = {false, false}, part[2] = {false, false};
        long long c0 = 0;
        int wpad = Bk;      // columns a kernel computes for this tile
        if (j < nk) {
            int g0, g1;
            bool tail;
            if (ALIGNED) {
                const lvsa_kv_tile kt = lvsa_kv_tile_of(j, 1, Bk, P, Tv, N);
                c0 = kt.c0; g0 = g1 = kt.g;
                wpad = (kt.width + LVSA_KV_PAD - 1) / LVSA_KV_PAD * LVSA_KV_PAD;
                tail = wpad != kt.width;          // padding columns are never allowed
            } else {
                c0 = (long long)j * Bk;
                const long long c1 = min(c0 + Bk, N) - 1;
                g0 = min((int)(c0 / P), Tf - 1); g1 = min((int)(c1 / P), Tf - 1);
                tail = (c0 + Bk > N);             // columns >= N are never allowed
            }
#pragma unroll
            for (int w = 0; w < 2; ++w) {
                part[w] = tail;
                for (int tq = fa[w]; tq <= fb[w]; ++tq) {
                    const uint32_t *row = a_bits + (size_t)tq * words;
                    for (int tk = g0; tk <= g1; ++tk) {
                        const bool b = bit_test(row, tk);
                        kept[w] |= b; part[w] |= !b;
                    }
                }
            }
        }
        const unsigned bal0 = __ballot_sync(0xffffffffu, kept[0]);
        const unsigned bal1 = __ballot_sync(0xffffffffu, kept[1]);
        const unsigned balu = bal0 | bal1;
        if (lane == 0) { warp_tot[0][wid] = __popc(bal0); warp_tot[1][wid] = __popc(bal1); warp_tot[2][wid] = __popc(balu); }
        __syncthreads();
        int woff[3] = {0, 0, 0}, tot[3] = {0, 0, 0};
        for (int w = 0; w < nwarps; ++w)
#pragma unroll
            for (int x = 0; x < 3; ++x) { const int c = warp_tot[x][w]; if (w < wid) woff[x] += c; tot[x] += c; }
        if (FILL) {
            const unsigned below = (1u << lane) - 1u;
            if (kept[0]) {
                const int pos = base[0] + run[0] + woff[0] + __popc(bal0 & below);
                indices[pos] = j; flags[pos] = part[0] ? LVSA_TILE_PARTIAL : LVSA_TILE_FULL; n_part += part[0];
                n_cols += wpad;
            }
            if (kept[1]) {
                const int pos = base[1] + run[1] + woff[1] + __popc(bal1 & below);
                indices[pos] = j; flags[pos] = part[1] ? LVSA_TILE_PARTIAL : LVSA_TILE_FULL; n_part += part[1];
                n_cols += wpad;
            }
            if (kept[0] || kept[1]) {
                const int st0 = kept[0] ? (part[0] ? LVSA_ST_PARTIAL : LVSA_ST_FULL) : LVSA_ST_SKIP;
                const int st1 = kept[1] ? (part[1] ? LVSA_ST_PARTIAL : LVSA_ST_FULL) : LVSA_ST_SKIP;
                const int pos = base[2] + run[2] + woff[2] + __popc(balu & below);
                // the width field has 2 bits: 32-column units (tiles wider than 128 do not exist)
                const unsigned wbits = (unsigned)(min(wpad, 128) / 32 - 1);
                item_tiles[pos] = (int32_t)((unsigned)j | ((unsigned)st0 << LVSA_ITEM_J_BITS) |
                                            ((unsigned)st1 << (LVSA_ITEM_J_BITS + 2)) | (wbits << LVSA_ITEM_W_SHIFT));
                item_col0[pos] = (int32_t)c0;
            }
        }
#pragma unroll
        for (int x = 0; x < 3; ++x) run[x] += tot[x];
        __syncthreads();
    }
    if (!FILL && tid == 0) { counts[i0] = run[0]; if (has1) counts[i1] = run[1]; icounts[g] = run[2]; }
    if (FILL) {
        // one global atomic per block and counter (all blocks add to the same two addresses)
        __shared__ int part_s;
        __shared__ unsigned long long cols_s;
        if (tid == 0) { part_s = 0; cols_s = 0ull; }
        __syncthreads();
        n_part = __reduce_add_sync(0xffffffffu, n_part);
        for (int o = 16; o > 0; o >>= 1) n_cols += __shfl_xor_sync(0xffffffffu, n_cols, o);
        if (lane == 0) { if (n_part) atomicAdd(&part_s, n_part); if (n_cols) atomicAdd(&cols_s, (unsigned long long)n_cols); }
        __syncthreads();
        if (tid == 0) { if (part_s) atomicAdd(&meta[1], part_s); if (cols_s) atomicAdd(kept_cols, cols_s); }
    }
}

// Work lists of the 4-CTA-cluster kernel (LVSA_KERNEL_TCGEN05_QUAD): one block per QUAD of adjacent
// q tiles (two work items); the list is the union of the kv lists of the four q tiles, each entry
// tagged with four 2-bit states (token-0 tiling only).  Same ordered compaction as above.
//   FILL = false: qcounts[u];  FILL = true: quad_tiles at quad_ptr[u].
template <bool FILL>
__global__ void lvsa_quads_kernel(long long N, int P, int Tf, int Bq, int Bk, int nq, int nk, int words,
                                  const uint32_t *__restrict__ a_bits, int32_t *__restrict__ quad_ptr,
                                  int32_t *__restrict__ qcounts, int32_t *__restrict__ quad_tiles,
                                  const int32_t *__restrict__ meta, int32_t *__restrict__ indptr_end,
                                  int32_t *__restrict__ item_ptr_end) {
    __shared__ int warp_tot[32];
    const int u = blockIdx.x, tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int nwarps = blockDim.x >> 5;
    if (FILL && meta[7]) {   // as in lvsa_tiles_kernel: poison every list end (the quad scan may be the one that overflowed)
        if (u == 0 && tid == 0) { quad_ptr[gridDim.x] = -1; *indptr_end = -1; *item_ptr_end = -1; }
        return;
    }
    int fa[4], fb[4];
#pragma unroll
    for (int w = 0; w < 4; ++w) {
        const int i = 4 * u + w;
        const long long r0 = (long long)i * Bq;
        const long long r1 = min(r0 + Bq, N) - 1;
        fa[w] = min((int)(min(r0, N - 1) / P), Tf - 1);
        fb[w] = i < nq ? min((int)(r1 / P), Tf - 1) : fa[w] - 1;   // empty range: no such q tile
    }
    int run = 0;
    const int base = FILL ? quad_ptr[u] : 0;
    for (int j0 = 0; j0 < nk; j0 += blockDim.x) {
        const int j = j0 + tid;
        unsigned st = 0u;   // four 2-bit states
        if (j < nk) {
            const long long c0 = (long long)j * Bk;
            const long long c1 = min(c0 + Bk, N) - 1;
            const int g0 = min((int)(c0 / P), Tf - 1), g1 = min((int)(c1 / P), Tf - 1);
            const bool tail = (c0 + Bk > N);
#pragma unroll
            for (int w = 0; w < 4; ++w) {
                bool kept = false, part = tail;
                for (int tq = fa[w]; tq <= fb[w]; ++tq) {
                    const uint32_t *row = a_bits + (size_t)tq * words;
                    for (int tk = g0; tk <= g1; ++tk) {
                        const bool b = bit_test(row, tk);
                        kept |= b; part |= !b;
                    }
                }
                st |= (unsigned)(kept ? (part ? LVSA_ST_PARTIAL : LVSA_ST_FULL) : LVSA_ST_SKIP) << (2 * w);
            }
        }
        const unsigned bal = __ballot_sync(0xffffffffu, st != 0u);
        if (lane == 0) warp_tot[wid] = __popc(bal);
        __syncthreads();
        int woff = 0, tot = 0;
        for (int w = 0; w < nwarps; ++w) { const int c = warp_tot[w]; if (w < wid) woff += c; tot += c; }
        if (FILL && st != 0u)
            quad_tiles[base + run + woff + __popc(bal & ((1u << lane) - 1u))] = (int32_t)((unsigned)j | (st << LVSA_QUAD_J_BITS));
        run += tot;
        __syncthreads();
    }
    if (!FILL && tid == 0) qcounts[u] = run;
}

// Single-block exclusive scan: out[0..n] from counts[0..n-1]; total also to *total_out.
// If the total exceeds `cap` (the host's allocation bound) meta[7] is raised, the fill passes write
// nothing and poison the list ends (the attention kernels trap on a poisoned index); the host reports
// it at the next lvsa_index_info / copy_host and lvsa_attn_fwd then refuses the index.
__global__ void lvsa_scan_kernel(const int32_t *__restrict__ counts_a, int n_a, int32_t *__restrict__ out_a,
                                 int32_t *__restrict__ total_a, long long cap_a,
                                 const int32_t *__restrict__ counts_b, int n_b, int32_t *__restrict__ out_b,
                                 int32_t *__restrict__ total_b, long long cap_b,
                                 int32_t *__restrict__ overflow) {
    // block 0 scans the per-q-tile counts (-> indptr), block 1 the per-item counts (-> item_ptr)
    const int32_t *counts = blockIdx.x == 0 ? counts_a : counts_b;
    const int n = blockIdx.x == 0 ? n_a : n_b;
    int32_t *out = blockIdx.x == 0 ? out_a : out_b;
    int32_t *total_out = blockIdx.x == 0 ? total_a : total_b;
    const long long cap = blockIdx.x == 0 ? cap_a : cap_b;
    __shared__ int warp_tot[32];
    __shared__ int carry_s;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5, nwarps = blockDim.x >> 5;
    if (tid == 0) carry_s = 0;
    __syncthreads();
    for (int i0 = 0; i0 < n; i0 += blockDim.x) {
        const int i = i0 + tid;
        const int v = (i < n) ? counts[i] : 0;
        int incl = v;
        for (int o = 1; o < 32; o <<= 1) {
            const int y = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += y;
        }
        if (lane == 31) warp_tot[wid] = incl;
        __syncthreads();
        int woff = 0, tot = 0;
        for (int w = 0; w < nwarps; ++w) { const int c = warp_tot[w]; if (w < wid) woff += c; tot += c; }
        const int carry = carry_s;
        if (i < n) out[i] = carry + woff + incl - v;
        __syncthreads();
        if (tid == 0) carry_s = carry + tot;
        __syncthreads();
    }
    if (tid == 0) { out[n] = carry_s; *total_out = carry_s; if (carry_s > cap) *overflow = 1; }
}

}  // namespace


// Host side.  The whole build is enqueued on `stream` with no host synchronisation: buffers come
// from one stream-ordered arena sized by an upper bound on the number of kept tiles, and the
// counts the host wants to report (nnz, ...) are fetched lazily by lvsa_index_fetch_meta.
//
// Bound (allocation only; the pattern itself is computed on the device): a q tile touches at
// most fq = floor((Bq-1)/P) + 2 frames, each attends to |A| <= min(T, m + 2W + 1) frames
// (PAPER.md:66 closed form, m = |G| <= ceil(T / T_per)), and a frame overlaps at most
// kf = floor((P-1)/Bk) + 2 kv tiles.
static size_t align_up(size_t x) { return (x + 255) & ~(size_t)255; }

lvsa_status_t lvsa_index_build_device(lvsa_index *ix, cudaStream_t stream) {
    const lvsa_params_t &p = ix->p;
    const int T = p.T, words = ix->words;
    const int W = p.window > T ? T : p.window;  // W >= T already spans [0, T-1]; avoids 2W overflow

    long long m_bound = T;
    if (p.anchors >= 0 && p.anchors < T) {
        if (p.anchors == 0) m_bound = 0;
        else { const long long T_per = (T + p.anchors - 1) / p.anchors; m_bound = (T + T_per - 1) / T_per; }
    }
    m_bound += p.initial_anchors;
    long long a_bound = m_bound + 2ll * W + 1; if (a_bound > T) a_bound = T;
    const long long fq = (p.tile_q - 1) / p.P + 2, kf = (p.P - 1) / p.tile_k + 2;
    long long per_q = fq * a_bound * kf;
    if (p.n_text > 0) per_q += (p.n_text - 1) / p.tile_k + 2;      // the text columns every row keeps
    if (per_q > ix->nk) per_q = ix->nk;
    ix->n_items = (ix->nq + ix->group - 1) / ix->group;
    long long per_item = per_q * ix->group; if (per_item > ix->nk) per_item = ix->nk;
    // q tiles that hold text rows keep every kv tile
    const long long text_q = p.n_text > 0 ? (p.n_text - 1) / p.tile_q + 2 : 0;
    ix->cap_nnz = per_q * ix->nq + text_q * ix->nk;
    ix->cap_item_tiles = per_item * ix->n_items + text_q * ix->nk;
#ifdef LVSA_TEST_CAP_SHRINK   // test-only build (tests/test_gpu_overflow.py): an allocation bound that is too small
    ix->cap_nnz /= LVSA_TEST_CAP_SHRINK; ix->cap_item_tiles /= LVSA_TEST_CAP_SHRINK;
#endif
    if (ix->cap_nnz >= (1ll << 31) || ix->cap_item_tiles >= (1ll << 31)) {
        lvsa_set_error("index too large for int32 offsets");
        return LVSA_EUNSUPPORTED;
    }

    size_t off = 0;
    auto take = [&](size_t bytes) { const size_t o = off; off += align_up(bytes); return o; };
    const size_t o_wlo = take(sizeof(int32_t) * T), o_whi = take(sizeof(int32_t) * T);
    const size_t o_abits = take(sizeof(uint32_t) * (size_t)ix->Tf * words), o_meta = take(sizeof(int32_t) * 8);
    const size_t o_indptr = take(sizeof(int32_t) * ((size_t)ix->nq + 1));
    const size_t o_counts = take(sizeof(int32_t) * ((size_t)ix->nq + 1));
    const size_t o_icounts = take(sizeof(int32_t) * ((size_t)ix->n_items + 1));
    const size_t o_indices = take(sizeof(int32_t) * (size_t)(ix->cap_nnz + 1));
    const size_t o_flags = take((size_t)(ix->cap_nnz + 1));
    const size_t o_item_ptr = take(sizeof(int32_t) * ((size_t)ix->n_items + 1));
    const size_t o_item_tiles = take(sizeof(int32_t) * (size_t)(ix->cap_item_tiles + 1));
    const size_t o_item_col0 = take(sizeof(int32_t) * (size_t)(ix->cap_item_tiles + 1));
    const size_t o_kept_cols = take(sizeof(unsigned long long));
    // work lists of the 4-CTA-cluster kernel, built only when that kernel was asked for
    const bool quads = p.kernel == LVSA_KERNEL_TCGEN05_QUAD || p.kernel == LVSA_KERNEL_TCGEN05_HYBRID;
    ix->n_quads = quads ? (ix->nq + 3) / 4 : 0;
    long long per_quad = per_q * 4; if (per_quad > ix->nk) per_quad = ix->nk;
    ix->cap_quad_tiles = quads ? per_quad * ix->n_quads + text_q * ix->nk : 0;
    if (ix->cap_quad_tiles >= (1ll << 31)) { lvsa_set_error("index too large for int32 offsets"); return LVSA_EUNSUPPORTED; }
    const size_t o_qcounts = take(sizeof(int32_t) * ((size_t)ix->n_quads + 1));
    const size_t o_quad_ptr = take(sizeof(int32_t) * ((size_t)ix->n_quads + 1));
    const size_t o_quad_tiles = take(sizeof(int32_t) * (size_t)(ix->cap_quad_tiles + 1));
    const size_t o_quad_meta = take(sizeof(int32_t) * 2);

    static bool pool_ready[LVSA_MAX_DEVICES] = {};
    if (!pool_ready[ix->device]) {
        cudaMemPool_t pool;
        LVSA_CUDA_TRY(cudaDeviceGetDefaultMemPool(&pool, ix->device));
        unsigned long long keep = ~0ull;   // keep freed arenas cached: rebuilds then allocate in microseconds
        LVSA_CUDA_TRY(cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep));
        pool_ready[ix->device] = true;
    }
    LVSA_CUDA_TRY(cudaMallocAsync(&ix->arena, off, stream));
    ix->arena_bytes = off;
    ix->build_stream = stream;
    ix->last_stream = stream;
    uint8_t *a = static_cast<uint8_t *>(ix->arena);
    ix->d_wlo = (int32_t *)(a + o_wlo); ix->d_whi = (int32_t *)(a + o_whi);
    ix->d_abits = (uint32_t *)(a + o_abits); ix->d_meta = (int32_t *)(a + o_meta);
    ix->d_indptr = (int32_t *)(a + o_indptr);
    int32_t *d_counts = (int32_t *)(a + o_counts), *d_icounts = (int32_t *)(a + o_icounts);
    ix->d_indices = (int32_t *)(a + o_indices); ix->d_flags = a + o_flags;
    ix->d_item_ptr = (int32_t *)(a + o_item_ptr); ix->d_item_tiles = (int32_t *)(a + o_item_tiles);
    ix->d_item_col0 = (int32_t *)(a + o_item_col0);
    ix->d_kept_cols = (unsigned long long *)(a + o_kept_cols);
    int32_t *d_qcounts = (int32_t *)(a + o_qcounts), *d_quad_meta = (int32_t *)(a + o_quad_meta);
    ix->d_quad_ptr = (int32_t *)(a + o_quad_ptr); ix->d_quad_tiles = (int32_t *)(a + o_quad_tiles);

    LVSA_CUDA_TRY(cudaMemsetAsync(ix->d_meta, 0, sizeof(int32_t) * 8, stream));
    LVSA_CUDA_TRY(cudaMemsetAsync(ix->d_kept_cols, 0, sizeof(unsigned long long), stream));
    lvsa_frames_kernel<<<1, 256, sizeof(uint32_t) * words, stream>>>(
        T, W, p.anchors, p.step, p.tie_break == LVSA_TIE_HI, p.initial_anchors, p.n_text > 0, words, ix->d_wlo, ix->d_whi,
        ix->d_abits, ix->d_meta);
    const int n_items = (int)ix->n_items;
    const bool aligned = p.kv_tiling == LVSA_KV_TILES_FRAME_ALIGNED;
    auto count_k = aligned ? lvsa_tiles_kernel<false, true> : lvsa_tiles_kernel<false, false>;
    auto fill_k = aligned ? lvsa_tiles_kernel<true, true> : lvsa_tiles_kernel<true, false>;
    count_k<<<n_items, 256, 0, stream>>>(
        (long long)ix->N, p.P, T, ix->Tf, p.tile_q, p.tile_k, ix->nq, ix->nk, words, ix->d_abits, nullptr, nullptr,
        d_counts, d_icounts, nullptr, nullptr, nullptr, nullptr, ix->d_meta, ix->d_kept_cols);
    lvsa_scan_kernel<<<2, 1024, 0, stream>>>(d_counts, ix->nq, ix->d_indptr, ix->d_meta + 0, (long long)ix->cap_nnz,
                                             d_icounts, n_items, ix->d_item_ptr, ix->d_meta + 2,
                                             (long long)ix->cap_item_tiles, ix->d_meta + 7);
    fill_k<<<n_items, 256, 0, stream>>>(
        (long long)ix->N, p.P, T, ix->Tf, p.tile_q, p.tile_k, ix->nq, ix->nk, words, ix->d_abits, ix->d_indptr,
        ix->d_item_ptr, nullptr, nullptr, ix->d_indices, ix->d_flags, ix->d_item_tiles, ix->d_item_col0, ix->d_meta,
        ix->d_kept_cols);
    if (quads) {
        const int nqd = (int)ix->n_quads;
        lvsa_quads_kernel<false><<<nqd, 256, 0, stream>>>((long long)ix->N, p.P, ix->Tf, p.tile_q, p.tile_k, ix->nq, ix->nk,
                                                          words, ix->d_abits, nullptr, d_qcounts, nullptr, ix->d_meta,
                                                          nullptr, nullptr);
        // block 0 scans the quad counts (total -> quad_meta[0]); block 1 has nothing to do
        lvsa_scan_kernel<<<2, 1024, 0, stream>>>(d_qcounts, nqd, ix->d_quad_ptr, d_quad_meta, (long long)ix->cap_quad_tiles,
                                                 d_qcounts, 0, d_qcounts + nqd, d_quad_meta + 1, 1ll << 40, ix->d_meta + 7);
        lvsa_quads_kernel<true><<<nqd, 256, 0, stream>>>((long long)ix->N, p.P, ix->Tf, p.tile_q, p.tile_k, ix->nq, ix->nk,
                                                         words, ix->d_abits, ix->d_quad_ptr, nullptr, ix->d_quad_tiles, ix->d_meta,
                                                         ix->d_indptr + ix->nq, ix->d_item_ptr + n_items);
    }
    LVSA_CUDA_TRY(cudaGetLastError());
    ix->meta_fetched = false;
    return LVSA_OK;
}

// Reads the device-side counters (nnz, PARTIAL count, item entries, T_per, phase, |G|) once;
// synchronises the build stream.  Called by lvsa_index_info / lvsa_index_copy_host.
lvsa_status_t lvsa_index_fetch_meta(const lvsa_index *ix) {
    if (ix->meta_fetched) return LVSA_OK;
    int32_t meta[8];
    unsigned long long kept_cols = 0;
    LVSA_CUDA_TRY(cudaMemcpyAsync(meta, ix->d_meta, sizeof(meta), cudaMemcpyDeviceToHost, ix->build_stream));
    LVSA_CUDA_TRY(cudaMemcpyAsync(&kept_cols, ix->d_kept_cols, sizeof(kept_cols), cudaMemcpyDeviceToHost, ix->build_stream));
    LVSA_CUDA_TRY(cudaStreamSynchronize(ix->build_stream));
    if (meta[7] != 0) {
        ix->overflowed = true;   // lvsa_attn_fwd refuses this index from now on
        lvsa_set_error("internal: kept-tile count exceeds the allocation bound");
        return LVSA_ECUDA;
    }
    ix->nnz = meta[0]; ix->n_partial = meta[1]; ix->n_item_tiles = meta[2];
    ix->T_per = meta[4]; ix->phase = meta[5]; ix->n_global = meta[6];
    ix->kept_cols = (int64_t)kept_cols;
    ix->meta_fetched = true;
    return LVSA_OK;
}
