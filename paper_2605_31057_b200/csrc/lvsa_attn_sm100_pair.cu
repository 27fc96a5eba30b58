// CTA-pair LVSA attention forward for sm_100a (d = 128, 128 x 128 tiles): one cluster of two CTAs
// per work item (pair of adjacent q tiles), tcgen05.mma.cta_group::2 with M = 256 across the pair.
//
// Computes Eq. 2 over the kept kv tiles listed by the block index, like the
// one-CTA-per-item kernel (lvsa_attn_sm100.cu); what changes is where the operands and accumulators live:
//   * CTA r of the pair owns q tile r of the item: its 128 rows of Q (shared memory), of S / P and
//     of O (its own TMEM).  Every MMA is one instruction for both CTAs, issued by the leader (CTA 0).
//   * B operands are split over the pair: CTA r loads kv rows [64 r, 64 r + 64) of K_j (the N
//     extent of S = Q K^T) and channels [64 r, 64 r + 64) of V_j (the N extent of O += P V), 16 KB
//     each instead of 32 KB; the tensor cores read both halves from both shared memories.
//   * with one q tile per CTA, TMEM holds THREE S/P buffers and O (512 columns).  Tile t uses buffer
//     t % 3; S(t+2) is issued right after PV(t-1), so it is computed while the softmax of tile t runs
//     and never waits for a P of the warpgroup that will consume it.  This removes the serial chain
//     softmax(t) -> PV(t) -> S(next tile of the same rows) -> softmax that bounds the one-CTA kernel
//     (DESIGN.md 7.2): measured tensor pipe 71 % busy instead of 61 %.
// Roles per CTA (12 warps): warps 0-3 / 4-7 softmax warpgroups 0 / 1, one thread per query row;
// warpgroup w takes the tiles with (running tile count) % 2 == w, so the exponentials of two
// consecutive tiles overlap.  Both accumulate into the same O and therefore share one reference
// maximum per row (shared memory); the short "row max, decide" phase is ordered by a token that
// passes between the warpgroups.  Warp 8 TMA producer, warp 9 MMA issuer (leader CTA only),
// warps 10-11 idle (setmaxnreg acts on whole warpgroups).
//
// Cross-CTA signalling: TMA completions of both CTAs are counted on the leader's FULL barriers
// (cta_group::2 loads); tcgen05.commit multicasts MMA completions to the barriers of both CTAs;
// the peer's softmax warps arrive remotely on the leader's P barriers.
#include <cuda.h>
#include <cuda_bf16.h>

#include <mutex>

#include "lvsa_internal.h"
#include "sm100_ptx.cuh"
#include "lvsa_softmax.cuh"

using namespace sm100;

namespace {

constexpr int D = 128, BT = 128, CH = 64;
constexpr int TILE_BYTES = BT * D * 2;          // 32 KB: one Q tile
constexpr int SPAN_BYTES = BT * 128;            // 16 KB: [128 rows][128 B] swizzle span
constexpr int STAGE_BYTES = 16384;              // half a K tile (64 rows x 256 B) or half a V tile (128 rows x 128 B)
constexpr int NTHREADS = 384;
constexpr float RESCALE_THRESHOLD = 8.0f;       // log2 units
#ifndef LVSA_PAIR_STAGES
#define LVSA_PAIR_STAGES 10
#endif

template <int NS>
struct SmemP {
    static constexpr int Q_OFF = 0;                            // 32 KB
    static constexpr int RING_OFF = TILE_BYTES;                // NS x 16 KB
    static constexpr int OUT_OFF = RING_OFF + NS * STAGE_BYTES;  // 32 KB: output staging, two [128 rows][128 B] spans
    static constexpr int BAR_OFF = OUT_OFF + TILE_BYTES;
    // barriers (8 B each).  "L": only the leader's copy is used (arrivals come from both CTAs).
    static constexpr int Q_FULL = 0 /*L*/, Q_EMPTY = 1, S_FULL = 2 /*3*/, PA_FULL = 5 /*3, L*/, PB_FULL = 8 /*3, L*/,
                         PV_DONE = 11 /*2*/, O_FULL = 13, O_FREE = 14 /*L*/, KV_FULL = 15 /*NS, L*/,
                         KV_EMPTY = 15 + NS /*NS*/, NBARS = 15 + 2 * NS;
    static constexpr int TMEM_SLOT_OFF = BAR_OFF + 8 * NBARS;
    static constexpr int XCH_OFF = TMEM_SLOT_OFF + 16;         // float m_ref[128], l[2][128]
    static constexpr int BYTES = XCH_OFF + 3 * 128 * 4;
};

__device__ __forceinline__ uint32_t range_mask32(int lo, int hi, int w) {
    const int a = max(lo, 32 * w), b = min(hi, 32 * w + 32);
    if (a >= b) return 0u;
    const int n = b - a;
    return (n == 32 ? 0xffffffffu : ((1u << n) - 1u)) << (a - 32 * w);
}

template <int REGS> __device__ __forceinline__ void reg_inc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(REGS)); }
template <int REGS> __device__ __forceinline__ void reg_dec() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(REGS)); }

template <int V> struct StaticInt { __device__ constexpr operator int() const { return V; } };

// 32-column chunks of the kv tile that are computed: 4 for a 128-column tile, fewer for a narrow
// frame-aligned tile (reading R25)
__device__ __forceinline__ int entry_chunks(int entry) { return (int)((uint32_t)entry >> LVSA_ITEM_W_SHIFT) + 1; }

// VARW = false: every kv tile is 128 columns from token j * 128 (LVSA_KV_TILES_TOKEN0); the list entry
// alone describes it and the widths are compile-time constants.  VARW = true: frame-aligned kv tiles
// (LVSA_KV_TILES_FRAME_ALIGNED, reading R25): the first token comes from item_col0[] and the width
// (32 .. 128 columns) from the entry, in the producer, the issuer and the softmax warps.
//
// MODE_QUAD: clusters of FOUR CTAs = two MMA pairs working on the two work items of a quad of adjacent
// q tiles (token-0 tiles).  Every K/V tile is loaded ONCE per cluster: CTA r of pair 0 issues the TMA
// load of "its" half with a multicast mask naming CTA r of both pairs, so the same bytes land at the
// same shared-memory offset of both, and each destination's completion is counted on the FULL barrier
// of its own pair's leader (cta_group::2 load, barrier address with the peer bit cleared).  The two
// pairs walk the quad's union list in lock step as far as the ring goes: a stage is refilled when the
// MMAs of BOTH pairs have read it (KV_EMPTY takes one commit from each issuer, multicast to all four
// CTAs).  Everything else (Q, S/P/O, softmax, epilogue) stays private to a pair.
enum { MODE_TOKEN0 = 0, MODE_VARW = 1, MODE_QUAD = 2 };
template <int NS, int MODE>
__global__ void __cluster_dims__(MODE == MODE_QUAD ? 4 : 2, 1, 1) __launch_bounds__(NTHREADS, 1)
lvsa_attn_sm100_pair_kernel(const __grid_constant__ CUtensorMap tmap_q,
                            const __grid_constant__ CUtensorMap tmap_k,   // box 64 rows
                            const __grid_constant__ CUtensorMap tmap_v,   // box 128 rows
                            const __grid_constant__ CUtensorMap tmap_o,   // out, box 128 rows x 64 channels
                            float *__restrict__ lse,
                            const int32_t *__restrict__ item_ptr, const int32_t *__restrict__ item_tiles,
                            const int32_t *__restrict__ item_col0,
                            const uint32_t *__restrict__ a_bits, int words, long long N, int P, int T,
                            int H, int h0, int hc, int n_items, long long work0, long long n_work, float scale_log2) {
    using SM = SmemP<NS>;
    constexpr bool VARW = MODE == MODE_VARW, QUAD = MODE == MODE_QUAD;
    constexpr int CL = QUAD ? 4 : 2;                   // CTAs per cluster
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    const uint32_t base = smem_u32(smem_raw);
    if ((base & 1023u) != 0u) __trap();   // SWIZZLE_128B tiles and UMMA descriptors need 1024 B
    // an index whose build overflowed its allocation bound has unfilled lists and a poisoned end (lvsa_index.cu)
    if (threadIdx.x == 0 && item_ptr[n_items] < 0) __trap();
    uint8_t *base_gen = smem_raw;
    const uint32_t sQ = base + SM::Q_OFF, sRing = base + SM::RING_OFF, sBar = base + SM::BAR_OFF;
    const uint32_t sOut = base + SM::OUT_OFF;
    auto bar = [&](int i) { return sBar + 8u * (uint32_t)i; };
    volatile uint32_t *tmem_slot_gen = reinterpret_cast<volatile uint32_t *>(base_gen + SM::TMEM_SLOT_OFF);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, wg = tid >> 7;
    const uint32_t crank = cluster_ctarank();
    const uint32_t rank = crank & 1u;                  // 0 = leader of my pair; also the q tile of the item I own
    const uint32_t pid = QUAD ? (crank >> 1) : 0u;     // my pair inside the cluster
    const uint32_t lead = crank & ~1u;                 // cluster rank of my pair's leader
    const uint16_t pair_mask = (uint16_t)(3u << (2u * pid));              // commit targets: my pair
    const uint16_t ring_mask = QUAD ? (uint16_t)0xF : pair_mask;          // ... or every CTA that shares the ring
    const long long pair = blockIdx.x / CL, n_pairs = gridDim.x / CL;     // cluster index / number of clusters
    // which list entry bits hold MY q tile's state, and the rows my pair owns in work unit `item`
    constexpr int J_MASK = QUAD ? LVSA_QUAD_J_MASK : LVSA_ITEM_J_MASK;
    const int st_shift = QUAD ? LVSA_QUAD_J_BITS + 2 * (int)(2u * pid + rank) : LVSA_ITEM_J_BITS + 2 * (int)rank;
    auto unit_row0 = [&](int item) { return ((long long)(QUAD ? 2 * item + (int)pid : item)) * 256 + (long long)rank * 128; };

    if (warp == 8 && lane == 0) {
        mbar_init(bar(SM::Q_FULL), 1); mbar_init(bar(SM::Q_EMPTY), 1);
        for (int b = 0; b < 3; ++b) {
            mbar_init(bar(SM::S_FULL + b), 1);
            mbar_init(bar(SM::PA_FULL + b), 8);     // 4 warps x 2 CTAs
            mbar_init(bar(SM::PB_FULL + b), 8);
        }
        mbar_init(bar(SM::PV_DONE), 1); mbar_init(bar(SM::PV_DONE + 1), 1); mbar_init(bar(SM::O_FULL), 1);
        mbar_init(bar(SM::O_FREE), 16);             // 8 warps x 2 CTAs
        for (int s = 0; s < NS; ++s) { mbar_init(bar(SM::KV_FULL + s), 1); mbar_init(bar(SM::KV_EMPTY + s), QUAD ? 2 : 1); }
        fence_barrier_init();
        prefetch_tmap(&tmap_q); prefetch_tmap(&tmap_k); prefetch_tmap(&tmap_v); prefetch_tmap(&tmap_o);
    }
    if (warp == 9) tmem_alloc_pair<512>(base + SM::TMEM_SLOT_OFF);
    tc_fence_before();
    cluster_sync_all();                                // barrier inits and TMEM visible in both CTAs
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_gen;

    if (wg < 2) {
        // =============================================================== softmax warpgroup `wg`
        // Warpgroup w processes the kv tiles with (running tile count) % 2 == w (S/P buffer = count % 3),
        // one thread per query row (128 logits), while the other warpgroup works on the next tile.
        // Both accumulate into the same O, so they share one reference maximum per row (m_ref, in
        // shared memory).  Decisions about m_ref are taken in tile order: a token passes between the
        // warpgroups (named barriers TOK0 / TOK1); only the short "load S, row max, decide" phase is
        // ordered, the exponentials of consecutive tiles overlap.
        reg_inc<208>();
        const int w = wg, rw = tid & 127;
        const uint32_t lane_off = (uint32_t)((warp & 3) * 32) << 16;
        const uint32_t tO = tmem_base + 384 + lane_off;                      // O, all 128 columns of my row
        const uint32_t tOh = tO + w * CH;                                    // the 64 columns I write out
        float *xch = reinterpret_cast<float *>(base_gen + SM::XCH_OFF);      // [0,128): m_ref, [128,384): l exchange
        float *m_ref = xch + rw;
        float *l_mine = xch + 128 + w * 128 + rw, *l_other = xch + 128 + (w ^ 1) * 128 + rw;
        const uint64_t scale2 = lvsa_sm::pack2(scale_log2, scale_log2);
        auto tok_wait = [&]() { asm volatile("bar.sync %0, 256;" ::"r"(1 + w) : "memory"); };
        auto tok_pass = [&]() { asm volatile("bar.arrive %0, 256;" ::"r"(1 + (w ^ 1)) : "memory"); };
        auto pair_sync = [&]() { asm volatile("bar.sync 3, 256;" ::: "memory"); };
        auto wg_sync = [&]() { asm volatile("bar.sync %0, 128;" ::"r"(4 + w) : "memory"); };    // my warpgroup only
        const uint32_t pa_full0 = map_to_cta(bar(SM::PA_FULL), lead);        // my pair leader's barriers
        const uint32_t pb_full0 = map_to_cta(bar(SM::PB_FULL), lead);
        const uint32_t ofree = map_to_cta(bar(SM::O_FREE), lead);
        if (w == 1) tok_pass();     // the first token: tile 0 belongs to warpgroup 0
        uint32_t tc = 0;            // kv tiles of this CTA so far (all items); tile tc belongs to warpgroup tc & 1
        uint32_t oc = 0;            // items finished
        for (long long work = work0 + pair; work < n_work; work += n_pairs) {   // works [work0, n_work) of this launch
            const int item = (int)(work % n_items);
            const int bh = (int)(work / n_items), h = h0 + bh % hc, b = bh / hc;   // heads [h0, h0 + hc) of H
            const long long my_row = unit_row0(item) + rw;
            const int fq = (int)min((long long)(T - 1), my_row / P);
            const uint32_t *arow = a_bits + (size_t)fq * words;
            const int e0 = item_ptr[item], e1 = item_ptr[item + 1];
            float m_run = -INFINITY, l_run = 0.f;   // m_run: my copy of m_ref; l_run: my tiles' part of the row sum
            // the list entries are fetched one tile ahead so that the load never sits in front of a decision
            const int e_first = e0 + (int)((w - tc) & 1u);
            int entry_nx = e_first < e1 ? __ldg(item_tiles + e_first) : 0;
            int col0_nx = (VARW && e_first < e1) ? __ldg(item_col0 + e_first) : 0;
            for (int e = e_first; e < e1; e += 2) {
                const uint32_t t_me = tc + (uint32_t)(e - e0);               // running index of this tile
                const int entry = entry_nx;
                // first token of the kv tile (PARTIAL tiles need it) and its 32-column chunks
                const int tile_col0 = VARW ? col0_nx : (entry & J_MASK) * BT;
                if (e + 2 < e1) { entry_nx = __ldg(item_tiles + e + 2); if (VARW) col0_nx = __ldg(item_col0 + e + 2); }
                const int st = (entry >> st_shift) & 3;
                const int nch = VARW ? entry_chunks(entry) : 4;
                const bool first = (e == e0);

                // three S/P buffers in rotation: S(t+2) is computed while the softmax of tile t runs, and is
                // issued right after PV(t-1), i.e. it never waits for a P of this warpgroup
                const uint32_t buf = t_me % 3u;
                const uint32_t tS = tmem_base + buf * 128 + lane_off;
                const uint32_t pa_full = pa_full0 + 8u * buf, pb_full = pb_full0 + 8u * buf;
                mbar_wait(bar(SM::S_FULL + buf), (t_me / 3u) & 1u);
                tc_fence_after();
                if (st == LVSA_ST_SKIP) {
                    // the pair's MMAs cover both q tiles for every listed kv tile; a tile that is not in
                    // MY q tile's list contributes nothing: P = 0.  The token still moves on.
                    uint32_t z[32];
#pragma unroll
                    for (int x = 0; x < 32; ++x) z[x] = 0u;
                    tmem_st_32x32b_x32(tS, z);
                    tmem_st_32x32b_x32(tS + 32, z);
                    tok_wait();
                    if (first) *m_ref = -INFINITY;
                    tok_pass();
                    tmem_wait_st();
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) { mbar_arrive_cluster(pa_full); mbar_arrive_cluster(pb_full); }
                    continue;
                }
                // The body below is instantiated twice: with the chunk count as a compile-time 4 (a
                // 128-column tile: no per-chunk tests, the four TMEM loads issue back to back) and with
                // the run-time count of a narrow frame-aligned tile.
                auto tile_body = [&](auto nch_) {
                    const int nchv = nch_;
                    float s[BT];
#pragma unroll
                    for (int c = 0; c < 4; ++c) {
                        if (c < nchv) {          // warp-uniform
                            uint32_t r[32];
                            tmem_ld_32x32b_x32(tS + c * 32, r);
#pragma unroll
                            for (int x = 0; x < 32; ++x) s[c * 32 + x] = __uint_as_float(r[x]);
                        } else {                // columns a narrow tile does not have
#pragma unroll
                            for (int x = 0; x < 32; ++x) s[c * 32 + x] = -INFINITY;
                        }
                    }
                    tmem_wait_ld();

                    uint32_t cm[4] = {~0u, ~0u, ~0u, ~0u};   // columns of this tile my row may attend to
                    if (st == LVSA_ST_PARTIAL) {
                        cm[0] = cm[1] = cm[2] = cm[3] = 0u;
                        // 32-bit arithmetic in coordinates relative to the tile's first token (N < 2^31)
                        const int Ni = (int)N;
                        int g = min((int)((unsigned)tile_col0 / (unsigned)P), T - 1);
                        // token-0 tiles: the columns run to the end of the tile (or N) across frame boundaries;
                        // frame-aligned tiles: they stop at the end of the tile's frame (the rest is padding)
                        const int lim = (!VARW || g == T - 1) ? Ni - tile_col0 : (g + 1) * P - tile_col0;
                        const int cend = min(32 * nchv, lim);
                        for (int fs = g * P - tile_col0, fe; fs < cend; fs = fe, ++g) {
                            fe = (g == T - 1) ? Ni - tile_col0 : fs + P;
                            if ((arow[g >> 5] >> (g & 31)) & 1u) {
                                const int lo = max(fs, 0), hi = min(fe, cend);
#pragma unroll
                                for (int x = 0; x < 4; ++x) cm[x] |= range_mask32(lo, hi, x);
                            }
                        }
                        // most rows of a PARTIAL tile are not masked at all (the flag is per q tile): a chunk
                        // whose 32 columns are all allowed is left alone
#pragma unroll
                        for (int c4 = 0; c4 < 4; ++c4)
                            if (cm[c4] != ~0u) {
#pragma unroll
                                for (int x = 0; x < 32; ++x)
                                    if (!((cm[c4] >> x) & 1u)) s[c4 * 32 + x] = -INFINITY;
                            }
                    }
                    const float rm = lvsa_sm::row_max<BT>(s) * scale_log2;

                    // ---- ordered phase: read the shared reference, decide, write it back
                    tok_wait();
                    bool grow;
                    float m_new;
                    if (first) {
                        grow = false; m_new = rm; m_run = rm;          // the first tile of the item sets the reference
                    } else {
                        const float m_sh = *m_ref;                      // may have been raised by the other warpgroup
                        if (m_sh != m_run) { l_run *= fast_exp2(m_run - m_sh); m_run = m_sh; }   // exp2(-inf - x) = 0, l_run = 0 then
                        grow = rm > m_run + RESCALE_THRESHOLD;
                        m_new = grow ? rm : m_run;
                    }
                    *m_ref = m_new;
                    tok_pass();
                    // ---- end of the ordered phase

                    if (__any_sync(0xffffffffu, grow)) {
                        // O is rescaled in place once every PV issued so far has landed (the other
                        // warpgroup's tile t_me - 1 included).  PV(t) commits to PV_DONE[t & 1].  S_FULL of this
                        // tile implies PV(t_me - 3) completed, the previous phase of that barrier, so the
                        // parity wait is unambiguous.  PV(t_me) cannot be issued before this warpgroup
                        // publishes P below.
                        mbar_wait(bar(SM::PV_DONE + ((t_me - 1u) & 1u)), ((t_me - 1u) >> 1) & 1u);
                        tc_fence_after();
                        const float corr = grow ? fast_exp2(m_run - m_new) : 1.f;
                        if (grow) { l_run *= corr; m_run = m_new; }
#pragma unroll 1
                        for (int c = 0; c < 8; ++c) {
                            uint32_t r[16];
                            tmem_ld_32x32b_x16(tO + c * 16, r);
                            tmem_wait_ld();
#pragma unroll
                            for (int x = 0; x < 16; ++x) r[x] = __float_as_uint(__uint_as_float(r[x]) * corr);
                            tmem_st_32x32b_x16(tO + c * 16, r);
                        }
                    }
                    const float m_use = (m_run == -INFINITY) ? 0.f : m_run;
                    const uint64_t negm2 = lvsa_sm::pack2(-m_use, -m_use);
                    uint64_t lsum = lvsa_sm::pack2(0.f, 0.f);
                    auto publish = [&](uint32_t which) {
                        tmem_wait_st();
                        tc_fence_before();
                        __syncwarp();
                        if (lane == 0) mbar_arrive_cluster(which);
                    };
                    // P for the nch chunks of the tile; the first half of P (or all of a narrow tile) is
                    // published as soon as it is in TMEM so that the PV MMAs can start.  Masked logits are
                    // -inf: the MUFU gives exact zeros; a fully masked chunk skips the exponentials.
                    const int pa_at = min(1, nchv - 1);
                    if (st == LVSA_ST_FULL) {
#pragma unroll
                        for (int c = 0; c < 4; ++c) {
                            if (c < nchv) {
                                uint32_t pk[16];
                                lvsa_sm::exp_chunk32(s, c * 32, scale2, negm2, pk, lsum);
                                tmem_st_32x32b_x16(tS + c * 16, pk);
                                if (c == pa_at) publish(pa_full);
                            }
                        }
                    } else
#pragma unroll
                    for (int c = 0; c < 4; ++c) {
                        if (c < nchv) {
                            uint32_t pk[16];
                            if (cm[c] == 0u) {
#pragma unroll
                                for (int x = 0; x < 16; ++x) pk[x] = 0u;
                            } else {
                                lvsa_sm::exp_chunk32(s, c * 32, scale2, negm2, pk, lsum);
                            }
                            tmem_st_32x32b_x16(tS + c * 16, pk);
                            if (c == pa_at) publish(pa_full);
                        }
                    }
                    publish(pb_full);
                    {
                        float la, lb;
                        lvsa_sm::unpack2(lsum, la, lb);
                        l_run += la + lb;
                    }
                };
                if (!VARW || nch == 4) tile_body(StaticInt<4>{});
                else tile_body(nch);
            }
            tc += (uint32_t)(e1 - e0);
            if (e0 < e1) {
                // epilogue: O / l -> bf16 -> global; I write 64 of the 128 columns of my row.
                // All PVs of the item have landed, so every decision about m_ref has been taken.
                mbar_wait(bar(SM::O_FULL), oc & 1u); ++oc;
                tc_fence_after();
                const float m_fin = *m_ref;
                if (m_fin != m_run) { l_run *= fast_exp2(m_run - m_fin); m_run = m_fin; }
                *l_mine = l_run;
                pair_sync();
                const float l_tot = l_run + *l_other;
                pair_sync();   // m_ref and the exchange slots are free again for the next item
                const bool row_ok = my_row < N;
                const float inv = 1.f / l_tot;
                // My 64 channels go to my warpgroup's span of the staging buffer, [128 rows][128 B] in the
                // SWIZZLE_128B layout of the output tensor map (16-byte chunk j of row r sits at chunk
                // j ^ (r & 7): conflict-free for the 8 rows a store phase covers), and one TMA store per
                // warpgroup writes the span out (rows >= N are clipped by the tensor map).
                if (rw == 0) tma_store_wait_read();        // the previous item's store has read the span
                wg_sync();
                const uint32_t srow = sOut + (uint32_t)w * SPAN_BYTES + (uint32_t)rw * 128u;
#pragma unroll
                for (int c = 0; c < 2; ++c) {
                    uint32_t r[32];
                    tmem_ld_32x32b_x32(tOh + c * 32, r);
                    tmem_wait_ld();
#pragma unroll
                    for (int x = 0; x < 4; ++x) {
                        const uint32_t v0 = pack_bf16x2(__uint_as_float(r[8 * x + 0]) * inv, __uint_as_float(r[8 * x + 1]) * inv);
                        const uint32_t v1 = pack_bf16x2(__uint_as_float(r[8 * x + 2]) * inv, __uint_as_float(r[8 * x + 3]) * inv);
                        const uint32_t v2 = pack_bf16x2(__uint_as_float(r[8 * x + 4]) * inv, __uint_as_float(r[8 * x + 5]) * inv);
                        const uint32_t v3 = pack_bf16x2(__uint_as_float(r[8 * x + 6]) * inv, __uint_as_float(r[8 * x + 7]) * inv);
                        st_shared_v4(srow + (uint32_t)(((4 * c + x) ^ (rw & 7)) * 16), v0, v1, v2, v3);
                    }
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive_cluster(ofree);
                fence_proxy_async_smem();                  // my generic-proxy writes, before the async-proxy read
                wg_sync();
                if (rw == 0) {
                    tma_store_4d(&tmap_o, sOut + (uint32_t)w * SPAN_BYTES, w * CH, h, (int)unit_row0(item), b);
                    tma_store_commit();
                }
                if (w == 0 && row_ok && lse != nullptr)
                    lse[((size_t)b * H + h) * N + my_row] = m_run * 0.6931471805599453f + __logf(l_tot);
            }
        }
        // drain the token that is left on one of the two barriers
        if ((tc & 1u) == (uint32_t)w) tok_wait();
        if (rw == 0) tma_store_wait_all();                 // my output stores have left shared memory
    } else {
        reg_dec<88>();
        if (warp == 8 && lane == 0) {
            // =========================================================== TMA producer (both CTAs)
            // Loads MY half of every operand; completion bytes are counted on the LEADER's barriers.
            // The leader arms each barrier with the bytes of both halves.  Ring order = the order the
            // issuer consumes: K(0), K(1), then per tile j: K(j+2), V(j).
            const uint32_t q_full_L = map_to_cta(bar(SM::Q_FULL), lead);
            uint32_t kv_it = 0, qi = 0;
            // col0 = first token of the kv tile; nt = its computed columns.  K: CTA r supplies columns
            // [r nt/2, (r+1) nt/2) of S, i.e. kv rows col0 + r nt/2 ... (the 64-row box over-reads for a
            // narrow tile; the MMA uses the first nt/2 rows).  V: all rows of the tile, my 64 channels.
            auto push = [&](const CUtensorMap *tm, bool is_k, int e, int h, int b) {
                const int col0 = VARW ? __ldg(item_col0 + e) : (__ldg(item_tiles + e) & J_MASK) * BT;
                const int nt = VARW ? 32 * entry_chunks(__ldg(item_tiles + e)) : BT;
                const uint32_t stage = kv_it % NS, n = kv_it / NS;
                mbar_wait(bar(SM::KV_EMPTY + stage), (n & 1u) ^ 1u);
                if (rank == 0) mbar_expect_tx(bar(SM::KV_FULL + stage), 2 * STAGE_BYTES);
                const uint32_t dst = sRing + stage * STAGE_BYTES;
                if (QUAD) {
                    // pair 0 loads for the whole cluster: my half goes to CTA `rank` of both pairs; the barrier
                    // operand is my own KV_FULL with the peer bit cleared = "the leader of the destination's pair"
                    if (pid == 0) {
                        const uint32_t full_rel = bar(SM::KV_FULL + stage) & 0xFEFFFFFFu;
                        const uint16_t mc = (uint16_t)(0x5u << rank);
                        if (is_k) {
                            tma_load_4d_pair_mc(dst, tm, full_rel, mc, 0, h, col0 + 64 * (int)rank, b);
                            tma_load_4d_pair_mc(dst + 8192, tm, full_rel, mc, 64, h, col0 + 64 * (int)rank, b);
                        } else {
                            tma_load_4d_pair_mc(dst, tm, full_rel, mc, 64 * (int)rank, h, col0, b);
                        }
                    }
                } else {
                    const uint32_t full_L = map_to_cta(bar(SM::KV_FULL + stage), lead);
                    if (is_k) {   // kv rows [col0 + 64 rank, +64), channels [0,64) and [64,128): two 8 KB spans
                        tma_load_4d_pair(dst, tm, full_L, 0, h, col0 + (nt / 2) * (int)rank, b);
                        tma_load_4d_pair(dst + 8192, tm, full_L, 64, h, col0 + (nt / 2) * (int)rank, b);
                    } else {      // channels [64 rank, +64) of all 128 kv rows: one 16 KB span
                        tma_load_4d_pair(dst, tm, full_L, 64 * (int)rank, h, col0, b);
                    }
                }
                ++kv_it;
            };
            for (long long work = work0 + pair; work < n_work; work += n_pairs) {   // works [work0, n_work) of this launch
                const int item = (int)(work % n_items);
                const int bh = (int)(work / n_items), h = h0 + bh % hc, b = bh / hc;   // heads [h0, h0 + hc) of H
                const long long row0 = unit_row0(item);
                const int e0 = item_ptr[item], e1 = item_ptr[item + 1];
                mbar_wait(bar(SM::Q_EMPTY), (qi & 1u) ^ 1u);
                if (rank == 0) mbar_expect_tx(bar(SM::Q_FULL), 2 * TILE_BYTES);
                // rows past N (a q tile that does not exist) are zero-filled by TMA
                tma_load_4d_pair(sQ, &tmap_q, q_full_L, 0, h, (int)row0, b);
                tma_load_4d_pair(sQ + SPAN_BYTES, &tmap_q, q_full_L, 64, h, (int)row0, b);
                ++qi;
                if (e0 < e1) push(&tmap_k, true, e0, h, b);
                if (e0 + 1 < e1) push(&tmap_k, true, e0 + 1, h, b);
                for (int e = e0; e < e1; ++e) {
                    if (e + 2 < e1) push(&tmap_k, true, e + 2, h, b);
                    push(&tmap_v, false, e, h, b);
                }
            }
        } else if (warp == 9 && rank == 0) {
            // =========================================================== MMA issuer (leader CTA)
            constexpr uint32_t IDESC_S0 = umma_idesc_bf16(256, 0, 0);   // N is filled in per tile
            constexpr uint32_t IDESC_O = umma_idesc_bf16(256, D, 1);
            const uint64_t dQ = umma_smem_desc_sw128(sQ, 16);
            const uint64_t dRing = umma_smem_desc_sw128(sRing, 16);
            const uint32_t tO = tmem_base + 384;
            // S(buf) = Q K^T: A = Q (128 rows per CTA, two 16 KB spans), B = my/peer K half (64 rows
            // per CTA, two 8 KB spans); 8 k-blocks of 16 channels
            auto issue_S = [&](uint32_t buf, uint32_t stage, bool last_of_item, int nt) {
                // a full tile takes the compile-time descriptor (N = 128), a narrow one builds its own
                constexpr uint32_t IDESC_S128 = IDESC_S0 | ((uint32_t)(BT >> 3) << 17);
                const uint32_t IDESC_S = nt == BT ? IDESC_S128 : (IDESC_S0 | ((uint32_t)(nt >> 3) << 17));
#pragma unroll
                for (int kk = 0; kk < 8; ++kk) {
                    const uint32_t offA = (uint32_t)((kk >> 2) * SPAN_BYTES + (kk & 3) * 32) >> 4;
                    const uint32_t offB = (uint32_t)((kk >> 2) * 8192 + (kk & 3) * 32) >> 4;
                    umma_ss_pair(tmem_base + buf * 128, dQ + (uint64_t)offA,
                                 dRing + (uint64_t)(((stage * STAGE_BYTES) >> 4) + offB), IDESC_S, kk > 0);
                }
                umma_commit_pair(bar(SM::S_FULL + buf), pair_mask);
                umma_commit_pair(bar(SM::KV_EMPTY + stage), ring_mask);
                if (last_of_item) umma_commit_pair(bar(SM::Q_EMPTY), pair_mask);   // Q is last read by S of the final tile
            };
            // O += P(buf) V: A = P from TMEM (2 bf16 per column), B = V half (MN-major, 64 channels per
            // CTA = one 128 B span; 16 kv rows = 2048 B per k-block)
            // nt / 16 k-blocks of 16 kv rows; half 0 = blocks 0..3, half 1 = blocks 4..7 (as far as the tile has them)
            auto issue_PV = [&](uint32_t buf, uint32_t stage, bool accumulate, int half, int nt) {
                if (nt == BT) {
#pragma unroll
                    for (int kk = 4 * half; kk < 4 * half + 4; ++kk)
                        umma_ts_pair(tO, tmem_base + buf * 128 + kk * 8,
                                     dRing + (uint64_t)((stage * STAGE_BYTES + (uint32_t)kk * 2048u) >> 4), IDESC_O,
                                     (accumulate || kk > 0) ? 1u : 0u);
                } else {
#pragma unroll
                    for (int kk = 4 * half; kk < 4 * half + 4; ++kk)
                        if (kk * 16 < nt)
                            umma_ts_pair(tO, tmem_base + buf * 128 + kk * 8,
                                         dRing + (uint64_t)((stage * STAGE_BYTES + (uint32_t)kk * 2048u) >> 4), IDESC_O,
                                         (accumulate || kk > 0) ? 1u : 0u);
                }
            };
            // the width is made warp-uniform explicitly (shuffle from lane 0): it feeds the instruction
            // descriptor, which lives in a uniform register, and a value the compiler cannot prove uniform
            // costs a per-instruction waterfall loop
            auto uniform_nt = [&](int raw_entry) { return __shfl_sync(0xffffffffu, 32 * entry_chunks(raw_entry), 0); };
            auto tile_nt = [&](int e) { return VARW ? uniform_nt(__ldg(item_tiles + e)) : BT; };
            uint32_t kv_it = 0, qi = 0, tc = 0, oc = 0;
            auto next_stage = [&](uint32_t &stage) {
                stage = kv_it % NS;
                const uint32_t n = kv_it / NS;
                ++kv_it;
                mbar_wait(bar(SM::KV_FULL + stage), n & 1u);
            };
            for (long long work = work0 + pair; work < n_work; work += n_pairs) {   // works [work0, n_work) of this launch
                const int item = (int)(work % n_items);
                const int e0 = __shfl_sync(0xffffffffu, __ldg(item_ptr + item), 0);
                const int e1 = __shfl_sync(0xffffffffu, __ldg(item_ptr + item + 1), 0);
                const int n = e1 - e0;
                mbar_wait(bar(SM::Q_FULL), qi & 1u); ++qi;
                // S of the first two tiles; the buffer of tile t is t % 3 (running count), its previous
                // P (tile t - 3) was read by a PV issued earlier
                // widths of tiles j, j+1, j+2 (nt0, nt1, nt2); the entry of tile j+3 is fetched one
                // iteration before it is needed, so no load sits in front of an MMA issue
                int nt0 = n > 0 ? tile_nt(e0) : 0, nt1 = n > 1 ? tile_nt(e0 + 1) : 0, nt2 = n > 2 ? tile_nt(e0 + 2) : 0;
                for (int j = 0; j < 2 && j < n; ++j) {
                    uint32_t stage;
                    next_stage(stage);
                    tc_fence_after();
                    const int nt = j == 0 ? nt0 : nt1;
                    if (elect_one_sync()) issue_S((tc + j) % 3u, stage, j == n - 1, nt);
                    __syncwarp();
                }
                for (int j = 0; j < n; ++j, ++tc) {
                    const uint32_t buf = tc % 3u, par = (tc / 3u) & 1u;
                    const int nt_pv = nt0;
                    // entry of tile j + 3: loaded now, shuffled (which waits for the load) at the end of the iteration
                    const int raw3 = (VARW && j + 3 < n) ? __ldg(item_tiles + e0 + j + 3) : 0;
                    if (j + 2 < n) {
                        const int nt = nt2;
                        uint32_t stage;
                        next_stage(stage);
                        tc_fence_after();
                        if (elect_one_sync()) issue_S((tc + 2u) % 3u, stage, j + 2 == n - 1, nt);   // after PV(tc-1): its buffer is free
                        __syncwarp();
                    }
                    uint32_t stageV;
                    next_stage(stageV);
                    if (j == 0) mbar_wait(bar(SM::O_FREE), (oc & 1u) ^ 1u);
                    mbar_wait(bar(SM::PA_FULL + buf), par);
                    tc_fence_after();
                    if (elect_one_sync()) issue_PV(buf, stageV, j > 0, 0, nt_pv);
                    __syncwarp();
                    mbar_wait(bar(SM::PB_FULL + buf), par);
                    tc_fence_after();
                    if (elect_one_sync()) {
                        issue_PV(buf, stageV, j > 0, 1, nt_pv);
                        umma_commit_pair(bar(SM::PV_DONE + (tc & 1u)), pair_mask);
                        umma_commit_pair(bar(SM::KV_EMPTY + stageV), ring_mask);
                    }
                    __syncwarp();
                    nt0 = nt1; nt1 = nt2; nt2 = VARW ? uniform_nt(raw3) : BT;
                }
                if (n > 0) {
                    if (elect_one_sync()) umma_commit_pair(bar(SM::O_FULL), pair_mask);
                    __syncwarp();
                    ++oc;
                } else if (elect_one_sync()) {
                    umma_commit_pair(bar(SM::Q_EMPTY), pair_mask);
                }
                __syncwarp();
            }
        }
    }
    tc_fence_before();
    cluster_sync_all();     // the peer may still signal my barriers / read my shared memory until here
    if (warp == 9) tmem_dealloc_pair<512>(tmem_base);
}

}  // namespace

// host side -------------------------------------------------------------------------------
lvsa_status_t lvsa_make_tmap_bf16(CUtensorMap *m, const void *base, const lvsa_index *ix, int box_rows, int which);

// One-time setup per DEVICE (the shared-memory attribute and the SM count belong to a device, not
// to the process); `device` must be the current device.
static int g_pair_n_sm[LVSA_MAX_DEVICES] = {};
static int g_quad_clusters[LVSA_MAX_DEVICES] = {};   // 4-CTA clusters that can be resident at once
// HYBRID's internal stream and fork/join events: created here, per device, so that no launch ever
// creates a resource (a first HYBRID call may already be under stream capture).  `join` is created
// last and is the "ready" mark: a set-up that failed half-way is retried, not used.
struct HybridSide { cudaStream_t side = nullptr; cudaEvent_t fork = nullptr, join = nullptr; };
static HybridSide g_hybrid[LVSA_MAX_DEVICES];
static std::mutex g_hybrid_mutex;
static std::mutex g_prepare_mutex;
lvsa_status_t lvsa_attn_sm100_pair_prepare(int device) {
    if (device < 0 || device >= LVSA_MAX_DEVICES) { lvsa_set_error("device ordinal out of range"); return LVSA_EUNSUPPORTED; }
    std::lock_guard<std::mutex> prepare_lock(g_prepare_mutex);
    if (g_pair_n_sm[device] != 0) return LVSA_OK;
    {
        HybridSide &hs = g_hybrid[device];
        if (hs.join == nullptr) {
            if (hs.side == nullptr) LVSA_CUDA_TRY(cudaStreamCreateWithFlags(&hs.side, cudaStreamNonBlocking));
            if (hs.fork == nullptr) LVSA_CUDA_TRY(cudaEventCreateWithFlags(&hs.fork, cudaEventDisableTiming));
            LVSA_CUDA_TRY(cudaEventCreateWithFlags(&hs.join, cudaEventDisableTiming));
        }
    }
    using SM = SmemP<LVSA_PAIR_STAGES>;
    LVSA_CUDA_TRY(cudaFuncSetAttribute(lvsa_attn_sm100_pair_kernel<LVSA_PAIR_STAGES, MODE_TOKEN0>,
                                       cudaFuncAttributeMaxDynamicSharedMemorySize, SM::BYTES));
    LVSA_CUDA_TRY(cudaFuncSetAttribute(lvsa_attn_sm100_pair_kernel<LVSA_PAIR_STAGES, MODE_VARW>,
                                       cudaFuncAttributeMaxDynamicSharedMemorySize, SM::BYTES));
    LVSA_CUDA_TRY(cudaFuncSetAttribute(lvsa_attn_sm100_pair_kernel<LVSA_PAIR_STAGES, MODE_QUAD>,
                                       cudaFuncAttributeMaxDynamicSharedMemorySize, SM::BYTES));
    int n = 0;
    LVSA_CUDA_TRY(cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, device));
    // A 4-CTA cluster needs four free SMs of one GPC, so fewer than n / 4 of them may fit at once; the
    // persistent grid must not be larger than that (a cluster that is not resident would only start
    // when another one has finished ALL its work).
    {
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3((unsigned)(n / 4 * 4)); cfg.blockDim = dim3(NTHREADS); cfg.dynamicSmemBytes = SM::BYTES;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = 4; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        cfg.attrs = at; cfg.numAttrs = 1;
        int nc = 0;
        LVSA_CUDA_TRY(cudaOccupancyMaxActiveClusters(&nc, lvsa_attn_sm100_pair_kernel<LVSA_PAIR_STAGES, MODE_QUAD>, &cfg));
        g_quad_clusters[device] = nc > 0 ? nc : 1;
    }
    g_pair_n_sm[device] = n;
    return LVSA_OK;
}

// HYBRID (LVSA_KERNEL_TCGEN05_HYBRID): 4-CTA clusters on the SMs they can cover, CTA pairs on the rest,
// as two launches that run side by side (the second on an internal stream, forked from and joined back to
// the caller's stream with events, which also works under stream capture).  The work is split statically
// at a quad boundary in proportion to the SMs of the two parts.
#ifndef LVSA_HYBRID_QUAD_SPEED
#define LVSA_HYBRID_QUAD_SPEED 1.04   // measured: work per SM and second of the 4-CTA clusters relative to the pairs
#endif

static bool is_quad(const lvsa_index *ix) { return ix->p.kernel == LVSA_KERNEL_TCGEN05_QUAD || ix->p.kernel == LVSA_KERNEL_TCGEN05_HYBRID; }

// HYBRID's static split over hc heads: quads [0, wq1) go to the 4-CTA clusters, items [item0, item_works) to
// the CTA pairs on the SMs the clusters cannot cover.  Returns false when everything goes to the clusters
// (one launch, no fork).
struct HybridSplit { long long wq1, item0, nqc, pairs_left; };
static bool hybrid_split(const lvsa_index *ix, int hc, HybridSplit *sp) {
    const int dev = ix->device;
    const long long item_works = ix->n_items * hc * ix->p.B, quad_works = ix->n_quads * hc * ix->p.B;
    sp->nqc = g_quad_clusters[dev]; sp->pairs_left = (g_pair_n_sm[dev] - 4 * sp->nqc) / 2;
    // the pairs' share of the quads, rounded to whole quads; the pair launch starts at the first item of quad wq1
    const double share = sp->pairs_left <= 0 ? 0.0 : 2.0 * sp->pairs_left / (4.0 * sp->nqc * LVSA_HYBRID_QUAD_SPEED + 2.0 * sp->pairs_left);
    sp->wq1 = quad_works - (long long)(quad_works * share + 0.5);
    if (sp->wq1 < 0) sp->wq1 = 0;
    sp->item0 = (sp->wq1 / ix->n_quads) * ix->n_items + 2 * (sp->wq1 % ix->n_quads);
    return !(sp->wq1 == quad_works || sp->item0 >= item_works);
}

// kernels one launch_heads call over hc heads enqueues (after prepare)
int lvsa_attn_sm100_pair_num_launches(const lvsa_index *ix, int hc) {
    if (ix->p.kernel != LVSA_KERNEL_TCGEN05_HYBRID) return 1;
    HybridSplit sp;
    if (!hybrid_split(ix, hc, &sp)) return 1;
    return sp.wq1 > 0 ? 2 : 1;
}

int lvsa_attn_sm100_pair_grid(const lvsa_index *ix, int hc) {
    if (ix->p.kernel == LVSA_KERNEL_TCGEN05_HYBRID) return g_pair_n_sm[ix->device] / 2 * 2;   // both parts together
    const bool quad = is_quad(ix);
    const int cl = quad ? 4 : 2;
    const long long n_work = (quad ? ix->n_quads : ix->n_items) * hc * ix->p.B;
    long long n_clusters = quad ? g_quad_clusters[ix->device] : g_pair_n_sm[ix->device] / cl;
    if (n_work < n_clusters) n_clusters = n_work;
    return (int)(cl * n_clusters);
}
// Heads [h0, h0 + hc) only (all batches): the host entry point pipelines head groups against the
// PCIe copies.  q, k, v, out, lse are the FULL tensors.
lvsa_status_t lvsa_attn_sm100_pair_launch_heads(const lvsa_index *ix, const void *q, const void *k, const void *v,
                                                void *out, float *lse, int h0, int hc, cudaStream_t stream) {
    constexpr int NS = LVSA_PAIR_STAGES;
    using SM = SmemP<NS>;
    CUtensorMap mq, mk, mv, mo;
    lvsa_status_t st;
    if ((st = lvsa_make_tmap_bf16(&mq, q, ix, 128, LVSA_T_Q)) != LVSA_OK) return st;
    if ((st = lvsa_make_tmap_bf16(&mk, k, ix, 64, LVSA_T_K)) != LVSA_OK) return st;
    if ((st = lvsa_make_tmap_bf16(&mv, v, ix, BT, LVSA_T_V)) != LVSA_OK) return st;
    if ((st = lvsa_make_tmap_bf16(&mo, out, ix, 128, LVSA_T_OUT)) != LVSA_OK) return st;
    if ((st = lvsa_attn_sm100_pair_prepare(ix->device)) != LVSA_OK) return st;
    const float scale_log2 = ix->p.softmax_scale * 1.4426950408889634f;
    // one launch over the works [work0, work_end) of its kind (quads for MODE_QUAD, items otherwise)
    auto launch = [&](int mode, long long work0, long long work_end, long long n_clusters, cudaStream_t s) {
        if (work_end <= work0) return;
        if (work_end - work0 < n_clusters) n_clusters = work_end - work0;
        const bool quad = mode == MODE_QUAD;
        auto kern = quad ? lvsa_attn_sm100_pair_kernel<NS, MODE_QUAD>
                  : mode == MODE_VARW ? lvsa_attn_sm100_pair_kernel<NS, MODE_VARW> : lvsa_attn_sm100_pair_kernel<NS, MODE_TOKEN0>;
        kern<<<(unsigned)((quad ? 4 : 2) * n_clusters), NTHREADS, SM::BYTES, s>>>(
            mq, mk, mv, mo, lse, quad ? ix->d_quad_ptr : ix->d_item_ptr, quad ? ix->d_quad_tiles : ix->d_item_tiles,
            ix->d_item_col0, ix->d_abits, ix->words, (long long)ix->N, ix->p.P, ix->Tf, ix->p.H, h0, hc,
            (int)(quad ? ix->n_quads : ix->n_items), work0, work_end, scale_log2);
    };
    const int dev = ix->device;
    const long long item_works = ix->n_items * hc * ix->p.B, quad_works = ix->n_quads * hc * ix->p.B;
    if (ix->p.kernel == LVSA_KERNEL_TCGEN05_HYBRID) {
        HybridSplit sp;
        const bool forks = hybrid_split(ix, hc, &sp);
        const long long nqc = sp.nqc, pairs_left = sp.pairs_left, wq1 = sp.wq1, item0 = sp.item0;
        if (!forks) {
            launch(MODE_QUAD, 0, quad_works, nqc, stream);
        } else {
            std::lock_guard<std::mutex> lock(g_hybrid_mutex);
            HybridSide &hs = g_hybrid[dev];   // created by lvsa_attn_sm100_pair_prepare (above)
            LVSA_CUDA_TRY(cudaEventRecord(hs.fork, stream));
            LVSA_CUDA_TRY(cudaStreamWaitEvent(hs.side, hs.fork, 0));
            launch(MODE_QUAD, 0, wq1, nqc, stream);                      // first: the clusters need whole GPC quarters
            launch(MODE_TOKEN0, item0, item_works, pairs_left, hs.side);
            LVSA_CUDA_TRY(cudaEventRecord(hs.join, hs.side));
            LVSA_CUDA_TRY(cudaStreamWaitEvent(stream, hs.join, 0));
        }
    } else if (ix->p.kernel == LVSA_KERNEL_TCGEN05_QUAD) {
        launch(MODE_QUAD, 0, quad_works, g_quad_clusters[dev], stream);
    } else {
        launch(ix->p.kv_tiling == LVSA_KV_TILES_FRAME_ALIGNED ? MODE_VARW : MODE_TOKEN0, 0, item_works, g_pair_n_sm[dev] / 2, stream);
    }
    LVSA_CUDA_TRY(cudaGetLastError());
    return LVSA_OK;
}

lvsa_status_t lvsa_attn_sm100_pair_launch(const lvsa_index *ix, const void *q, const void *k, const void *v,
                                          void *out, float *lse, cudaStream_t stream) {
    return lvsa_attn_sm100_pair_launch_heads(ix, q, k, v, out, lse, 0, ix->p.H, stream);
}
