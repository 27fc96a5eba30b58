// Warp-specialised, persistent LVSA attention forward for sm_100a (d = 128, 128 x 128 tiles).
//
// Computes Eq. 2 over the kept kv tiles listed by the block index.  One CTA per SM
// loops over work items (head, pair of adjacent q tiles = 256 query rows); both q tiles share
// every K/V tile load.  Roles (12 warps):
//   warps 0-3  softmax warpgroup 0 : rows of q tile 0   (TMEM lanes = rows; thread = one row)
//   warps 4-7  softmax warpgroup 1 : rows of q tile 1
//   warp  8    TMA producer        : Q once per item, then K_j, V_j of each listed tile into a ring
//   warps 9,10 MMA issuers         : S_w = Q_w K_j^T and O_w += P_w V_j (tcgen05, TMEM accumulators),
//                                    warp 9 for q tile 0, warp 10 for q tile 1
// TMEM (512 columns): S0 [0,128) S1 [128,256) O0 [256,384) O1 [384,512); P_w (bf16) overwrites the
// first 64 columns of S_w and is the A operand of the second MMA straight from TMEM.
// The tensor pipe executes MMAs in issue order, which is what makes the S/P aliasing and the
// "rescale O right after S arrives" step safe.
#include <cuda.h>
#include <cuda_bf16.h>

#include "lvsa_internal.h"
#include "sm100_ptx.cuh"
#include "lvsa_softmax.cuh"

using namespace sm100;

namespace {

constexpr int D = 128, BT = 128;
constexpr int TILE_BYTES = BT * D * 2;          // 32 KB: one Q, K or V tile
constexpr int HALF_BYTES = BT * 128;            // 16 KB: [128 rows][128 B] swizzle span
constexpr int NTHREADS = 384;
constexpr float RESCALE_THRESHOLD = 8.0f;       // log2 units: rescale O only if the max grew by > 2^8
#ifndef LVSA_POLY_PAIRS
#define LVSA_POLY_PAIRS 0                       // of every 16 logit pairs, how many take the FMA-pipe exp2
#endif

template <int NS>
struct Smem {
    static constexpr int Q_OFF = 0;                          // 2 x 32 KB
    static constexpr int RING_OFF = 2 * TILE_BYTES;          // NS x 32 KB
    static constexpr int BAR_OFF = RING_OFF + NS * TILE_BYTES;
    // barriers (8 B each)
    static constexpr int Q_FULL = 0, Q_EMPTY = 1, S_FULL = 2 /*2*/, P_FULL = 4 /*2*/, O_FULL = 6 /*2*/,
                         O_FREE = 8 /*2*/, P2_FULL = 10 /*2*/, TURN = 12 /*2*/, KV_FULL = 14 /*NS*/, KV_EMPTY = 14 + NS /*NS*/,
                         NBARS = 14 + 2 * NS;
    static constexpr int TMEM_SLOT_OFF = BAR_OFF + 8 * NBARS;
    static constexpr int BYTES = TMEM_SLOT_OFF + 16 + 1024 /*alignment slack*/;
};

__device__ __forceinline__ uint32_t range_mask32(int lo, int hi, int w) {
    const int a = max(lo, 32 * w), b = min(hi, 32 * w + 32);
    if (a >= b) return 0u;
    const int n = b - a;
    return (n == 32 ? 0xffffffffu : ((1u << n) - 1u)) << (a - 32 * w);
}

template <int REGS> __device__ __forceinline__ void reg_inc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(REGS)); }
template <int REGS> __device__ __forceinline__ void reg_dec() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(REGS)); }

__device__ __forceinline__ int entry_state(int entry, int w) { return (entry >> (LVSA_ITEM_J_BITS + 2 * w)) & 3; }

template <int NS>
__global__ void __launch_bounds__(NTHREADS, 1)
lvsa_attn_sm100_ws_kernel(const __grid_constant__ CUtensorMap tmap_q,
                          const __grid_constant__ CUtensorMap tmap_k,
                          const __grid_constant__ CUtensorMap tmap_v,
                          __nv_bfloat16 *__restrict__ out, float *__restrict__ lse,
                          const int32_t *__restrict__ item_ptr, const int32_t *__restrict__ item_tiles,
                          const uint32_t *__restrict__ a_bits, int words, long long N, int P, int T,
                          int H, int n_items, long long n_work, float scale_log2) {
    using SM = Smem<NS>;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t *base_gen = smem_raw + (base - smem_u32(smem_raw));
    const uint32_t sQ = base + SM::Q_OFF, sRing = base + SM::RING_OFF, sBar = base + SM::BAR_OFF;
    auto bar = [&](int i) { return sBar + 8u * (uint32_t)i; };
    volatile uint32_t *tmem_slot_gen = reinterpret_cast<volatile uint32_t *>(base_gen + SM::TMEM_SLOT_OFF);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, wg = tid >> 7;

    if (warp == 8 && lane == 0) {
        mbar_init(bar(SM::Q_FULL), 1); mbar_init(bar(SM::Q_EMPTY), 2);
        for (int w = 0; w < 2; ++w) {
            mbar_init(bar(SM::S_FULL + w), 1); mbar_init(bar(SM::P_FULL + w), 4);
            mbar_init(bar(SM::P2_FULL + w), 4);
            mbar_init(bar(SM::O_FULL + w), 1); mbar_init(bar(SM::O_FREE + w), 4);
            mbar_init(bar(SM::TURN + w), 1);
        }
        for (int s = 0; s < NS; ++s) { mbar_init(bar(SM::KV_FULL + s), 1); mbar_init(bar(SM::KV_EMPTY + s), 2); }
        fence_barrier_init();
        prefetch_tmap(&tmap_q); prefetch_tmap(&tmap_k); prefetch_tmap(&tmap_v);
    }
    if (warp == 9) tmem_alloc<512>(base + SM::TMEM_SLOT_OFF);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_gen;

    if (wg < 2) {
        // =============================================================== softmax warpgroup `wg`
        reg_inc<208>();
        const int w = wg, rw = tid & 127;
        const uint32_t lane_off = (uint32_t)((warp & 3) * 32) << 16;
        const uint32_t tS = tmem_base + w * 128 + lane_off;
        const uint32_t tO = tmem_base + 256 + w * 128 + lane_off;
        uint32_t sc = 0, oc = 0;
        for (long long work = blockIdx.x; work < n_work; work += gridDim.x) {
            const int item = (int)(work % n_items);
            const int bh = (int)(work / n_items), h = bh % H, b = bh / H;
            const long long my_row = (long long)item * 256 + w * 128 + rw;
            const int fq = (int)min((long long)(T - 1), my_row / P);
            const uint32_t *arow = a_bits + (size_t)fq * words;
            const int e0 = item_ptr[item], e1 = item_ptr[item + 1];
            float m_run = -INFINITY, l_run = 0.f;
            int cnt = 0;
            int entry_next = (e0 < e1) ? __ldg(item_tiles + e0) : 0;
            for (int e = e0; e < e1; ++e) {
                const int entry = entry_next;
                if (e + 1 < e1) entry_next = __ldg(item_tiles + e + 1);
                const int st = entry_state(entry, w);
                if (st == LVSA_ST_SKIP) continue;
                const long long col0 = (long long)(entry & LVSA_ITEM_J_MASK) * BT;

                mbar_wait(bar(SM::S_FULL + w), sc & 1u); ++sc;
                tc_fence_after();
#ifdef LVSA_DIAG_NOSOFTMAX   // timing diagnostic only (wrong results): MMA/TMA pipeline alone
                tc_fence_before(); __syncwarp();
                if (lane == 0) { mbar_arrive(bar(SM::P_FULL + w)); mbar_arrive(bar(SM::P2_FULL + w)); }
                ++cnt; l_run = 1.f; m_run = 0.f;
                continue;
#endif
                float s[BT];
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    uint32_t r[32];
                    tmem_ld_32x32b_x32(tS + c * 32, r);
#pragma unroll
                    for (int x = 0; x < 32; ++x) s[c * 32 + x] = __uint_as_float(r[x]);
                }
                tmem_wait_ld();

                if (st == LVSA_ST_PARTIAL) {
                    uint32_t cm[4] = {0u, 0u, 0u, 0u};
                    const long long cend = min(col0 + BT, N);
                    // frame g covers tokens [g P, (g+1) P); the last frame row (the text pseudo-frame when
                    // n_text > 0, R23) runs to N
                    int g = min((int)(col0 / P), T - 1);
                    for (long long fs = (long long)g * P, fe; fs < cend; fs = fe, ++g) {
                        fe = (g == T - 1) ? N : fs + P;
                        if ((arow[g >> 5] >> (g & 31)) & 1u) {
                            const int lo = (int)(max(fs, col0) - col0), hi = (int)(min(fe, cend) - col0);
#pragma unroll
                            for (int x = 0; x < 4; ++x) cm[x] |= range_mask32(lo, hi, x);
                        }
                    }
#pragma unroll
                    for (int c = 0; c < BT; ++c)
                        if (!((cm[c >> 5] >> (c & 31)) & 1u)) s[c] = -INFINITY;
                }

                const float rm = lvsa_sm::row_max<BT>(s) * scale_log2;
                if (cnt == 0) {
                    m_run = rm;
                } else {
                    const bool grow = rm > m_run + RESCALE_THRESHOLD;
                    if (__any_sync(0xffffffffu, grow)) {
                        // PV_w of the previous tile has completed (its commit precedes S_FULL's):
                        // O_w can be rescaled in place before this tile's P is published.
                        const float corr = grow ? fast_exp2(m_run - rm) : 1.f;
                        if (grow) { m_run = rm; l_run *= corr; }
#pragma unroll
                        for (int c = 0; c < 4; ++c) {
                            uint32_t r[32];
                            tmem_ld_32x32b_x32(tO + c * 32, r);
                            tmem_wait_ld();
#pragma unroll
                            for (int x = 0; x < 32; ++x) r[x] = __float_as_uint(__uint_as_float(r[x]) * corr);
                            tmem_st_32x32b_x32(tO + c * 32, r);
                        }
                    }
                }
                const float m_use = (m_run == -INFINITY) ? 0.f : m_run;
                // P = exp2(S * scale - m) as bf16 over S's first 64 columns, published in two
                // halves so that the first four k-blocks of O += P V can start while the second
                // half of the exponentials is still being computed.
                const uint64_t scale2 = lvsa_sm::pack2(scale_log2, scale_log2);
                const uint64_t negm2 = lvsa_sm::pack2(-m_use, -m_use);
                uint64_t lsum = lvsa_sm::pack2(0.f, 0.f);
                auto publish = [&](int which) {
                    tmem_wait_st();
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) mbar_arrive(bar(which + w));
                };
                if (st == LVSA_ST_FULL) {
#pragma unroll
                    for (int c = 0; c < 4; ++c) {
                        uint32_t pk[16];
                        lvsa_sm::exp_chunk32<LVSA_POLY_PAIRS>(s, c * 32, scale2, negm2, pk, lsum);
                        tmem_st_32x32b_x16(tS + c * 16, pk);
                        if (c == 1) publish(SM::P_FULL);
                    }
                } else {   // masked logits are -inf: the MUFU path gives exact zeros
#pragma unroll
                    for (int c = 0; c < 4; ++c) {
                        uint32_t pk[16];
                        lvsa_sm::exp_chunk32<0>(s, c * 32, scale2, negm2, pk, lsum);
                        tmem_st_32x32b_x16(tS + c * 16, pk);
                        if (c == 1) publish(SM::P_FULL);
                    }
                }
                publish(SM::P2_FULL);
                {
                    float la, lb;
                    lvsa_sm::unpack2(lsum, la, lb);
                    l_run += la + lb;
                }
                ++cnt;
            }
            if (cnt > 0) {
                // epilogue: O_w / l -> bf16 -> global, lse = ln2 m + ln l
                mbar_wait(bar(SM::O_FULL + w), oc & 1u); ++oc;
                tc_fence_after();
                const bool row_ok = my_row < N;
                const float inv = 1.f / l_run;
                __nv_bfloat16 *orow = out + (((size_t)b * N + (row_ok ? my_row : 0)) * H + h) * D;
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    uint32_t r[32];
                    tmem_ld_32x32b_x32(tO + c * 32, r);
                    tmem_wait_ld();
                    uint4 *dst = reinterpret_cast<uint4 *>(orow + c * 32);
#pragma unroll
                    for (int x = 0; x < 4; ++x) {
                        uint4 v;
                        v.x = pack_bf16x2(__uint_as_float(r[8 * x + 0]) * inv, __uint_as_float(r[8 * x + 1]) * inv);
                        v.y = pack_bf16x2(__uint_as_float(r[8 * x + 2]) * inv, __uint_as_float(r[8 * x + 3]) * inv);
                        v.z = pack_bf16x2(__uint_as_float(r[8 * x + 4]) * inv, __uint_as_float(r[8 * x + 5]) * inv);
                        v.w = pack_bf16x2(__uint_as_float(r[8 * x + 6]) * inv, __uint_as_float(r[8 * x + 7]) * inv);
                        if (row_ok) dst[x] = v;
                    }
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(bar(SM::O_FREE + w));
                if (row_ok && lse != nullptr)
                    lse[((size_t)b * H + h) * N + my_row] = m_run * 0.6931471805599453f + __logf(l_run);
            }
        }
    } else {
        reg_dec<88>();
        if (warp == 8 && lane == 0) {
            // =========================================================== TMA producer
            uint32_t kv_it = 0, qi = 0;
            for (long long work = blockIdx.x; work < n_work; work += gridDim.x) {
                const int item = (int)(work % n_items);
                const int bh = (int)(work / n_items), h = bh % H, b = bh / H;
                const long long row0 = (long long)item * 256;
                const int e0 = item_ptr[item], e1 = item_ptr[item + 1];
                mbar_wait(bar(SM::Q_EMPTY), (qi & 1u) ^ 1u);
                const int nload = (row0 + 128 >= N) ? 1 : 2;
                mbar_expect_tx(bar(SM::Q_FULL), nload * TILE_BYTES);
                for (int w = 0; w < nload; ++w)
                    for (int hh = 0; hh < 2; ++hh)
                        tma_load_4d(sQ + w * TILE_BYTES + hh * HALF_BYTES, &tmap_q, bar(SM::Q_FULL), hh * 64, h,
                                    (int)(row0 + w * 128), b);
                ++qi;
                int entry_next = (e0 < e1) ? __ldg(item_tiles + e0) : 0;
                for (int e = e0; e < e1; ++e) {
                    const int entry = entry_next;
                    if (e + 1 < e1) entry_next = __ldg(item_tiles + e + 1);
                    const int col0 = (entry & LVSA_ITEM_J_MASK) * BT;
#pragma unroll
                    for (int t = 0; t < 2; ++t) {   // t = 0: K_j, t = 1: V_j
                        const uint32_t stage = kv_it % NS, n = kv_it / NS;
                        mbar_wait(bar(SM::KV_EMPTY + stage), (n & 1u) ^ 1u);
                        mbar_expect_tx(bar(SM::KV_FULL + stage), TILE_BYTES);
                        const uint32_t dst = sRing + stage * TILE_BYTES;
                        const CUtensorMap *tm = t == 0 ? &tmap_k : &tmap_v;
                        tma_load_4d(dst, tm, bar(SM::KV_FULL + stage), 0, h, col0, b);
                        tma_load_4d(dst + HALF_BYTES, tm, bar(SM::KV_FULL + stage), 64, h, col0, b);
                        ++kv_it;
                    }
                }
            }
        } else if (warp == 9 || warp == 10) {
            // =========================================================== MMA issuers
            // One issuing warp per q tile (w = 0: warp 9, w = 1: warp 10).  A single warp issuing all
            // 32 MMAs of a kv tile plus their descriptor moves was itself the limiter (measured with
            // the softmax disabled: tensor pipe 73 % busy, issuer never idle).  The two chains
            // softmax_w -> PV_w -> S_w are independent; they only share the K/V ring and Q, whose
            // "empty" barriers therefore take one commit from each issuer.
            // The whole warp runs the control flow (waits included); one elected lane issues.
            // Under elect.sync the compiler keeps descriptors in uniform registers with no
            // per-lane waterfall around every tcgen05.mma.
            const int w = warp - 9;
            constexpr uint32_t IDESC_S = umma_idesc_bf16(128, BT, 0);
            constexpr uint32_t IDESC_O = umma_idesc_bf16(128, D, 1);
            const uint64_t dQ = umma_smem_desc_sw128(sQ + w * TILE_BYTES, 16);
            const uint64_t dRingK = umma_smem_desc_sw128(sRing, 16);
            const uint64_t dRingV = umma_smem_desc_sw128(sRing, HALF_BYTES);
            const uint32_t tS = tmem_base + w * 128, tO = tmem_base + 256 + w * 128;
            auto issue_S = [&](uint32_t stageK) {
#pragma unroll
                for (int kk = 0; kk < 8; ++kk) {
                    const uint32_t off = (uint32_t)((kk >> 2) * HALF_BYTES + (kk & 3) * 32) >> 4;
                    umma_ss(tS, dQ + (uint64_t)off, dRingK + (uint64_t)(((stageK * TILE_BYTES) >> 4) + off),
                            IDESC_S, kk > 0);
                }
                umma_commit(bar(SM::S_FULL + w));
            };
            auto issue_PV = [&](uint32_t stageV, bool accumulate, int half) {
#pragma unroll
                for (int kk = 4 * half; kk < 4 * half + 4; ++kk)
                    umma_ts(tO, tS + kk * 8, dRingV + (uint64_t)(((stageV * TILE_BYTES) >> 4) + ((kk * 2048) >> 4)),
                            IDESC_O, (accumulate || kk > 0) ? 1u : 0u);
            };
            uint32_t kv_it = 0, qi = 0, pc = 0, oc = 0, turn = 0;
            for (long long work = blockIdx.x; work < n_work; work += gridDim.x) {
                const int item = (int)(work % n_items);
                const int e0 = __shfl_sync(0xffffffffu, __ldg(item_ptr + item), 0);
                const int e1 = __shfl_sync(0xffffffffu, __ldg(item_ptr + item + 1), 0);
                if (e0 == e1) continue;   // cannot happen (t in A(t)), kept for symmetry with the producer
                bool started = false;
                mbar_wait(bar(SM::Q_FULL), qi & 1u); ++qi;
                int entry = __shfl_sync(0xffffffffu, __ldg(item_tiles + e0), 0);
                {   // S(0)
                    const uint32_t stageK = kv_it % NS, n = kv_it / NS;
                    mbar_wait(bar(SM::KV_FULL + stageK), n & 1u);
                    tc_fence_after();
                    if (elect_one_sync()) {
                        if (entry_state(entry, w) != LVSA_ST_SKIP) issue_S(stageK);
                        umma_commit(bar(SM::KV_EMPTY + stageK));
                    }
                    __syncwarp();
                    ++kv_it;
                }
                for (int e = e0; e < e1; ++e) {
                    const bool has_next = e + 1 < e1;
                    const int entry_n = has_next ? __shfl_sync(0xffffffffu, __ldg(item_tiles + e + 1), 0) : 0;
                    const uint32_t stageV = kv_it % NS, nV = kv_it / NS;
                    ++kv_it;
                    uint32_t stageK = 0, nK = 0;
                    if (has_next) { stageK = kv_it % NS; nK = kv_it / NS; ++kv_it; }
                    const bool do_pv = entry_state(entry, w) != LVSA_ST_SKIP;
                    const bool do_s = has_next && entry_state(entry_n, w) != LVSA_ST_SKIP;
                    // Q_w is last read by the S MMAs of the final tile, all issued by now
                    if (!has_next && elect_one_sync()) umma_commit(bar(SM::Q_EMPTY));
                    __syncwarp();
                    // Both issuers wait for every stage, used or not: a stage's KV_EMPTY takes one
                    // commit from each, so neither may run a whole ring ahead of the other.
                    mbar_wait(bar(SM::KV_FULL + stageV), nV & 1u);
#ifndef LVSA_NO_TURNS
                    // The issuers take turns, q tile 0 first: that keeps the two softmax warpgroups
                    // half a period apart, so each has the MUFU to itself while the tensor pipe
                    // works for the other (left to themselves the two chains fall into step and the
                    // exponentials of both q tiles collide: measured 40 ms instead of 35 ms).
                    mbar_wait(bar(SM::TURN + w), (turn & 1u) ^ (w == 0 ? 1u : 0u));
                    ++turn;
#endif
                    if (do_pv) {
                        if (!started) mbar_wait(bar(SM::O_FREE + w), (oc & 1u) ^ 1u);
                        mbar_wait(bar(SM::P_FULL + w), pc & 1u);
                        tc_fence_after();
                        if (elect_one_sync()) issue_PV(stageV, started, 0);
                        __syncwarp();
                        mbar_wait(bar(SM::P2_FULL + w), pc & 1u);
                        ++pc;
                        tc_fence_after();
                    }
                    if (has_next) {
                        mbar_wait(bar(SM::KV_FULL + stageK), nK & 1u);
                        tc_fence_after();
                    }
                    if (elect_one_sync()) {
                        if (do_pv) issue_PV(stageV, started, 1);
                        if (do_s) issue_S(stageK);
                        // a stage this issuer never read (skipped q tile) is released at once
                        umma_commit(bar(SM::KV_EMPTY + stageV));
                        if (has_next) umma_commit(bar(SM::KV_EMPTY + stageK));
#ifndef LVSA_NO_TURNS
                        mbar_arrive(bar(SM::TURN + (w ^ 1)));
#endif
                    }
                    __syncwarp();
                    started |= do_pv;
                    entry = entry_n;
                }
                if (started) {
                    if (elect_one_sync()) umma_commit(bar(SM::O_FULL + w));
                    __syncwarp();
                    ++oc;
                }
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 9) tmem_dealloc<512>(tmem_base);
}

}  // namespace

// host side -------------------------------------------------------------------------------
lvsa_status_t lvsa_make_tmap_bf16(CUtensorMap *m, const void *base, long long N, int H, int d, int B,
                                  int box_rows);

// One-time setup (opt-in shared memory size, SM count), kept out of the launch path so that a
// launch is nothing but tensor-map encoding and the launch itself (CUDA-graph capturable).
static int g_n_sm = 0;
lvsa_status_t lvsa_attn_sm100_ws_prepare(int device) {
    if (g_n_sm != 0) return LVSA_OK;
    using SM = Smem<5>;
    LVSA_CUDA_TRY(cudaFuncSetAttribute(lvsa_attn_sm100_ws_kernel<5>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                       SM::BYTES));
    int n = 0;
    LVSA_CUDA_TRY(cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, device));
    g_n_sm = n;
    return LVSA_OK;
}

lvsa_status_t lvsa_attn_sm100_ws_launch(const lvsa_index *ix, const void *q, const void *k, const void *v,
                                        void *out, float *lse, cudaStream_t stream) {
    constexpr int NS = 5;
    using SM = Smem<NS>;
    CUtensorMap mq, mk, mv;
    lvsa_status_t st;
    if ((st = lvsa_make_tmap_bf16(&mq, q, ix->N, ix->p.H, D, ix->p.B, 128)) != LVSA_OK) return st;
    if ((st = lvsa_make_tmap_bf16(&mk, k, ix->N, ix->p.H, D, ix->p.B, BT)) != LVSA_OK) return st;
    if ((st = lvsa_make_tmap_bf16(&mv, v, ix->N, ix->p.H, D, ix->p.B, BT)) != LVSA_OK) return st;
    auto kern = lvsa_attn_sm100_ws_kernel<NS>;
    if ((st = lvsa_attn_sm100_ws_prepare(ix->device)) != LVSA_OK) return st;
    const int n_sm = g_n_sm;
    const long long n_work = (long long)ix->n_items * ix->p.H * ix->p.B;
    const int grid = (int)(n_work < n_sm ? n_work : n_sm);
    const float scale_log2 = ix->p.softmax_scale * 1.4426950408889634f;
    kern<<<grid, NTHREADS, SM::BYTES, stream>>>(
        mq, mk, mv, (__nv_bfloat16 *)out, lse, ix->d_item_ptr, ix->d_item_tiles, ix->d_abits, ix->words,
        (long long)ix->N, ix->p.P, ix->Tf, ix->p.H, (int)ix->n_items, n_work, scale_log2);
    LVSA_CUDA_TRY(cudaGetLastError());
    return LVSA_OK;
}
