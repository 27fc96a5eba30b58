// CTA-pair LVSA attention forward for sm_100a (d = 128, 128 x 128 tiles): one cluster of two CTAs
// per work item (pair of adjacent q tiles), tcgen05.mma.cta_group::2 with M = 256 across the pair.
//
// Computes Eq. 2 over the kept kv tiles listed by the block index, like
// lvsa_attn_sm100_ws.cu; what changes is where the operands and accumulators live:
//   * CTA r of the pair owns q tile r of the item: its 128 rows of Q (shared memory), of S / P and
//     of O (its own TMEM).  Every MMA is one instruction for both CTAs, issued by the leader (CTA 0).
//   * B operands are split over the pair: CTA r loads kv rows [64 r, 64 r + 64) of K_j (the N
//     extent of S = Q K^T) and channels [64 r, 64 r + 64) of V_j (the N extent of O += P V), 16 KB
//     each instead of 32 KB; the tensor cores read both halves from both shared memories.
//   * with one q tile per CTA, TMEM holds TWO S/P buffers and O (384 of 512 columns): S(j+1) is
//     computed while the softmax of tile j runs, which removes the serial chain
//     softmax(j) -> PV(j) -> S(j+1) -> softmax(j+1) that bounds the one-CTA kernel.
// Roles per CTA (12 warps): warps 0-3 / 4-7 softmax warpgroups for kv columns [0,64) / [64,128) of
// every tile (two threads per query row; the row maximum is exchanged through shared memory),
// warp 8 TMA producer, warp 9 MMA issuer (leader CTA only), warps 10-11 idle.
//
// Cross-CTA signalling: TMA completions of both CTAs are counted on the leader's FULL barriers
// (cta_group::2 loads); tcgen05.commit multicasts MMA completions to the barriers of both CTAs;
// the peer's softmax warps arrive remotely on the leader's P barriers.
#include <cuda.h>
#include <cuda_bf16.h>

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
#ifndef LVSA_POLY_PAIRS
#define LVSA_POLY_PAIRS 0
#endif
#ifndef LVSA_PAIR_STAGES
#define LVSA_PAIR_STAGES 10
#endif

template <int NS>
struct SmemP {
    static constexpr int Q_OFF = 0;                            // 32 KB
    static constexpr int RING_OFF = TILE_BYTES;                // NS x 16 KB
    static constexpr int BAR_OFF = RING_OFF + NS * STAGE_BYTES;
    // barriers (8 B each).  "L": only the leader's copy is used (arrivals come from both CTAs).
    static constexpr int Q_FULL = 0 /*L*/, Q_EMPTY = 1, S_FULL = 2 /*2*/, PA_FULL = 4 /*2, L*/, PB_FULL = 6 /*2, L*/,
                         PV_DONE = 8, O_FULL = 9, O_FREE = 10 /*L*/, KV_FULL = 11 /*NS, L*/, KV_EMPTY = 11 + NS /*NS*/,
                         NBARS = 11 + 2 * NS;
    static constexpr int TMEM_SLOT_OFF = BAR_OFF + 8 * NBARS;
    static constexpr int XCH_OFF = TMEM_SLOT_OFF + 16;         // float [2 halves][128 rows]
    static constexpr int BYTES = XCH_OFF + 2 * 128 * 4;
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
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(NTHREADS, 1)
lvsa_attn_sm100_pair_kernel(const __grid_constant__ CUtensorMap tmap_q,
                            const __grid_constant__ CUtensorMap tmap_k,   // box 64 rows
                            const __grid_constant__ CUtensorMap tmap_v,   // box 128 rows
                            __nv_bfloat16 *__restrict__ out, float *__restrict__ lse,
                            const int32_t *__restrict__ item_ptr, const int32_t *__restrict__ item_tiles,
                            const uint32_t *__restrict__ a_bits, int words, long long N, int P, int T,
                            int H, int n_items, long long n_work, float scale_log2) {
    using SM = SmemP<NS>;
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    const uint32_t base = smem_u32(smem_raw);
    if ((base & 1023u) != 0u) __trap();   // SWIZZLE_128B tiles and UMMA descriptors need 1024 B
    uint8_t *base_gen = smem_raw;
    const uint32_t sQ = base + SM::Q_OFF, sRing = base + SM::RING_OFF, sBar = base + SM::BAR_OFF;
    auto bar = [&](int i) { return sBar + 8u * (uint32_t)i; };
    volatile uint32_t *tmem_slot_gen = reinterpret_cast<volatile uint32_t *>(base_gen + SM::TMEM_SLOT_OFF);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, wg = tid >> 7;
    const uint32_t rank = cluster_ctarank();           // 0 = leader; also the q tile of the item I own
    const long long pair = blockIdx.x >> 1, n_pairs = gridDim.x >> 1;

    if (warp == 8 && lane == 0) {
        mbar_init(bar(SM::Q_FULL), 1); mbar_init(bar(SM::Q_EMPTY), 1);
        for (int b = 0; b < 2; ++b) {
            mbar_init(bar(SM::S_FULL + b), 1);
            mbar_init(bar(SM::PA_FULL + b), 8);     // 4 warps x 2 CTAs
            mbar_init(bar(SM::PB_FULL + b), 8);
        }
        mbar_init(bar(SM::PV_DONE), 1); mbar_init(bar(SM::O_FULL), 1);
        mbar_init(bar(SM::O_FREE), 16);             // 8 warps x 2 CTAs
        for (int s = 0; s < NS; ++s) { mbar_init(bar(SM::KV_FULL + s), 1); mbar_init(bar(SM::KV_EMPTY + s), 1); }
        fence_barrier_init();
        prefetch_tmap(&tmap_q); prefetch_tmap(&tmap_k); prefetch_tmap(&tmap_v);
    }
    if (warp == 9) tmem_alloc_pair<512>(base + SM::TMEM_SLOT_OFF);
    tc_fence_before();
    cluster_sync_all();                                // barrier inits and TMEM visible in both CTAs
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_gen;
