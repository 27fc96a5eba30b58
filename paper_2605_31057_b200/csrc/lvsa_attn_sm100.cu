// Block-sparse LVSA attention forward for sm_100a: TMA -> swizzled smem -> tcgen05.mma with TMEM
// accumulators -> online exp2 softmax -> P (bf16) back into TMEM -> tcgen05.mma O += P V.
// Computes Eq. 2 over the kept kv tiles of the block index, with element-level
// masking on PARTIAL tiles (frame(k) in A(frame(q)) and k < N) and LSE output.
//
// Work item = a group of adjacent q tiles covering 128 * NWG query rows that share every K/V
// tile load (tile 128: two q tiles, two warpgroups; tile 64: two q tiles in one warpgroup).
// Each softmax thread owns one query row: TMEM lane = row, columns = kv positions.
//
// This file holds kernel "v0" (bring-up: one role at a time, every step fenced by a CTA
// barrier) and is the reference point for the pipelined kernel.  See DESIGN.md "Kernels".
#include <cuda.h>
#include <cuda_bf16.h>

#include "lvsa_internal.h"
#include "sm100_ptx.cuh"

using namespace sm100;

namespace {

template <int D, int BT>
struct Cfg {
    static constexpr int NWG = (BT == 128) ? 2 : 1;        // warpgroups; each owns 128 query rows
    static constexpr int ROWS = 128 * NWG;                 // query rows per work item (= 2 q tiles)
    static constexpr int HALVES = D / 64;                  // 128-byte swizzle spans per row
    static constexpr int Q_HALF_BYTES = 128 * 128;         // [128 rows][128 B]
    static constexpr int Q_WG_BYTES = Q_HALF_BYTES * HALVES;
    static constexpr int KV_HALF_BYTES = BT * 128;         // [BT rows][128 B]
    static constexpr int KV_BYTES = KV_HALF_BYTES * HALVES;
    static constexpr int S_COLS = BT, O_COLS = D;
    static constexpr int TMEM_COLS = NWG * (S_COLS + O_COLS);   // 512 / 128
    static constexpr int SMEM_DATA = NWG * Q_WG_BYTES + 2 * KV_BYTES;
    static constexpr int SMEM_BYTES = SMEM_DATA + 1024 /*align*/ + 128 /*barriers*/;
    static_assert(TMEM_COLS == 512 || TMEM_COLS == 128, "TMEM allocation must be a power of two");
};

__device__ __forceinline__ uint32_t range_mask32(int lo, int hi, int w) {
    // bits of [lo, hi) that fall into word w
    const int a = max(lo, 32 * w), b = min(hi, 32 * w + 32);
    if (a >= b) return 0u;
    const int n = b - a;
    return (n == 32 ? 0xffffffffu : ((1u << n) - 1u)) << (a - 32 * w);
}

template <int D, int BT>
__global__ void __launch_bounds__(Cfg<D, BT>::NWG * 128, 1)
lvsa_attn_sm100_v0_kernel(const __grid_constant__ CUtensorMap tmap_q,
                          const __grid_constant__ CUtensorMap tmap_k,
                          const __grid_constant__ CUtensorMap tmap_v,
                          __nv_bfloat16 *__restrict__ out, float *__restrict__ lse,
                          const int32_t *__restrict__ item_ptr, const int32_t *__restrict__ item_tiles,
                          const uint32_t *__restrict__ a_bits, int words, long long N, int P, int T,
                          int H, long long sn, long long sh, long long sb, float scale_log2) {
    using C = Cfg<D, BT>;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t sQ = smem_base;                                  // [NWG][HALVES][128][128 B]
    const uint32_t sK = sQ + C::NWG * C::Q_WG_BYTES;                // [HALVES][BT][128 B]
    const uint32_t sV = sK + C::KV_BYTES;
    const uint32_t sBar = sV + C::KV_BYTES;
    const uint32_t bar_q = sBar, bar_kv = sBar + 8, bar_s = sBar + 16, bar_o = sBar + 24;
    const uint32_t tmem_slot = sBar + 32;
    uint8_t *smem_gen = smem_raw + (smem_base - smem_u32(smem_raw));
    volatile uint32_t *tmem_slot_gen = reinterpret_cast<volatile uint32_t *>(smem_gen + C::SMEM_DATA + 32);

    const int item = blockIdx.x, h = blockIdx.y, b = blockIdx.z;
    const int tid = threadIdx.x, warp = tid >> 5, wg = tid >> 7, rw = tid & 127;
    // an index whose build overflowed its allocation bound has unfilled lists and a poisoned end (lvsa_index.cu)
    if (tid == 0 && item_ptr[gridDim.x] < 0) __trap();

    if (warp == 0) tmem_alloc<C::TMEM_COLS>(tmem_slot);
    if (tid == 32) {
        mbar_init(bar_q, 1); mbar_init(bar_kv, 1); mbar_init(bar_s, 1); mbar_init(bar_o, 1);
        fence_barrier_init();
        prefetch_tmap(&tmap_q); prefetch_tmap(&tmap_k); prefetch_tmap(&tmap_v);
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_gen;
    const uint32_t lane_off = (uint32_t)((warp & 3) * 32) << 16;
    const uint32_t tS = tmem_base + wg * C::S_COLS;                     // S (fp32) / P (bf16) of my WG
    const uint32_t tO = tmem_base + C::NWG * C::S_COLS + wg * C::O_COLS;

    const long long row0 = (long long)item * C::ROWS;
    if (tid == 0) {
        // a warpgroup whose first row is past N has no q tile (odd nq): nothing to load for it
        const int nload = (C::NWG == 2 && row0 + 128 >= N) ? 1 : C::NWG;
        mbar_expect_tx(bar_q, nload * C::Q_WG_BYTES);
        for (int w = 0; w < nload; ++w)
            for (int hh = 0; hh < C::HALVES; ++hh)
                tma_load_4d(sQ + w * C::Q_WG_BYTES + hh * C::Q_HALF_BYTES, &tmap_q, bar_q, hh * 64, h,
                            (int)(row0 + w * 128), b);
    }

    const long long my_row = row0 + wg * 128 + rw;
    const int my_qt = (BT == 128) ? wg : (rw >> 6);                    // which q tile of the item
    const int fq = (int)min((long long)(T - 1), my_row / P);
    const uint32_t *arow = a_bits + (size_t)fq * words;

    constexpr uint32_t IDESC_S = umma_idesc_bf16(128, BT, 0);
    constexpr uint32_t IDESC_O = umma_idesc_bf16(128, D, 1);

    float m_run = -INFINITY, l_run = 0.f;
    bool started = false;     // has my WG's O accumulator been written yet (WG-uniform)
    bool started_w[2] = {false, false};

    const int e0 = item_ptr[item], e1 = item_ptr[item + 1];
    mbar_wait(bar_q, 0);

    for (int e = e0; e < e1; ++e) {
        const uint32_t ph = (uint32_t)(e - e0) & 1u;
        const int entry = item_tiles[e];
        const int j = entry & LVSA_ITEM_J_MASK;
        const int st0 = (entry >> LVSA_ITEM_J_BITS) & 3, st1 = (entry >> (LVSA_ITEM_J_BITS + 2)) & 3;
        const bool act_w[2] = {(BT == 128) ? (st0 != LVSA_ST_SKIP) : true,
                               (BT == 128) ? (st1 != LVSA_ST_SKIP) : false};
        const bool wg_active = act_w[wg];
        const int st_row = my_qt == 0 ? st0 : st1;
        const long long col0 = (long long)j * BT;

        if (tid == 0) {
            mbar_expect_tx(bar_kv, 2 * C::KV_BYTES);
            for (int hh = 0; hh < C::HALVES; ++hh) {
                tma_load_4d(sK + hh * C::KV_HALF_BYTES, &tmap_k, bar_kv, hh * 64, h, (int)col0, b);
                tma_load_4d(sV + hh * C::KV_HALF_BYTES, &tmap_v, bar_kv, hh * 64, h, (int)col0, b);
            }
            mbar_wait(bar_kv, ph);
            tc_fence_after();
            for (int w = 0; w < C::NWG; ++w) {
                if (!act_w[w]) continue;
#pragma unroll
                for (int kk = 0; kk < D / 16; ++kk) {
                    const uint32_t off = (kk >> 2) * C::Q_HALF_BYTES + (kk & 3) * 32;
                    const uint32_t offk = (kk >> 2) * C::KV_HALF_BYTES + (kk & 3) * 32;
                    umma_ss(tmem_base + w * C::S_COLS,
                            umma_smem_desc_sw128(sQ + w * C::Q_WG_BYTES + off, 16),
                            umma_smem_desc_sw128(sK + offk, 16), IDESC_S, kk > 0);
                }
            }
            umma_commit(bar_s);
        }
        mbar_wait(bar_s, ph);
        tc_fence_after();

        if (wg_active) {
            float s[BT];
#pragma unroll
            for (int c = 0; c < BT / 32; ++c) {
                uint32_t r[32];
                tmem_ld_32x32b_x32(tS + lane_off + c * 32, r);
#pragma unroll
                for (int x = 0; x < 32; ++x) s[c * 32 + x] = __uint_as_float(r[x]);
            }
            tmem_wait_ld();
            if (st_row != LVSA_ST_FULL) {
                uint32_t cm[BT / 32];
#pragma unroll
                for (int w = 0; w < BT / 32; ++w) cm[w] = 0u;
                if (st_row == LVSA_ST_PARTIAL) {
                    const long long cend = min(col0 + BT, N);
                    // frame g covers tokens [g P, (g+1) P); the last frame row (the text pseudo-frame when
                    // n_text > 0, R23) runs to N
                    int g = min((int)(col0 / P), T - 1);
                    for (long long fs = (long long)g * P, fe; fs < cend; fs = fe, ++g) {
                        fe = (g == T - 1) ? N : fs + P;
                        if ((arow[g >> 5] >> (g & 31)) & 1u) {
                            const int lo = (int)(max(fs, col0) - col0);
                            const int hi = (int)(min(fe, cend) - col0);
#pragma unroll
                            for (int w = 0; w < BT / 32; ++w) cm[w] |= range_mask32(lo, hi, w);
                        }
                    }
                }
#pragma unroll
                for (int c = 0; c < BT; ++c)
                    if (!((cm[c >> 5] >> (c & 31)) & 1u)) s[c] = -INFINITY;
            }
            float mx = s[0];
#pragma unroll
            for (int c = 1; c < BT; ++c) mx = fmaxf(mx, s[c]);
            const float m_new = fmaxf(m_run, mx * scale_log2);
            const float m_use = (m_new == -INFINITY) ? 0.f : m_new;
            const float corr = fast_exp2(m_run - m_use);
            float lsum = 0.f;
#pragma unroll
            for (int c = 0; c < BT / 32; ++c) {
                uint32_t pk[16];
#pragma unroll
                for (int x = 0; x < 16; ++x) {
                    const float p0 = fast_exp2(fmaf(s[c * 32 + 2 * x], scale_log2, -m_use));
                    const float p1 = fast_exp2(fmaf(s[c * 32 + 2 * x + 1], scale_log2, -m_use));
                    lsum += p0 + p1;
                    pk[x] = pack_bf16x2(p0, p1);
                }
                tmem_st_32x32b_x16(tS + lane_off + c * 16, pk);
            }
            l_run = l_run * corr + lsum;
            const bool need = __any_sync(0xffffffffu, m_new > m_run) && started;
            if (need) {
#pragma unroll
                for (int c = 0; c < D / 32; ++c) {
                    uint32_t r[32];
                    tmem_ld_32x32b_x32(tO + lane_off + c * 32, r);
                    tmem_wait_ld();
#pragma unroll
                    for (int x = 0; x < 32; ++x) r[x] = __float_as_uint(__uint_as_float(r[x]) * corr);
                    tmem_st_32x32b_x32(tO + lane_off + c * 32, r);
                }
            }
            m_run = m_new;
            tmem_wait_st();
        }
        tc_fence_before();
        __syncthreads();
        if (tid == 0) {
            tc_fence_after();
            for (int w = 0; w < C::NWG; ++w) {
                if (!act_w[w]) continue;
#pragma unroll
                for (int kk = 0; kk < BT / 16; ++kk) {
                    umma_ts(tmem_base + C::NWG * C::S_COLS + w * C::O_COLS,
                            tmem_base + w * C::S_COLS + kk * 8,
                            umma_smem_desc_sw128(sV + kk * 2048, C::KV_HALF_BYTES), IDESC_O,
                            (started_w[w] || kk > 0) ? 1u : 0u);
                }
            }
            umma_commit(bar_o);
        }
        started_w[0] |= act_w[0]; started_w[1] |= act_w[1];
        started = started_w[wg];
        mbar_wait(bar_o, ph);
        tc_fence_after();
    }

    // epilogue: O / l -> bf16 -> global; lse = ln2 * m + ln l.  The TMEM loads are warp-collective,
    // so rows >= N of a tail tile load too and only skip the stores.
    if (started) {
        const bool row_ok = my_row < N;
        const float inv = 1.f / l_run;
        __nv_bfloat16 *orow = out + (size_t)b * sb + (size_t)(row_ok ? my_row : 0) * sn + (size_t)h * sh;
#pragma unroll
        for (int c = 0; c < D / 32; ++c) {
            uint32_t r[32];
            tmem_ld_32x32b_x32(tO + lane_off + c * 32, r);
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
        if (row_ok && lse != nullptr)
            lse[((size_t)b * H + h) * N + my_row] = m_run * 0.6931471805599453f + __logf(l_run);
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc<C::TMEM_COLS>(tmem_base);
}

// ------------------------------------------------------------------------------------ host
typedef CUresult (*PFN_encodeTiled)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *,
                                    const cuuint64_t *, const cuuint64_t *, const cuuint32_t *,
                                    const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                    CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

PFN_encodeTiled get_encode() {
    static PFN_encodeTiled fn = nullptr;
    if (fn == nullptr) {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = (PFN_encodeTiled)p;
    }
    return fn;
}

}  // namespace

// bf16 tensor with axes (d, H, N, B), d contiguous; element strides of the token / head / batch axes
// from lvsa_layout_strides (NHD or HND).  Tensor-map dims (fastest first): d, H, N, B whatever the
// memory order (TMA strides need not be sorted).  Box: 64 x 1 x rows x 1 with SWIZZLE_128B, i.e.
// smem tile [rows][128 B]; rows >= N are zero-filled.
lvsa_status_t lvsa_make_tmap_bf16(CUtensorMap *m, const void *base, const lvsa_index *ix, int box_rows, int which) {
    const long long N = ix->N;
    const int H = ix->p.H, d = ix->p.d, B = ix->p.B;
    const lvsa_strides sd = lvsa_tensor_strides(ix, which);   // LVSA_T_Q / K / V / OUT
    PFN_encodeTiled enc = get_encode();
    if (enc == nullptr) { lvsa_set_error("cuTensorMapEncodeTiled entry point not found"); return LVSA_ECUDA; }
    cuuint64_t dims[4] = {(cuuint64_t)d, (cuuint64_t)H, (cuuint64_t)N, (cuuint64_t)B};
    cuuint64_t strides[3] = {(cuuint64_t)sd.h * 2, (cuuint64_t)sd.n * 2, (cuuint64_t)sd.b * 2};
    cuuint32_t box[4] = {64, 1, (cuuint32_t)box_rows, 1};
    cuuint32_t estr[4] = {1, 1, 1, 1};
    CUresult r = enc(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4, const_cast<void *>(base), dims, strides, box, estr,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                     CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        lvsa_set_error("cuTensorMapEncodeTiled failed with CUresult " + std::to_string((int)r));
        return LVSA_ECUDA;
    }
    return LVSA_OK;
}

namespace {

template <int D, int BT>
lvsa_status_t launch_v0(const lvsa_index *ix, const void *q, const void *k, const void *v, void *out,
                        float *lse, cudaStream_t stream) {
    using C = Cfg<D, BT>;
    CUtensorMap mq, mk, mv;
    lvsa_status_t st;
    if ((st = lvsa_make_tmap_bf16(&mq, q, ix, 128, LVSA_T_Q)) != LVSA_OK) return st;
    if ((st = lvsa_make_tmap_bf16(&mk, k, ix, BT, LVSA_T_K)) != LVSA_OK) return st;
    if ((st = lvsa_make_tmap_bf16(&mv, v, ix, BT, LVSA_T_V)) != LVSA_OK) return st;
    auto kern = lvsa_attn_sm100_v0_kernel<D, BT>;
    // the attribute is per device: set once per (instantiation, device)
    static bool ready[LVSA_MAX_DEVICES] = {};
    if (!ready[ix->device]) {
        LVSA_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES));
        ready[ix->device] = true;
    }
    const float scale_log2 = ix->p.softmax_scale * 1.4426950408889634f;
    const lvsa_strides sd = lvsa_tensor_strides(ix, LVSA_T_OUT);   // the kernel stores `out` with plain stores
    dim3 grid((unsigned)ix->n_items, ix->p.H, ix->p.B);
    kern<<<grid, C::NWG * 128, C::SMEM_BYTES, stream>>>(
        mq, mk, mv, (__nv_bfloat16 *)out, lse, ix->d_item_ptr, ix->d_item_tiles, ix->d_abits, ix->words,
        (long long)ix->N, ix->p.P, ix->Tf, ix->p.H, sd.n, sd.h, sd.b, scale_log2);
    LVSA_CUDA_TRY(cudaGetLastError());
    return LVSA_OK;
}

}  // namespace

int lvsa_attn_sm100_supported(const lvsa_index *ix) {
    // compute-capability major per device, queried once (cudaGetDeviceProperties costs milliseconds
    // and this runs in every index build)
    static int cc_major[LVSA_MAX_DEVICES] = {};
    const int dev = ix->device;
    if (dev < 0 || dev >= LVSA_MAX_DEVICES) return 0;
    if (cc_major[dev] == 0) {
        int v = 0;
        if (cudaDeviceGetAttribute(&v, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) return 0;
        cc_major[dev] = v;
    }
    if (cc_major[dev] != 10) return 0;
    return (ix->p.d == 128 && ix->p.tile_q == 128) || (ix->p.d == 64 && ix->p.tile_q == 64);
}

// d = 128: the CTA-pair kernel unless the index asks for the one-CTA-per-item kernel
int lvsa_attn_uses_pair_kernel(const lvsa_index *ix) {
    return ix->p.d == 128 && ix->p.kernel != LVSA_KERNEL_TCGEN05_V0;
}

lvsa_status_t lvsa_attn_sm100_launch(const lvsa_index *ix, const void *q, const void *k,
                                     const void *v, void *out, float *lse, cudaStream_t stream) {
    if (ix->p.H > 65535 || ix->p.B > 65535) {
        lvsa_set_error("tcgen05 kernel: H and B must be <= 65535");
        return LVSA_EUNSUPPORTED;
    }
    if (ix->p.d == 128) {
        if (lvsa_attn_uses_pair_kernel(ix)) return lvsa_attn_sm100_pair_launch(ix, q, k, v, out, lse, stream);
        return launch_v0<128, 128>(ix, q, k, v, out, lse, stream);
    }
    return launch_v0<64, 64>(ix, q, k, v, out, lse, stream);
}
