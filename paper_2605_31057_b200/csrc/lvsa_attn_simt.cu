// SIMT fp32 attention forward over the block index (bring-up / fp32 path).
// Computes Eq. 2 with every product and sum in fp32 on the CUDA cores; consumes
// the CSR + FULL/PARTIAL flags + A(t) bitsets exactly as the tensor-core kernel does, so index
// semantics, element masking and LSE can be checked with a tight tolerance.  It is the kernel
// behind LVSA_DTYPE_FP32 and an in-repo GPU cross-check for the tcgen05 kernel.
//
// One CTA per (q tile, head, batch); 8 warps; warp w owns rows w, w+8, ... of the tile.  A kv
// tile is staged in shared memory as fp32; lane c scores key c of each 32-key chunk (full
// d-length dot product), the chunk is folded into the row's online softmax with warp shuffles,
// and lane l accumulates output channels l, l+32, ...
#include <cuda_bf16.h>

#include "lvsa_internal.h"

namespace {

template <typename T> __device__ __forceinline__ float to_f32(T x);
template <> __device__ __forceinline__ float to_f32<float>(float x) { return x; }
template <> __device__ __forceinline__ float to_f32<__nv_bfloat16>(__nv_bfloat16 x) { return __bfloat162float(x); }
template <typename T> __device__ __forceinline__ T from_f32(float x);
template <> __device__ __forceinline__ float from_f32<float>(float x) { return x; }
template <> __device__ __forceinline__ __nv_bfloat16 from_f32<__nv_bfloat16>(float x) { return __float2bfloat16_rn(x); }

constexpr int SIMT_WARPS = 8;

template <int D, int BT, typename T>
__global__ void __launch_bounds__(SIMT_WARPS * 32)
lvsa_attn_simt_kernel(const T *__restrict__ q, const T *__restrict__ k, const T *__restrict__ v,
                      T *__restrict__ out, float *__restrict__ lse,
                      const int32_t *__restrict__ indptr, const int32_t *__restrict__ indices,
                      const uint8_t *__restrict__ flags, const uint32_t *__restrict__ a_bits,
                      int words, long long N, int P, int Tf, int H, lvsa_strides sq, lvsa_strides sk, lvsa_strides sv,
                      lvsa_strides so, int aligned, int Tv, float scale) {
    constexpr int R = BT / SIMT_WARPS;  // rows per warp
    constexpr int CH = D / 32;          // output channels per lane
    constexpr int KS = D + 1;           // padded K row (lane c reads row c: conflict-free)
    extern __shared__ float smem[];
    float *Qs = smem;                   // [BT][D]
    float *Ks = Qs + BT * D;            // [BT][D+1]
    float *Vs = Ks + BT * KS;           // [BT][D]
    const int i = blockIdx.x, h = blockIdx.y, b = blockIdx.z;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    // an index whose build overflowed its allocation bound has unfilled lists and a poisoned end (lvsa_index.cu)
    if (tid == 0 && indptr[gridDim.x] < 0) __trap();
    const long long row0 = (long long)i * BT;
    // token / head / batch strides per operand: lvsa_params_t.layout or .stride_q/k/v/out
    const T *qb = q + (size_t)b * (size_t)sq.b + (size_t)h * (size_t)sq.h;
    const T *kb = k + (size_t)b * (size_t)sk.b + (size_t)h * (size_t)sk.h;
    const T *vb = v + (size_t)b * (size_t)sv.b + (size_t)h * (size_t)sv.h;

    for (int e = tid; e < BT * D; e += blockDim.x) {
        const int r = e / D, c = e % D;
        const long long n = row0 + r;
        Qs[e] = (n < N) ? to_f32<T>(qb[(size_t)n * (size_t)sq.n + c]) : 0.f;
    }

    float m[R], l[R], acc[R][CH];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        m[r] = -INFINITY; l[r] = 0.f;
#pragma unroll
        for (int c = 0; c < CH; ++c) acc[r][c] = 0.f;
    }

    const int e0 = indptr[i], e1 = indptr[i + 1];
    for (int e = e0; e < e1; ++e) {
        const int j = indices[e];
        const bool partial = flags[e] != LVSA_TILE_FULL;
        // geometry of kv tile j under the index's tiling (token-0 tiles or frame-aligned tiles, R25)
        const lvsa_kv_tile kt = lvsa_kv_tile_of(j, aligned, BT, P, Tv, N);
        const long long col0 = kt.c0;
        const int nchunks = (kt.width + 31) / 32;   // 32-column chunks that hold valid columns
        __syncthreads();
        for (int x = tid; x < BT * D; x += blockDim.x) {
            const int r = x / D, c = x % D;
            const long long n = col0 + r;
            const bool ok = r < kt.width;
            Ks[r * KS + c] = ok ? to_f32<T>(kb[(size_t)n * (size_t)sk.n + c]) : 0.f;
            Vs[r * D + c] = ok ? to_f32<T>(vb[(size_t)n * (size_t)sv.n + c]) : 0.f;
        }
        __syncthreads();
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int rl = wid + r * SIMT_WARPS;
            const long long nq = row0 + rl;
            if (nq >= N) continue;  // warp-uniform
            const uint32_t *arow = a_bits + (size_t)min((int)(nq / P), Tf - 1) * words;   // text rows: frame Tf-1
            const float *qrow = Qs + rl * D;
            for (int cc = 0; cc < nchunks; ++cc) {
                const int cl = cc * 32 + lane;
                const float *krow = Ks + cl * KS;
                float s = 0.f;
#pragma unroll 8
                for (int c = 0; c < D; ++c) s = fmaf(qrow[c], krow[c], s);
                s *= scale;
                if (partial) {
                    const long long nk_ = col0 + cl;
                    bool ok = cl < kt.width;
                    if (ok) { const int f = min((int)(nk_ / P), Tf - 1); ok = (arow[f >> 5] >> (f & 31)) & 1u; }
                    if (!ok) s = -INFINITY;
                }
                float cmax = s;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) cmax = fmaxf(cmax, __shfl_xor_sync(0xffffffffu, cmax, o));
                const float m_new = fmaxf(m[r], cmax);
                if (m_new == -INFINITY) continue;  // nothing allowed so far (warp-uniform)
                const float corr = expf(m[r] - m_new);  // m = -inf -> 0
                const float p = expf(s - m_new);        // s = -inf -> 0
                float psum = p;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) psum += __shfl_xor_sync(0xffffffffu, psum, o);
                l[r] = l[r] * corr + psum;
                m[r] = m_new;
#pragma unroll
                for (int c = 0; c < CH; ++c) acc[r][c] *= corr;
                for (int c2 = 0; c2 < 32; ++c2) {
                    const float pc = __shfl_sync(0xffffffffu, p, c2);
                    const float *vrow = Vs + (cc * 32 + c2) * D + lane;
#pragma unroll
                    for (int c = 0; c < CH; ++c) acc[r][c] = fmaf(pc, vrow[32 * c], acc[r][c]);
                }
            }
        }
    }

    T *ob = out + (size_t)b * (size_t)so.b + (size_t)h * (size_t)so.h;
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int rl = wid + r * SIMT_WARPS;
        const long long nq = row0 + rl;
        if (nq >= N) continue;
        const float inv = 1.f / l[r];
#pragma unroll
        for (int c = 0; c < CH; ++c)
            ob[(size_t)nq * (size_t)so.n + lane + 32 * c] = from_f32<T>(acc[r][c] * inv);
        if (lse != nullptr && lane == 0)
            lse[((size_t)b * H + h) * N + nq] = m[r] + logf(l[r]);
    }
}

template <int D, int BT, typename T>
lvsa_status_t launch(const lvsa_index *ix, const void *q, const void *k, const void *v, void *out,
                     float *lse, cudaStream_t stream) {
    const size_t smem = sizeof(float) * ((size_t)BT * D + (size_t)BT * (D + 1) + (size_t)BT * D);
    auto kern = lvsa_attn_simt_kernel<D, BT, T>;
    LVSA_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    const float scale = ix->p.softmax_scale;
    dim3 grid(ix->nq, ix->p.H, ix->p.B);
    kern<<<grid, SIMT_WARPS * 32, smem, stream>>>(
        (const T *)q, (const T *)k, (const T *)v, (T *)out, lse, ix->d_indptr, ix->d_indices,
        ix->d_flags, ix->d_abits, ix->words, (long long)ix->N, ix->p.P, ix->Tf, ix->p.H,
        lvsa_tensor_strides(ix, LVSA_T_Q), lvsa_tensor_strides(ix, LVSA_T_K), lvsa_tensor_strides(ix, LVSA_T_V),
        lvsa_tensor_strides(ix, LVSA_T_OUT), ix->p.kv_tiling == LVSA_KV_TILES_FRAME_ALIGNED, ix->p.T, scale);
    LVSA_CUDA_TRY(cudaGetLastError());
    return LVSA_OK;
}

}  // namespace

lvsa_status_t lvsa_attn_simt_launch(const lvsa_index *ix, const void *q, const void *k,
                                    const void *v, void *out, float *lse, cudaStream_t stream) {
    const bool bf16 = ix->p.dtype == LVSA_DTYPE_BF16;
    if (ix->p.H > 65535 || ix->p.B > 65535) {
        lvsa_set_error("SIMT kernel: H and B must be <= 65535");
        return LVSA_EUNSUPPORTED;
    }
    if (ix->p.d == 64 && ix->p.tile_q == 64)
        return bf16 ? launch<64, 64, __nv_bfloat16>(ix, q, k, v, out, lse, stream)
                    : launch<64, 64, float>(ix, q, k, v, out, lse, stream);
    if (ix->p.d == 128 && ix->p.tile_q == 128)
        return bf16 ? launch<128, 128, __nv_bfloat16>(ix, q, k, v, out, lse, stream)
                    : launch<128, 128, float>(ix, q, k, v, out, lse, stream);
    lvsa_set_error("SIMT kernel: only (d, tile) = (64, 64) or (128, 128)");
    return LVSA_EUNSUPPORTED;
}
