// Internal declarations of liblvsa (CUDA path).  Not part of the C ABI; include/lvsa.h is.
// Nothing here is shared with oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <string>

#include "lvsa.h"

// Work-item entry encoding for the attention kernels (one int32 per kv-tile visit of a q-tile
// group).  bits [0,26): kv tile j.  bits [26,28): state for the group's q tile 0, bits [28,30):
// state for q tile 1.  States:
// bits [30,32): (computed columns of the kv tile) / 32 - 1, i.e. 3 for a 128-column tile, less for a
// narrow frame-aligned tile (lvsa_params_t.kv_tiling).
constexpr int LVSA_ST_SKIP = 0, LVSA_ST_FULL = 1, LVSA_ST_PARTIAL = 2;
constexpr int LVSA_ITEM_J_BITS = 26;
constexpr int LVSA_ITEM_J_MASK = (1 << LVSA_ITEM_J_BITS) - 1;
constexpr int LVSA_ITEM_W_SHIFT = 30;
// Work-list entry of the 4-CTA-cluster kernel: bits [0,24): kv tile j; bits [24 + 2w, 26 + 2w): state
// of the quad's q tile w (w = 0..3).
constexpr int LVSA_QUAD_J_BITS = 24;
constexpr int LVSA_QUAD_J_MASK = (1 << LVSA_QUAD_J_BITS) - 1;

// Geometry of kv tile j under either tiling (include/lvsa.h, readings R14 / R25): first token, valid
// width, and the frame row of its first token.  T = video frames, Tf = T + (text pseudo-frame).
struct lvsa_kv_tile { long long c0; int width; int g; };
__host__ __device__ inline int lvsa_kv_tiles_per_frame(int P, int Bk) { return (P + Bk - 1) / Bk; }
__host__ __device__ inline lvsa_kv_tile lvsa_kv_tile_of(int j, int frame_aligned, int Bk, int P, int T, long long N) {
    lvsa_kv_tile t;
    if (!frame_aligned) {
        t.c0 = (long long)j * Bk;
        t.width = (int)((t.c0 + Bk <= N) ? Bk : N - t.c0);
        const long long f = t.c0 / P;
        t.g = (int)(f < T ? f : T);
        return t;
    }
    const int kpf = lvsa_kv_tiles_per_frame(P, Bk);
    const int tau = j / kpf;
    if (tau < T) {                      // video frame tau, tile k of it
        const int k = j - tau * kpf;
        t.c0 = (long long)tau * P + (long long)k * Bk;
        t.width = (k + 1) * Bk <= P ? Bk : P - k * Bk;
        t.g = tau;
    } else {                            // text pseudo-frame (R23)
        const int k = j - T * kpf;
        t.c0 = (long long)T * P + (long long)k * Bk;
        t.width = (int)((t.c0 + Bk <= N) ? Bk : N - t.c0);
        t.g = T;
    }
    return t;
}

struct lvsa_index {
    lvsa_params_t p;  // with defaults resolved
    int64_t N = 0;
    int32_t nq = 0, nk = 0, words = 0;
    int32_t Tf = 0;   // frame rows of A: T video frames (+ 1 text pseudo-frame when n_text > 0, R23)
    // counters computed on the device; fetched lazily (lvsa_index_fetch_meta) so that the build
    // itself never synchronises
    mutable int32_t T_per = 0, phase = 0, n_global = 0;
    mutable int64_t nnz = 0, n_partial = 0;
    mutable bool meta_fetched = false;
    mutable bool overflowed = false;   // the device raised meta[7]: lists unfilled and poisoned
    int device = 0;
    // one stream-ordered arena holds every device buffer below
    void *arena = nullptr;
    size_t arena_bytes = 0;
    int64_t cap_nnz = 0, cap_item_tiles = 0;   // allocation bounds (entries)
    cudaStream_t build_stream = nullptr;
    mutable cudaStream_t last_stream = nullptr;   // last stream that used the index
    mutable bool multi_stream = false;            // used on more than one stream: free synchronously
    // device buffers (views into the arena)
    int32_t *d_wlo = nullptr, *d_whi = nullptr;
    uint32_t *d_abits = nullptr;   // [T][words]
    int32_t *d_meta = nullptr;     // small scratch: {nnz, n_partial, n_item_tiles, n_global}
    int32_t *d_indptr = nullptr;   // [nq+1]
    int32_t *d_indices = nullptr;  // [nnz]
    uint8_t *d_flags = nullptr;    // [nnz]
    // attention work items: groups of LVSA_GROUP adjacent q tiles that share kv-tile loads
    int32_t group = 2;
    int64_t n_items = 0;
    mutable int64_t n_item_tiles = 0;
    int32_t *d_item_ptr = nullptr;    // [n_items+1]
    int32_t *d_item_tiles = nullptr;  // [n_item_tiles], encoding above
    int32_t *d_item_col0 = nullptr;   // [n_item_tiles], first token of the entry's kv tile
    int64_t n_quads = 0, cap_quad_tiles = 0;   // LVSA_KERNEL_TCGEN05_QUAD only
    int32_t *d_quad_ptr = nullptr;    // [n_quads+1]
    int32_t *d_quad_tiles = nullptr;  // entries as above
    mutable int64_t kept_cols = 0;    // sum of computed kv columns over the kept pairs
    unsigned long long *d_kept_cols = nullptr;
};

// Element strides of the token, head and batch axes of q, k, v, out (d is contiguous):
// NHD = [B, N, H, d], HND = [B, H, N, d] (lvsa_params_t.layout).
struct lvsa_strides { long long n, h, b; };
inline lvsa_strides lvsa_layout_strides(const lvsa_index *ix) {
    const long long N = ix->N, H = ix->p.H, d = ix->p.d;
    if (ix->p.layout == LVSA_LAYOUT_HND) return {d, N * d, H * N * d};
    return {H * d, d, N * H * d};
}
// Strides of one operand: lvsa_params_t.stride_q/k/v/out when given (any non-zero entry), else the layout's.
enum { LVSA_T_Q = 0, LVSA_T_K = 1, LVSA_T_V = 2, LVSA_T_OUT = 3 };
inline bool lvsa_has_custom_strides(const lvsa_params_t &p) {
    const int64_t *t[4] = {p.stride_q, p.stride_k, p.stride_v, p.stride_out};
    for (int i = 0; i < 4; ++i) if (t[i][0] | t[i][1] | t[i][2]) return true;
    return false;
}
inline lvsa_strides lvsa_tensor_strides(const lvsa_index *ix, int which) {
    const int64_t *t = which == LVSA_T_Q ? ix->p.stride_q : which == LVSA_T_K ? ix->p.stride_k
                     : which == LVSA_T_V ? ix->p.stride_v : ix->p.stride_out;
    if (t[0] | t[1] | t[2]) return {(long long)t[0], (long long)t[1], (long long)t[2]};
    return lvsa_layout_strides(ix);
}
constexpr int LVSA_MAX_DEVICES = 64;   // per-device one-time state is kept in arrays of this size

void lvsa_set_error(const std::string &msg);
lvsa_status_t lvsa_cuda_fail(cudaError_t e, const char *what);

#define LVSA_CUDA_TRY(expr)                                          \
    do {                                                             \
        cudaError_t _e = (expr);                                     \
        if (_e != cudaSuccess) return lvsa_cuda_fail(_e, #expr);     \
    } while (0)

// lvsa_index.cu
lvsa_status_t lvsa_index_build_device(lvsa_index *ix, cudaStream_t stream);
lvsa_status_t lvsa_index_fetch_meta(const lvsa_index *ix);

// lvsa_attn_simt.cu
lvsa_status_t lvsa_attn_simt_launch(const lvsa_index *ix, const void *q, const void *k,
                                    const void *v, void *out, float *lse, cudaStream_t stream);

// lvsa_attn_sm100.cu
lvsa_status_t lvsa_attn_sm100_launch(const lvsa_index *ix, const void *q, const void *k,
                                     const void *v, void *out, float *lse, cudaStream_t stream);
int lvsa_attn_sm100_supported(const lvsa_index *ix);

// lvsa_attn_sm100_pair.cu (CTA-pair kernel, cta_group::2, d = 128)
lvsa_status_t lvsa_attn_sm100_pair_launch(const lvsa_index *ix, const void *q, const void *k,
                                          const void *v, void *out, float *lse, cudaStream_t stream);
lvsa_status_t lvsa_attn_sm100_pair_launch_heads(const lvsa_index *ix, const void *q, const void *k,
                                                const void *v, void *out, float *lse, int h0, int hc,
                                                cudaStream_t stream);
lvsa_status_t lvsa_attn_sm100_pair_prepare(int device);
int lvsa_attn_sm100_pair_grid(const lvsa_index *ix, int hc);   // CTAs of a launch over hc heads (after prepare)
int lvsa_attn_sm100_pair_num_launches(const lvsa_index *ix, int hc);   // kernels of that launch (after prepare)
int lvsa_attn_uses_pair_kernel(const lvsa_index *ix);   // lvsa_attn_sm100.cu

// lvsa_capi.cu: one-time kernel setup for the index's kernel (used by the schedule driver)
lvsa_status_t lvsa_attn_prepare(const lvsa_index *ix);
