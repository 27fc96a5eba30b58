// lvsa_build_csr_static: the block index (steps a1-a5, same definitions as lvsa_index.cu) for
// callers that must not allocate device memory.
//
// Who that is.  A diffusion server usually hands the whole GPU to one allocator at start-up (a
// framework's caching pool, or a fixed memory plan made when the model was loaded).  A plugin that
// then asks the CUDA driver for memory of its own in the middle of the denoising loop can be
// refused although the pool still has room, stalls every stream of the process while the driver
// maps the pages, and breaks the host's accounting of what is resident.  The handle-based builder
// (lvsa_build_block_index_ex) takes a stream-ordered arena per index; this entry point takes
// nothing: the caller brings the three output arrays, and the intermediate data of the build (the
// A(t) bitsets and the per-q-tile counts, which the handle-based path keeps in its arena) live in
// ONE fixed array below that is part of the library image.  The price is a size limit
// (LVSA_STATIC_MAX_FRAMES, LVSA_STATIC_MAX_Q_TILES) and no concurrency: every call on a device
// uses the same array.
//
// The kernels here are a CSR-only restatement of lvsa_frames_kernel / lvsa_tiles_kernel /
// lvsa_scan_kernel (no work items, no quad lists, token-0 kv tiles); tests/test_zz_no_alloc.py
// holds the two paths bit-identical.  Shares nothing with oracle/.
#include <mutex>
#include <string>

#include "lvsa_internal.h"

namespace {

constexpr int MAX_FRAMES = LVSA_STATIC_MAX_FRAMES;     // rows of A, text pseudo-frame included
constexpr int MAX_WORDS = (MAX_FRAMES + 31) / 32;
constexpr int MAX_Q_TILES = LVSA_STATIC_MAX_Q_TILES;
// layout of the scratch array: [control words | a_bits | counts]
constexpr size_t OFF_CTRL = 0;                         // int32[64]: [0] = "nnz does not fit" flag
constexpr size_t OFF_ABITS = 256;
constexpr size_t OFF_COUNTS = OFF_ABITS + sizeof(uint32_t) * MAX_FRAMES * MAX_WORDS;
constexpr size_t SCRATCH_BYTES = OFF_COUNTS + sizeof(int32_t) * MAX_Q_TILES;
static_assert(OFF_COUNTS % 256 == 0, "sections of the scratch array stay 256-byte aligned");
static_assert(SCRATCH_BYTES <= LVSA_STATIC_SCRATCH_BYTES, "the header states the size of the array");

// The scratch memory.  Every GPU that loads liblvsa holds these bytes until the process exits.
// In HOST code this name is only a handle for cudaGetSymbolAddress, never a device address: the
// kernels below get the address looked up in scratch_of_current_device().
static __device__ __align__(256) unsigned char lvsa_static_scratch[LVSA_STATIC_SCRATCH_BYTES];

__device__ __forceinline__ bool in_set(const uint32_t *bits, int x) { return (bits[x >> 5] >> (x & 31)) & 1u; }

// One block.  G^s (Eq. 3; dedicated anchors R22), the adaptive window,
// Algorithm 1 and A(t) (Def. 2) as bitsets, row T = text pseudo-frame
// (R23).  Also clears the control word the previous call may have left raised.
__global__ void static_frames_kernel(int T, int W, int a, int s, int tie_hi, int k0, int has_text, int words,
                                     uint32_t *__restrict__ a_bits, int32_t *__restrict__ ctrl) {
    __shared__ uint32_t g_bits[MAX_WORDS];
    __shared__ int n_global_s;
    const int tid = threadIdx.x;
    if (tid == 0) ctrl[0] = 0;
    for (int w = tid; w < words; w += blockDim.x) g_bits[w] = 0u;
    __syncthreads();
    const bool all_tiles = (a == LVSA_ANCHORS_ALL_TILES);
    if (!all_tiles && a > 0) {
        const int T_per = (T + a - 1) / a, m = (T + T_per - 1) / T_per, phase = s % T_per;
        for (int i = tid; i < m; i += blockDim.x) {
            const int f = (phase + i * T_per) % T;
            atomicOr(&g_bits[f >> 5], 1u << (f & 31));
        }
    }
    if (!all_tiles)
        for (int f = tid; f < min(k0, T); f += blockDim.x) atomicOr(&g_bits[f >> 5], 1u << (f & 31));
    __syncthreads();
    if (tid == 0) {
        int c = 0;
        for (int w = 0; w < words; ++w) c += __popc(g_bits[w]);
        n_global_s = c;
    }
    __syncthreads();
    const int target = min(2 * W + 1, T - n_global_s);
    for (int t = tid; t < T; t += blockDim.x) {
        int l = 0, h = T - 1;
        if (!all_tiles) {
            l = max(0, min(t - W, T - 1 - 2 * W));
            h = min(T - 1, max(t + W, 2 * W));
            int nonglobal = 0;
            for (int x = l; x <= h; ++x) nonglobal += !in_set(g_bits, x);
            while (nonglobal < target && (l > 0 || h < T - 1)) {
                const int room_lo = l, room_hi = T - 1 - h;
                int nw;
                if (room_lo > room_hi || (room_lo == room_hi && !tie_hi)) nw = --l;
                else nw = ++h;
                nonglobal += !in_set(g_bits, nw);
            }
        }
        for (int w = 0; w < words; ++w) {
            const int b0 = max(l, 32 * w), b1 = min(h, 32 * w + 31);
            uint32_t span = 0u;
            if (b0 <= b1) {
                const int n = b1 - b0 + 1;
                span = (n == 32 ? 0xffffffffu : ((1u << n) - 1u)) << (b0 - 32 * w);
            }
            uint32_t bits = g_bits[w] | span;
            if (has_text && (T >> 5) == w) bits |= 1u << (T & 31);
            a_bits[(size_t)t * words + w] = bits;
        }
    }
    if (has_text)
        for (int w = tid; w < words; w += blockDim.x) {
            const int n = min(32, T + 1 - 32 * w);
            a_bits[(size_t)T * words + w] = n <= 0 ? 0u : (n == 32 ? 0xffffffffu : ((1u << n) - 1u));
        }
}

// One block per q tile i.  kv tile j is kept iff some (row of i, column of j) pair is allowed and
// PARTIAL iff some pair is not, or j holds columns >= N (R14).  Threads take kv tiles in ascending
// chunks, so the fill pass writes each q tile's list in ascending order.
template <bool FILL>
__global__ void static_tiles_kernel(long long N, int P, int Tf, int Bq, int Bk, int nk, int words,
                                    const uint32_t *__restrict__ a_bits, int32_t *__restrict__ counts,
                                    const int32_t *__restrict__ indptr, int32_t *__restrict__ indices,
                                    uint8_t *__restrict__ flags, const int32_t *__restrict__ ctrl) {
    __shared__ int warp_tot[32];
    const int i = blockIdx.x, tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int nwarps = blockDim.x >> 5;
    if (FILL && ctrl[0]) return;      // the list does not fit the caller's arrays: write nothing
    const long long r0 = (long long)i * Bq, r1 = min(r0 + Bq, N) - 1;
    const int fa = min((int)(r0 / P), Tf - 1), fb = min((int)(r1 / P), Tf - 1);
    const int base = FILL ? indptr[i] : 0;
    int run = 0;
    for (int j0 = 0; j0 < nk; j0 += blockDim.x) {
        const int j = j0 + tid;
        bool kept = false, part = false;
        if (j < nk) {
            const long long c0 = (long long)j * Bk, c1 = min(c0 + Bk, N) - 1;
            const int g0 = min((int)(c0 / P), Tf - 1), g1 = min((int)(c1 / P), Tf - 1);
            part = (c0 + Bk > N);
            for (int tq = fa; tq <= fb; ++tq) {
                const uint32_t *row = a_bits + (size_t)tq * words;
                for (int tk = g0; tk <= g1; ++tk) {
                    const bool b = in_set(row, tk);
                    kept |= b; part |= !b;
                }
            }
        }
        const unsigned bal = __ballot_sync(0xffffffffu, kept);
        if (lane == 0) warp_tot[wid] = __popc(bal);
        __syncthreads();
        int woff = 0, tot = 0;
        for (int w = 0; w < nwarps; ++w) { const int c = warp_tot[w]; if (w < wid) woff += c; tot += c; }
        if (FILL && kept) {
            const int pos = base + run + woff + __popc(bal & ((1u << lane) - 1u));
            indices[pos] = j;
            flags[pos] = part ? LVSA_TILE_PARTIAL : LVSA_TILE_FULL;
        }
        run += tot;
        __syncthreads();
    }
    if (!FILL && tid == 0) counts[i] = run;
}

// One block: indptr[0..nq] = exclusive scan of counts; *nnz = total; raises ctrl[0] when the total
// does not fit `capacity` entries.
__global__ void static_scan_kernel(const int32_t *__restrict__ counts, int nq, long long capacity,
                                   int32_t *__restrict__ indptr, int32_t *__restrict__ nnz, int32_t *__restrict__ ctrl) {
    __shared__ int warp_tot[32];
    __shared__ int carry_s;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5, nwarps = blockDim.x >> 5;
    if (tid == 0) carry_s = 0;
    __syncthreads();
    for (int i0 = 0; i0 < nq; i0 += blockDim.x) {
        const int i = i0 + tid;
        const int v = i < nq ? counts[i] : 0;
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
        if (i < nq) indptr[i] = carry + woff + incl - v;
        __syncthreads();
        if (tid == 0) carry_s = carry + tot;
        __syncthreads();
    }
    if (tid == 0) { indptr[nq] = carry_s; *nnz = carry_s; if (carry_s > capacity) ctrl[0] = 1; }
}

// Device address of lvsa_static_scratch on the CURRENT device, looked up once per device.
std::mutex g_setup_mutex;
unsigned char *g_scratch_addr[LVSA_MAX_DEVICES] = {};

lvsa_status_t scratch_of_current_device(unsigned char **out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return lvsa_cuda_fail(e, "cudaGetDevice (no usable CUDA device; there is no CPU fallback)");
    if (dev < 0 || dev >= LVSA_MAX_DEVICES) { lvsa_set_error("device ordinal out of range"); return LVSA_EUNSUPPORTED; }
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    if (g_scratch_addr[dev] == nullptr) {
        void *p = nullptr;
        LVSA_CUDA_TRY(cudaGetSymbolAddress(&p, lvsa_static_scratch));
        if (p == nullptr) { lvsa_set_error("cudaGetSymbolAddress returned a null address"); return LVSA_ECUDA; }
        g_scratch_addr[dev] = static_cast<unsigned char *>(p);
    }
    *out = g_scratch_addr[dev];
    return LVSA_OK;
}

}  // namespace

extern "C" lvsa_status_t lvsa_build_csr_static(const lvsa_params_t *params, void *stream_, int32_t *indptr,
                                               int32_t *indices, uint8_t *flags, int64_t capacity, int32_t *nnz) {
    lvsa_set_error("");
    if (params == nullptr || indptr == nullptr || indices == nullptr || flags == nullptr || nnz == nullptr) {
        lvsa_set_error("NULL argument");
        return LVSA_EINVAL;
    }
    if (((uintptr_t)indptr | (uintptr_t)indices | (uintptr_t)nnz) & 3u) {
        lvsa_set_error("indptr, indices, nnz must be 4-byte aligned");
        return LVSA_EINVAL;
    }
    lvsa_params_t p = *params;
    if (p.T <= 0 || p.P <= 0) { lvsa_set_error("T, P must be > 0"); return LVSA_EINVAL; }
    if (p.window < 0) { lvsa_set_error("window must be >= 0"); return LVSA_EINVAL; }
    if (p.anchors < LVSA_ANCHORS_ALL_TILES) { lvsa_set_error("anchors must be >= -1"); return LVSA_EINVAL; }
    if (p.step < 0) { lvsa_set_error("step must be >= 0"); return LVSA_EINVAL; }
    if (p.initial_anchors < 0 || p.n_text < 0) { lvsa_set_error("initial_anchors, n_text must be >= 0"); return LVSA_EINVAL; }
    if (p.tie_break != LVSA_TIE_LO && p.tie_break != LVSA_TIE_HI) { lvsa_set_error("bad tie_break"); return LVSA_EINVAL; }
    if (capacity < 0) { lvsa_set_error("capacity must be >= 0"); return LVSA_EINVAL; }
    const long long N = (long long)p.T * p.P + p.n_text;
    if (N >= (1ll << 31)) { lvsa_set_error("T*P + n_text must be < 2^31"); return LVSA_EINVAL; }
    if (p.d != 64 && p.d != 128) { lvsa_set_error("head dim must be 64 or 128"); return LVSA_EUNSUPPORTED; }
    if (p.tile_q == 0) p.tile_q = p.d;
    if (p.tile_k == 0) p.tile_k = p.d;
    if (p.tile_q != p.d || p.tile_k != p.d) {
        lvsa_set_error("tiles must be 128x128 for d = 128 and 64x64 for d = 64");
        return LVSA_EUNSUPPORTED;
    }
    if (p.kv_tiling != LVSA_KV_TILES_TOKEN0) {
        lvsa_set_error("lvsa_build_csr_static builds token-0 kv tiles only");
        return LVSA_EUNSUPPORTED;
    }
    const int Tf = p.T + (p.n_text > 0 ? 1 : 0);
    const long long nq = (N + p.tile_q - 1) / p.tile_q, nk = (N + p.tile_k - 1) / p.tile_k;
    if (Tf > MAX_FRAMES) {
        lvsa_set_error("lvsa_build_csr_static: " + std::to_string(Tf) + " frame rows exceed LVSA_STATIC_MAX_FRAMES = " +
                       std::to_string(MAX_FRAMES) + " (use lvsa_build_block_index_ex, which allocates)");
        return LVSA_EUNSUPPORTED;
    }
    if (nq > MAX_Q_TILES) {
        lvsa_set_error("lvsa_build_csr_static: " + std::to_string(nq) + " q tiles exceed LVSA_STATIC_MAX_Q_TILES = " +
                       std::to_string(MAX_Q_TILES) + " (use lvsa_build_block_index_ex, which allocates)");
        return LVSA_EUNSUPPORTED;
    }
    unsigned char *scratch = nullptr;
    lvsa_status_t st = scratch_of_current_device(&scratch);
    if (st != LVSA_OK) return st;
    int32_t *ctrl = reinterpret_cast<int32_t *>(scratch + OFF_CTRL);
    uint32_t *a_bits = reinterpret_cast<uint32_t *>(scratch + OFF_ABITS);
    int32_t *counts = reinterpret_cast<int32_t *>(scratch + OFF_COUNTS);

    cudaStream_t stream = (cudaStream_t)stream_;
    const int T = p.T, words = (Tf + 31) / 32;
    const int W = p.window > T ? T : p.window;   // W >= T already spans [0, T-1]; avoids 2W overflow
    static_frames_kernel<<<1, 256, 0, stream>>>(T, W, p.anchors, p.step, p.tie_break == LVSA_TIE_HI, p.initial_anchors,
                                                p.n_text > 0, words, a_bits, ctrl);
    static_tiles_kernel<false><<<(int)nq, 256, 0, stream>>>(N, p.P, Tf, p.tile_q, p.tile_k, (int)nk, words, a_bits, counts,
                                                            nullptr, nullptr, nullptr, ctrl);
    static_scan_kernel<<<1, 1024, 0, stream>>>(counts, (int)nq, (long long)capacity, indptr, nnz, ctrl);
    static_tiles_kernel<true><<<(int)nq, 256, 0, stream>>>(N, p.P, Tf, p.tile_q, p.tile_k, (int)nk, words, a_bits, nullptr,
                                                           indptr, indices, flags, ctrl);
    LVSA_CUDA_TRY(cudaGetLastError());
    return LVSA_OK;
}
