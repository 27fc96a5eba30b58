// C ABI of liblvsa (include/lvsa.h): argument checks, handle lifetime, kernel selection.
#include <math.h>
#include <stdlib.h>
#include <string.h>

#include <mutex>
#include <new>

#include "lvsa_internal.h"

static thread_local std::string g_last_error;

void lvsa_set_error(const std::string &msg) { g_last_error = msg; }

lvsa_status_t lvsa_cuda_fail(cudaError_t e, const char *what) {
    g_last_error = std::string(what) + ": " + cudaGetErrorName(e) + " (" + cudaGetErrorString(e) + ")";
    return LVSA_ECUDA;
}

// staging buffers of lvsa_attn_fwd_host: one workspace per DEVICE, process lifetime (or until
// lvsa_workspace_release), guarded by one mutex
struct HostWorkspace { void *ptr = nullptr; size_t cap = 0; };
static HostWorkspace g_ws[LVSA_MAX_DEVICES];
static std::mutex g_ws_mutex;

// streams and events of the pipelined host entry point (per device, created on first use)
struct HostPipe {
    static constexpr int MAXG = 16;
    cudaStream_t s_in = nullptr, s_out = nullptr;
    cudaEvent_t ev_in[MAXG] = {}, ev_c[MAXG] = {}, ev_edge = nullptr;
};
static HostPipe g_host[LVSA_MAX_DEVICES];

// the index belongs to one device; every call that uses it must run with that device current
static lvsa_status_t check_device(const lvsa_index *ix) {
    int dev = -1;
    LVSA_CUDA_TRY(cudaGetDevice(&dev));
    if (dev != ix->device) {
        lvsa_set_error("the index was built on device " + std::to_string(ix->device) + " but device " +
                       std::to_string(dev) + " is current");
        return LVSA_EINVAL;
    }
    return LVSA_OK;
}

// records that `stream` used the index (its arena is stream-ordered memory)
static bool index_touch_stream(const lvsa_index *index, cudaStream_t stream) {
    if (index->last_stream != stream) {
        index->multi_stream = true;
        index->last_stream = stream;
        return true;
    }
    return false;
}

static size_t elem_size(const lvsa_index *ix) { return ix->p.dtype == LVSA_DTYPE_FP32 ? 4 : 2; }

static int use_tcgen05(const lvsa_index *ix) {
    if (ix->p.kernel == LVSA_KERNEL_SIMT) return 0;
    if (ix->p.kernel == LVSA_KERNEL_TCGEN05 || ix->p.kernel == LVSA_KERNEL_TCGEN05_V0 ||
        ix->p.kernel == LVSA_KERNEL_TCGEN05_QUAD || ix->p.kernel == LVSA_KERNEL_TCGEN05_HYBRID) return 1;
    return ix->p.dtype == LVSA_DTYPE_BF16;
}

lvsa_status_t lvsa_attn_prepare(const lvsa_index *ix) {
    if (use_tcgen05(ix) && lvsa_attn_uses_pair_kernel(ix)) return lvsa_attn_sm100_pair_prepare(ix->device);
    return LVSA_OK;   // the other kernels set their attributes at their first launch
}

extern "C" {

const char *lvsa_last_error(void) { return g_last_error.c_str(); }

const char *lvsa_version(void) {
    return "liblvsa 0.3 (sm_100a; kernels: index-builder (handle-based; static-scratch CSR), attn-simt-fp32, "
           "attn-tcgen05-bf16 (CTA-pair cta_group::2: token-0 and frame-aligned kv tiles; 4-CTA-cluster multicast quad; "
           "hybrid quad+pair; one-CTA v0))";
}

lvsa_status_t lvsa_build_block_index_ex(const lvsa_params_t *params, void *stream, lvsa_index_t **out) {
    g_last_error.clear();
    if (out == nullptr || params == nullptr) { lvsa_set_error("NULL params/out"); return LVSA_EINVAL; }
    *out = nullptr;
    lvsa_params_t p = *params;
    if (p.T <= 0 || p.P <= 0 || p.H <= 0 || p.d <= 0) { lvsa_set_error("T, P, H, d must be > 0"); return LVSA_EINVAL; }
    if (p.B == 0) p.B = 1;
    if (p.B < 0) { lvsa_set_error("B must be > 0"); return LVSA_EINVAL; }
    if (p.window < 0) { lvsa_set_error("window must be >= 0"); return LVSA_EINVAL; }
    if (p.anchors < LVSA_ANCHORS_ALL_TILES) { lvsa_set_error("anchors must be >= -1"); return LVSA_EINVAL; }
    if (p.step < 0 || p.layer < 0) { lvsa_set_error("step and layer must be >= 0"); return LVSA_EINVAL; }
    if ((long long)p.T * p.P + (long long)(p.n_text > 0 ? p.n_text : 0) >= (1ll << 31)) { lvsa_set_error("T*P + n_text must be < 2^31"); return LVSA_EINVAL; }
    if (p.initial_anchors < 0) { lvsa_set_error("initial_anchors must be >= 0"); return LVSA_EINVAL; }
    if (p.n_text < 0) { lvsa_set_error("n_text must be >= 0"); return LVSA_EINVAL; }
    if (p.tie_break != LVSA_TIE_LO && p.tie_break != LVSA_TIE_HI) { lvsa_set_error("bad tie_break"); return LVSA_EINVAL; }
    if (p.dtype != LVSA_DTYPE_BF16 && p.dtype != LVSA_DTYPE_FP32) { lvsa_set_error("bad dtype"); return LVSA_EINVAL; }
    if (p.kernel < LVSA_KERNEL_AUTO || p.kernel > LVSA_KERNEL_TCGEN05_HYBRID) { lvsa_set_error("bad kernel"); return LVSA_EINVAL; }
    if (p.layout != LVSA_LAYOUT_NHD && p.layout != LVSA_LAYOUT_HND) { lvsa_set_error("bad layout"); return LVSA_EINVAL; }
    if (p.host_groups < 0) { lvsa_set_error("host_groups must be >= 0"); return LVSA_EINVAL; }
    if (p.kv_tiling != LVSA_KV_TILES_TOKEN0 && p.kv_tiling != LVSA_KV_TILES_FRAME_ALIGNED) { lvsa_set_error("bad kv_tiling"); return LVSA_EINVAL; }
    {   // free strides: all-zero triplet = derive from layout; else d contiguous, 16-byte multiples, TMA range
        const int64_t *st[4] = {p.stride_q, p.stride_k, p.stride_v, p.stride_out};
        const char *nm[4] = {"stride_q", "stride_k", "stride_v", "stride_out"};
        const int64_t es = p.dtype == LVSA_DTYPE_FP32 ? 4 : 2;
        for (int t = 0; t < 4; ++t) {
            if (!(st[t][0] | st[t][1] | st[t][2])) continue;
            for (int a = 0; a < 3; ++a) {
                const int64_t v = st[t][a];
                if (v < 0 || (v * es) % 16 != 0 || v * es >= (1ll << 40)) {
                    lvsa_set_error(std::string(nm[t]) + ": strides must be >= 0, multiples of 16 bytes and below 2^40 bytes");
                    return LVSA_EINVAL;
                }
            }
            if (st[t][0] < p.d) { lvsa_set_error(std::string(nm[t]) + ": the token stride must be >= d (d is contiguous)"); return LVSA_EINVAL; }
            if (st[t][1] == 0 && p.H > 1) { lvsa_set_error(std::string(nm[t]) + ": the head stride must be > 0 when H > 1"); return LVSA_EINVAL; }
            if (st[t][2] == 0 && p.B > 1) { lvsa_set_error(std::string(nm[t]) + ": the batch stride must be > 0 when B > 1"); return LVSA_EINVAL; }
        }
    }
    if (p.T > 4096) { lvsa_set_error("T > 4096 frames is not supported"); return LVSA_EUNSUPPORTED; }
    if (p.d != 64 && p.d != 128) { lvsa_set_error("head dim must be 64 or 128"); return LVSA_EUNSUPPORTED; }
    if (p.tile_q == 0) p.tile_q = p.d;
    if (p.tile_k == 0) p.tile_k = p.d;
    if (p.tile_q != p.d || p.tile_k != p.d) {
        lvsa_set_error("tiles must be 128x128 for d = 128 and 64x64 for d = 64");
        return LVSA_EUNSUPPORTED;
    }
    if ((p.kernel == LVSA_KERNEL_TCGEN05_QUAD || p.kernel == LVSA_KERNEL_TCGEN05_HYBRID) && (p.d != 128 || p.kv_tiling != LVSA_KV_TILES_TOKEN0)) {
        lvsa_set_error("the 4-CTA-cluster kernel takes d = 128 and token-0 kv tiles only");
        return LVSA_EUNSUPPORTED;
    }
    if (p.dtype == LVSA_DTYPE_FP32 && (p.kernel == LVSA_KERNEL_TCGEN05 || p.kernel == LVSA_KERNEL_TCGEN05_V0 ||
                                       p.kernel == LVSA_KERNEL_TCGEN05_QUAD || p.kernel == LVSA_KERNEL_TCGEN05_HYBRID)) {
        lvsa_set_error("the tcgen05 kernel takes bf16 only");
        return LVSA_EUNSUPPORTED;
    }
    if (!(p.softmax_scale > 0.f)) p.softmax_scale = 1.0f / sqrtf((float)p.d);

    lvsa_index *ix = new (std::nothrow) lvsa_index();
    if (ix == nullptr) { lvsa_set_error("out of host memory"); return LVSA_ENOMEM; }
    ix->p = p;
    ix->N = (int64_t)p.T * p.P + p.n_text;
    ix->Tf = p.T + (p.n_text > 0 ? 1 : 0);
    ix->nq = (int32_t)((ix->N + p.tile_q - 1) / p.tile_q);
    ix->nk = (int32_t)((ix->N + p.tile_k - 1) / p.tile_k);
    if (p.kv_tiling == LVSA_KV_TILES_FRAME_ALIGNED) {   // ceil(P/Bk) tiles per frame + the text tiles (R25)
        const long long nk = (long long)p.T * lvsa_kv_tiles_per_frame(p.P, p.tile_k) + (p.n_text + p.tile_k - 1) / p.tile_k;
        if (nk >= (1ll << LVSA_ITEM_J_BITS)) { delete ix; lvsa_set_error("too many kv tiles"); return LVSA_EUNSUPPORTED; }
        ix->nk = (int32_t)nk;
    }
    ix->words = (ix->Tf + 31) / 32;
    ix->group = 2;
    if ((long long)ix->nq * ix->nk >= (1ll << 31)) {
        lvsa_index_destroy(ix);
        lvsa_set_error("nq*nk must be < 2^31");
        return LVSA_EUNSUPPORTED;
    }
    cudaError_t e = cudaGetDevice(&ix->device);
    if (e != cudaSuccess) { lvsa_index_destroy(ix); return lvsa_cuda_fail(e, "cudaGetDevice (no usable CUDA device; there is no CPU fallback)"); }
    if (ix->device < 0 || ix->device >= LVSA_MAX_DEVICES) { lvsa_index_destroy(ix); lvsa_set_error("device ordinal out of range"); return LVSA_EUNSUPPORTED; }
    lvsa_status_t st = lvsa_index_build_device(ix, (cudaStream_t)stream);
    if (st != LVSA_OK) { lvsa_index_destroy(ix); return st; }
    if (use_tcgen05(ix) && p.kv_tiling == LVSA_KV_TILES_FRAME_ALIGNED && !lvsa_attn_uses_pair_kernel(ix)) {
        lvsa_index_destroy(ix);
        lvsa_set_error("frame-aligned kv tiles: CTA-pair kernel (d = 128) or SIMT kernel only");
        return LVSA_EUNSUPPORTED;
    }
    if (use_tcgen05(ix) && !lvsa_attn_sm100_supported(ix)) {
        lvsa_index_destroy(ix);
        lvsa_set_error("tcgen05 kernel: device is not sm_100 or shape unsupported");
        return LVSA_EUNSUPPORTED;
    }
    *out = ix;
    return LVSA_OK;
}

lvsa_index_t *lvsa_build_block_index(int T, int P, int H, int d, int window, int anchors, int step,
                                     int layer) {
    lvsa_params_t p;
    memset(&p, 0, sizeof(p));
    p.T = T; p.P = P; p.H = H; p.d = d; p.window = window; p.anchors = anchors; p.step = step;
    p.layer = layer;
    lvsa_index_t *ix = nullptr;
    if (lvsa_build_block_index_ex(&p, nullptr, &ix) != LVSA_OK) return nullptr;
    return ix;
}

lvsa_status_t lvsa_attn_fwd(const void *q, const void *k, const void *v, const lvsa_index_t *index,
                            void *out, float *lse, void *stream) {
    if (q == nullptr || k == nullptr || v == nullptr || index == nullptr || out == nullptr) {
        lvsa_set_error("NULL argument");
        return LVSA_EINVAL;
    }
    if (((uintptr_t)q | (uintptr_t)k | (uintptr_t)v | (uintptr_t)out) & 15u) {
        lvsa_set_error("q, k, v, out must be 16-byte aligned");
        return LVSA_EINVAL;
    }
    if ((uintptr_t)lse & 3u) { lvsa_set_error("lse must be 4-byte aligned"); return LVSA_EINVAL; }
    lvsa_status_t dst = check_device(index);
    if (dst != LVSA_OK) return dst;
    if (index->overflowed) {   // known from an earlier lvsa_index_info / copy_host; unknown yet: the kernel traps
        lvsa_set_error("internal: the index build exceeded its allocation bound; the index is unusable");
        return LVSA_ECUDA;
    }
    index_touch_stream(index, (cudaStream_t)stream);   // the arena is stream-ordered memory
    if (use_tcgen05(index)) return lvsa_attn_sm100_launch(index, q, k, v, out, lse, (cudaStream_t)stream);
    return lvsa_attn_simt_launch(index, q, k, v, out, lse, (cudaStream_t)stream);
}

// The pipelined body of lvsa_attn_fwd_host: everything it enqueues goes to `stream`, hp.s_in and
// hp.s_out; the caller synchronises all three whatever this returns.
static lvsa_status_t host_pipeline(lvsa_index *ix, HostPipe &hp, int G, const void *qh, const void *kh, const void *vh,
                                   void *oh, float *lseh, void *s_q, void *s_k, void *s_v, void *s_o,
                                   float *s_lse, cudaStream_t stream) {
    const int H = ix->p.H;
    const size_t es = elem_size(ix);
    const int per = (H + G - 1) / G;
    // One head group = a strided 2-D block of the tensor: NHD [B*N rows][H*d] -> hc*d wide columns of
    // every token row; HND [B rows][H*N*d] -> hc*N*d contiguous elements of every batch.
    const bool hnd = ix->p.layout == LVSA_LAYOUT_HND;
    const size_t pitch = hnd ? (size_t)H * ix->N * ix->p.d * es : (size_t)H * ix->p.d * es;
    const size_t rows = hnd ? (size_t)ix->p.B : (size_t)ix->p.B * ix->N;
    const size_t per_head = hnd ? (size_t)ix->N * ix->p.d * es : (size_t)ix->p.d * es;
    size_t width_cur = 0;   // bytes per row of the head group being copied (set in the loops below)
    // HND: the group is B contiguous runs, copied one by one (a 2-D copy would need the batch stride as its
    // pitch, and cudaMemcpy2D refuses pitches above cudaDevAttrMaxPitch = 2^31 - 1 bytes: H*N*d*2 exceeds
    // that from about 8.4 M token-heads).  NHD: one 2-D copy, pitch = H*d elements.
    auto copy_group = [&](uint8_t *dst, const uint8_t *src, cudaMemcpyKind kind, cudaStream_t s) -> lvsa_status_t {
        if (!hnd) {
            LVSA_CUDA_TRY(cudaMemcpy2DAsync(dst, pitch, src, pitch, width_cur, rows, kind, s));
            return LVSA_OK;
        }
        for (size_t b = 0; b < rows; ++b)
            LVSA_CUDA_TRY(cudaMemcpyAsync(dst + b * pitch, src + b * pitch, width_cur, kind, s));
        return LVSA_OK;
    };
    // copies start after whatever the caller already enqueued on `stream`
    LVSA_CUDA_TRY(cudaEventRecord(hp.ev_edge, stream));
    LVSA_CUDA_TRY(cudaStreamWaitEvent(hp.s_in, hp.ev_edge, 0));
    LVSA_CUDA_TRY(cudaStreamWaitEvent(hp.s_out, hp.ev_edge, 0));
    int ng = 0;
    for (int h0 = 0; h0 < H; h0 += per, ++ng) {
        const int hc = h0 + per <= H ? per : H - h0;
        const size_t off = (size_t)h0 * per_head;
        width_cur = (size_t)hc * per_head;
        const void *src[3] = {qh, kh, vh};
        void *dst[3] = {s_q, s_k, s_v};
        for (int t = 0; t < 3; ++t) {
            lvsa_status_t cst = copy_group((uint8_t *)dst[t] + off, (const uint8_t *)src[t] + off, cudaMemcpyHostToDevice, hp.s_in);
            if (cst != LVSA_OK) return cst;
        }
        LVSA_CUDA_TRY(cudaEventRecord(hp.ev_in[ng], hp.s_in));
    }
    ng = 0;
    for (int h0 = 0; h0 < H; h0 += per, ++ng) {
        const int hc = h0 + per <= H ? per : H - h0;
        const size_t off = (size_t)h0 * per_head;
        width_cur = (size_t)hc * per_head;
        LVSA_CUDA_TRY(cudaStreamWaitEvent(stream, hp.ev_in[ng], 0));
        lvsa_status_t st = lvsa_attn_sm100_pair_launch_heads(ix, s_q, s_k, s_v, s_o, s_lse, h0, hc, stream);
        if (st != LVSA_OK) return st;
        LVSA_CUDA_TRY(cudaEventRecord(hp.ev_c[ng], stream));
        LVSA_CUDA_TRY(cudaStreamWaitEvent(hp.s_out, hp.ev_c[ng], 0));
        lvsa_status_t cst = copy_group((uint8_t *)oh + off, (const uint8_t *)s_o + off, cudaMemcpyDeviceToHost, hp.s_out);
        if (cst != LVSA_OK) return cst;
        if (lseh != nullptr)   // lse is [B, H, N]: heads h0.. of every batch are contiguous runs of hc * N floats
            LVSA_CUDA_TRY(cudaMemcpy2DAsync(lseh + (size_t)h0 * ix->N, sizeof(float) * (size_t)H * ix->N,
                                            s_lse + (size_t)h0 * ix->N, sizeof(float) * (size_t)H * ix->N,
                                            sizeof(float) * (size_t)hc * ix->N, (size_t)ix->p.B,
                                            cudaMemcpyDeviceToHost, hp.s_out));
    }
    LVSA_CUDA_TRY(cudaEventRecord(hp.ev_edge, hp.s_out));
    LVSA_CUDA_TRY(cudaStreamWaitEvent(stream, hp.ev_edge, 0));
    return LVSA_OK;
}

static lvsa_status_t host_plain(lvsa_index *ix, size_t bytes, size_t lbytes, const void *qh, const void *kh,
                                const void *vh, void *oh, float *lseh, void *s_q, void *s_k, void *s_v, void *s_o,
                                float *s_lse, cudaStream_t stream) {
    LVSA_CUDA_TRY(cudaMemcpyAsync(s_q, qh, bytes, cudaMemcpyHostToDevice, stream));
    LVSA_CUDA_TRY(cudaMemcpyAsync(s_k, kh, bytes, cudaMemcpyHostToDevice, stream));
    LVSA_CUDA_TRY(cudaMemcpyAsync(s_v, vh, bytes, cudaMemcpyHostToDevice, stream));
    lvsa_status_t st = lvsa_attn_fwd(s_q, s_k, s_v, ix, s_o, s_lse, stream);
    if (st != LVSA_OK) return st;
    LVSA_CUDA_TRY(cudaMemcpyAsync(oh, s_o, bytes, cudaMemcpyDeviceToHost, stream));
    if (lseh != nullptr) LVSA_CUDA_TRY(cudaMemcpyAsync(lseh, s_lse, lbytes, cudaMemcpyDeviceToHost, stream));
    return LVSA_OK;
}

lvsa_status_t lvsa_attn_fwd_host(const void *qh, const void *kh, const void *vh, lvsa_index_t *ix,
                                 void *oh, float *lseh, void *stream_) {
    if (qh == nullptr || kh == nullptr || vh == nullptr || ix == nullptr || oh == nullptr) {
        lvsa_set_error("NULL argument");
        return LVSA_EINVAL;
    }
    lvsa_status_t dst = check_device(ix);
    if (dst != LVSA_OK) return dst;
    if (lvsa_has_custom_strides(ix->p)) {
        lvsa_set_error("lvsa_attn_fwd_host takes layout-derived strides only (stride_q/k/v/out must be zero)");
        return LVSA_EUNSUPPORTED;
    }
    cudaStream_t stream = (cudaStream_t)stream_;
    const size_t bytes = (size_t)ix->p.B * ix->N * ix->p.H * ix->p.d * elem_size(ix);
    const size_t lbytes = sizeof(float) * (size_t)ix->p.B * ix->p.H * ix->N;
    // device staging buffers: one workspace per device, grown on demand, shared by every index
    // handle (a per-step rebuild of the index must not re-allocate gigabytes)
    const size_t ab = (bytes + 255) & ~(size_t)255;
    const size_t need = 4 * ab + lbytes;
    std::lock_guard<std::mutex> lock(g_ws_mutex);
    HostWorkspace &ws = g_ws[ix->device];
    if (ws.ptr == nullptr || ws.cap < need) {
        if (ws.ptr != nullptr) { cudaFree(ws.ptr); ws.ptr = nullptr; ws.cap = 0; }
        LVSA_CUDA_TRY(cudaMalloc(&ws.ptr, need));
        ws.cap = need;
    }
    uint8_t *wsp = static_cast<uint8_t *>(ws.ptr);
    void *s_q = wsp, *s_k = wsp + ab, *s_v = wsp + 2 * ab, *s_o = wsp + 3 * ab;
    float *s_lse = reinterpret_cast<float *>(wsp + 4 * ab);
    // Pipelined path (CTA-pair kernel, bf16): heads are independent, so the call is cut into groups
    // of heads; the H2D copy of group g+1 and the D2H copy of group g-1 overlap the kernel of
    // group g.  lvsa_params_t.host_groups: 0 = one head per group (at most MAXG groups), 1 = off.
    int G = ix->p.host_groups == 0 ? HostPipe::MAXG : ix->p.host_groups;
    if (G > ix->p.H) G = ix->p.H;
    if (G > HostPipe::MAXG) G = HostPipe::MAXG;
    const bool piped = G > 1 && use_tcgen05(ix) && lvsa_attn_uses_pair_kernel(ix);
    HostPipe &hp = g_host[ix->device];
    lvsa_status_t st;
    if (piped) {
        if (hp.ev_edge == nullptr) {
            LVSA_CUDA_TRY(cudaStreamCreateWithFlags(&hp.s_in, cudaStreamNonBlocking));
            LVSA_CUDA_TRY(cudaStreamCreateWithFlags(&hp.s_out, cudaStreamNonBlocking));
            for (int i = 0; i < HostPipe::MAXG; ++i) {
                LVSA_CUDA_TRY(cudaEventCreateWithFlags(&hp.ev_in[i], cudaEventDisableTiming));
                LVSA_CUDA_TRY(cudaEventCreateWithFlags(&hp.ev_c[i], cudaEventDisableTiming));
            }
            LVSA_CUDA_TRY(cudaEventCreateWithFlags(&hp.ev_edge, cudaEventDisableTiming));
        }
        index_touch_stream(ix, stream);
        st = host_pipeline(ix, hp, G, qh, kh, vh, oh, lseh, s_q, s_k, s_v, s_o, s_lse, stream);
    } else {
        st = host_plain(ix, bytes, lbytes, qh, kh, vh, oh, lseh, s_q, s_k, s_v, s_o, s_lse, stream);
    }
    // Whatever happened, nothing this call enqueued may still touch the caller's host buffers or the
    // workspace when it returns: wait for all three streams, then report the first error.
    const std::string first_error = st != LVSA_OK ? std::string(lvsa_last_error()) : std::string();
    cudaError_t e_in = piped ? cudaStreamSynchronize(hp.s_in) : cudaSuccess;
    cudaError_t e_main = cudaStreamSynchronize(stream);
    cudaError_t e_out = piped ? cudaStreamSynchronize(hp.s_out) : cudaSuccess;
    if (st != LVSA_OK) { lvsa_set_error(first_error); return st; }
    LVSA_CUDA_TRY(e_in);
    LVSA_CUDA_TRY(e_main);
    LVSA_CUDA_TRY(e_out);
    return LVSA_OK;
}

void lvsa_workspace_release(void) {
    std::lock_guard<std::mutex> lock(g_ws_mutex);
    int cur = -1;
    cudaGetDevice(&cur);
    for (int dev = 0; dev < LVSA_MAX_DEVICES; ++dev) {
        if (g_ws[dev].ptr == nullptr) continue;
        cudaSetDevice(dev);
        cudaFree(g_ws[dev].ptr);
        g_ws[dev].ptr = nullptr; g_ws[dev].cap = 0;
        // the streams and events of the pipelined host path go with the workspace (re-created on demand)
        HostPipe &hp = g_host[dev];
        if (hp.s_in != nullptr) cudaStreamDestroy(hp.s_in);
        if (hp.s_out != nullptr) cudaStreamDestroy(hp.s_out);
        for (int i = 0; i < HostPipe::MAXG; ++i) {
            if (hp.ev_in[i] != nullptr) cudaEventDestroy(hp.ev_in[i]);
            if (hp.ev_c[i] != nullptr) cudaEventDestroy(hp.ev_c[i]);
        }
        if (hp.ev_edge != nullptr) cudaEventDestroy(hp.ev_edge);
        hp = HostPipe();
    }
    if (cur >= 0) cudaSetDevice(cur);
}

void lvsa_index_destroy(lvsa_index_t *ix) {
    if (ix == nullptr) return;
    if (ix->arena != nullptr) {
        // the arena and its streams belong to the index's device: make it current around the free
        int cur = -1;
        const bool sw = cudaGetDevice(&cur) == cudaSuccess && cur != ix->device;
        if (sw) cudaSetDevice(ix->device);
        // stream-ordered free behind the work that used the index; if several streams used it,
        // wait for the device first
        if (ix->multi_stream) cudaDeviceSynchronize();
        if (cudaFreeAsync(ix->arena, ix->last_stream) != cudaSuccess) {
            cudaGetLastError();                 // e.g. the stream is gone: free synchronously instead
            cudaDeviceSynchronize();
            cudaFree(ix->arena);
        }
        if (sw) cudaSetDevice(cur);
    }
    delete ix;
}

lvsa_status_t lvsa_index_info(const lvsa_index_t *ix, lvsa_index_info_t *info) {
    if (ix == nullptr || info == nullptr) { lvsa_set_error("NULL argument"); return LVSA_EINVAL; }
    memset(info, 0, sizeof(*info));
    if (!ix->meta_fetched) {   // the counters still have to come from the index's device
        lvsa_status_t dst = check_device(ix);
        if (dst != LVSA_OK) return dst;
    }
    lvsa_status_t fst = lvsa_index_fetch_meta(ix);
    if (fst != LVSA_OK) return fst;
    const lvsa_params_t &p = ix->p;
    info->T = p.T; info->P = p.P; info->H = p.H; info->d = p.d; info->B = p.B;
    info->window = p.window; info->anchors = p.anchors; info->step = p.step; info->layer = p.layer;
    info->tile_q = p.tile_q; info->tile_k = p.tile_k; info->nq = ix->nq; info->nk = ix->nk;
    info->T_per = ix->T_per; info->phase = ix->phase; info->n_global = ix->n_global;
    info->words = ix->words; info->dtype = p.dtype; info->n_text = p.n_text;
    info->initial_anchors = p.initial_anchors; info->layout = p.layout; info->kv_tiling = p.kv_tiling;
    info->kept_cols = ix->kept_cols;
    info->kernel = !use_tcgen05(ix) ? LVSA_KERNEL_SIMT
                 : (p.kernel == LVSA_KERNEL_TCGEN05_V0 || p.kernel == LVSA_KERNEL_TCGEN05_QUAD || p.kernel == LVSA_KERNEL_TCGEN05_HYBRID ? p.kernel : LVSA_KERNEL_TCGEN05);
    info->N = ix->N; info->nnz = ix->nnz; info->n_partial = ix->n_partial;
    info->n_items = ix->n_items; info->n_item_tiles = ix->n_item_tiles;
    return LVSA_OK;
}

lvsa_status_t lvsa_index_copy_host(const lvsa_index_t *ix, int32_t *indptr, int32_t *indices,
                                   uint8_t *flags, int32_t *w_lo, int32_t *w_hi, uint32_t *a_bits) {
    if (ix == nullptr) { lvsa_set_error("NULL index"); return LVSA_EINVAL; }
    const int T = ix->p.T;
    lvsa_status_t dst = check_device(ix);
    if (dst != LVSA_OK) return dst;
    lvsa_status_t fst = lvsa_index_fetch_meta(ix);
    if (fst != LVSA_OK) return fst;
    if (indptr) LVSA_CUDA_TRY(cudaMemcpy(indptr, ix->d_indptr, sizeof(int32_t) * ((size_t)ix->nq + 1), cudaMemcpyDeviceToHost));
    if (indices && ix->nnz) LVSA_CUDA_TRY(cudaMemcpy(indices, ix->d_indices, sizeof(int32_t) * (size_t)ix->nnz, cudaMemcpyDeviceToHost));
    if (flags && ix->nnz) LVSA_CUDA_TRY(cudaMemcpy(flags, ix->d_flags, (size_t)ix->nnz, cudaMemcpyDeviceToHost));
    if (w_lo) LVSA_CUDA_TRY(cudaMemcpy(w_lo, ix->d_wlo, sizeof(int32_t) * T, cudaMemcpyDeviceToHost));
    if (w_hi) LVSA_CUDA_TRY(cudaMemcpy(w_hi, ix->d_whi, sizeof(int32_t) * T, cudaMemcpyDeviceToHost));
    if (a_bits) LVSA_CUDA_TRY(cudaMemcpy(a_bits, ix->d_abits, sizeof(uint32_t) * (size_t)ix->Tf * ix->words, cudaMemcpyDeviceToHost));
    return LVSA_OK;
}

lvsa_status_t lvsa_index_copy_kv_tiles(const lvsa_index_t *ix, int32_t *col0, int32_t *width) {
    if (ix == nullptr) { lvsa_set_error("NULL index"); return LVSA_EINVAL; }
    const int aligned = ix->p.kv_tiling == LVSA_KV_TILES_FRAME_ALIGNED;
    for (int j = 0; j < ix->nk; ++j) {
        const lvsa_kv_tile t = lvsa_kv_tile_of(j, aligned, ix->p.tile_k, ix->p.P, ix->p.T, ix->N);
        if (col0) col0[j] = (int32_t)t.c0;
        if (width) width[j] = t.width;
    }
    return LVSA_OK;
}

// ---------------------------------------------------------------- whole-schedule driver (f1)
struct lvsa_schedule {
    int n_phases = 0;
    lvsa_index **phase = nullptr;   // [n_phases], index of step r = phase r
};

lvsa_status_t lvsa_schedule_create(const lvsa_params_t *params, void *stream, lvsa_schedule_t **out) {
    if (params == nullptr || out == nullptr) { lvsa_set_error("NULL argument"); return LVSA_EINVAL; }
    *out = nullptr;
    // a1: T_per = ceil(T / a); no rotation without anchors or on the all-tiles path
    int n = 1;
    if (params->T > 0 && params->anchors > 0) n = (params->T + params->anchors - 1) / params->anchors;
    lvsa_schedule *sc = new (std::nothrow) lvsa_schedule();
    if (sc == nullptr) { lvsa_set_error("out of host memory"); return LVSA_ENOMEM; }
    sc->phase = new (std::nothrow) lvsa_index *[n]();
    if (sc->phase == nullptr) { delete sc; lvsa_set_error("out of host memory"); return LVSA_ENOMEM; }
    sc->n_phases = n;
    for (int r = 0; r < n; ++r) {
        lvsa_params_t p = *params;
        p.step = r;
        lvsa_status_t st = lvsa_build_block_index_ex(&p, stream, &sc->phase[r]);
        if (st != LVSA_OK) { lvsa_schedule_destroy(sc); return st; }
    }
    // one-time kernel attribute setup now, so that later launches are pure launches (graph capture)
    lvsa_status_t st = lvsa_attn_prepare(sc->phase[0]);
    if (st != LVSA_OK) { lvsa_schedule_destroy(sc); return st; }
    *out = sc;
    return LVSA_OK;
}

int lvsa_schedule_num_phases(const lvsa_schedule_t *sc) { return sc == nullptr ? 0 : sc->n_phases; }

const lvsa_index_t *lvsa_schedule_index(const lvsa_schedule_t *sc, int step) {
    if (sc == nullptr || step < 0) { lvsa_set_error("NULL schedule or negative step"); return nullptr; }
    return sc->phase[step % sc->n_phases];
}

lvsa_status_t lvsa_schedule_attn_fwd(const lvsa_schedule_t *sc, int step, const void *q, const void *k,
                                     const void *v, void *out, float *lse, void *stream) {
    const lvsa_index_t *ix = lvsa_schedule_index(sc, step);
    if (ix == nullptr) return LVSA_EINVAL;
    return lvsa_attn_fwd(q, k, v, ix, out, lse, stream);
}

void lvsa_schedule_destroy(lvsa_schedule_t *sc) {
    if (sc == nullptr) return;
    if (sc->phase != nullptr) {
        for (int r = 0; r < sc->n_phases; ++r) lvsa_index_destroy(sc->phase[r]);
        delete[] sc->phase;
    }
    delete sc;
}

int lvsa_attn_fwd_launches(const lvsa_index_t *ix) {
    if (ix == nullptr) return 0;
    if (ix->p.kernel != LVSA_KERNEL_TCGEN05_HYBRID) return 1;
    // HYBRID forks into a 4-CTA-cluster launch and a CTA-pair launch when both parts get work
    if (check_device(ix) != LVSA_OK || lvsa_attn_sm100_pair_prepare(ix->device) != LVSA_OK) return -1;
    return lvsa_attn_sm100_pair_num_launches(ix, ix->p.H);
}

int lvsa_index_build_launches(const lvsa_index_t *ix) {
    if (ix == nullptr) return 0;
    // frames, count, scan, fill (+ count, scan, fill of the quad lists); lvsa_index.cu
    return ix->n_quads != 0 ? 7 : 4;
}

int lvsa_attn_fwd_grid(const lvsa_index_t *ix) {
    if (ix == nullptr) { lvsa_set_error("NULL index"); return -1; }
    if (!use_tcgen05(ix) || !lvsa_attn_uses_pair_kernel(ix)) return 0;
    if (check_device(ix) != LVSA_OK || lvsa_attn_sm100_pair_prepare(ix->device) != LVSA_OK) return -1;
    return lvsa_attn_sm100_pair_grid(ix, ix->p.H);
}

}  // extern "C"
