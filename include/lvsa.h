/*
 * lvsa.h — C ABI of the B200-native LVSA block-sparse attention forward.
 *
 * The operation is the one PAPER.md section 2 defines (arxiv/paper_2605_31057):
 *   Attn(q_{t,i}) = sum_{tau in A(t)} sum_p softmax_{(tau,p)}( q_{t,i} . k_{tau,p} / sqrt(d) ) v_{tau,p}
 *                                                                        (Eq. 2)
 *   A(t) = G^s  u  [w_lo(t), w_hi(t)]                                     (Def. 2)
 *   G^s  = { (s mod T_per + i T_per) mod T : i < ceil(T/T_per) }          (Eq. 3)
 *   T_per = ceil( T / (C - (2W+1)) )
 *   (w_lo, w_hi) = Algorithm 1 applied to the adaptive window of PAPER.md:68
 *
 * Token layout (reading R12): N = T*P tokens, token n = t*P + p.
 * Everything runs on ONE GPU (sm_100a).  There is no CPU fallback: without a usable CUDA
 * device every call below that touches the device returns LVSA_ECUDA / NULL.
 * No exception crosses this boundary; the only global state is a thread-local error string.
 */
#ifndef LVSA_H_
#define LVSA_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct lvsa_index lvsa_index_t; /* opaque; owns its device and host buffers */

typedef enum {
    LVSA_OK = 0,
    LVSA_EINVAL = 1,       /* bad argument (sizes <= 0, W < 0, a < -1, step < 0, NULL, T*P >= 2^31 ...) */
    LVSA_EUNSUPPORTED = 2, /* legal but not built: head dim / tile / dtype outside {64/64, 128/128} */
    LVSA_ECUDA = 3,        /* CUDA runtime or driver failure; lvsa_last_error() has the string */
    LVSA_ENOMEM = 4
} lvsa_status_t;

#define LVSA_ANCHORS_ALL_TILES (-1) /* anchors value selecting the all-tiles (dense, Eq. 1) path */

enum { LVSA_TILE_FULL = 0, LVSA_TILE_PARTIAL = 1 };            /* values of flags[]            */
enum { LVSA_TIE_LO = 0, LVSA_TIE_HI = 1 };                     /* Algorithm 1 line 5 tie-break */
enum { LVSA_DTYPE_BF16 = 0, LVSA_DTYPE_FP32 = 1 };             /* element type of q,k,v,out    */
/* LVSA_KERNEL_TCGEN05: the production tensor-core kernel (d = 128: persistent CTA-pair kernel,
 * cta_group::2; d = 64: the one-CTA-per-item kernel).  LVSA_KERNEL_TCGEN05_V0: the simple
 * one-CTA-per-item tcgen05 kernel for d = 128 too (a second implementation of the same maths, kept
 * as an A/B and cross-check variant; same results within the stated tolerance).
 * LVSA_KERNEL_TCGEN05_QUAD (d = 128, token-0 kv tiles): the CTA-pair kernel run as clusters of FOUR CTAs,
 * two MMA pairs working on adjacent work items that receive every K/V tile from ONE TMA load
 * (multicast), which halves the L2 -> SM traffic.
 * LVSA_KERNEL_TCGEN05_HYBRID: 4-CTA clusters on the SMs they can cover (a cluster needs four SMs of one GPC:
 * 132 of 148 on B200) and CTA pairs on the rest, as two launches side by side on the caller's stream and an
 * internal one (forked and joined with events; capturable). */
enum { LVSA_KERNEL_AUTO = 0, LVSA_KERNEL_SIMT = 1, LVSA_KERNEL_TCGEN05 = 2, LVSA_KERNEL_TCGEN05_V0 = 3,
       LVSA_KERNEL_TCGEN05_QUAD = 4, LVSA_KERNEL_TCGEN05_HYBRID = 5 };
/* Memory order of q, k, v, out (PAPER.md:31 fixes only N = T*P, not the order of the axes):
 * NHD = [B, N, H, d] (default), HND = [B, H, N, d]; d is always fastest.  lse is [B, H, N] in both.
 * Neither is faster: measured on B200 at H = 12 and H = 40 (token stride 3 KB / 10 KB vs 256 B) the time
 * differs by under 0.5 % and the DRAM traffic is the same (profiles/r03_README.md), so use the order the
 * producer of q, k, v has and do not transpose for this library. */
enum { LVSA_LAYOUT_NHD = 0, LVSA_LAYOUT_HND = 1 };
/* How the key/value tokens are cut into kv tiles (cost only: the result is Eq. 2 either way; the paper
 * does not say how tokens map to blocks):
 *   TOKEN0        : tile j = tokens [j*tile_k, (j+1)*tile_k), from token 0 (reading R14).
 *   FRAME_ALIGNED : kv tiles restart at every frame boundary: a frame of P tokens (the text pseudo-frame:
 *                   n_text) is cut into ceil(P/tile_k) tiles, all tile_k wide except the frame's last
 *                   (reading R25).  Every kv tile then lies inside one frame, so a query row attends to a
 *                   tile as a whole or not at all; the kernels compute a tile over its width rounded up
 *                   to LVSA_KV_PAD columns.  Accepted by the CTA-pair kernel (d = 128) and the SIMT
 *                   kernel; LVSA_EUNSUPPORTED with the one-CTA-per-item tcgen05 kernel (d = 64, _V0). */
enum { LVSA_KV_TILES_TOKEN0 = 0, LVSA_KV_TILES_FRAME_ALIGNED = 1 };
#define LVSA_KV_PAD 32 /* column granularity of a narrow kv tile (FRAME_ALIGNED) */

/* Parameters of lvsa_build_block_index_ex.  Zero means "default" where a default is named. */
typedef struct lvsa_params {
    int32_t T;          /* latent frames, >= 1                                                  */
    int32_t P;          /* tokens per frame, >= 1; T*P < 2^31                                    */
    int32_t H;          /* heads, >= 1                                                           */
    int32_t d;          /* head dim: 64 or 128                                                   */
    int32_t B;          /* batch, default 1                                                      */
    int32_t window;     /* W >= 0                                                  */
    int32_t anchors;    /* a = C-(2W+1) >= 0; a >= T: every frame is an anchor;
                           a == 0: no anchors; LVSA_ANCHORS_ALL_TILES: dense                    */
    int32_t step;       /* denoising step s >= 0 (Eq. 3)                                        */
    int32_t layer;      /* >= 0; recorded, does not change the pattern (reading R4)   */
    int32_t tile_q;     /* default: 128 when d = 128, 64 when d = 64; must equal tile_k         */
    int32_t tile_k;
    int32_t tie_break;  /* LVSA_TIE_LO (default) or LVSA_TIE_HI                                 */
    int32_t dtype;      /* LVSA_DTYPE_BF16 (default, tensor-core kernel) or LVSA_DTYPE_FP32
                           (SIMT kernel only)                                                   */
    int32_t kernel;     /* LVSA_KERNEL_AUTO: tcgen05 for bf16, SIMT for fp32; or one of the
                           LVSA_KERNEL_* values above                                           */
    float softmax_scale;/* default 1/sqrt(d) (Eq. 1)                                            */
    int32_t initial_anchors; /* k0 >= 0 dedicated initial anchors: frames 0..k0-1 join G^s at every
                           step (reading R22).  0 = the paper's pattern */
    int32_t n_text;     /* >= 0 extra tokens after the T*P video tokens (HunyuanVideo's text tokens
                           inside self-attention).  Every query attends to them and they
                           attend to every token (reading R23).  N = T*P + n_text.          */
    int32_t layout;     /* LVSA_LAYOUT_NHD (default) or LVSA_LAYOUT_HND: memory order of q,k,v,out     */
    int32_t host_groups;/* lvsa_attn_fwd_host only: number of head groups the call is pipelined over
                           (0 = default: one head per group, at most 16 groups; 1 = unpipelined)      */
    int32_t kv_tiling;  /* LVSA_KV_TILES_TOKEN0 (default) or LVSA_KV_TILES_FRAME_ALIGNED               */
    /* Free strides (PAPER.md:31 fixes only N = T*P, not where the tokens of q, k, v live).  Per tensor,
     * the ELEMENT strides of the {token, head, batch} axes; the d elements of one (token, head) are always
     * contiguous.  An all-zero triplet (the default) means "derive from `layout`".  With them a fused
     * projection output [B, N, 3, H, d] feeds q, k, v without a copy: pass the three base pointers and
     * {3*H*d, d, N*3*H*d} for each.  Every stride must be >= 0, a multiple of 16 bytes (8 bf16 / 4 fp32
     * elements), the token stride >= d, and the byte strides < 2^40 (TMA); else LVSA_EINVAL.  lse stays
     * [B, H, N].  lvsa_attn_fwd_host takes layout-derived strides only (LVSA_EUNSUPPORTED otherwise). */
    int64_t stride_q[3], stride_k[3], stride_v[3], stride_out[3];
} lvsa_params_t;

typedef struct lvsa_index_info {
    int32_t T, P, H, d, B;
    int32_t window, anchors, step, layer;
    int32_t tile_q, tile_k;
    int32_t nq, nk;          /* ceil(N/tile_q), ceil(N/tile_k)                                  */
    int32_t T_per;           /* 0 when there are no anchors                                     */
    int32_t phase;           /* s mod T_per                                                     */
    int32_t n_global;        /* |G^s|                                                           */
    int32_t words;           /* uint32 words per A(t) bitset = ceil(T'/32), T' = T + (n_text>0) */
    int32_t dtype, kernel;
    int32_t n_text;          /* text tokens after the video tokens (R23)                        */
    int32_t initial_anchors; /* dedicated initial anchors k0 (R22)                              */
    int32_t layout;          /* LVSA_LAYOUT_*                                                   */
    int32_t kv_tiling;       /* LVSA_KV_TILES_*                                                 */
    int32_t reserved0;       /* 0                                                               */
    int64_t N;               /* T*P + n_text                                                    */
    int64_t nnz;             /* kept (q tile, kv tile) pairs                                    */
    int64_t kept_cols;       /* sum over the kept pairs of the kv columns a kernel computes for
                                them (tile_k, or the width rounded up to LVSA_KV_PAD for a narrow
                                FRAME_ALIGNED tile): computed work = tile_q * kept_cols * 4d flop
                                per head and batch                                              */
    int64_t n_partial;       /* of which PARTIAL                                                */
    int64_t n_items;         /* work items of the attention kernel (q-tile groups)              */
    int64_t n_item_tiles;    /* kv-tile visits over all items (>= nnz / rows-per-item ratio)    */
} lvsa_index_info_t;

/*
 * lvsa_build_block_index — steps a1..a5 of the hot path on the GPU (Alg. 1
 * :74-89, Eq. 3 :97, Def. 2 :49; tile mapping per DESIGN.md reading R14).
 * Builds, for denoising step `step`, the per-frame attended sets A(t) and the CSR of kept
 * kv tiles per q tile (tile = 128 tokens for d = 128, 64 for d = 64; q tiles start at token 0, kv
 * tiles too unless lvsa_params_t.kv_tiling says FRAME_ALIGNED):
 *   indptr[nq+1], indices[nnz] ascending within a q tile, flags[nnz] in {FULL, PARTIAL}.
 * A kv tile is kept iff some (valid query row, valid key column) pair is allowed; it is PARTIAL
 * iff some (valid row, column of the tile) pair is not (frame not attended, or column >= N).
 * All arithmetic is integer and runs in CUDA kernels on the current device's default stream.
 * The call only ENQUEUES the four builder kernels and returns: it never synchronises.  Device
 * buffers come from one stream-ordered allocation sized by an upper bound on nnz (no device
 * round trip); the counters (nnz, ...) are read back lazily by lvsa_index_info /
 * lvsa_index_copy_host, which do synchronise.  Use the index on the stream it was built on (or
 * order other streams after it).  Returns NULL on error (lvsa_last_error()).
 * The handle is owned by the library; free it with lvsa_index_destroy.  Its contents never change
 * and it may be used by any number of lvsa_attn_fwd calls, but a handle is NOT thread-safe: the
 * library records on it which stream used it last (to free its stream-ordered memory behind that
 * work), so calls that share one handle must be serialised by the caller.  Different handles may
 * be used from different threads.  The index belongs to the device that was current when it was
 * built; every later call with it must be made with that device current (else LVSA_EINVAL).
 */
lvsa_index_t *lvsa_build_block_index(int T, int P, int H, int d, int window, int anchors,
                                     int step, int layer);

/* Same with every knob; `stream` is the cudaStream_t the builder kernels run on (NULL = default). */
lvsa_status_t lvsa_build_block_index_ex(const lvsa_params_t *params, void *stream,
                                        lvsa_index_t **out);

/*
 * lvsa_build_csr_static — the same block index (steps a1..a5: Alg. 1 :74-89, Eq. 3
 * :97, Def. 2 :49; token-0 kv tiles, reading R14) for callers that are not allowed to allocate
 * device memory.
 *
 * When to use it.  An inference server commonly gives the whole GPU to one allocator when the model
 * is loaded (a framework's caching pool, or a fixed memory plan).  Code that runs inside such a
 * process during the denoising loop (an attention plugin, a step callback) should then not ask the
 * CUDA driver for memory itself: the request can fail although the pool has room, it stalls the other
 * streams of the process while it is served, and the memory is invisible to the host's accounting.
 * lvsa_build_block_index(_ex) allocates an arena per index; THIS call allocates nothing, neither
 * directly (no cudaMalloc / cudaMallocAsync / cudaFree) nor through a library routine.  The caller
 * passes the output arrays; the intermediate data of the build (the A(t) bitsets and the per-q-tile
 * counts) go to a fixed LVSA_STATIC_SCRATCH_BYTES array inside the library image, which every GPU that
 * loads liblvsa holds until the process exits.
 *
 *   params   : as lvsa_build_block_index_ex.  Used: T, P, d, tile_q, tile_k, window, anchors, step,
 *              tie_break, initial_anchors, n_text.  kv_tiling must be LVSA_KV_TILES_TOKEN0.  The other
 *              fields (H, B, layer, dtype, kernel, softmax_scale, layout, host_groups) do not change
 *              the index and are ignored.
 *   indptr   : DEVICE, int32[nq + 1], nq = ceil((T*P + n_text) / tile_q).  Always written.
 *   indices  : DEVICE, int32[capacity]: kept kv tiles, ascending within a q tile.
 *   flags    : DEVICE, uint8[capacity]: LVSA_TILE_FULL / LVSA_TILE_PARTIAL per entry.
 *   capacity : entries `indices` and `flags` can hold (nq * ceil(N / tile_k) always suffices).
 *   nnz      : DEVICE, int32[1]: receives the number of kept (q tile, kv tile) pairs.  If it is
 *              larger than `capacity`, indices and flags were left untouched (indptr is still valid):
 *              call again with larger arrays.  The host learns this only by reading *nnz.
 *   stream   : cudaStream_t the four kernels are enqueued on (NULL = default stream).
 * The caller owns all four arrays; the library keeps no reference.  The call only enqueues and never
 * synchronises.  The result is bit-identical to lvsa_index_copy_host of an index built from the same
 * parameters.
 *
 * Limits: T + (n_text > 0) <= LVSA_STATIC_MAX_FRAMES and nq <= LVSA_STATIC_MAX_Q_TILES (about 2.1 M
 * tokens at 128-token tiles; the largest shape of the paper has 1475 q tiles), else LVSA_EUNSUPPORTED
 * with a message that names the limit; argument errors are LVSA_EINVAL as for the _ex call.  All of
 * these are checked on the host before anything is enqueued.
 *
 * Sharing.  All calls on one device use the same scratch array, and it keeps what the last call left
 * in it (each call resets the words that must start at zero, on the stream, before using them).  Two
 * calls whose kernels can overlap on the GPU (different streams with no ordering between them, or two
 * host threads) race on it and give wrong indices: order them.  The outputs of a finished call do not
 * depend on the array any more.
 *
 * First call.  The first call made on a device (with that device current) looks up the device address
 * of the array (cudaGetSymbolAddress) and remembers it; make that first call during set-up, outside
 * any stream capture.  Later calls on that device only launch kernels.
 */
#define LVSA_STATIC_MAX_FRAMES 512
#define LVSA_STATIC_MAX_Q_TILES 16384
#define LVSA_STATIC_SCRATCH_BYTES (97 * 1024)
lvsa_status_t lvsa_build_csr_static(const lvsa_params_t *params, void *stream, int32_t *indptr,
                                    int32_t *indices, uint8_t *flags, int64_t capacity, int32_t *nnz);

/*
 * lvsa_attn_fwd — step a6/a7: Eq. 2 over the kept tiles, exactly (element-level masking on
 * PARTIAL tiles).
 *   q, k, v : DEVICE pointers, contiguous [B, N, H, d] (or [B, H, N, d] when the index was built
 *             with LVSA_LAYOUT_HND; or with the strides given in lvsa_params_t.stride_q/k/v), d
 *             fastest, bf16 (or fp32 when the index was built with LVSA_DTYPE_FP32); 16-byte aligned.
 *             Read-only.
 *   out     : DEVICE pointer, same shape, layout and dtype as q.  Every element is written.
 *   lse     : DEVICE pointer, fp32 [B, H, N], 4-byte aligned, lse = ln sum_{kept} exp(q.k/sqrt d)
 *             (natural log), or NULL.
 *   stream  : cudaStream_t of the caller (NULL = default stream).
 * The call only enqueues work on `stream` and returns; it never synchronises and allocates
 * nothing.  Caller owns all five buffers; the library keeps no reference after the kernels ran.
 * bf16 inputs: products and sums accumulate in fp32, softmax statistics in fp32, P rounded to
 * bf16 before P.V, bf16 output.
 */
lvsa_status_t lvsa_attn_fwd(const void *q, const void *k, const void *v,
                            const lvsa_index_t *index, void *out, float *lse, void *stream);

/*
 * lvsa_attn_fwd_host — the same call for HOST buffers (pinned or pageable): copies q, k, v to
 * a device workspace owned by the library (one per process, allocated on first use, grown on
 * demand, shared by all indices; freed by lvsa_workspace_release), runs lvsa_attn_fwd on
 * `stream`, copies out (and lse if not NULL) back, and synchronises `stream` before returning.
 * With the CTA-pair kernel (bf16, d = 128) the call is pipelined over groups of heads (by default
 * one head per group, at most 16 groups; lvsa_params_t.host_groups overrides): the host-to-device
 * copy of the next group and the device-to-host copy of the previous one run on two internal
 * streams while the kernel of the current group runs on `stream`.  Results are identical to the
 * unpipelined call.  Calls through the workspace are serialised by a mutex.  If a CUDA call fails
 * part-way, the call waits for everything it enqueued before it returns the error, so no copy is
 * still reading or writing the caller's host buffers afterwards.
 */
lvsa_status_t lvsa_attn_fwd_host(const void *q_host, const void *k_host, const void *v_host,
                                 lvsa_index_t *index, void *out_host, float *lse_host,
                                 void *stream);

/*
 * Whole-schedule driver.  The pattern of step s depends on s only
 * through s mod T_per (Eq. 3), so a schedule of S denoising steps x L layers uses at
 * most T_per distinct indices.  Where the paper recomputes the metadata on the CPU at every step
 * (PAPER.md:104-110), lvsa_schedule_create builds all T_per indices once, on `stream`, without
 * synchronising; lvsa_schedule_attn_fwd then only launches the attention kernel, which makes a
 * whole S x L replay capturable in a CUDA graph (no allocation, no synchronisation, no index
 * build inside the captured region).  `params->step` is ignored.
 */
typedef struct lvsa_schedule lvsa_schedule_t;
lvsa_status_t lvsa_schedule_create(const lvsa_params_t *params, void *stream, lvsa_schedule_t **out);
/* number of distinct phases = T_per (1 when there are no rotating anchors); 0 on NULL */
int lvsa_schedule_num_phases(const lvsa_schedule_t *sched);
/* the index of denoising step `step` >= 0 (borrowed: owned by the schedule); NULL on error */
const lvsa_index_t *lvsa_schedule_index(const lvsa_schedule_t *sched, int step);
/* lvsa_attn_fwd with the index of `step`; same argument rules; enqueue only */
lvsa_status_t lvsa_schedule_attn_fwd(const lvsa_schedule_t *sched, int step, const void *q,
                                     const void *k, const void *v, void *out, float *lse,
                                     void *stream);
void lvsa_schedule_destroy(lvsa_schedule_t *sched);

/* Frees the device workspace of lvsa_attn_fwd_host (synchronises the device).  Safe to call
 * at any time when no lvsa_attn_fwd_host call is in flight; the next host call re-allocates. */
void lvsa_workspace_release(void);

/* Frees the index.  Its device buffers are stream-ordered memory: they are released behind the
 * work already enqueued on the stream that last used the index, without synchronising (if the
 * index was used on more than one stream the device is synchronised first). */
void lvsa_index_destroy(lvsa_index_t *index);

lvsa_status_t lvsa_index_info(const lvsa_index_t *index, lvsa_index_info_t *info);

/* Copies the index to HOST arrays sized from lvsa_index_info (any pointer may be NULL):
 * indptr[nq+1], indices[nnz], flags[nnz], w_lo[T], w_hi[T], a_bits[T'*words] with T' = T +
 * (n_text > 0 ? 1 : 0) rows (bit x of row t set iff x in A(t), little-endian words; row T is the
 * text pseudo-frame, R23).  Synchronises. */
lvsa_status_t lvsa_index_copy_host(const lvsa_index_t *index, int32_t *indptr, int32_t *indices,
                                   uint8_t *flags, int32_t *w_lo, int32_t *w_hi,
                                   uint32_t *a_bits);

/* The kv tiling of the index as HOST arrays of nk entries each (lvsa_index_info: nk): col0[j] = first
 * token of kv tile j, width[j] = its tokens (<= tile_k).  Either pointer may be NULL.  Pure host
 * arithmetic from the parameters; no device work. */
lvsa_status_t lvsa_index_copy_kv_tiles(const lvsa_index_t *index, int32_t *col0, int32_t *width);

/* Number of kernels lvsa_attn_fwd enqueues per call for this index (bench.py's gpu_launches): 1, or 2
 * for LVSA_KERNEL_TCGEN05_HYBRID when both of its parts get work (needs the index's device current;
 * -1 on error, 0 on NULL). */
int lvsa_attn_fwd_launches(const lvsa_index_t *index);

/* Number of kernels the build of this index enqueued: 4 (frames, count, scan, fill), 7 with the work lists
 * of the 4-CTA-cluster kernels (QUAD / HYBRID); two small memsets come on top. */
int lvsa_index_build_launches(const lvsa_index_t *index);

/* Number of CTAs the (persistent) tensor-core attention kernel is launched with for this index on its
 * device: 2 x the CTA pairs, or 4 x the 4-CTA clusters that can be resident at once
 * (LVSA_KERNEL_TCGEN05_QUAD; a cluster needs four SMs of one GPC, so some SMs stay idle).  0 for the
 * kernels that launch one CTA per work item, -1 on error. */
int lvsa_attn_fwd_grid(const lvsa_index_t *index);

/* Last error message of the calling thread ("" if none).  Never NULL. */
const char *lvsa_last_error(void);

/* Library version / build string (arch, kernel variants compiled in). */
const char *lvsa_version(void);

#ifdef __cplusplus
}
#endif
#endif /* LVSA_H_ */
