"""Thin ctypes binding over csrc/liblvsa.so (include/lvsa.h).  Argument marshalling only:
every step of the hot path (index build, attention) runs in the library's CUDA kernels.
PyTorch is used by callers for device memory and streams; this module only reads
`tensor.data_ptr()` and the current stream handle.

There is no CPU fallback.  If the library cannot be built or loaded, importing the symbols
raises; if there is no CUDA device, the library calls return LVSA_ECUDA and this module raises
LvsaError.  Nothing here imports oracle/.
"""
from __future__ import annotations

import ctypes as C
from dataclasses import dataclass

import numpy as np

from . import build as _build

ALL_TILES = -1
TILE_FULL, TILE_PARTIAL = 0, 1
TIE_LO, TIE_HI = 0, 1
DTYPE_BF16, DTYPE_FP32 = 0, 1
KERNEL_AUTO, KERNEL_SIMT, KERNEL_TCGEN05, KERNEL_TCGEN05_V0, KERNEL_TCGEN05_QUAD, KERNEL_TCGEN05_HYBRID = 0, 1, 2, 3, 4, 5
LAYOUT_NHD, LAYOUT_HND = 0, 1
KV_TILES_TOKEN0, KV_TILES_FRAME_ALIGNED = 0, 1
KV_PAD = 32
OK, EINVAL, EUNSUPPORTED, ECUDA, ENOMEM = 0, 1, 2, 3, 4


class LvsaError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"lvsa status {status}: {msg}")
        self.status = status


class Params(C.Structure):
    _fields_ = [(n, C.c_int32) for n in
                ("T", "P", "H", "d", "B", "window", "anchors", "step", "layer", "tile_q", "tile_k",
                 "tie_break", "dtype", "kernel")] + [("softmax_scale", C.c_float),
                                                     ("initial_anchors", C.c_int32),
                                                     ("n_text", C.c_int32),
                                                     ("layout", C.c_int32),
                                                     ("host_groups", C.c_int32),
                                                     ("kv_tiling", C.c_int32),
                                                     ("stride_q", C.c_int64 * 3), ("stride_k", C.c_int64 * 3),
                                                     ("stride_v", C.c_int64 * 3), ("stride_out", C.c_int64 * 3)]


class IndexInfo(C.Structure):
    _fields_ = [(n, C.c_int32) for n in
                ("T", "P", "H", "d", "B", "window", "anchors", "step", "layer", "tile_q", "tile_k",
                 "nq", "nk", "T_per", "phase", "n_global", "words", "dtype", "kernel", "n_text",
                 "initial_anchors", "layout", "kv_tiling", "reserved0")] + \
               [(n, C.c_int64) for n in ("N", "nnz", "kept_cols", "n_partial", "n_items", "n_item_tiles")]


EXPORTS = ("lvsa_build_block_index", "lvsa_build_block_index_ex", "lvsa_attn_fwd",
           "lvsa_attn_fwd_host", "lvsa_index_destroy", "lvsa_index_info", "lvsa_index_copy_host",
           "lvsa_index_copy_kv_tiles", "lvsa_attn_fwd_launches", "lvsa_attn_fwd_grid", "lvsa_workspace_release", "lvsa_schedule_create",
           "lvsa_schedule_num_phases", "lvsa_schedule_index", "lvsa_schedule_attn_fwd", "lvsa_schedule_destroy", "lvsa_last_error", "lvsa_version",
           "lvsa_build_csr_static", "lvsa_index_build_launches")

_lib = None


def lib() -> C.CDLL:
    """Loads (building first if the .so is missing or older than its sources) liblvsa.so."""
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        L.lvsa_build_block_index.restype = C.c_void_p
        L.lvsa_build_block_index.argtypes = [C.c_int] * 8
        L.lvsa_build_block_index_ex.restype = C.c_int
        L.lvsa_build_block_index_ex.argtypes = [C.POINTER(Params), C.c_void_p, C.POINTER(C.c_void_p)]
        L.lvsa_attn_fwd.restype = C.c_int
        L.lvsa_attn_fwd.argtypes = [C.c_void_p] * 7
        L.lvsa_attn_fwd_host.restype = C.c_int
        L.lvsa_attn_fwd_host.argtypes = [C.c_void_p] * 7
        L.lvsa_index_destroy.restype = None
        L.lvsa_index_destroy.argtypes = [C.c_void_p]
        L.lvsa_index_info.restype = C.c_int
        L.lvsa_index_info.argtypes = [C.c_void_p, C.POINTER(IndexInfo)]
        L.lvsa_index_copy_host.restype = C.c_int
        L.lvsa_index_copy_host.argtypes = [C.c_void_p] * 7
        L.lvsa_index_copy_kv_tiles.restype = C.c_int
        L.lvsa_index_copy_kv_tiles.argtypes = [C.c_void_p] * 3
        L.lvsa_attn_fwd_grid.restype = C.c_int
        L.lvsa_attn_fwd_grid.argtypes = [C.c_void_p]
        L.lvsa_attn_fwd_launches.restype = C.c_int
        L.lvsa_attn_fwd_launches.argtypes = [C.c_void_p]
        L.lvsa_index_build_launches.restype = C.c_int
        L.lvsa_index_build_launches.argtypes = [C.c_void_p]
        L.lvsa_workspace_release.restype = None
        L.lvsa_workspace_release.argtypes = []
        L.lvsa_schedule_create.restype = C.c_int
        L.lvsa_schedule_create.argtypes = [C.POINTER(Params), C.c_void_p, C.POINTER(C.c_void_p)]
        L.lvsa_schedule_num_phases.restype = C.c_int
        L.lvsa_schedule_num_phases.argtypes = [C.c_void_p]
        L.lvsa_schedule_index.restype = C.c_void_p
        L.lvsa_schedule_index.argtypes = [C.c_void_p, C.c_int]
        L.lvsa_schedule_attn_fwd.restype = C.c_int
        L.lvsa_schedule_attn_fwd.argtypes = [C.c_void_p, C.c_int] + [C.c_void_p] * 6
        L.lvsa_schedule_destroy.restype = None
        L.lvsa_schedule_destroy.argtypes = [C.c_void_p]
        L.lvsa_build_csr_static.restype = C.c_int
        L.lvsa_build_csr_static.argtypes = [C.POINTER(Params), C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                            C.c_int64, C.c_void_p]
        L.lvsa_last_error.restype = C.c_char_p
        L.lvsa_version.restype = C.c_char_p
        _lib = L
    return _lib


def lvsa_last_error() -> str:
    return lib().lvsa_last_error().decode()


def lvsa_version() -> str:
    return lib().lvsa_version().decode()


def _check(status: int):
    if status != OK:
        raise LvsaError(status, lvsa_last_error())


@dataclass
class HostIndex:
    indptr: np.ndarray
    indices: np.ndarray
    flags: np.ndarray
    w_lo: np.ndarray
    w_hi: np.ndarray
    a_bits: np.ndarray


class BlockIndex:
    """One lvsa_index_t handle: owned (destroyed with the object) unless borrowed from a schedule."""

    def __init__(self, handle: int, owned: bool = True):
        self._h = C.c_void_p(handle)
        self._owned = owned

    @property
    def handle(self) -> C.c_void_p:
        if not self._h:
            raise ValueError("index already destroyed")
        return self._h

    def info(self) -> IndexInfo:
        info = IndexInfo()
        _check(lib().lvsa_index_info(self.handle, C.byref(info)))
        return info

    def copy_host(self) -> HostIndex:
        i = self.info()
        indptr = np.zeros(i.nq + 1, np.int32)
        indices = np.zeros(i.nnz, np.int32)
        flags = np.zeros(i.nnz, np.uint8)
        w_lo = np.zeros(i.T, np.int32)
        w_hi = np.zeros(i.T, np.int32)
        a_bits = np.zeros((i.T + (1 if i.n_text > 0 else 0), i.words), np.uint32)
        ptr = lambda a: a.ctypes.data_as(C.c_void_p)
        _check(lib().lvsa_index_copy_host(self.handle, ptr(indptr), ptr(indices), ptr(flags),
                                          ptr(w_lo), ptr(w_hi), ptr(a_bits)))
        return HostIndex(indptr, indices, flags, w_lo, w_hi, a_bits)

    def kv_tiles(self):
        """(col0, width) of every kv tile of the index's tiling (host arithmetic in the library)."""
        nk = self.info().nk
        col0, width = np.zeros(nk, np.int32), np.zeros(nk, np.int32)
        _check(lib().lvsa_index_copy_kv_tiles(self.handle, col0.ctypes.data_as(C.c_void_p),
                                              width.ctypes.data_as(C.c_void_p)))
        return col0, width

    def grid(self) -> int:
        """CTAs of the persistent attention launch for this index (0: one CTA per work item)."""
        return int(lib().lvsa_attn_fwd_grid(self.handle))

    def launches(self) -> int:
        return int(lib().lvsa_attn_fwd_launches(self.handle))

    def build_launches(self) -> int:
        """Kernels the build of this index enqueued (4, or 7 with the quad work lists)."""
        return int(lib().lvsa_index_build_launches(self.handle))

    def destroy(self):
        if self._h:
            if self._owned:
                lib().lvsa_index_destroy(self._h)
            self._h = C.c_void_p(None)

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def lvsa_build_block_index(T: int, P: int, H: int, d: int, window: int, anchors: int, step: int,
                           layer: int) -> BlockIndex:
    h = lib().lvsa_build_block_index(T, P, H, d, window, anchors, step, layer)
    if not h:
        raise LvsaError(-1, lvsa_last_error())
    return BlockIndex(h)


def lvsa_build_block_index_ex(stream: int = 0, **kw) -> BlockIndex:
    p = Params()
    for k, v in kw.items():
        if not hasattr(p, k):
            raise TypeError(f"unknown lvsa_params_t field {k!r}")
        setattr(p, k, v)
    out = C.c_void_p()
    _check(lib().lvsa_build_block_index_ex(C.byref(p), C.c_void_p(stream), C.byref(out)))
    return BlockIndex(out.value)


STATIC_MAX_FRAMES, STATIC_MAX_Q_TILES = 512, 16384


def lvsa_build_csr_static(indptr, indices, flags, nnz, stream: int | None = None, **kw) -> None:
    """The block index written into the caller's CUDA tensors, for callers that must not allocate device
    memory inside the denoising loop (a plugin in a server whose allocator owns the GPU): indptr int32
    [nq + 1], indices int32 [capacity], flags uint8 [capacity], nnz int32 [1]; capacity =
    min(len(indices), len(flags)).  `kw` are lvsa_params_t fields.  Enqueues on `stream` (default: torch's
    current stream) and returns; read `nnz` to learn whether the list fitted (include/lvsa.h).  Calls
    that can overlap on the GPU race on the library's fixed scratch array."""
    p = Params()
    for k, v in kw.items():
        if not hasattr(p, k):
            raise TypeError(f"unknown lvsa_params_t field {k!r}")
        setattr(p, k, v)
    if stream is None:
        import torch
        stream = torch.cuda.current_stream().cuda_stream
    cap = min(indices.numel(), flags.numel())
    _check(lib().lvsa_build_csr_static(C.byref(p), C.c_void_p(stream), _dev_ptr(indptr), _dev_ptr(indices),
                                       _dev_ptr(flags), C.c_int64(cap), _dev_ptr(nnz)))


def _dev_ptr(t, strided: bool = False) -> C.c_void_p:
    if t is None:
        return C.c_void_p(None)
    if strided:     # a view whose strides the index was built with (lvsa_params_t.stride_*): d must be contiguous
        if not t.is_cuda or t.stride(-1) != 1:
            raise ValueError("a strided operand must be a CUDA tensor with a contiguous last axis")
    elif not t.is_cuda or not t.is_contiguous():
        raise ValueError("lvsa_attn_fwd takes contiguous CUDA tensors")
    return C.c_void_p(t.data_ptr())


def tensor_strides(t):
    """{token, head, batch} element strides of a [B, N, H, d] view, as lvsa_params_t.stride_q/k/v/out take
    them (e.g. q = fused[:, :, 0] of a [B, N, 3, H, d] projection output).  The last axis must be contiguous."""
    if t.dim() != 4 or t.stride(3) != 1:
        raise ValueError("expected a [B, N, H, d] view with a contiguous last axis")
    return (t.stride(1), t.stride(2), t.stride(0))


def lvsa_attn_fwd(q, k, v, index: BlockIndex, out, lse=None, stream: int | None = None, strided: bool = False):
    """q, k, v, out: CUDA tensors [B, N, H, d] (or [B, H, N, d] for an index built with
    layout=LAYOUT_HND); lse: CUDA fp32 [B, H, N] or None.  Enqueues on
    `stream` (default: torch's current stream) and returns without synchronising.
    strided=True: q, k, v, out may be views; the index must have been built with their strides
    (stride_q=tensor_strides(q), ...), which only the caller can vouch for."""
    if stream is None:
        import torch
        stream = torch.cuda.current_stream().cuda_stream
    _check(lib().lvsa_attn_fwd(_dev_ptr(q, strided), _dev_ptr(k, strided), _dev_ptr(v, strided), index.handle,
                               _dev_ptr(out, strided), _dev_ptr(lse), C.c_void_p(stream)))
    return out


def lvsa_attn_fwd_host(q, k, v, index: BlockIndex, out, lse=None, stream: int = 0):
    """Host-buffer variant: q, k, v, out (and lse) are CPU tensors (ideally pinned); copies run
    inside the call, which returns after the results are back on the host."""
    hp = lambda t: C.c_void_p(None) if t is None else C.c_void_p(t.data_ptr())
    for t in (q, k, v, out):
        if t.is_cuda or not t.is_contiguous():
            raise ValueError("lvsa_attn_fwd_host takes contiguous CPU tensors")
    _check(lib().lvsa_attn_fwd_host(hp(q), hp(k), hp(v), index.handle, hp(out), hp(lse),
                                    C.c_void_p(stream)))
    return out


def lvsa_workspace_release() -> None:
    lib().lvsa_workspace_release()


class Schedule:
    """Owns one lvsa_schedule_t: the T_per distinct block indices of a denoising schedule."""

    def __init__(self, handle: int):
        self._h = C.c_void_p(handle)

    @property
    def handle(self) -> C.c_void_p:
        if not self._h:
            raise ValueError("schedule already destroyed")
        return self._h

    def num_phases(self) -> int:
        return int(lib().lvsa_schedule_num_phases(self.handle))

    def index(self, step: int) -> BlockIndex:
        """Borrowed view of the index of `step` (do not destroy it)."""
        h = lib().lvsa_schedule_index(self.handle, C.c_int(step))
        if not h:
            raise LvsaError(EINVAL, lvsa_last_error())
        return BlockIndex(h, owned=False)

    def destroy(self) -> None:
        if self._h:
            lib().lvsa_schedule_destroy(self._h)
            self._h = C.c_void_p(None)


def lvsa_schedule_create(stream: int = 0, **kw) -> Schedule:
    p = Params()
    for k, v in kw.items():
        if not hasattr(p, k):
            raise TypeError(f"unknown lvsa_params_t field {k!r}")
        setattr(p, k, v)
    out = C.c_void_p()
    _check(lib().lvsa_schedule_create(C.byref(p), C.c_void_p(stream), C.byref(out)))
    return Schedule(out.value)


def lvsa_schedule_attn_fwd(sched: Schedule, step: int, q, k, v, out, lse=None, stream: int | None = None):
    if stream is None:
        import torch
        stream = torch.cuda.current_stream().cuda_stream
    _check(lib().lvsa_schedule_attn_fwd(sched.handle, C.c_int(step), _dev_ptr(q), _dev_ptr(k), _dev_ptr(v),
                                        _dev_ptr(out), _dev_ptr(lse), C.c_void_p(stream)))
    return out
