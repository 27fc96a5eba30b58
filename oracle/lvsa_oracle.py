"""ctypes front end of oracle/lvsa_oracle.c — TEST INFRASTRUCTURE, NOT THE PRODUCT.

Argument marshalling only; every number comes from the C file, which restates
PAPER.md (Def. 2 :49, Eq. 2 :42, Eq. 3 :97, :62, :68, Algorithm 1 :74-89) in fp64 /
exact integers.  Nothing here imports the CUDA package and the CUDA package never
imports this.  Allowed callers: tests/, __graft_entry__.smoke(), bench.py's
cpu_baseline and --impl reference legs.
"""
from __future__ import annotations

import ctypes as C
import os
import re
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lvsa_oracle.c")


def _cpu_flags() -> list[str]:
    """-mavx2 -mfma only when this host has them (the .so may travel to another box)."""
    try:
        with open("/proc/cpuinfo") as f:
            txt = f.read()
    except OSError:
        return []
    m = re.search(r"^flags\s*:\s*(.*)$", txt, re.M)
    have = set(m.group(1).split()) if m else set()
    return ["-mavx2", "-mfma"] if {"avx2", "fma"} <= have else []


_FLAGS = _cpu_flags()
_LIB = os.path.join(_HERE, "liblvsa_oracle_avx2.so" if _FLAGS else "liblvsa_oracle.so")

ALL_TILES = -1


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O3, OpenMP, no fast-math)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O3", *_FLAGS, "-fopenmp", "-shared", "-fPIC", "-std=gnu11",
               "-o", _LIB, _SRC, "-lm"]
        try:
            subprocess.run(cmd, check=True, capture_output=True, text=True)
        except subprocess.CalledProcessError as e:  # pragma: no cover
            raise RuntimeError("oracle build failed:\n" + e.stderr) from e
    return _LIB


_lib = None


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.lvsa_oracle_tile_index.restype = C.c_int64
        _lib.lvsa_oracle_tile_index_fa.restype = C.c_int64
        _lib.lvsa_oracle_kv_tiles_frame_aligned.restype = C.c_int64
        _lib.lvsa_oracle_time_rebuild.restype = C.c_double
    return _lib


def _p(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


@dataclass
class Pattern:
    T: int
    W: int
    a: int
    s: int
    A: np.ndarray        # [T, T] uint8, row t = attended set of query frame t (Def. 2)
    w_lo: np.ndarray     # [T] int32 (Algorithm 1 output)
    w_hi: np.ndarray     # [T] int32
    inG: np.ndarray      # [T] uint8, membership in G^s (Eq. 3)
    iters: np.ndarray    # [T] int32, Algorithm 1 while-loop trip count
    T_per: int
    phase: int
    n_global: int

    def a_bits(self) -> np.ndarray:
        """A(t) packed little-endian into uint32 words, [T, ceil(T/32)]."""
        T = self.T
        nw = (T + 31) // 32
        out = np.zeros((T, nw), dtype=np.uint32)
        for t in range(T):
            for x in np.nonzero(self.A[t])[0]:
                out[t, x // 32] |= np.uint32(1) << np.uint32(x % 32)
        return out


def pattern(T: int, W: int, a: int, s: int, tie_hi: int = 0, initial_anchors: int = 0) -> Pattern:
    """Def. 2 with Eq. 3 and Algorithm 1; initial_anchors = k0 dedicated first frames added to
    G^s (reading R22; 0 = the paper's pattern)."""
    A = np.zeros((T, T), np.uint8)
    lo = np.zeros(T, np.int32)
    hi = np.zeros(T, np.int32)
    inG = np.zeros(T, np.uint8)
    it = np.zeros(T, np.int32)
    meta = np.zeros(3, np.int32)
    lib().lvsa_oracle_pattern_ex(C.c_int(T), C.c_int(W), C.c_int(a), C.c_int(s), C.c_int(tie_hi),
                                 C.c_int(initial_anchors), _p(A), _p(lo), _p(hi), _p(inG), _p(it),
                                 _p(meta))
    return Pattern(T, W, a, s, A, lo, hi, inG, it, int(meta[0]), int(meta[1]), int(meta[2]))


def with_text(A: np.ndarray) -> np.ndarray:
    """Frame-level pattern with the text pseudo-frame appended (reading R23 of
    PAPER.md:132): every video frame attends to the text tokens, the text tokens attend to every
    frame and to themselves.  [T, T] -> [T+1, T+1]."""
    T = A.shape[0]
    Af = np.ones((T + 1, T + 1), np.uint8)
    Af[:T, :T] = A
    return Af


def tile_index(T: int, P: int, Bq: int, Bk: int, A: np.ndarray, n_text: int = 0):
    """CSR (indptr, indices, flags) of kept kv tiles per q tile; flags 1 = PARTIAL.
    n_text > 0: A is the [T+1, T+1] pattern of with_text and N = T*P + n_text."""
    A = np.ascontiguousarray(A, np.uint8)
    assert A.shape == (T + (n_text > 0), T + (n_text > 0))
    N = T * P + n_text
    nq = (N + Bq - 1) // Bq
    indptr = np.zeros(nq + 1, np.int32)
    nnz = lib().lvsa_oracle_tile_index(C.c_int(T), C.c_int(P), C.c_int(n_text), C.c_int(Bq), C.c_int(Bk),
                                       _p(A), _p(indptr), None, None, C.c_int64(0))
    indices = np.zeros(max(nnz, 1), np.int32)
    flags = np.zeros(max(nnz, 1), np.uint8)
    got = lib().lvsa_oracle_tile_index(C.c_int(T), C.c_int(P), C.c_int(n_text), C.c_int(Bq), C.c_int(Bk),
                                       _p(A), _p(indptr), _p(indices), _p(flags), C.c_int64(nnz))
    assert got == nnz
    return indptr, indices[:nnz], flags[:nnz]


def kv_tiles_frame_aligned(T: int, P: int, Bk: int, n_text: int = 0):
    """Frame-aligned kv tiling (reading R25): (col0, width) per kv tile, token order."""
    nk = lib().lvsa_oracle_kv_tiles_frame_aligned(C.c_int(T), C.c_int(P), C.c_int(n_text), C.c_int(Bk),
                                                  None, None, C.c_int64(0))
    col0 = np.zeros(max(nk, 1), np.int32)
    width = np.zeros(max(nk, 1), np.int32)
    got = lib().lvsa_oracle_kv_tiles_frame_aligned(C.c_int(T), C.c_int(P), C.c_int(n_text), C.c_int(Bk),
                                                   _p(col0), _p(width), C.c_int64(nk))
    assert got == nk
    return col0[:nk], width[:nk]


def tile_index_fa(T: int, P: int, Bq: int, Bk: int, A: np.ndarray, n_text: int = 0, pad: int = 32):
    """CSR (indptr, indices, flags) over the frame-aligned kv tiling; flags 1 = PARTIAL (some row of
    the q tile does not attend to the tile's frame, or the tile is narrower than its padded width)."""
    A = np.ascontiguousarray(A, np.uint8)
    assert A.shape == (T + (n_text > 0), T + (n_text > 0))
    N = T * P + n_text
    nq = (N + Bq - 1) // Bq
    indptr = np.zeros(nq + 1, np.int32)
    args = (C.c_int(T), C.c_int(P), C.c_int(n_text), C.c_int(Bq), C.c_int(Bk), C.c_int(pad), _p(A), _p(indptr))
    nnz = lib().lvsa_oracle_tile_index_fa(*args, None, None, C.c_int64(0))
    indices = np.zeros(max(nnz, 1), np.int32)
    flags = np.zeros(max(nnz, 1), np.uint8)
    got = lib().lvsa_oracle_tile_index_fa(*args, _p(indices), _p(flags), C.c_int64(nnz))
    assert got == nnz
    return indptr, indices[:nnz], flags[:nnz]


def csr_keyset_equal_tiles(T, P, Bq, A, col0, width, indptr, indices, flags, rows, n_text: int = 0,
                           pad: int = 32) -> bool:
    A = np.ascontiguousarray(A, np.uint8)
    rows = np.ascontiguousarray(rows, np.int64)
    col0 = np.ascontiguousarray(col0, np.int32)
    width = np.ascontiguousarray(width, np.int32)
    indptr = np.ascontiguousarray(indptr, np.int32)
    indices = np.ascontiguousarray(indices, np.int32)
    flags = np.ascontiguousarray(flags, np.uint8)
    return bool(lib().lvsa_oracle_csr_keyset_equal_tiles(
        C.c_int(T), C.c_int(P), C.c_int(n_text), C.c_int(Bq), C.c_int(pad), _p(A), _p(col0), _p(width),
        _p(indptr), _p(indices), _p(flags), _p(rows), C.c_int64(rows.size)))


def _as_input(x) -> tuple[np.ndarray, int]:
    """Accept a numpy fp32 array or raw bf16 bits (uint16); returns (array, is_bf16)."""
    x = np.ascontiguousarray(x)
    if x.dtype == np.uint16:
        return x, 1
    if x.dtype == np.float32:
        return x, 0
    raise TypeError(f"oracle inputs must be float32 or uint16 (raw bf16), got {x.dtype}")


def attn_rows(q, k, v, T: int, P: int, A: np.ndarray, rows, scale: float = 0.0,
              nthreads: int = 0, n_text: int = 0):
    """Eq. 2 for the query tokens in `rows`, every head.  q,k,v: [N, H, d].
    Returns (out [nrows,H,d] fp64, lse [nrows,H] fp64)."""
    q, b0 = _as_input(q)
    k, b1 = _as_input(k)
    v, b2 = _as_input(v)
    assert b0 == b1 == b2 and q.shape == k.shape == v.shape and q.ndim == 3
    N, H, d = q.shape
    assert N == T * P + n_text and A.shape[0] == T + (n_text > 0)
    A = np.ascontiguousarray(A, np.uint8)
    rows = np.ascontiguousarray(rows, np.int64)
    assert rows.size == 0 or (rows.min() >= 0 and rows.max() < N)
    out = np.zeros((rows.size, H, d), np.float64)
    lse = np.zeros((rows.size, H), np.float64)
    lib().lvsa_oracle_attn_rows(_p(q), _p(k), _p(v), C.c_int(b0), C.c_int(T), C.c_int(P),
                                C.c_int(n_text), C.c_int(H), C.c_int(d), _p(A), _p(rows), C.c_int64(rows.size),
                                C.c_double(scale), _p(out), _p(lse), C.c_int(nthreads))
    return out, lse


def csr_keyset_equal(T, P, Bq, Bk, A, indptr, indices, flags, rows, n_text: int = 0) -> bool:
    A = np.ascontiguousarray(A, np.uint8)
    rows = np.ascontiguousarray(rows, np.int64)
    indptr = np.ascontiguousarray(indptr, np.int32)
    indices = np.ascontiguousarray(indices, np.int32)
    flags = np.ascontiguousarray(flags, np.uint8)
    return bool(lib().lvsa_oracle_csr_keyset_equal(
        C.c_int(T), C.c_int(P), C.c_int(n_text), C.c_int(Bq), C.c_int(Bk), _p(A), _p(indptr), _p(indices),
        _p(flags), _p(rows), C.c_int64(rows.size)))


def time_rebuild(T: int, W: int, a: int, S: int, reps: int = 200):
    """Report-only: seconds per metadata rebuild, max / mean Algorithm-1 loop count."""
    mx = C.c_int32(0)
    mean = C.c_double(0.0)
    sec = lib().lvsa_oracle_time_rebuild(C.c_int(T), C.c_int(W), C.c_int(a), C.c_int(S),
                                         C.c_int(reps), C.byref(mx), C.byref(mean))
    return float(sec), int(mx.value), float(mean.value)


def num_threads() -> int:
    return int(lib().lvsa_oracle_num_threads())
