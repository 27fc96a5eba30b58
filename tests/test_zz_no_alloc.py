"""lvsa_build_csr_static: the block index for callers that must not allocate device memory.

Some users of this library run inside a process whose GPU memory already belongs to somebody else:
an inference server that gave the whole device to its caching allocator when it loaded the model,
and now calls the attention plugin once per denoising step.  Such a caller cannot let the library
take memory from the CUDA driver behind the allocator's back (the request may be refused, and it
stalls the other streams while it is served), so the handle-based builder, which allocates an arena
per index, is not for it.  lvsa_build_csr_static writes the same CSR into arrays the caller brings
and keeps its intermediate data in one fixed array inside the library (limits:
LVSA_STATIC_MAX_FRAMES frame rows, LVSA_STATIC_MAX_Q_TILES q tiles).

What is checked: the CSR is bit-identical to the one the handle-based path returns (integer work:
the tolerance of every index test here is zero), on two calls in a row that share the scratch array
- the second on a smaller problem, so data the first call left behind would show -, the driver's free
memory does not move between the calls, a list that does not fit is reported and does not poison
the next call, and sizes beyond the limits are refused on the host.

This file is named to be collected last: pytest -x stops at the first failure, and a failure here
must not hide the other tests.  It passes alone in a fresh process and after the other tests.
"""
import numpy as np
import pytest
import torch

from paper_2605_31057_b200 import binding, inputs


def handle_path_csr(**kw):
    """indptr, indices, flags through the existing path: lvsa_build_block_index_ex + copy_host."""
    ix = binding.lvsa_build_block_index_ex(H=1, **kw)
    host = ix.copy_host()
    ix.destroy()
    return host.indptr, host.indices, host.flags


class CallerArrays:
    """Output arrays the caller owns, allocated once, before the calls under test."""

    def __init__(self, nq_max, capacity):
        dev = torch.device("cuda:0")
        self.indptr = torch.full((nq_max + 1,), -7, dtype=torch.int32, device=dev)
        self.indices = torch.full((capacity,), -7, dtype=torch.int32, device=dev)
        self.flags = torch.full((capacity,), 77, dtype=torch.uint8, device=dev)
        self.nnz = torch.full((1,), -7, dtype=torch.int32, device=dev)


def num_tiles(kw):
    N = kw["T"] * kw["P"] + kw.get("n_text", 0)
    return -(-N // kw["d"])


@pytest.mark.gpu
def test_two_calls_in_a_row_match_the_handle_path_and_allocate_nothing():
    w = inputs.WORKLOADS["wan1.3b_1x"]
    first = dict(T=w.T, P=w.P, d=w.d, window=w.W, anchors=w.a, step=1)
    # smaller, with the optional parts of the pattern switched on (text row, dedicated anchors, tie-break)
    second = dict(T=9, P=200, d=128, window=1, anchors=3, step=5, n_text=70, initial_anchors=1,
                  tie_break=binding.TIE_HI)
    want = [handle_path_csr(**first), handle_path_csr(**second)]
    arr = CallerArrays(max(num_tiles(first), num_tiles(second)), max(len(want[0][1]), len(want[1][1])) + 5)
    torch.cuda.synchronize()

    got, free = [], []
    for kw in (first, second):
        binding.lvsa_build_csr_static(arr.indptr, arr.indices, arr.flags, arr.nnz, **kw)
        torch.cuda.synchronize()
        free.append(torch.cuda.mem_get_info()[0])     # before any torch work of our own
        nq, nnz = num_tiles(kw), int(arr.nnz.item())
        got.append((arr.indptr[:nq + 1].cpu().numpy(), arr.indices[:nnz].cpu().numpy(),
                    arr.flags[:nnz].cpu().numpy(), arr.indices[nnz:].cpu().numpy()))
    for (indptr, indices, flags), (g_indptr, g_indices, g_flags, g_rest) in zip(want, got):
        assert np.array_equal(g_indptr, indptr)
        assert np.array_equal(g_indices, indices)
        assert np.array_equal(g_flags, flags)
    # nothing was written past nnz in the second call: entries there are the first call's or the fill value
    assert len(want[1][1]) < len(want[0][1])
    assert np.array_equal(got[1][3][:len(want[0][1]) - len(want[1][1])], want[0][1][len(want[1][1]):])
    assert (got[1][3][len(want[0][1]) - len(want[1][1]):] == -7).all()
    assert free[0] == free[1], "the driver's free device memory moved between two calls"


@pytest.mark.gpu
def test_a_list_that_does_not_fit_is_reported_and_the_next_call_is_clean():
    kw = dict(T=12, P=50, d=64, window=1, anchors=2, step=3)
    indptr, indices, flags = handle_path_csr(**kw)
    nq = num_tiles(kw)
    small = CallerArrays(nq, len(indices) - 1)
    binding.lvsa_build_csr_static(small.indptr, small.indices, small.flags, small.nnz, **kw)
    assert int(small.nnz.item()) == len(indices) > small.indices.numel()
    assert (small.indices == -7).all() and (small.flags == 77).all()       # untouched
    assert np.array_equal(small.indptr.cpu().numpy(), indptr)               # still valid
    exact = CallerArrays(nq, len(indices))                                  # the raised flag must not stick
    binding.lvsa_build_csr_static(exact.indptr, exact.indices, exact.flags, exact.nnz, **kw)
    assert int(exact.nnz.item()) == len(indices)
    assert np.array_equal(exact.indices.cpu().numpy(), indices)
    assert np.array_equal(exact.flags.cpu().numpy(), flags)
    # the all-tiles path (Eq. 1) and a side stream
    dense = dict(T=5, P=128, d=128, anchors=binding.ALL_TILES)
    d_indptr, d_indices, d_flags = handle_path_csr(**dense)
    out = CallerArrays(num_tiles(dense), len(d_indices))
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        binding.lvsa_build_csr_static(out.indptr, out.indices, out.flags, out.nnz, **dense)
    side.synchronize()
    assert np.array_equal(out.indptr.cpu().numpy(), d_indptr)
    assert np.array_equal(out.indices.cpu().numpy(), d_indices)
    assert np.array_equal(out.flags.cpu().numpy(), d_flags)


class _FakeDeviceArray:
    """Stands in for a CUDA tensor where the call must fail on the host before touching the device."""
    is_cuda = True

    def __init__(self, n):
        self._buf = np.zeros(n, np.int32)

    def is_contiguous(self):
        return True

    def data_ptr(self):
        return self._buf.ctypes.data

    def numel(self):
        return self._buf.size


def test_sizes_beyond_the_fixed_scratch_are_refused_on_the_host():
    a = _FakeDeviceArray(16)
    call = lambda **kw: binding.lvsa_build_csr_static(a, a, a, a, stream=0, **kw)
    with pytest.raises(binding.LvsaError) as ei:
        call(T=binding.STATIC_MAX_FRAMES + 1, P=4, d=64)
    assert ei.value.status == binding.EUNSUPPORTED and "LVSA_STATIC_MAX_FRAMES" in str(ei.value)
    with pytest.raises(binding.LvsaError) as ei:                # the text row counts as a frame row
        call(T=binding.STATIC_MAX_FRAMES, P=4, d=64, n_text=3)
    assert ei.value.status == binding.EUNSUPPORTED and "LVSA_STATIC_MAX_FRAMES" in str(ei.value)
    with pytest.raises(binding.LvsaError) as ei:
        call(T=64, P=(binding.STATIC_MAX_Q_TILES * 128) // 64 + 2, d=128)
    assert ei.value.status == binding.EUNSUPPORTED and "LVSA_STATIC_MAX_Q_TILES" in str(ei.value)
    with pytest.raises(binding.LvsaError) as ei:
        call(T=4, P=4, d=64, kv_tiling=binding.KV_TILES_FRAME_ALIGNED)
    assert ei.value.status == binding.EUNSUPPORTED
    for bad in (dict(T=0, P=4, d=64), dict(T=4, P=4, d=64, window=-1), dict(T=4, P=4, d=64, anchors=-2),
                dict(T=4, P=4, d=64, step=-1), dict(T=4, P=4, d=64, tie_break=3)):
        with pytest.raises(binding.LvsaError) as ei:
            call(**bad)
        assert ei.value.status == binding.EINVAL, bad


def test_header_limits_match_binding_and_scratch_is_modest():
    import os
    import re
    src = open(os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "include", "lvsa.h")).read()
    assert int(re.search(r"#define LVSA_STATIC_MAX_FRAMES (\d+)", src).group(1)) == binding.STATIC_MAX_FRAMES
    assert int(re.search(r"#define LVSA_STATIC_MAX_Q_TILES (\d+)", src).group(1)) == binding.STATIC_MAX_Q_TILES
    kib = int(re.search(r"#define LVSA_STATIC_SCRATCH_BYTES \((\d+) \* 1024\)", src).group(1))
    assert kib <= 128
