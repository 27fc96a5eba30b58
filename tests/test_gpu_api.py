"""C-ABI behaviour on the GPU beyond parity: the host-buffer entry point and its workspace, handle
lifetime with stream-ordered memory, optional outputs, argument errors."""
import ctypes as C

import numpy as np
import pytest
import torch

from helpers import build_index, gpu_attn
from paper_2605_31057_b200 import binding, inputs

pytestmark = pytest.mark.gpu


def test_host_entry_point_matches_device_path_and_workspace_lifecycle():
    small, big = inputs.WORKLOADS["tiny_straddle"], inputs.WORKLOADS["small128"]
    for w in (small, big, small):            # the workspace grows for `big`, then is reused
        q, k, v = inputs.make_qkv(w, "cuda", torch.bfloat16)
        ix = build_index(w, 1)
        want, want_lse = gpu_attn(w, ix, q, k, v)
        qh, kh, vh = (x.cpu() for x in (q, k, v))                       # pageable host memory
        oh = torch.empty_like(qh)
        lh = torch.empty((w.B, w.H, w.N), dtype=torch.float32)
        binding.lvsa_attn_fwd_host(qh, kh, vh, ix, oh, lh)
        assert torch.equal(oh, want.cpu()) and torch.equal(lh, want_lse.cpu())
        qp, kp, vp = (x.pin_memory() for x in (qh, kh, vh))             # pinned, no lse
        op = torch.empty_like(qp).pin_memory()
        binding.lvsa_attn_fwd_host(qp, kp, vp, ix, op, None)
        assert torch.equal(op, want.cpu())
        ix.destroy()
    binding.lvsa_workspace_release()
    binding.lvsa_workspace_release()                                    # idempotent
    w = small
    q, k, v = inputs.make_qkv(w, "cuda", torch.bfloat16)
    ix = build_index(w, 0)
    want, _ = gpu_attn(w, ix, q, k, v)
    oh = torch.empty_like(q, device="cpu")
    binding.lvsa_attn_fwd_host(q.cpu(), k.cpu(), v.cpu(), ix, oh, None)  # re-allocates after release
    assert torch.equal(oh, want.cpu())
    ix.destroy()


@pytest.mark.parametrize("layout", ["nhd", "hnd"])
@pytest.mark.parametrize("host_groups", [0, 1, 3, 16])
def test_host_entry_point_head_groups(host_groups, layout):
    """The pipelined host path with several heads per group and a short last group (H = 20: 16 groups of
    2 heads -> 10 used; 3 groups of 7, 7, 6), B = 2 (strided lse copy with pitch H*N), lse requested, in
    both memory orders; bitwise equal to the device path."""
    w = inputs.Workload("host_b2_h20", 1, T=5, P=150, H=20, d=128, tile=128, W=1, a=2, B=2)
    q, k, v = inputs.make_qkv(w, "cuda", torch.bfloat16)
    kw = dict(host_groups=host_groups)
    if layout == "hnd":
        q, k, v = (x.transpose(1, 2).contiguous() for x in (q, k, v))
        kw["layout"] = binding.LAYOUT_HND
    ix = build_index(w, 1, **kw)
    want, want_lse = gpu_attn(w, ix, q, k, v)
    qh, kh, vh = (x.cpu().pin_memory() for x in (q, k, v))
    oh = torch.full_like(qh, float("nan"))
    lh = torch.full((w.B, w.H, w.N), float("nan"), dtype=torch.float32)
    binding.lvsa_attn_fwd_host(qh, kh, vh, ix, oh, lh)
    assert torch.equal(oh, want.cpu()) and torch.equal(lh, want_lse.cpu())
    ix.destroy()


def test_lse_is_optional_and_outputs_do_not_depend_on_it():
    w = inputs.WORKLOADS["small128"]
    q, k, v = inputs.make_qkv(w, "cuda", torch.bfloat16)
    ix = build_index(w, 2)
    a, _ = gpu_attn(w, ix, q, k, v, want_lse=True)
    b, none = gpu_attn(w, ix, q, k, v, want_lse=False)
    assert none is None and torch.equal(a, b)
    ix.destroy()


def test_index_rebuild_loop_reuses_its_arena():
    """Per-step rebuilds must not grow device memory: the arena comes from a
    stream-ordered pool and goes back to it in lvsa_index_destroy."""
    w = inputs.WORKLOADS["wan1.3b_1x"]
    for s in range(4):
        build_index(w, s).destroy()
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for s in range(300):
        ix = build_index(w, s)
        ix.destroy()
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free0 - free1 < 64 << 20, (free0, free1)


def test_index_used_on_two_streams_and_destroyed():
    w = inputs.WORKLOADS["small128"]
    q, k, v = inputs.make_qkv(w, "cuda", torch.bfloat16)
    ix = build_index(w, 1)
    want, _ = gpu_attn(w, ix, q, k, v)
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    out = torch.empty_like(q)
    binding.lvsa_attn_fwd(q, k, v, ix, out, None, stream=side.cuda_stream)
    ix.destroy()                      # used on two streams: destroy waits for the device first
    torch.cuda.synchronize()
    assert torch.equal(out, want)


def test_info_agrees_with_copied_index_and_is_idempotent():
    w = inputs.WORKLOADS["small128"]
    ix = build_index(w, 3)
    a, b = ix.info(), ix.info()
    host = ix.copy_host()
    assert a.nnz == b.nnz == len(host.indices) == int(host.indptr[-1])
    assert a.n_partial == int(host.flags.sum()) and a.n_items == (a.nq + 1) // 2
    assert a.n_item_tiles >= (a.nnz + 1) // 2
    ix.destroy()


def test_attn_fwd_argument_errors():
    w = inputs.WORKLOADS["tiny"]
    q, k, v = inputs.make_qkv(w, "cuda", torch.bfloat16)
    out = torch.empty_like(q)
    ix = build_index(w, 0)
    L = binding.lib()
    null, stream = C.c_void_p(None), C.c_void_p(torch.cuda.current_stream().cuda_stream)
    p = lambda t: C.c_void_p(t.data_ptr())
    assert L.lvsa_attn_fwd(null, p(k), p(v), ix.handle, p(out), null, stream) == binding.EINVAL
    assert L.lvsa_attn_fwd(p(q), p(k), p(v), null, p(out), null, stream) == binding.EINVAL
    assert L.lvsa_attn_fwd(C.c_void_p(q.data_ptr() + 2), p(k), p(v), ix.handle, p(out), null, stream) == binding.EINVAL
    assert "aligned" in binding.lvsa_last_error()
    lse = torch.empty((w.B, w.H, w.N + 1), device="cuda", dtype=torch.float32)
    assert L.lvsa_attn_fwd(p(q), p(k), p(v), ix.handle, p(out), C.c_void_p(lse.data_ptr() + 2), stream) == binding.EINVAL
    assert "lse" in binding.lvsa_last_error()
    assert L.lvsa_schedule_attn_fwd(null, 0, p(q), p(k), p(v), p(out), null, stream) == binding.EINVAL
    ix.destroy()
    ix.destroy()                      # second destroy of the Python wrapper is a no-op


def test_repeated_launches_are_bitwise_identical():
    """The result does not depend on timing: the MMAs of a q tile accumulate in list order and the
    rescale decisions are taken in tile order, so repeated launches must agree bit for bit (a race in
    the mbarrier / TMEM / shared-reference protocols would show up here)."""
    for name, n in (("small128", 40), ("wan1.3b_1x", 25)):
        w = inputs.WORKLOADS[name]
        q, k, v = inputs.make_qkv(w, "cuda", torch.bfloat16)
        ix = build_index(w, w.steps[0])
        ref, ref_lse = gpu_attn(w, ix, q, k, v)
        for _ in range(n):
            out, lse = gpu_attn(w, ix, q, k, v)
            assert torch.equal(out, ref) and torch.equal(lse, ref_lse)
        ix.destroy()
