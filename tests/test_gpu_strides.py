"""Free strides (lvsa_params_t.stride_q/k/v/out; SURVEY.md section 8(b) "layout / strides"; PAPER.md:31 fixes
only N = T*P): one fused projection output [B, N, 3, H, d] feeds q, k and v without a copy, and `out` may be a
slice of a wider buffer.  Against the fp64 oracle (which gets contiguous copies of the same values), and bit for
bit against the same kernel on contiguous operands."""
import numpy as np
import pytest
import torch

from helpers import (BF16_MAX_ABS, BF16_MEAN_ABS, FP32_MAX_ABS, LSE_MAX_ABS_BF16, LSE_MAX_ABS_FP32, build_index,
                     compare, gpu_attn, oracle_attn)
from paper_2605_31057_b200 import binding, inputs

KERNELS = {"pair": dict(dtype=binding.DTYPE_BF16, kernel=binding.KERNEL_TCGEN05),
           "v0": dict(dtype=binding.DTYPE_BF16, kernel=binding.KERNEL_TCGEN05_V0),
           "quad": dict(dtype=binding.DTYPE_BF16, kernel=binding.KERNEL_TCGEN05_QUAD),
           "simt_bf16": dict(dtype=binding.DTYPE_BF16, kernel=binding.KERNEL_SIMT),
           "simt_fp32": dict(dtype=binding.DTYPE_FP32, kernel=binding.KERNEL_SIMT)}


def fused_views(w, q, k, v, out_slots=2):
    """q, k, v as views of ONE [B, N, 3, H, d] buffer; out as slot 1 of a [B, N, out_slots, H, d] buffer."""
    fused = torch.stack((q, k, v), dim=2).contiguous()
    wide = torch.full((w.B, w.N, out_slots, w.H, w.d), float("nan"), device=q.device, dtype=q.dtype)
    return fused, fused[:, :, 0], fused[:, :, 1], fused[:, :, 2], wide, wide[:, :, 1]


def run_fused(w, step, rows, kern, tol):
    dt = torch.float32 if kern["dtype"] == binding.DTYPE_FP32 else torch.bfloat16
    q, k, v = inputs.make_qkv(w, "cuda", dt)
    fused, qv, kv, vv, wide, ov = fused_views(w, q, k, v)
    assert not qv.is_contiguous() and qv.data_ptr() != kv.data_ptr()
    ix = build_index(w, step, stride_q=binding.tensor_strides(qv), stride_k=binding.tensor_strides(kv),
                     stride_v=binding.tensor_strides(vv), stride_out=binding.tensor_strides(ov), **kern)
    lse = torch.full((w.B, w.H, w.N), float("nan"), device="cuda", dtype=torch.float32)
    before = fused.clone()
    binding.lvsa_attn_fwd(qv, kv, vv, ix, ov, lse, strided=True)
    torch.cuda.synchronize()
    ix.destroy()
    assert torch.equal(fused, before)                            # inputs are read-only
    assert torch.isnan(wide[:, :, 0]).all()                      # nothing written outside out's slot
    ixc = build_index(w, step, **kern)                           # the same kernel on contiguous operands
    want, want_lse = gpu_attn(w, ixc, q, k, v)
    ixc.destroy()
    assert torch.equal(ov, want) and torch.equal(lse, want_lse)
    max_abs, mean_abs, lse_abs = tol
    for b in range(w.B):
        ref, ref_lse = oracle_attn(w, q, k, v, step, rows, b=b)
        st = compare(ov, lse, ref, ref_lse, rows, b)
        assert st["nan"] == 0 and st["max_abs"] <= max_abs and st["mean_abs"] <= mean_abs, (w.name, st)
        assert st["lse_max_abs"] <= lse_abs, (w.name, st)


@pytest.mark.gpu
@pytest.mark.parametrize("kname", ["pair", "v0", "quad", "simt_bf16"])
def test_fused_qkv_buffer_all_rows_small128(kname):
    w = inputs.WORKLOADS["small128"]
    run_fused(w, w.steps[1], np.arange(w.N), KERNELS[kname], (BF16_MAX_ABS, BF16_MEAN_ABS, LSE_MAX_ABS_BF16))


@pytest.mark.gpu
def test_fused_qkv_buffer_tiny_fp32_and_batched():
    w = inputs.WORKLOADS["tiny"]
    run_fused(w, w.steps[1], np.arange(w.N), KERNELS["simt_fp32"], (FP32_MAX_ABS, FP32_MAX_ABS, LSE_MAX_ABS_FP32))
    wb = inputs.Workload("strides_b2", 1, T=5, P=150, H=3, d=128, tile=128, W=1, a=2, B=2)   # batch stride, ragged tail
    run_fused(wb, 1, np.arange(wb.N), KERNELS["pair"], (BF16_MAX_ABS, BF16_MEAN_ABS, LSE_MAX_ABS_BF16))


@pytest.mark.gpu
@pytest.mark.slow
def test_fused_qkv_buffer_sampled_rows_wan1x():
    w = inputs.WORKLOADS["wan1.3b_1x"]
    rows = inputs.sample_rows(w, n_uniform=768, n_edge=256)
    run_fused(w, w.steps[0], rows, KERNELS["pair"], (BF16_MAX_ABS, BF16_MEAN_ABS, LSE_MAX_ABS_BF16))


@pytest.mark.gpu
def test_host_entry_point_refuses_custom_strides():
    w = inputs.WORKLOADS["small128"]
    ix = build_index(w, 0, stride_q=(3 * w.H * w.d, w.d, w.N * 3 * w.H * w.d))
    h = torch.zeros((w.B, w.N, w.H, w.d), dtype=torch.bfloat16)
    with pytest.raises(binding.LvsaError) as ei:
        binding.lvsa_attn_fwd_host(h, h, h, ix, h.clone(), None)
    assert ei.value.status == binding.EUNSUPPORTED
    ix.destroy()


def test_stride_validation_needs_no_gpu():
    base = dict(T=4, P=64, H=2, d=128)
    ok_n, ok_h, ok_b = 3 * 2 * 128, 128, 4 * 64 * 3 * 2 * 128
    for bad in (dict(stride_q=(ok_n + 4, ok_h, ok_b)),         # not a multiple of 16 bytes
                dict(stride_k=(64, ok_h, ok_b)),                # token stride < d
                dict(stride_v=(-ok_n, ok_h, ok_b)),             # negative
                dict(stride_out=(ok_n, 0, ok_b)),               # H = 2 needs a head stride
                dict(stride_q=(ok_n, ok_h, 0), B=2),            # B = 2 needs a batch stride
                dict(stride_q=(1 << 40, ok_h, ok_b))):          # beyond the TMA stride range
        with pytest.raises(binding.LvsaError) as ei:
            binding.lvsa_build_block_index_ex(**base, **bad)
        assert ei.value.status == binding.EINVAL, bad
    with pytest.raises(ValueError):
        binding.tensor_strides(torch.zeros(2, 3, 4, 5).transpose(2, 3))
    assert binding.tensor_strides(torch.zeros(2, 7, 3, 4, 8)[:, :, 1]) == (3 * 4 * 8, 8, 7 * 3 * 4 * 8)
