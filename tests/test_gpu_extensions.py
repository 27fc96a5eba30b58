"""GPU parity for the extension rows of SURVEY.md section 8f, through the C ABI:
  f1 whole-schedule driver (+ CUDA-graph replay), f2 text tokens, f3 dedicated initial anchors."""
import math

import numpy as np
import pytest
import torch

from helpers import (BF16_MAX_ABS, BF16_MEAN_ABS, FP32_MAX_ABS, LSE_MAX_ABS_BF16, LSE_MAX_ABS_FP32,
                     build_index, compare, gpu_attn, oracle_attn)
from oracle import lvsa_oracle as orc
from paper_2605_31057_b200 import binding, inputs

pytestmark = pytest.mark.gpu


# ---------------------------------------------------------------- index, bit-exact
def check_index(T, P, d, W, a, step, k0=0, n_text=0, tie=0):
    ix = binding.lvsa_build_block_index_ex(T=T, P=P, H=2, d=d, window=W, anchors=a, step=step,
                                           tie_break=tie, initial_anchors=k0, n_text=n_text)
    info, host = ix.info(), ix.copy_host()
    p = orc.pattern(T, W, a, step, tie, initial_anchors=k0)
    A = orc.with_text(p.A) if n_text > 0 else p.A
    indptr, indices, flags = orc.tile_index(T, P, d, d, A, n_text=n_text)
    assert (info.T_per, info.phase, info.n_global) == (p.T_per, p.phase, p.n_global)
    assert info.N == T * P + n_text and info.n_text == n_text and info.initial_anchors == k0
    assert info.nnz == len(indices) and info.n_partial == int(flags.sum())
    assert np.array_equal(host.w_lo, p.w_lo) and np.array_equal(host.w_hi, p.w_hi)
    Tf = A.shape[0]
    bits = ((host.a_bits[:, :, None] >> np.arange(32, dtype=np.uint32)[None, None, :]) & 1).reshape(Tf, -1)
    assert np.array_equal(bits[:, :Tf], A) and not bits[:, Tf:].any()
    assert np.array_equal(host.indptr, indptr) and np.array_equal(host.indices, indices)
    assert np.array_equal(host.flags, flags)
    ix.destroy()


@pytest.mark.parametrize("T,P,d", [(8, 40, 64), (9, 200, 128), (7, 13, 64), (33, 100, 128), (31, 50, 64),
                                   (32, 50, 64), (1, 300, 128)])
def test_index_with_extensions_bit_exact(T, P, d):
    for W in (0, 1, 2):
        for a in (0, 2, 5, 100, binding.ALL_TILES):
            for step in (0, 1, 6):
                for k0, n_text in ((1, 0), (3, 0), (T + 1, 0), (0, 1), (0, 77), (0, 300), (2, 130)):
                    check_index(T, P, d, W, a, step, k0, n_text)


# ---------------------------------------------------------------- attention parity, all rows
KERNELS = {"tcgen05": dict(dtype=binding.DTYPE_BF16, kernel=binding.KERNEL_TCGEN05),
           "simt_bf16": dict(dtype=binding.DTYPE_BF16, kernel=binding.KERNEL_SIMT),
           "simt_fp32": dict(dtype=binding.DTYPE_FP32, kernel=binding.KERNEL_SIMT)}


def run_case(w, kname, steps, rows=None):
    torch_dtype = torch.float32 if kname == "simt_fp32" else torch.bfloat16
    q, k, v = inputs.make_qkv(w, "cuda", torch_dtype)
    rows = np.arange(w.N) if rows is None else rows
    mx, mean = (FP32_MAX_ABS, FP32_MAX_ABS) if kname == "simt_fp32" else (BF16_MAX_ABS, BF16_MEAN_ABS)
    lse_tol = LSE_MAX_ABS_BF16 if kname == "tcgen05" else LSE_MAX_ABS_FP32
    for s in steps:
        ix = build_index(w, s, **KERNELS[kname])
        out, lse = gpu_attn(w, ix, q, k, v)
        ref, ref_lse = oracle_attn(w, q, k, v, s, rows)
        st = compare(out, lse, ref, ref_lse, rows)
        assert st["nan"] == 0, (kname, s, st)
        assert st["max_abs"] <= mx and st["mean_abs"] <= mean and st["lse_max_abs"] <= lse_tol, (kname, s, st)
        ix.destroy()


@pytest.mark.parametrize("kname", ["simt_fp32", "simt_bf16", "tcgen05"])
@pytest.mark.parametrize("name", ["tiny_text", "small128_text", "small128_k0"])
def test_extensions_all_rows(name, kname):
    w = inputs.WORKLOADS[name]
    run_case(w, kname, w.steps)


@pytest.mark.parametrize("kname", ["simt_fp32", "tcgen05"])
def test_text_edge_shapes(kname):
    W = inputs.Workload
    cases = [W("text_only_tail", 1, T=2, P=128, H=1, d=128, tile=128, W=0, a=0, n_text=1),    # 1 text token
             W("text_gt_frame", 1, T=3, P=50, H=2, d=64, tile=64, W=0, a=1, n_text=200),      # text longer than a frame
             W("text_aligned", 1, T=4, P=64, H=1, d=64, tile=64, W=1, a=0, n_text=64),        # text = one whole tile
             W("text_and_k0", 1, T=10, P=30, H=2, d=64, tile=64, W=1, a=2, n_text=45, k0=2)]
    for w in cases:
        run_case(w, kname, (0, 1, 2))


@pytest.mark.slow
def test_hv_shaped_text_sampled_rows():
    w = inputs.WORKLOADS["hv1.5_1x_text"]
    rows = inputs.sample_rows(w, n_uniform=1024, n_edge=256)
    rows = np.unique(np.concatenate([rows, np.arange(w.T * w.P, w.N, 37)]))      # text rows too
    run_case(w, "tcgen05", w.steps[:1], rows=rows)


# ---------------------------------------------------------------- f1: schedule
def test_schedule_matches_per_step_indices_and_graph_replay():
    w = inputs.WORKLOADS["small128"]
    T_per = math.ceil(w.T / w.a)
    sched = binding.lvsa_schedule_create(T=w.T, P=w.P, H=w.H, d=w.d, window=w.W, anchors=w.a)
    assert sched.num_phases() == T_per
    q, k, v = inputs.make_qkv(w, "cuda", torch.bfloat16)
    S, L = T_per + 3, 2
    # f1 parity against the ORACLE (reading R24): the index the schedule holds
    # for step s is the oracle's index of step s, bit for bit, and what the schedule computes with it
    # is Eq. 2 within the stated tolerance -- for every step, beyond one period
    rows = np.arange(w.N)
    for s in range(S):
        p = orc.pattern(w.T, w.W, w.a, s)
        indptr, indices, flags = orc.tile_index(w.T, w.P, w.d, w.d, p.A)
        hp = sched.index(s).copy_host()
        assert np.array_equal(hp.indptr, indptr) and np.array_equal(hp.indices, indices)
        assert np.array_equal(hp.flags, flags) and np.array_equal(hp.a_bits, p.a_bits())
        assert np.array_equal(hp.w_lo, p.w_lo) and np.array_equal(hp.w_hi, p.w_hi)
        out = torch.full_like(q, float("nan"))
        lse = torch.full((w.B, w.H, w.N), float("nan"), device="cuda", dtype=torch.float32)
        binding.lvsa_schedule_attn_fwd(sched, s, q, k, v, out, lse)
        torch.cuda.synchronize()
        ref, ref_lse = oracle_attn(w, q, k, v, s, rows)
        st = compare(out, lse, ref, ref_lse, rows)
        assert st["nan"] == 0 and st["max_abs"] <= BF16_MAX_ABS and st["mean_abs"] <= BF16_MEAN_ABS, (s, st)
        assert st["lse_max_abs"] <= LSE_MAX_ABS_BF16 and st["rel_l2"] <= 2e-2, (s, st)
    # eager, one index per step (what the paper does per step): the schedule must also
    # agree bit for bit with the per-step path of the library
    want = []
    for s in range(S):
        ix = build_index(w, s)
        hs, hp = ix.copy_host(), sched.index(s).copy_host()
        assert np.array_equal(hs.indices, hp.indices) and np.array_equal(hs.flags, hp.flags)
        assert np.array_equal(hs.a_bits, hp.a_bits) and sched.index(s).info().phase == s % T_per
        out, lse = gpu_attn(w, ix, q, k, v)
        want.append((out.clone(), lse.clone()))
        ix.destroy()
    # schedule, eager
    outs = [torch.empty_like(q) for _ in range(S * L)]
    lses = [torch.empty((w.B, w.H, w.N), device="cuda", dtype=torch.float32) for _ in range(S * L)]
    for s in range(S):
        for layer in range(L):
            binding.lvsa_schedule_attn_fwd(sched, s, q, k, v, outs[s * L + layer], lses[s * L + layer])
    torch.cuda.synchronize()
    for s in range(S):
        for layer in range(L):
            assert torch.equal(outs[s * L + layer], want[s][0]) and torch.equal(lses[s * L + layer], want[s][1])
    # schedule, whole S x L replay captured in one CUDA graph
    for o in outs:
        o.zero_()
    g = torch.cuda.CUDAGraph()
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        with torch.cuda.graph(g, stream=side):
            for s in range(S):
                for layer in range(L):
                    binding.lvsa_schedule_attn_fwd(sched, s, q, k, v, outs[s * L + layer], lses[s * L + layer],
                                                   stream=side.cuda_stream)
    torch.cuda.current_stream().wait_stream(side)
    for _ in range(2):
        g.replay()
    torch.cuda.synchronize()
    for s in range(S):
        for layer in range(L):
            assert torch.equal(outs[s * L + layer], want[s][0])
    sched.destroy()


def test_schedule_without_rotation_has_one_phase():
    for a in (0, binding.ALL_TILES, 100):
        sched = binding.lvsa_schedule_create(T=6, P=70, H=1, d=64, window=1, anchors=a)
        assert sched.num_phases() == 1
        sched.destroy()
