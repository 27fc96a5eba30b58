"""GPU parity for the frame-aligned kv tiling (reading R25),
through the C ABI: index bit-exact against the oracle's second tile definition, attention against the
fp64 oracle (which does not know about tiles at all) element by element."""
import numpy as np
import pytest
import torch

from helpers import (BF16_MAX_ABS, BF16_MEAN_ABS, FP32_MAX_ABS, LSE_MAX_ABS_BF16, LSE_MAX_ABS_FP32,
                     build_index, compare, gpu_attn, oracle_attn)
from oracle import lvsa_oracle as orc
from paper_2605_31057_b200 import binding, inputs

pytestmark = pytest.mark.gpu

FA = dict(kv_tiling=binding.KV_TILES_FRAME_ALIGNED)
KERNELS = {"tcgen05": dict(dtype=binding.DTYPE_BF16, kernel=binding.KERNEL_TCGEN05),
           "simt_bf16": dict(dtype=binding.DTYPE_BF16, kernel=binding.KERNEL_SIMT),
           "simt_fp32": dict(dtype=binding.DTYPE_FP32, kernel=binding.KERNEL_SIMT)}


# ---------------------------------------------------------------- index, bit-exact
def check_index(T, P, d, W, a, step, k0=0, n_text=0, tie=0):
    ix = binding.lvsa_build_block_index_ex(T=T, P=P, H=2, d=d, window=W, anchors=a, step=step, tie_break=tie,
                                           initial_anchors=k0, n_text=n_text, kernel=binding.KERNEL_SIMT, **FA)
    info, host = ix.info(), ix.copy_host()
    p = orc.pattern(T, W, a, step, tie, initial_anchors=k0)
    A = orc.with_text(p.A) if n_text > 0 else p.A
    indptr, indices, flags = orc.tile_index_fa(T, P, d, d, A, n_text=n_text, pad=binding.KV_PAD)
    col0, width = orc.kv_tiles_frame_aligned(T, P, d, n_text)
    g_col0, g_width = ix.kv_tiles()
    assert info.kv_tiling == binding.KV_TILES_FRAME_ALIGNED and info.nk == len(col0)
    assert np.array_equal(g_col0, col0) and np.array_equal(g_width, width)
    assert info.nnz == len(indices) and info.n_partial == int(flags.sum())
    assert np.array_equal(host.indptr, indptr) and np.array_equal(host.indices, indices)
    assert np.array_equal(host.flags, flags)
    wpad = (width + binding.KV_PAD - 1) // binding.KV_PAD * binding.KV_PAD
    assert info.kept_cols == int(wpad[indices].sum())
    assert np.array_equal(host.w_lo, p.w_lo) and np.array_equal(host.w_hi, p.w_hi)
    ix.destroy()


@pytest.mark.parametrize("T,P,d", [(8, 40, 64), (9, 200, 128), (7, 13, 64), (12, 50, 64), (33, 100, 128),
                                   (40, 7, 64), (1, 300, 128), (5, 128, 128), (6, 161, 128), (5, 31, 128)])
def test_index_frame_aligned_bit_exact(T, P, d):
    for W in (0, 1, 2):
        for a in (0, 1, 3, 100, binding.ALL_TILES):
            for step in (0, 1, 5):
                check_index(T, P, d, W, a, step, tie=step & 1)
    for k0, n_text in ((1, 0), (0, 1), (0, 77), (2, 130), (0, 300)):
        check_index(T, P, d, 1, 2, 1, k0, n_text)


@pytest.mark.parametrize("name", ["wan1.3b_1x", "wan1.3b_6x", "wan14b_6x", "hv1.5_2x", "hv1.5_1x_text"])
def test_baseline_configs_frame_aligned_bit_exact(name):
    w = inputs.WORKLOADS[name]
    for s in w.steps[:2]:
        check_index(w.T, w.P, w.d, w.W, w.a, s, n_text=w.n_text)


def test_token0_kept_cols_and_kv_tiles():
    """The default tiling reports its geometry through the same calls: nk tiles of tile_k tokens from token 0."""
    w = inputs.WORKLOADS["small128"]
    ix = build_index(w, 0)
    info = ix.info()
    col0, width = ix.kv_tiles()
    assert info.kv_tiling == binding.KV_TILES_TOKEN0 and info.kept_cols == info.nnz * 128
    assert np.array_equal(col0, np.arange(info.nk) * 128)
    assert np.array_equal(width, np.minimum(128, w.N - col0))
    ix.destroy()


def test_unsupported_with_the_one_cta_kernel():
    for kw in (dict(d=64, kernel=binding.KERNEL_TCGEN05), dict(d=128, kernel=binding.KERNEL_TCGEN05_V0)):
        with pytest.raises(binding.LvsaError) as ei:
            binding.lvsa_build_block_index_ex(T=8, P=40, H=1, window=1, anchors=2, **FA, **kw)
        assert ei.value.status == binding.EUNSUPPORTED


# ---------------------------------------------------------------- attention parity
def run_case(w, kname, steps, rows=None, seed=None, anchors=None):
    torch_dtype = torch.float32 if kname == "simt_fp32" else torch.bfloat16
    q, k, v = inputs.make_qkv(w, "cuda", torch_dtype, seed=seed)
    rows = np.arange(w.N) if rows is None else rows
    mx, mean = (FP32_MAX_ABS, FP32_MAX_ABS) if kname == "simt_fp32" else (BF16_MAX_ABS, BF16_MEAN_ABS)
    lse_tol = LSE_MAX_ABS_BF16 if kname == "tcgen05" else LSE_MAX_ABS_FP32
    for s in steps:
        ix = build_index(w, s, anchors=anchors, **KERNELS[kname], **FA)
        out, lse = gpu_attn(w, ix, q, k, v)
        for b in range(w.B):
            ref, ref_lse = oracle_attn(w, q, k, v, s, rows, anchors=anchors, b=b)
            st = compare(out, lse, ref, ref_lse, rows, b)
            assert st["nan"] == 0, (kname, s, st)
            assert st["max_abs"] <= mx and st["mean_abs"] <= mean and st["lse_max_abs"] <= lse_tol, (kname, s, st)
            assert st["rel_l2"] <= 2e-2, (kname, s, st)
        ix.destroy()


@pytest.mark.parametrize("kname", ["simt_fp32", "simt_bf16", "tcgen05"])
@pytest.mark.parametrize("name", ["small128", "small128_text", "small128_k0"])
def test_all_rows_d128(name, kname):
    w = inputs.WORKLOADS[name]
    run_case(w, kname, w.steps[:3])


@pytest.mark.parametrize("name", ["tiny", "tiny_straddle", "tiny_text"])
def test_all_rows_d64_simt(name):
    w = inputs.WORKLOADS[name]
    run_case(w, "simt_fp32", w.steps[:3])


@pytest.mark.parametrize("kname", ["simt_fp32", "tcgen05"])
def test_edge_shapes(kname):
    W = inputs.Workload
    cases = [W("one_tile", 1, T=1, P=128, H=2, d=128, tile=128, W=0, a=0),            # exactly one full tile
             W("one_narrow", 1, T=1, P=100, H=1, d=128, tile=128, W=0, a=0),           # one tile, 100 -> 128 columns
             W("narrow32", 1, T=6, P=24, H=1, d=128, tile=128, W=1, a=1),              # every tile is 24 -> 32 wide
             W("narrow64", 1, T=5, P=161, H=2, d=128, tile=128, W=1, a=2),             # 128 + 33 -> 64
             W("narrow96", 1, T=4, P=200, H=1, d=128, tile=128, W=0, a=1),             # 128 + 72 -> 96
             W("aligned", 1, T=5, P=256, H=1, d=128, tile=128, W=1, a=1),              # frames are whole tiles
             W("odd_nq_b2", 1, T=5, P=150, H=2, d=128, tile=128, W=1, a=2, B=2),
             W("dense_window", 1, T=5, P=90, H=2, d=128, tile=128, W=2, a=0),          # 2W+1 >= T: Eq. 1
             W("text_tail", 1, T=3, P=140, H=1, d=128, tile=128, W=0, a=1, n_text=45),
             W("wan_frame", 1, T=3, P=1560, H=1, d=128, tile=128, W=0, a=1)]           # 12 x 128 + 24 per frame
    for w in cases:
        run_case(w, kname, (0, 1))
    run_case(cases[3], kname, (0,), anchors=binding.ALL_TILES)


def test_seeded_shape_sweep():
    rng = np.random.default_rng(20260601)
    W = inputs.Workload
    for case in range(20):
        w = W(f"fa_sweep{case}", 1, T=int(rng.integers(1, 12)), P=int(rng.integers(17, 420)), H=int(rng.integers(1, 4)),
              d=128, tile=128, W=int(rng.integers(0, 3)), a=int(rng.choice([0, 1, 2, 3, 5, binding.ALL_TILES])),
              B=int(rng.integers(1, 3)), n_text=int(rng.choice([0, 0, 1, 64, 150])), k0=int(rng.choice([0, 0, 1, 2])))
        run_case(w, "tcgen05", (int(rng.integers(0, 7)),), seed=2000 + case)


def test_structured_logits_growing_maximum():
    """The lazy rescale and the shared reference maximum with narrow tiles in the list."""
    w = inputs.Workload("fa_num", 1, T=9, P=200, H=2, d=128, tile=128, W=1, a=2)
    g = torch.Generator(device="cuda").manual_seed(11)
    q = torch.randn((1, w.N, w.H, w.d), generator=g, device="cuda") * 0.05
    k = torch.randn((1, w.N, w.H, w.d), generator=g, device="cuda") * 0.05
    v = torch.randn((1, w.N, w.H, w.d), generator=g, device="cuda")
    q[..., 0] = 1.0
    k[..., 0] = torch.linspace(0.0, 1.0, w.N, device="cuda")[None, :, None] * 40.0 * w.d ** 0.5
    q, k, v = (x.to(torch.bfloat16) for x in (q, k, v))
    rows = np.arange(w.N)
    for s in (0, 1):
        ix = build_index(w, s, **FA)
        out, lse = gpu_attn(w, ix, q, k, v)
        ref, ref_lse = oracle_attn(w, q, k, v, s, rows)
        st = compare(out, lse, ref, ref_lse, rows)
        assert st["nan"] == 0 and st["max_abs"] <= BF16_MAX_ABS and st["mean_abs"] <= BF16_MEAN_ABS, (s, st)
        assert st["rel_l2"] <= 5e-3 and st["lse_max_abs"] <= LSE_MAX_ABS_BF16, (s, st)
        ix.destroy()


@pytest.mark.slow
@pytest.mark.parametrize("name,n_rows", [("wan1.3b_1x", 1024), ("wan1.3b_6x", 2048), ("hv1.5_2x", 1024),
                                         ("wan14b_6x", 1024), ("hv1.5_1x_text", 1024)])
def test_large_configs_sampled_rows(name, n_rows):
    w = inputs.WORKLOADS[name]
    rows = inputs.sample_rows(w, n_uniform=n_rows - 256, n_edge=256)
    if w.n_text:
        rows = np.unique(np.concatenate([rows, np.arange(w.T * w.P, w.N, 41)]))
    run_case(w, "tcgen05", w.steps[:1], rows=rows)
