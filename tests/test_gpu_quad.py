"""GPU parity for the 4-CTA-cluster variants of the attention kernel (K/V tiles
shared by two MMA pairs through one multicast TMA load), through the C ABI, against the fp64 oracle element
by element: LVSA_KERNEL_TCGEN05_QUAD (clusters of four only) and LVSA_KERNEL_TCGEN05_HYBRID (clusters of four
plus CTA pairs on the SMs the clusters cannot cover, two launches side by side).  The index (CSR) is the same
as for the other kernels; the variants only consume a different work list (unions over four q tiles)."""
import numpy as np
import pytest
import torch

from helpers import (BF16_MAX_ABS, BF16_MEAN_ABS, LSE_MAX_ABS_BF16, build_index, compare, gpu_attn, oracle_attn)
from paper_2605_31057_b200 import binding, inputs

pytestmark = pytest.mark.gpu

KERNELS = {"quad": dict(dtype=binding.DTYPE_BF16, kernel=binding.KERNEL_TCGEN05_QUAD),
           "hybrid": dict(dtype=binding.DTYPE_BF16, kernel=binding.KERNEL_TCGEN05_HYBRID)}
QUAD = KERNELS["quad"]
W = inputs.Workload


def run_case(w, steps, rows=None, seed=None, anchors=None, hnd=False, QUAD=QUAD):
    q, k, v = inputs.make_qkv(w, "cuda", torch.bfloat16, seed=seed)
    rows = np.arange(w.N) if rows is None else rows
    for s in steps:
        if hnd:
            ix = build_index(w, s, anchors=anchors, layout=binding.LAYOUT_HND, **QUAD)
            out_t, lse = gpu_attn(w, ix, *(x.transpose(1, 2).contiguous() for x in (q, k, v)))
            out = out_t.transpose(1, 2)
        else:
            ix = build_index(w, s, anchors=anchors, **QUAD)
            out, lse = gpu_attn(w, ix, q, k, v)
        assert ix.info().kernel == QUAD["kernel"]
        for b in range(w.B):
            ref, ref_lse = oracle_attn(w, q, k, v, s, rows, anchors=anchors, b=b)
            st = compare(out, lse, ref, ref_lse, rows, b)
            assert st["nan"] == 0, (w.name, s, st)
            assert st["max_abs"] <= BF16_MAX_ABS and st["mean_abs"] <= BF16_MEAN_ABS, (w.name, s, st)
            assert st["lse_max_abs"] <= LSE_MAX_ABS_BF16 and st["rel_l2"] <= 2e-2, (w.name, s, st)
        ix.destroy()


@pytest.mark.parametrize("kname", list(KERNELS))
@pytest.mark.parametrize("name", ["small128", "small128_text", "small128_k0"])
def test_all_rows(name, kname):
    w = inputs.WORKLOADS[name]
    run_case(w, w.steps[:3], QUAD=KERNELS[kname])
    run_case(w, w.steps[:1], hnd=True, QUAD=KERNELS[kname])


@pytest.mark.parametrize("kname", list(KERNELS))
def test_edge_shapes(kname):
    cases = [W("one_tile", 1, T=1, P=128, H=2, d=128, tile=128, W=0, a=0),           # one q tile: three of four CTAs have no rows
             W("two_tiles", 1, T=2, P=128, H=1, d=128, tile=128, W=0, a=1),
             W("odd_nq", 1, T=3, P=128, H=1, d=128, tile=128, W=0, a=1),             # nq = 3
             W("nq5", 1, T=5, P=128, H=2, d=128, tile=128, W=1, a=0),                # nq = 5: second quad holds one q tile
             W("nq6_b2", 1, T=5, P=150, H=2, d=128, tile=128, W=1, a=2, B=2),        # nq = 6, ragged tail, B = 2
             W("dense_window", 1, T=5, P=90, H=2, d=128, tile=128, W=2, a=0),        # 2W+1 >= T: Eq. 1
             W("many_heads", 1, T=4, P=200, H=9, d=128, tile=128, W=1, a=1)]
    for w in cases:
        run_case(w, (0, 1), QUAD=KERNELS[kname])
    run_case(cases[4], (0,), anchors=binding.ALL_TILES, QUAD=KERNELS[kname])


@pytest.mark.parametrize("kname", list(KERNELS))
def test_seeded_shape_sweep(kname):
    rng = np.random.default_rng(20260602)
    for case in range(20):
        w = W(f"quad_sweep{case}", 1, T=int(rng.integers(1, 14)), P=int(rng.integers(17, 420)), H=int(rng.integers(1, 4)),
              d=128, tile=128, W=int(rng.integers(0, 3)), a=int(rng.choice([0, 1, 2, 3, 5, binding.ALL_TILES])),
              B=int(rng.integers(1, 3)), n_text=int(rng.choice([0, 0, 1, 64, 150])), k0=int(rng.choice([0, 0, 1, 2])))
        run_case(w, (int(rng.integers(0, 7)),), seed=3000 + case, QUAD=KERNELS[kname])


def test_structured_logits_growing_maximum():
    w = W("quad_num", 1, T=9, P=200, H=2, d=128, tile=128, W=1, a=2)
    g = torch.Generator(device="cuda").manual_seed(13)
    q = torch.randn((1, w.N, w.H, w.d), generator=g, device="cuda") * 0.05
    k = torch.randn((1, w.N, w.H, w.d), generator=g, device="cuda") * 0.05
    v = torch.randn((1, w.N, w.H, w.d), generator=g, device="cuda")
    q[..., 0] = 1.0
    k[..., 0] = torch.linspace(0.0, 1.0, w.N, device="cuda")[None, :, None] * 40.0 * w.d ** 0.5
    q, k, v = (x.to(torch.bfloat16) for x in (q, k, v))
    rows = np.arange(w.N)
    for s in (0, 1):
        ix = build_index(w, s, **QUAD)
        out, lse = gpu_attn(w, ix, q, k, v)
        ref, ref_lse = oracle_attn(w, q, k, v, s, rows)
        st = compare(out, lse, ref, ref_lse, rows)
        assert st["nan"] == 0 and st["max_abs"] <= BF16_MAX_ABS and st["mean_abs"] <= BF16_MEAN_ABS, (s, st)
        assert st["rel_l2"] <= 5e-3 and st["lse_max_abs"] <= LSE_MAX_ABS_BF16, (s, st)
        ix.destroy()


def test_grid_and_repeatability_and_host_entry_point():
    w = inputs.WORKLOADS["wan1.3b_1x"]
    q, k, v = inputs.make_qkv(w, "cuda", torch.bfloat16)
    ix = build_index(w, w.steps[0], **QUAD)
    ixp = build_index(w, w.steps[0])
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    assert ixp.grid() == sms // 2 * 2                                  # CTA pairs: every SM
    assert 0 < ix.grid() <= sms and ix.grid() % 4 == 0                 # resident 4-CTA clusters only
    ixh = build_index(w, w.steps[0], **KERNELS["hybrid"])
    assert ixh.grid() == sms // 2 * 2                                  # clusters of four + pairs: every SM
    hyb, hyb_lse = gpu_attn(w, ixh, q, k, v)
    # launch counts the library reports (bench.py's gpu_launches): HYBRID forks into two kernels when both
    # parts get work (B200: 132 SMs in clusters of four, 16 in pairs); 7 builder kernels with quad lists
    assert ixp.launches() == 1 and ix.launches() == 1
    assert ixh.launches() == (2 if ix.grid() < sms // 2 * 2 else 1)
    assert ixp.build_launches() == 4 and ix.build_launches() == 7 and ixh.build_launches() == 7
    # ... and HYBRID against the oracle itself, not only against its own graph replay
    rows_h = inputs.sample_rows(w, n_uniform=192, n_edge=64)
    ref_h, ref_h_lse = oracle_attn(w, q, k, v, w.steps[0], rows_h)
    st = compare(hyb, hyb_lse, ref_h, ref_h_lse, rows_h)
    assert st["nan"] == 0 and st["max_abs"] <= BF16_MAX_ABS and st["mean_abs"] <= BF16_MEAN_ABS, st
    assert st["lse_max_abs"] <= LSE_MAX_ABS_BF16 and st["rel_l2"] <= 2e-2, st
    # CUDA-graph capture of the two side-by-side launches (fork / join with events on an internal stream)
    g, side, out_g = torch.cuda.CUDAGraph(), torch.cuda.Stream(), torch.zeros_like(q)
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        with torch.cuda.graph(g, stream=side):
            binding.lvsa_attn_fwd(q, k, v, ixh, out_g, None, stream=side.cuda_stream)
    torch.cuda.current_stream().wait_stream(side)
    g.replay(); torch.cuda.synchronize()
    assert torch.equal(out_g, hyb)
    ixh.destroy()
    ref, ref_lse = gpu_attn(w, ix, q, k, v)
    for _ in range(10):                                                # timing-independent result
        out, lse = gpu_attn(w, ix, q, k, v)
        assert torch.equal(out, ref) and torch.equal(lse, ref_lse)
    pair, _ = gpu_attn(w, ixp, q, k, v)                                 # same maths as the pair kernel
    assert float((pair.float() - ref.float()).abs().max()) <= 2e-3
    oh = torch.full_like(q, float("nan"), device="cpu").pin_memory()
    lh = torch.full((w.B, w.H, w.N), float("nan"), dtype=torch.float32).pin_memory()
    binding.lvsa_attn_fwd_host(q.cpu().pin_memory(), k.cpu().pin_memory(), v.cpu().pin_memory(), ix, oh, lh)
    assert torch.equal(oh, ref.cpu()) and torch.equal(lh, ref_lse.cpu())
    ix.destroy(); ixp.destroy()


@pytest.mark.slow
@pytest.mark.parametrize("kname", list(KERNELS))
@pytest.mark.parametrize("name", ["wan1.3b_1x", "wan1.3b_6x", "wan14b_6x", "hv1.5_2x"])
def test_large_configs_sampled_rows(name, kname):
    """Every shape bench.py / profiles/ report a QUAD or HYBRID time for (the four large BASELINE.json configs):
    1024 sampled rows, edge rows included, against the oracle at full size."""
    w = inputs.WORKLOADS[name]
    rows = inputs.sample_rows(w, n_uniform=768, n_edge=256)
    run_case(w, w.steps[:1], rows=rows, QUAD=KERNELS[kname])
