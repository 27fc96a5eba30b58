"""Seeded synthetic inputs and the workload table — shared by tests, bench.py and smoke().

This module holds NONE of the method's arithmetic (no anchor sets, windows, masks or
softmax): only shapes, seeds, random tensors and row samples.  It is the one module both
the oracle-side tests and the CUDA-side callers may import.

The paper measures on Wan 2.1 / HunyuanVideo 1.5 latents; those models,
prompts and latents are not available, so i.i.d. N(0,1) tensors of the same shapes stand in
for them (BASELINE.json configs).
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np
import torch

SEED_BASE = 26053105700  # + config index (1..5), reading R19


@dataclass(frozen=True)
class Workload:
    name: str
    index: int            # 1-based position in BASELINE.json:configs
    T: int                # latent frames
    P: int                # tokens per frame (H_p * W_p)
    H: int                # heads
    d: int                # head dim
    tile: int             # Bq = Bk
    W: int                # window half width (reading R1 / R3)
    a: int                # anchor target C - (2W+1) (readings R1-R3)
    steps: tuple = ()     # denoising steps the config asks for
    layers: tuple = ()    # layers the config asks for
    n_layers: int = 0
    B: int = 1
    n_text: int = 0       # text tokens after the video tokens (reading R23); 0 = none
    k0: int = 0           # dedicated initial anchors (reading R22); 0 = the paper's pattern

    @property
    def N(self) -> int:
        return self.T * self.P + self.n_text

    @property
    def seed(self) -> int:
        return SEED_BASE + self.index


WORKLOADS = {
    "tiny": Workload("tiny", 1, T=8, P=64, H=2, d=64, tile=64, W=1, a=2,
                     steps=tuple(range(10)), layers=(0, 1, 2, 3), n_layers=4),
    "wan1.3b_1x": Workload("wan1.3b_1x", 2, T=21, P=1560, H=12, d=128, tile=128, W=2, a=16,
                           steps=(25,), layers=(15,), n_layers=30),
    "wan1.3b_6x": Workload("wan1.3b_6x", 3, T=121, P=1560, H=12, d=128, tile=128, W=2, a=16,
                           steps=(0, 25, 49), layers=(0, 15, 29), n_layers=30),
    "wan14b_6x": Workload("wan14b_6x", 4, T=121, P=1560, H=40, d=128, tile=128, W=2, a=16,
                          steps=(25,), layers=(20,), n_layers=40),
    "hv1.5_2x": Workload("hv1.5_2x", 5, T=65, P=1590, H=16, d=128, tile=128, W=2, a=28,
                         steps=(0, 25, 49), layers=(27,), n_layers=54),
    # the paper's second measured resolution, 720x1280 -> 45 x 80 latent tokens per frame, at the 6x
    # horizon (Table 4); not a BASELINE.json config, same readings as wan1.3b_6x
    "wan1.3b_6x_720p": Workload("wan1.3b_6x_720p", 3, T=121, P=3600, H=12, d=128, tile=128, W=2, a=16,
                                steps=(25,), layers=(15,), n_layers=30),
    # non-contract variants used by the parity tests (ragged tiles, straddling frames)
    "tiny_straddle": Workload("tiny_straddle", 1, T=8, P=40, H=2, d=64, tile=64, W=1, a=2,
                              steps=tuple(range(10)), layers=(0,), n_layers=4),
    "small128": Workload("small128", 2, T=9, P=200, H=3, d=128, tile=128, W=1, a=2,
                         steps=(0, 1, 2, 3, 4), layers=(0,), n_layers=1),
    # extension rows: text tokens inside self-attention (f2; the paper's
    # prompts are "around 500 tokens") and dedicated initial anchors (f3)
    "tiny_text": Workload("tiny_text", 1, T=8, P=40, H=2, d=64, tile=64, W=1, a=2,
                          steps=(0, 1, 2, 3), layers=(0,), n_layers=1, n_text=30),
    "small128_text": Workload("small128_text", 2, T=9, P=200, H=3, d=128, tile=128, W=1, a=2,
                              steps=(0, 1, 2), layers=(0,), n_layers=1, n_text=77),
    "small128_k0": Workload("small128_k0", 2, T=9, P=200, H=3, d=128, tile=128, W=1, a=2,
                            steps=(0, 1, 2), layers=(0,), n_layers=1, k0=2),
    "hv1.5_1x_text": Workload("hv1.5_1x_text", 5, T=33, P=1590, H=16, d=128, tile=128, W=2, a=12,
                              steps=(0, 25), layers=(27,), n_layers=54, n_text=512),
}


def make_qkv(w: Workload, device: str = "cpu", dtype: torch.dtype = torch.bfloat16,
             seed: int | None = None):
    """q, k, v of shape [B, N, H, d]: randn in fp32 from a seeded generator on `device`
    (Philox on CUDA), drawn in the order q, k, v, then rounded to `dtype` (R19)."""
    g = torch.Generator(device=device)
    g.manual_seed(w.seed if seed is None else seed)
    out = []
    for _ in range(3):
        x = torch.randn((w.B, w.N, w.H, w.d), generator=g, device=device, dtype=torch.float32)
        out.append(x.to(dtype))
        del x
    return tuple(out)


def to_oracle_array(x: torch.Tensor) -> np.ndarray:
    """Host copy of one batch element as the oracle takes it: raw bf16 bits (uint16) or fp32,
    shape [N, H, d].  Value-preserving; no arithmetic."""
    assert x.dim() == 3
    x = x.detach().cpu().contiguous()
    if x.dtype == torch.bfloat16:
        return x.view(torch.int16).numpy().view(np.uint16)
    return x.to(torch.float32).numpy()


def sample_rows(w: Workload, n_uniform: int = 3584, n_edge: int = 512,
                seed: int | None = None) -> np.ndarray:
    """Query rows for sampled parity at large sizes: uniform rows plus forced edge rows
    (frame boundaries t*P-1 / t*P, tile boundaries, the first and last row, the tail tile)."""
    rng = np.random.default_rng(w.seed if seed is None else seed)
    N, P, tile = w.N, w.P, w.tile
    n_uniform = min(n_uniform, N)
    rows = set(rng.choice(N, size=n_uniform, replace=False).tolist())
    edge = {0, N - 1}
    tail0 = (N // tile) * tile if N % tile else N - tile
    edge.update(range(max(tail0, 0), N, max(1, (N - tail0) // 8)))
    if w.n_text > 0:
        edge.update((w.T * P - 1, w.T * P))          # last video row, first text row
    ts = rng.permutation(np.arange(1, w.T))
    for t in ts:
        if len(edge) >= n_edge:
            break
        b = int(t) * P
        edge.update((b - 1, b))                      # last row of frame t-1, first of frame t
        q0 = (b // tile) * tile
        edge.update((q0, min(q0 + tile - 1, N - 1)))  # ends of the straddling q tile
    rows.update(e for e in edge if 0 <= e < N)
    return np.array(sorted(rows), dtype=np.int64)


def probe_qkv(w: Workload, device: str = "cpu", dtype: torch.dtype = torch.bfloat16):
    """Closed-form probe inputs: Q = 0, K random, V[n, c] = 1 if n // P == c else 0 (needs
    T <= d).  What the output must equal is stated, and checked, in the tests."""
    assert w.T <= w.d
    _, k, _ = make_qkv(w, device, dtype)
    q = torch.zeros_like(k)
    frame = torch.arange(w.N, device=device) // w.P
    v1 = torch.zeros((w.N, w.d), device=device, dtype=dtype)
    v1[torch.arange(w.N, device=device), frame] = 1
    v = v1[None, :, None, :].expand(w.B, w.N, w.H, w.d).contiguous()
    return q, k, v
