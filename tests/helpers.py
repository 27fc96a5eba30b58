"""Shared test plumbing: runs the CUDA path through the C-ABI binding and the oracle on the same
seeded inputs.  The two sides only meet here, in the comparison."""
import numpy as np
import torch

from oracle import lvsa_oracle as orc
from paper_2605_31057_b200 import binding, inputs

# north_star tolerance for bf16 inputs / fp32 accumulation vs the fp64 oracle
BF16_MAX_ABS, BF16_MEAN_ABS = 1e-2, 1e-3
FP32_MAX_ABS = 1e-5
LSE_MAX_ABS_BF16, LSE_MAX_ABS_FP32 = 2e-3, 1e-5


def build_index(w, step, layer=0, anchors=None, window=None, **kw):
    return binding.lvsa_build_block_index_ex(
        T=w.T, P=w.P, H=w.H, d=w.d, B=w.B, window=w.W if window is None else window,
        anchors=w.a if anchors is None else anchors, step=step, layer=layer,
        initial_anchors=w.k0, n_text=w.n_text, **kw)


def gpu_attn(w, ix, q, k, v, want_lse=True):
    out = torch.full_like(q, float("nan"))
    lse = torch.full((w.B, w.H, w.N), float("nan"), device=q.device, dtype=torch.float32) if want_lse else None
    binding.lvsa_attn_fwd(q, k, v, ix, out, lse)
    torch.cuda.synchronize()
    return out, lse


def oracle_attn(w, q, k, v, step, rows, anchors=None, window=None, b=0):
    p = orc.pattern(w.T, w.W if window is None else window, w.a if anchors is None else anchors, step,
                    initial_anchors=w.k0)
    A = orc.with_text(p.A) if w.n_text > 0 else p.A
    qa, ka, va = (inputs.to_oracle_array(x[b]) for x in (q, k, v))
    return orc.attn_rows(qa, ka, va, w.T, w.P, A, rows, n_text=w.n_text)


def compare(out_gpu, lse_gpu, out_ref, lse_ref, rows, b=0):
    """out_gpu [B,N,H,d] torch; out_ref [nrows,H,d] fp64.  Returns error statistics."""
    rows_t = torch.as_tensor(rows, device=out_gpu.device)
    og = out_gpu[b].index_select(0, rows_t).double().cpu().numpy()
    err = np.abs(og - out_ref)
    st = dict(max_abs=float(err.max()), mean_abs=float(err.mean()),
              rel_l2=float(np.linalg.norm(og - out_ref) / max(np.linalg.norm(out_ref), 1e-300)),
              nan=int(np.isnan(og).sum()))
    if lse_gpu is not None:
        lg = lse_gpu[b].index_select(1, rows_t).double().cpu().numpy().T    # [nrows, H]
        st["lse_max_abs"] = float(np.abs(lg - lse_ref).max())
        st["nan"] += int(np.isnan(lg).sum())
    return st
