"""CPU-only checks of the C-ABI boundary: the library builds/loads, exports every symbol that
include/lvsa.h declares, and fails loudly (no CPU fallback) when there is no CUDA device."""
import ctypes as C
import os
import re

import pytest
import torch

from paper_2605_31057_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "lvsa.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(lvsa_[a-z_0-9]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    L = binding.lib()
    names = declared_symbols()
    assert set(binding.EXPORTS) <= set(names) and len(names) >= 10
    for n in names:
        assert hasattr(L, n), n
    assert "sm_100a" in binding.lvsa_version()


def test_struct_sizes_match_header():
    # 14 int32 + float + 2 int32; 21 int32 + pad + 5 int64
    assert C.sizeof(binding.Params) == 17 * 4
    assert C.sizeof(binding.IndexInfo) == 22 * 4 + 5 * 8


def test_argument_validation_needs_no_gpu():
    bad = [dict(T=0, P=4, H=1, d=64), dict(T=4, P=4, H=1, d=64, window=-1),
           dict(T=4, P=4, H=1, d=64, anchors=-2), dict(T=4, P=4, H=1, d=64, step=-1),
           dict(T=4, P=4, H=1, d=64, layer=-1), dict(T=1 << 16, P=1 << 16, H=1, d=64),
           dict(T=4, P=4, H=1, d=64, tie_break=7), dict(T=4, P=4, H=1, d=64, initial_anchors=-1),
           dict(T=4, P=4, H=1, d=64, n_text=-1)]
    for kw in bad:
        with pytest.raises(binding.LvsaError) as ei:
            binding.lvsa_build_block_index_ex(**kw)
        assert ei.value.status == binding.EINVAL, kw
    with pytest.raises(binding.LvsaError) as ei:
        binding.lvsa_schedule_create(T=4, P=4, H=1, d=64, window=-1)
    assert ei.value.status == binding.EINVAL
    for kw in [dict(T=4, P=4, H=1, d=96), dict(T=4, P=4, H=1, d=128, tile_q=64, tile_k=64),
               dict(T=4, P=4, H=1, d=64, dtype=binding.DTYPE_FP32, kernel=binding.KERNEL_TCGEN05)]:
        with pytest.raises(binding.LvsaError) as ei:
            binding.lvsa_build_block_index_ex(**kw)
        assert ei.value.status == binding.EUNSUPPORTED, kw


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-device failure mode")
def test_no_cpu_fallback_without_a_device():
    with pytest.raises(binding.LvsaError) as ei:
        binding.lvsa_build_block_index(8, 64, 2, 64, 1, 2, 0, 0)
    assert "cuda" in str(ei.value).lower()
