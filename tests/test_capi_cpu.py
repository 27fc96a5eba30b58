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


def test_header_constants_match_binding():
    """The enum values the binding hard-codes are the header's."""
    src = open(os.path.join(ROOT, "include", "lvsa.h")).read()
    vals = {k: int(v) for k, v in re.findall(r"\b(LVSA_[A-Z0-9_]+)\s*=\s*(-?\d+)", src)}
    for name in ("KERNEL_AUTO", "KERNEL_SIMT", "KERNEL_TCGEN05", "KERNEL_TCGEN05_V0", "KERNEL_TCGEN05_QUAD", "KERNEL_TCGEN05_HYBRID", "LAYOUT_NHD", "LAYOUT_HND",
                 "KV_TILES_TOKEN0", "KV_TILES_FRAME_ALIGNED",
                 "DTYPE_BF16", "DTYPE_FP32", "TIE_LO", "TIE_HI", "TILE_FULL", "TILE_PARTIAL", "OK", "EINVAL",
                 "EUNSUPPORTED", "ECUDA", "ENOMEM"):
        assert vals["LVSA_" + name] == getattr(binding, name), name
    assert int(re.search(r"#define LVSA_KV_PAD (\d+)", src).group(1)) == binding.KV_PAD
    # no debug hooks or environment switches in the product library
    csrc = os.path.join(ROOT, "paper_2605_31057_b200", "csrc")
    for f in os.listdir(csrc):
        if f.endswith((".cu", ".cuh", ".h")):
            assert "getenv" not in open(os.path.join(csrc, f)).read(), f
    assert not hasattr(binding.lib(), "lvsa_debug_set_dump")
    # ... and none in the Python side that picks the library: build.py / binding.py read no environment
    pkg = os.path.join(ROOT, "paper_2605_31057_b200")
    for f in ("build.py", "binding.py", "__init__.py", "inputs.py"):
        src = open(os.path.join(pkg, f)).read()
        assert "environ" not in src and "getenv" not in src, f
    assert binding._build.build() == binding._build.LIB


def test_version_names_the_variants_compiled_in():
    v = binding.lvsa_version()
    for word in ("static-scratch", "quad", "hybrid", "frame-aligned", "CTA-pair", "simt"):
        assert word in v, word


def test_struct_sizes_match_header():
    # 14 int32 + float + 5 int32 + 4 x 3 int64; 24 int32 + 6 int64 (include/lvsa.h)
    assert C.sizeof(binding.Params) == 20 * 4 + 12 * 8 and binding.Params.stride_q.offset == 80
    assert C.sizeof(binding.IndexInfo) == 24 * 4 + 6 * 8
    assert binding.IndexInfo.N.offset == 24 * 4


def test_argument_validation_needs_no_gpu():
    bad = [dict(T=0, P=4, H=1, d=64), dict(T=4, P=4, H=1, d=64, window=-1),
           dict(T=4, P=4, H=1, d=64, anchors=-2), dict(T=4, P=4, H=1, d=64, step=-1),
           dict(T=4, P=4, H=1, d=64, layer=-1), dict(T=1 << 16, P=1 << 16, H=1, d=64),
           dict(T=4, P=4, H=1, d=64, tie_break=7), dict(T=4, P=4, H=1, d=64, initial_anchors=-1),
           dict(T=4, P=4, H=1, d=64, n_text=-1), dict(T=4, P=4, H=1, d=64, layout=2),
           dict(T=4, P=4, H=1, d=64, kernel=6), dict(T=4, P=4, H=1, d=64, host_groups=-1),
           dict(T=4, P=4, H=1, d=64, kv_tiling=2)]
    for kw in bad:
        with pytest.raises(binding.LvsaError) as ei:
            binding.lvsa_build_block_index_ex(**kw)
        assert ei.value.status == binding.EINVAL, kw
    with pytest.raises(binding.LvsaError) as ei:
        binding.lvsa_schedule_create(T=4, P=4, H=1, d=64, window=-1)
    assert ei.value.status == binding.EINVAL
    for kw in [dict(T=4, P=4, H=1, d=96), dict(T=4, P=4, H=1, d=128, tile_q=64, tile_k=64),
               dict(T=4, P=4, H=1, d=64, dtype=binding.DTYPE_FP32, kernel=binding.KERNEL_TCGEN05),
               dict(T=4, P=4, H=1, d=128, dtype=binding.DTYPE_FP32, kernel=binding.KERNEL_TCGEN05_V0),
               dict(T=4, P=4, H=1, d=64, kernel=binding.KERNEL_TCGEN05_QUAD),
               dict(T=4, P=4, H=1, d=128, kernel=binding.KERNEL_TCGEN05_QUAD, kv_tiling=binding.KV_TILES_FRAME_ALIGNED)]:
        with pytest.raises(binding.LvsaError) as ei:
            binding.lvsa_build_block_index_ex(**kw)
        assert ei.value.status == binding.EUNSUPPORTED, kw


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-device failure mode")
def test_no_cpu_fallback_without_a_device():
    with pytest.raises(binding.LvsaError) as ei:
        binding.lvsa_build_block_index(8, 64, 2, 64, 1, 2, 0, 0)
    assert "cuda" in str(ei.value).lower()
