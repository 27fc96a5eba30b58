"""Fault injection: an index whose build overflowed its allocation bound must fail loudly.

The builder sizes its arena from an upper bound on the kept tiles (lvsa_index.cu).  If that bound were ever
wrong, the fill passes write nothing; before this test existed lvsa_attn_fwd would then have walked unfilled
lists with status LVSA_OK.  Now the list ends are poisoned on the device, every attention kernel traps on a
poisoned index, lvsa_index_info / copy_host report the overflow, and lvsa_attn_fwd refuses an index once the
host knows.  The bound cannot be made wrong through the API, so the test compiles a separate library with
-DLVSA_TEST_CAP_SHRINK (build.build_variant; never the product path) and runs each case in a subprocess of
its own, because a device trap poisons the CUDA context of the process it happens in."""
import os
import subprocess
import sys
import textwrap

import pytest

from paper_2605_31057_b200 import build

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

PRELUDE = """
import sys, torch
sys.path.insert(0, {root!r})
from paper_2605_31057_b200 import build, binding
build.build = lambda *a, **k: {lib!r}            # this process loads the fault-injection build
w = dict(T=9, P=200, H=2, d={d}, window=1, anchors=2, step=1, dtype={dtype}, kernel={kernel})
N = w["T"] * w["P"]
dt = torch.float32 if {dtype} == binding.DTYPE_FP32 else torch.bfloat16
q = torch.randn((1, N, w["H"], w["d"]), device="cuda").to(dt)
out = torch.zeros_like(q)
ix = binding.lvsa_build_block_index_ex(**w)
"""


@pytest.fixture(scope="module")
def shrunk_lib(tmp_path_factory):
    out = str(tmp_path_factory.mktemp("lvsa_variant") / "liblvsa_cap_shrink.so")
    return build.build_variant(out, ["-DLVSA_TEST_CAP_SHRINK=64"])


def run(script):
    return subprocess.run([sys.executable, "-c", textwrap.dedent(script)], capture_output=True, text=True, timeout=600)


CASES = {"pair": dict(d=128, dtype=0, kernel=2), "v0": dict(d=128, dtype=0, kernel=3), "d64": dict(d=64, dtype=0, kernel=2),
         "quad": dict(d=128, dtype=0, kernel=4), "hybrid": dict(d=128, dtype=0, kernel=5), "simt": dict(d=64, dtype=1, kernel=1)}


@pytest.mark.parametrize("case", list(CASES))
def test_kernel_traps_on_an_overflowed_index(shrunk_lib, case):
    r = run(PRELUDE.format(root=ROOT, lib=shrunk_lib, **CASES[case]) + """
binding.lvsa_attn_fwd(q, q, q, ix, out, None)       # the host does not know yet: the call enqueues
try:
    torch.cuda.synchronize()
    print("NO-ERROR")
except Exception as e:
    print("DEVICE-ERROR", type(e).__name__, str(e)[:120].replace("\\n", " "))
""")
    assert "DEVICE-ERROR" in r.stdout and "NO-ERROR" not in r.stdout, (r.stdout[-2000:], r.stderr[-2000:])


def test_host_reports_and_then_refuses(shrunk_lib):
    r = run(PRELUDE.format(root=ROOT, lib=shrunk_lib, d=128, dtype=0, kernel=2) + """
try:
    ix.info()
    print("INFO-OK")
except binding.LvsaError as e:
    print("INFO-ERROR", e.status, e)
try:
    binding.lvsa_attn_fwd(q, q, q, ix, out, None)
    print("FWD-ENQUEUED")
except binding.LvsaError as e:
    print("FWD-REFUSED", e.status, e)
torch.cuda.synchronize()                              # nothing ran: the context is healthy
print("SYNC-OK", float(out.abs().max()))
""")
    assert "INFO-ERROR 3" in r.stdout and "allocation bound" in r.stdout, (r.stdout[-2000:], r.stderr[-2000:])
    assert "FWD-REFUSED 3" in r.stdout and "FWD-ENQUEUED" not in r.stdout, r.stdout[-2000:]
    assert "SYNC-OK 0.0" in r.stdout, r.stdout[-2000:]


def test_the_product_library_is_not_the_fault_injection_build():
    src = open(os.path.join(ROOT, "paper_2605_31057_b200", "csrc", "build.log")).read() if os.path.exists(
        os.path.join(ROOT, "paper_2605_31057_b200", "csrc", "build.log")) else ""
    assert "LVSA_TEST_CAP_SHRINK" not in src
    assert "LVSA_TEST_CAP_SHRINK" not in " ".join(build.NVCC_FLAGS)
