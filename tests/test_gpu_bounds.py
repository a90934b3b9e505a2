"""The product kernels with their index computations turned into device asserts
(-DGSR_BOUNDS_CHECK, csrc/gsr_aprod.cu): window offsets, star numbers and instrumental columns
(Algorithms 1-2).  compute-sanitizer is not available on the GPU pool, so this
instrumented build is what checks the indices: a second library is compiled into a temporary
directory and a fresh process runs the cfg1/10 parity of __graft_entry__.smoke() and two seeds
of the fuzz test through it.  A failed device assert aborts that process."""
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_bounds_checked_build_passes_parity_and_fuzz(tmp_path):
    from paper_2212_11675_b200 import build
    lib = build.build(extra_flags=["-DGSR_BOUNDS_CHECK"], out=str(tmp_path / "libgsr_b200_bounds.so"))
    # the asserts are really in this build and not in the product one
    dump = lambda p: subprocess.run(["cuobjdump", "-sass", p], capture_output=True, text=True).stdout
    assert "__assertfail" in dump(lib) or "assert" in subprocess.run(
        ["strings", lib], capture_output=True, text=True).stdout
    env = dict(os.environ, GSR_B200_LIB=lib)
    code = ("import __graft_entry__ as e, paper_2212_11675_b200.binding as b; "
            f"assert b.LIB_PATH == {lib!r}; e.smoke()")
    out = subprocess.run([sys.executable, "-c", code], cwd=ROOT, env=env, capture_output=True, text=True,
                         timeout=900)
    assert out.returncode == 0 and "smoke ok" in out.stdout, out.stderr[-3000:]
    out = subprocess.run([sys.executable, "-m", "pytest", "-q", "-x", "-m", "gpu", "tests/test_gpu_fuzz.py",
                          "-k", "11 or 12"], cwd=ROOT, env=env, capture_output=True, text=True, timeout=900)
    assert out.returncode == 0 and "2 passed" in out.stdout, out.stdout[-3000:] + out.stderr[-3000:]
