"""CPU-only: the C-ABI library builds, loads and exports every symbol include/gsr.h declares.
No compute calls (there is no GPU here); argument checks that need no device are exercised."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2212_11675_b200 import build, binding
    build.build()
    return binding.lib()


def _declared():
    src = open(os.path.join(ROOT, "include", "gsr.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(gsr_[a-z0-9_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(lib):
    from paper_2212_11675_b200 import binding
    names = _declared()
    assert len(names) >= 14
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(binding.EXPORTS) == names      # the binding mirrors the header one to one


def test_strerror_and_null_checks(lib):
    from paper_2212_11675_b200 import binding as b
    assert b.strerror(0) == "ok"
    for code in (-1, -2, -3, -4, -5):
        assert b.strerror(code) and "unknown" not in b.strerror(code)
    assert "unknown" in b.strerror(-99)
    assert lib.gsr_matrix_destroy(None) == 0
    assert lib.gsr_matrix_begin(None, None, None) == b.GSR_EINVAL
    h = C.c_void_p()
    d = b.gsr_dims(10, 1, 3, 1, 1)                 # D < 4
    assert lib.gsr_matrix_begin(C.byref(h), C.byref(d), None) == b.GSR_EINVAL and not h.value
    d = b.gsr_dims(10, 1, 8, 1, 2)                 # n_glob != 1
    assert lib.gsr_matrix_begin(C.byref(h), C.byref(d), None) == b.GSR_EINVAL
    assert lib.gsr_aprod1(None, None, None, None) == b.GSR_EINVAL
    assert lib.gsr_lsqr_solve(None, None, None, 1, 0.0, 0.0, 0.0, None, None) == b.GSR_EINVAL
    assert lib.gsr_launch_count() == 0


def test_no_gpu_fails_loudly_not_silently(lib):
    """Without a CUDA device the product path reports an error; it never computes on the CPU."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_2212_11675_b200 import binding as b
    h = C.c_void_p()
    d = b.gsr_dims(10, 1, 8, 1, 1)
    rc = lib.gsr_matrix_begin(C.byref(h), C.byref(d), None)
    assert rc in (b.GSR_ECUDA, b.GSR_EUNSUPPORTED) and not h.value


def test_product_path_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2212_11675_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cuh")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in txt.lower() or f == "inputs.py", f
    txt = open(os.path.join(pkg, "inputs.py")).read()
    assert "import oracle" not in txt and "from oracle" not in txt
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            assert "paper_2212_11675_b200" not in open(os.path.join(ROOT, "oracle", f)).read() \
                or f.endswith(".c")
