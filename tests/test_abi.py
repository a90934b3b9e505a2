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


@pytest.mark.parametrize("dims,code", [
    ((10, 1, 8, 27521, 1), "GSR_EUNSUPPORTED"),           # I: x's instrumental block + windows > 227 KB
    ((10, 1, 8, 70000, 1), "GSR_EUNSUPPORTED"),           # I > 65535 (uint16 instrumental columns)
    ((10, 1, 987_140, 3328, 1), "GSR_EUNSUPPORTED"),  # more than 4096 attitude bins at bw = 241
    ((10, 1, 724_996, 10_000, 1), "GSR_EUNSUPPORTED"),    # ... at bw = 177 (I = 10 000)
    ((10, 429_496_800, 8, 1, 1), "GSR_EINVAL"),           # n_cols >= 2^31
    ((0xFFFFFFF0, 1, 8, 1, 1), "GSR_EINVAL"),             # n_rows >= 2^32 - 16
    ((-1, 1, 8, 1, 1), "GSR_EINVAL"),
    ((10, 0, 8, 1, 1), "GSR_EINVAL"),
    ((10, 1, 8, 0, 1), "GSR_EINVAL"),
])
def test_size_limits_documented_in_the_header(lib, dims, code):
    """include/gsr.h "Size limits": each is refused before any device work."""
    from paper_2212_11675_b200 import binding as b
    h = C.c_void_p()
    d = b.gsr_dims(*dims)
    assert lib.gsr_matrix_begin(C.byref(h), C.byref(d), None) == getattr(b, code) and not h.value


def test_sizes_just_inside_the_limits_pass_the_checks(lib):
    """The same checks accept the largest sizes the header names (on a box without a GPU the call
    then fails at the device query, which is not a size error)."""
    import torch
    from paper_2212_11675_b200 import binding as b
    for dims in ((10, 1, 8, 27520, 1), (10, 1, 987_139, 3328, 1), (10, 1, 724_995, 10_000, 1)):
        h = C.c_void_p()
        d = b.gsr_dims(*dims)
        rc = lib.gsr_matrix_begin(C.byref(h), C.byref(d), None)
        if torch.cuda.is_available():
            assert rc == b.GSR_OK
            lib.gsr_matrix_destroy(h)
        else:
            assert rc == b.GSR_ECUDA


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
