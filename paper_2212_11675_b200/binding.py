"""Thin ctypes binding of libgsr_b200.so (include/gsr.h): argument marshalling only.

Every step of the path runs in the library's CUDA kernels.  PyTorch is used for device memory
(`tensor.data_ptr()`) and streams (`torch.cuda.current_stream().cuda_stream`).  There is no
CPU fallback: if the shared library is missing or a call fails, GsrError is raised.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

_HERE = os.path.dirname(os.path.abspath(__file__))
# GSR_B200_LIB: another build of the SAME sources (the -DGSR_BOUNDS_CHECK one of build.build);
# never a fallback -- if the named file is missing, loading fails
LIB_PATH = os.environ.get("GSR_B200_LIB") or os.path.join(_HERE, "libgsr_b200.so")

GSR_OK, GSR_EINVAL, GSR_ENOMEM, GSR_ECUDA, GSR_ESTATE, GSR_EUNSUPPORTED, GSR_ERANGE = 0, -1, -2, -3, -4, -5, -6
GSR_OPT_FORCE_ITNLIM, GSR_OPT_DETERMINISTIC, GSR_OPT_FUSED, GSR_OPT_FIXED_POINT = 1, 2, 3, 4
GSR_OPT_APROD2_SPLIT, GSR_OPT_WHILE_GRAPH = 5, 6

EXPORTS = [
    "gsr_matrix_create", "gsr_matrix_begin", "gsr_matrix_append_rows", "gsr_matrix_finalize",
    "gsr_matrix_destroy", "gsr_matrix_dims", "gsr_matrix_device_bytes", "gsr_aprod1",
    "gsr_aprod2", "gsr_precondition", "gsr_lsqr_solve", "gsr_set_option", "gsr_strerror",
    "gsr_debug_expand_rows", "gsr_time_product", "gsr_launch_count", "gsr_lsqr_standard_errors", "gsr_lsqr_last_loop_ms", "gsr_lsqr_set_damp",
    "gsr_debug_fused_pass", "gsr_debug_graph_builds", "gsr_debug_while_graph", "gsr_matrix_set_constraints", "gsr_comm_unique_id", "gsr_comm_create", "gsr_comm_destroy", "gsr_matrix_set_comm",
    "gsr_matrix_begin_streamed", "gsr_matrix_host_bytes", "gsr_matrix_streamed_bytes",
    "gsr_norm2_static", "gsr_matrix_internal_rows", "gsr_vector_to_internal", "gsr_vector_from_internal",
    "gsr_aprod1_internal", "gsr_aprod2_internal",
]
GSR_NORM2_STATIC_MAX_LEN = 1 << 29


class GsrError(RuntimeError):
    def __init__(self, code: int, what: str):
        self.code = code
        # no strerror() lookup when the library itself is what is missing (it would recurse)
        msg = strerror(code) if _lib is not None else "libgsr_b200.so not loaded"
        super().__init__(f"{what}: {msg} ({code})")


class gsr_dims(C.Structure):
    _fields_ = [("n_rows", C.c_int64), ("n_stars", C.c_int64), ("n_dfa", C.c_int64),
                ("n_instr", C.c_int64), ("n_glob", C.c_int32)]


class gsr_lsqr_result(C.Structure):
    _fields_ = [("istop", C.c_int32), ("istop_natural", C.c_int32), ("itn", C.c_int64),
                ("itn_natural", C.c_int64), ("rnorm", C.c_double), ("arnorm", C.c_double),
                ("anorm", C.c_double), ("acond", C.c_double), ("xnorm", C.c_double),
                ("bnorm", C.c_double)]


@dataclass
class LsqrResult:
    istop: int
    itn: int
    istop_natural: int
    itn_natural: int
    rnorm: float
    arnorm: float
    anorm: float
    acond: float
    xnorm: float
    bnorm: float


_lib = None


def lib():
    """Load libgsr_b200.so; fail loudly when it has not been built (no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise GsrError(GSR_EUNSUPPORTED,
                           f"{LIB_PATH} is missing -- run __graft_entry__.build() "
                           "(python -m paper_2212_11675_b200.build)")
        L = C.CDLL(LIB_PATH)
        vp, i64, dbl = C.c_void_p, C.c_int64, C.c_double
        L.gsr_matrix_create.argtypes = [C.POINTER(vp), C.POINTER(gsr_dims), vp, vp, vp, vp, vp]
        L.gsr_matrix_begin.argtypes = [C.POINTER(vp), C.POINTER(gsr_dims), vp]
        L.gsr_matrix_begin_streamed.argtypes = [C.POINTER(vp), C.POINTER(gsr_dims), i64, i64, vp]
        L.gsr_matrix_host_bytes.argtypes = [vp]
        L.gsr_matrix_host_bytes.restype = i64
        L.gsr_matrix_streamed_bytes.argtypes = [vp]
        L.gsr_matrix_streamed_bytes.restype = i64
        L.gsr_matrix_append_rows.argtypes = [vp, i64, i64, vp, vp, vp, vp]
        L.gsr_matrix_finalize.argtypes = [vp]
        L.gsr_matrix_destroy.argtypes = [vp]
        L.gsr_matrix_dims.argtypes = [vp, C.POINTER(gsr_dims), C.POINTER(i64)]
        L.gsr_matrix_device_bytes.argtypes = [vp]
        L.gsr_matrix_device_bytes.restype = i64
        L.gsr_aprod1.argtypes = [vp, vp, vp, vp]
        L.gsr_aprod2.argtypes = [vp, vp, vp, vp]
        L.gsr_precondition.argtypes = [vp, vp, vp]
        L.gsr_lsqr_solve.argtypes = [vp, vp, vp, i64, dbl, dbl, dbl, C.POINTER(gsr_lsqr_result), vp]
        L.gsr_lsqr_standard_errors.argtypes = [vp, vp, vp]
        L.gsr_lsqr_set_damp.argtypes = [vp, dbl]
        L.gsr_lsqr_last_loop_ms.argtypes = [vp]
        L.gsr_lsqr_last_loop_ms.restype = dbl
        L.gsr_matrix_set_constraints.argtypes = [vp, i64, vp, vp, vp]
        L.gsr_comm_unique_id.argtypes = [vp, i64]
        L.gsr_comm_create.argtypes = [C.POINTER(vp), C.c_int, C.c_int, vp, i64]
        L.gsr_comm_destroy.argtypes = [vp]
        L.gsr_matrix_set_comm.argtypes = [vp, vp, i64, i64]
        L.gsr_set_option.argtypes = [vp, C.c_int, i64]
        L.gsr_strerror.argtypes = [C.c_int]
        L.gsr_strerror.restype = C.c_char_p
        L.gsr_debug_expand_rows.argtypes = [vp, i64, i64, vp, vp]
        L.gsr_time_product.argtypes = [vp, C.c_int, C.c_int, C.POINTER(C.c_float), vp]
        L.gsr_launch_count.argtypes = []
        L.gsr_launch_count.restype = i64
        L.gsr_debug_fused_pass.argtypes = [vp, vp, dbl, vp, vp, vp]
        L.gsr_debug_graph_builds.argtypes = [vp]
        L.gsr_debug_graph_builds.restype = i64
        L.gsr_debug_while_graph.argtypes = [vp]
        L.gsr_debug_while_graph.restype = C.c_int
        L.gsr_norm2_static.argtypes = [vp, i64, vp, vp]
        L.gsr_matrix_internal_rows.argtypes = [vp]
        L.gsr_matrix_internal_rows.restype = i64
        for name in ("gsr_vector_to_internal", "gsr_vector_from_internal", "gsr_aprod1_internal",
                     "gsr_aprod2_internal"):
            getattr(L, name).argtypes = [vp, vp, vp, vp]
        _lib = L
    return _lib


def strerror(code: int) -> str:
    try:
        return lib().gsr_strerror(int(code)).decode()
    except GsrError:
        return "library not built"


def _check(rc: int, what: str):
    if rc != GSR_OK:
        raise GsrError(rc, what)


def _ptr(a):
    """Address of a torch tensor (host or device), numpy array, int address or None."""
    if a is None:
        return None
    if isinstance(a, int):
        return a
    if hasattr(a, "data_ptr"):
        assert a.is_contiguous()
        return a.data_ptr()
    assert a.flags["C_CONTIGUOUS"]
    return a.ctypes.data


def _stream(stream):
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream if torch.cuda.is_available() else None
    return getattr(stream, "cuda_stream", stream)


def _dims(n_rows, n_stars, n_dfa, n_instr):
    return gsr_dims(int(n_rows), int(n_stars), int(n_dfa), int(n_instr), 1)


# ---- functions with the C names ------------------------------------------------------------

def gsr_matrix_create(n_rows, n_stars, n_dfa, n_instr, star_idx, att_start, instr_col, values,
                      stream=None) -> int:
    h = C.c_void_p()
    d = _dims(n_rows, n_stars, n_dfa, n_instr)
    _check(lib().gsr_matrix_create(C.byref(h), C.byref(d), _ptr(star_idx), _ptr(att_start),
                                   _ptr(instr_col), _ptr(values), _stream(stream)), "gsr_matrix_create")
    return h.value


def gsr_matrix_begin(n_rows, n_stars, n_dfa, n_instr, stream=None) -> int:
    h = C.c_void_p()
    d = _dims(n_rows, n_stars, n_dfa, n_instr)
    _check(lib().gsr_matrix_begin(C.byref(h), C.byref(d), _stream(stream)), "gsr_matrix_begin")
    return h.value


def gsr_matrix_begin_streamed(n_rows, n_stars, n_dfa, n_instr, resident_bytes, chunk_bytes,
                              stream=None) -> int:
    h = C.c_void_p()
    d = _dims(n_rows, n_stars, n_dfa, n_instr)
    _check(lib().gsr_matrix_begin_streamed(C.byref(h), C.byref(d), int(resident_bytes), int(chunk_bytes),
                                           _stream(stream)), "gsr_matrix_begin_streamed")
    return h.value


def gsr_matrix_host_bytes(h) -> int:
    return int(lib().gsr_matrix_host_bytes(h))


def gsr_matrix_streamed_bytes(h) -> int:
    return int(lib().gsr_matrix_streamed_bytes(h))


def gsr_matrix_append_rows(h, row0, nrows, star_idx, att_start, instr_col, values):
    _check(lib().gsr_matrix_append_rows(h, int(row0), int(nrows), _ptr(star_idx), _ptr(att_start),
                                        _ptr(instr_col), _ptr(values)), "gsr_matrix_append_rows")


def gsr_matrix_finalize(h):
    _check(lib().gsr_matrix_finalize(h), "gsr_matrix_finalize")


def gsr_matrix_destroy(h):
    _check(lib().gsr_matrix_destroy(h), "gsr_matrix_destroy")


def gsr_matrix_dims(h):
    d, n = gsr_dims(), C.c_int64()
    _check(lib().gsr_matrix_dims(h, C.byref(d), C.byref(n)), "gsr_matrix_dims")
    return d, n.value


def gsr_matrix_device_bytes(h) -> int:
    return int(lib().gsr_matrix_device_bytes(h))


def gsr_aprod1(h, x_dev, y_dev, stream=None):
    _check(lib().gsr_aprod1(h, _ptr(x_dev), _ptr(y_dev), _stream(stream)), "gsr_aprod1")


def gsr_aprod2(h, y_dev, x_dev, stream=None):
    _check(lib().gsr_aprod2(h, _ptr(y_dev), _ptr(x_dev), _stream(stream)), "gsr_aprod2")


def gsr_matrix_internal_rows(h) -> int:
    return int(lib().gsr_matrix_internal_rows(h))


def gsr_vector_to_internal(h, y_dev, yint_dev, stream=None):
    _check(lib().gsr_vector_to_internal(h, _ptr(y_dev), _ptr(yint_dev), _stream(stream)), "gsr_vector_to_internal")


def gsr_vector_from_internal(h, yint_dev, y_dev, stream=None):
    _check(lib().gsr_vector_from_internal(h, _ptr(yint_dev), _ptr(y_dev), _stream(stream)),
           "gsr_vector_from_internal")


def gsr_aprod1_internal(h, x_dev, yint_dev, stream=None):
    _check(lib().gsr_aprod1_internal(h, _ptr(x_dev), _ptr(yint_dev), _stream(stream)), "gsr_aprod1_internal")


def gsr_aprod2_internal(h, yint_dev, x_dev, stream=None):
    _check(lib().gsr_aprod2_internal(h, _ptr(yint_dev), _ptr(x_dev), _stream(stream)), "gsr_aprod2_internal")


def gsr_precondition(h, p_out=None, stream=None):
    _check(lib().gsr_precondition(h, _ptr(p_out), _stream(stream)), "gsr_precondition")


def gsr_lsqr_solve(h, b, x, itnlim, atol=0.0, btol=0.0, conlim=0.0, stream=None) -> LsqrResult:
    r = gsr_lsqr_result()
    _check(lib().gsr_lsqr_solve(h, _ptr(b), _ptr(x), int(itnlim), float(atol), float(btol),
                                float(conlim), C.byref(r), _stream(stream)), "gsr_lsqr_solve")
    return LsqrResult(r.istop, r.itn, r.istop_natural, r.itn_natural, r.rnorm, r.arnorm, r.anorm,
                      r.acond, r.xnorm, r.bnorm)


def gsr_lsqr_set_damp(h, damp: float):
    _check(lib().gsr_lsqr_set_damp(h, float(damp)), "gsr_lsqr_set_damp")


def gsr_lsqr_last_loop_ms(h) -> float:
    return float(lib().gsr_lsqr_last_loop_ms(h))


def gsr_lsqr_standard_errors(h, se, stream=None):
    _check(lib().gsr_lsqr_standard_errors(h, _ptr(se), _stream(stream)), "gsr_lsqr_standard_errors")


def gsr_matrix_set_constraints(h, n_con, row_ptr, col, val):
    """row_ptr int64 [n_con+1], col int32 [nnz], val float64 [nnz] (numpy, torch or None)."""
    _check(lib().gsr_matrix_set_constraints(h, int(n_con), _ptr(row_ptr), _ptr(col), _ptr(val)),
           "gsr_matrix_set_constraints")


GSR_COMM_ID_BYTES = 128


def gsr_comm_unique_id() -> bytes:
    """Rank 0: a fresh NCCL unique id, to be broadcast to the other ranks by the caller."""
    buf = C.create_string_buffer(GSR_COMM_ID_BYTES)
    _check(lib().gsr_comm_unique_id(buf, GSR_COMM_ID_BYTES), "gsr_comm_unique_id")
    return buf.raw


def gsr_comm_create(rank: int, world: int, unique_id: bytes) -> int:
    c = C.c_void_p()
    buf = C.create_string_buffer(bytes(unique_id), GSR_COMM_ID_BYTES)
    _check(lib().gsr_comm_create(C.byref(c), int(rank), int(world), buf, GSR_COMM_ID_BYTES), "gsr_comm_create")
    return c.value


def gsr_comm_destroy(c):
    _check(lib().gsr_comm_destroy(c), "gsr_comm_destroy")


def gsr_matrix_set_comm(h, comm, n_rows_global, n_cols_global):
    _check(lib().gsr_matrix_set_comm(h, comm, int(n_rows_global), int(n_cols_global)), "gsr_matrix_set_comm")


def gsr_set_option(h, key, value):
    _check(lib().gsr_set_option(h, int(key), int(value)), "gsr_set_option")


def gsr_debug_expand_rows(h, row0, nrows):
    import numpy as np
    cols = np.empty((nrows, 24), dtype=np.int64)
    vals = np.empty((nrows, 24), dtype=np.float64)
    _check(lib().gsr_debug_expand_rows(h, int(row0), int(nrows), _ptr(cols), _ptr(vals)),
           "gsr_debug_expand_rows")
    return cols, vals


def gsr_time_product(h, which, reps, stream=None) -> float:
    ms = C.c_float()
    _check(lib().gsr_time_product(h, int(which), int(reps), C.byref(ms), _stream(stream)),
           "gsr_time_product")
    return float(ms.value)


def gsr_debug_fused_pass(h, x_dev, ca, y_dev, t_dev, stream=None):
    """y <- A x + ca y ; t += A^T y_new through the solver's fused kernels (caller row order)."""
    _check(lib().gsr_debug_fused_pass(h, _ptr(x_dev), float(ca), _ptr(y_dev), _ptr(t_dev),
                                      _stream(stream)), "gsr_debug_fused_pass")


def gsr_debug_graph_builds(h) -> int:
    return int(lib().gsr_debug_graph_builds(h))


def gsr_debug_while_graph(h) -> int:
    return int(lib().gsr_debug_while_graph(h))


def gsr_norm2_static(v_dev, out_dev, stream=None, length=None):
    """out_dev[0] = ||v_dev||_2 without any device allocation (include/gsr.h): for callers that
    run while the device is full or that cannot afford cudaMalloc's device-wide synchronisation.
    The scratch is one fixed array per GPU shared by all calls: keep the calls of a device on one
    stream.  At most GSR_NORM2_STATIC_MAX_LEN elements; `length` defaults to v_dev.numel()."""
    n = int(v_dev.numel() if length is None else length)
    _check(lib().gsr_norm2_static(_ptr(v_dev), n, _ptr(out_dev), _stream(stream)),
           f"gsr_norm2_static(len={n}, limit={GSR_NORM2_STATIC_MAX_LEN})")


def gsr_launch_count() -> int:
    return int(lib().gsr_launch_count())


class GsrMatrix:
    """RAII convenience around the handle (still only marshalling)."""

    def __init__(self, handle: int):
        self.h = handle
        d, n = gsr_matrix_dims(handle)
        self.m, self.n = d.n_rows, n
        self.n_stars, self.n_dfa, self.n_instr = d.n_stars, d.n_dfa, d.n_instr

    @classmethod
    def create(cls, cfg, star, att, instr, vals, stream=None):
        return cls(gsr_matrix_create(cfg.n_rows, cfg.n_stars, cfg.n_dfa, cfg.n_instr, star, att,
                                     instr, vals, stream))

    def close(self):
        if self.h:
            gsr_matrix_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()
