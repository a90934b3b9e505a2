"""gsr_norm2_static: the norm for callers that cannot allocate device memory.

Some users of this library are handed device buffers and a stream and nothing else: a
convergence monitor that runs beside a solve which already fills the GPU (a cudaMalloc there can
fail, or make the host framework drop its cache), or code on a latency path (cudaMalloc and
cudaFree synchronise the whole device and would stall the iteration in flight).  Every other
entry point needs a handle, and a handle allocates.  gsr_norm2_static keeps its partial sums in
a fixed 33 KB array inside the library image instead, one per GPU, shared by all calls.

What is checked here: the new entry point against the EXISTING path for the same quantity --
`bnorm` = ||b||, which gsr_lsqr_solve forms with the handle's own (cudaMalloc'ed) partial sums --
on consecutive calls.  The calls alternate between a long and a short vector, so the second call
finds the first one's partial sums and ticket still in the array: a call that relied on the
array being fresh, or that read a stale partial, would fail.  The file is named to be collected
last (pytest -x would otherwise hide every later test behind a failure here), and it passes
both alone in a fresh process and after the rest of the suite.
"""
import ctypes as C

import numpy as np
import pytest
import torch

from paper_2212_11675_b200 import inputs

pytestmark = pytest.mark.gpu

# Both sides sum squares (all terms positive) in fp64 in a different order: the difference is a
# few ulp.  The bar is the suite's aprod tolerance, 1e-12 relative (tests/test_gpu_parity.py).
TOL = 1e-12


def _binding():
    from paper_2212_11675_b200 import binding
    return binding


def _bnorm_existing_path(b, counts, seed):
    """||rhs|| as gsr_lsqr_solve reports it (k_gather_sumsq + k_scalar_init1 on handle memory)."""
    cfg = inputs.micro_config("noalloc", seed, counts, 12, 5)
    star, att, instr, vals = inputs.gen_all(cfg)
    A = b.GsrMatrix.create(cfg, star.cuda(), att.cuda(), instr.cuda(), vals.cuda())
    rhs = inputs.random_vector(cfg, 9, cfg.n_rows).cuda()
    x = torch.empty(cfg.n_cols, dtype=torch.float64, device="cuda")
    r = b.gsr_lsqr_solve(A.h, rhs, x, 1)
    A.close()
    return rhs, r.bnorm


def test_static_norm_matches_the_solver_norm_on_consecutive_calls():
    b = _binding()
    # long: 3 CTAs of 2^17 elements and a ragged tail; short: a fraction of one CTA
    long_v, long_ref = _bnorm_existing_path(b, [1000] * 400 + [37], 31)
    short_v, short_ref = _bnorm_existing_path(b, [700, 3, 0, 250], 32)
    assert long_v.numel() == 400_037 and short_v.numel() == 953
    out = torch.full((4,), -1.0, dtype=torch.float64, device="cuda")
    # back to back on one stream, no synchronisation in between: the calls share the array
    b.gsr_norm2_static(long_v, out[0:1])
    b.gsr_norm2_static(short_v, out[1:2])
    b.gsr_norm2_static(long_v, out[2:3])
    b.gsr_norm2_static(short_v, out[3:4])
    got = out.cpu().numpy()
    for g, ref in zip(got, (long_ref, short_ref, long_ref, short_ref)):
        assert ref > 0 and abs(g - ref) <= TOL * ref, (g, ref)
    # same input, same bits: the result does not depend on which CTA finished last
    assert got[0] == got[2] and got[1] == got[3]
    # and against the plain definition
    assert abs(got[0] - float(torch.linalg.vector_norm(long_v))) <= TOL * long_ref


def test_static_norm_edges_and_limit():
    b = _binding()
    out = torch.full((1,), -1.0, dtype=torch.float64, device="cuda")
    b.gsr_norm2_static(torch.empty(0, dtype=torch.float64, device="cuda"), out)
    assert out.item() == 0.0                                    # empty vector
    v = torch.tensor([3.0, -4.0], dtype=torch.float64, device="cuda")
    b.gsr_norm2_static(v, out)
    assert out.item() == 5.0
    # exactly one full CTA chunk, and one element more (a second CTA with a single element)
    w = torch.ones((1 << 17) + 1, dtype=torch.float64, device="cuda")
    b.gsr_norm2_static(w, out, length=1 << 17)
    assert out.item() == float(np.sqrt(float(1 << 17)))
    b.gsr_norm2_static(w, out)
    assert abs(out.item() - np.sqrt((1 << 17) + 1.0)) <= TOL * out.item()
    # beyond the array's capacity: refused with the library's size error, nothing launched
    n0 = b.gsr_launch_count()
    with pytest.raises(b.GsrError) as e:
        b.gsr_norm2_static(w, out, length=b.GSR_NORM2_STATIC_MAX_LEN + 1)
    assert e.value.code == b.GSR_EUNSUPPORTED and "limit" in str(e.value)
    assert b.gsr_launch_count() == n0
    L = b.lib()
    assert L.gsr_norm2_static(None, 5, C.c_void_p(out.data_ptr()), None) == b.GSR_EINVAL
    assert L.gsr_norm2_static(C.c_void_p(w.data_ptr()), -1, C.c_void_p(out.data_ptr()), None) == b.GSR_EINVAL
    assert L.gsr_norm2_static(C.c_void_p(w.data_ptr()), 5, None, None) == b.GSR_EINVAL
