"""The two products on vectors in the library's internal row order (gsr_aprod1_internal,
gsr_aprod2_internal with gsr_vector_to_internal / _from_internal; Algorithms 1-2,
PAPER.md:145-392) against the oracle, element-wise at the aprod bar, on the edge-case systems of
tests/test_gpu_parity.py, with constraint rows, and on a streamed (out-of-core) handle."""
import numpy as np
import pytest
import torch

from paper_2212_11675_b200 import inputs
from tests.test_gpu_parity import APROD_TOL, CASES, Sys, _binding

pytestmark = pytest.mark.gpu


def _check_products(b, h, o, cfg, m_total, n):
    mi = b.gsr_matrix_internal_rows(h)
    assert mi >= m_total and (mi - (m_total - cfg.n_rows)) % 32 == 0     # whole tiles + constraint rows
    x = inputs.random_vector(cfg, 1, n)
    y0 = inputs.random_vector(cfg, 2, m_total)
    # round trip: bit exact, padding positions zero
    yi = torch.full((mi,), 7.0, dtype=torch.float64, device="cuda")
    b.gsr_vector_to_internal(h, y0.cuda(), yi)
    back = torch.full((m_total,), -3.0, dtype=torch.float64, device="cuda")
    b.gsr_vector_from_internal(h, yi, back)
    assert torch.equal(back.cpu(), y0)
    assert abs(float(yi.sum()) - float(y0.sum())) <= 1e-9 * float(y0.abs().sum() + 1)
    assert int((yi == 0).sum()) >= mi - m_total
    # aprod1: y0 + A x
    y_ref, scale = o.aprod1(x.numpy(), y0.numpy(), want_scale=True)
    b.gsr_aprod1_internal(h, x.cuda(), yi)
    b.gsr_vector_from_internal(h, yi, back)
    err = np.abs(back.cpu().numpy() - y_ref)
    assert np.all(err <= APROD_TOL * scale), float((err / scale).max())
    # aprod2: x0 + A^T y
    y = inputs.random_vector(cfg, 3, m_total)
    x0 = inputs.random_vector(cfg, 4, n)
    x_ref, xs = o.aprod2(y.numpy(), x0.numpy(), want_scale=True)
    b.gsr_vector_to_internal(h, y.cuda(), yi)
    for split in (1, 0):
        xd = x0.cuda()
        b.gsr_set_option(h, b.GSR_OPT_APROD2_SPLIT, split)
        b.gsr_aprod2_internal(h, yi, xd)
        err = np.abs(xd.cpu().numpy() - x_ref)
        assert np.all(err <= APROD_TOL * np.maximum(xs, 1e-300)), (split, float((err / xs).max()))
    b.gsr_set_option(h, b.GSR_OPT_APROD2_SPLIT, -1)


@pytest.mark.parametrize("name", list(CASES))
def test_internal_order_products_match_the_oracle(name):
    b = _binding()
    s = Sys(CASES[name], edge_att=True)
    try:
        _check_products(b, s.A.h, s.o, s.cfg, s.m, s.n)
    finally:
        s.A.close()


def test_internal_order_products_with_constraint_rows():
    b = _binding()
    s = Sys(CASES["ragged_empty_stars"])
    try:
        rng = np.random.default_rng(3)
        n_con = 5
        ptr = np.arange(0, 4 * n_con + 1, 4, dtype=np.int64)
        col = rng.integers(0, s.n, 4 * n_con).astype(np.int32)
        val = rng.standard_normal(4 * n_con)
        s.o.set_constraints(ptr, col, val)
        b.gsr_matrix_set_constraints(s.A.h, n_con, ptr, col, val)
        _check_products(b, s.A.h, s.o, s.cfg, s.m + n_con, s.n)
    finally:
        s.A.close()


def test_internal_order_calls_before_finalize_are_refused():
    b = _binding()
    h = b.gsr_matrix_begin(10, 1, 8, 2)
    try:
        assert b.gsr_matrix_internal_rows(h) == -1
        t = torch.zeros(64, dtype=torch.float64, device="cuda")
        for fn in (b.gsr_vector_to_internal, b.gsr_vector_from_internal, b.gsr_aprod1_internal,
                   b.gsr_aprod2_internal):
            with pytest.raises(b.GsrError) as e:
                fn(h, t, t)
            assert e.value.code == b.GSR_ESTATE
    finally:
        b.gsr_matrix_destroy(h)
