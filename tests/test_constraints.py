"""Row f3: constraint equations as extra CSR rows below the observations (the
"constraints computation" that ends Algorithms 1 and 2).
CPU: the oracle against a dense augmented matrix (numpy).  GPU: the C ABI against the oracle."""
import numpy as np
import pytest
import scipy.sparse as sp

from paper_2212_11675_b200 import inputs
from tests.helpers import csr_from_raw, make_oracle, small_system


def _constraints(n, n_con, nnz_row, seed, empty_row=True):
    rng = np.random.default_rng(seed)
    C = np.zeros((n_con, n))
    for r in range(n_con):
        if empty_row and r == 1:
            continue                                  # an all-zero constraint row is legal
        idx = rng.choice(n, min(nnz_row, n), replace=False)
        C[r, idx] = rng.standard_normal(idx.size)
    Cs = sp.csr_matrix(C)
    return C, Cs.indptr.astype(np.int64), Cs.indices.astype(np.int32), Cs.data.astype(np.float64)


def test_oracle_with_constraints_equals_dense_augmented_matrix():
    cfg, star, att, instr, vals = small_system()
    o = make_oracle(cfg, star, att, instr, vals)
    A = csr_from_raw(cfg, star, att, instr, vals)[0].toarray()
    C, ptr, col, val = _constraints(o.n, 5, 17, 3)
    o.set_constraints(ptr, col, val)
    Aug = np.vstack([A, C])
    rng = np.random.default_rng(4)
    x, y = rng.standard_normal(o.n), rng.standard_normal(o.m_total)
    y0, x0 = rng.standard_normal(o.m_total), rng.standard_normal(o.n)
    assert np.allclose(o.aprod1(x, y0), y0 + Aug @ x, rtol=0, atol=1e-13)
    assert np.allclose(o.aprod2(y, x0), x0 + Aug.T @ y, rtol=0, atol=1e-13)
    # adjoint identity on the augmented operator
    lhs = np.dot(o.aprod1(x, np.zeros(o.m_total)), y)
    rhs = np.dot(x, o.aprod2(y, np.zeros(o.n)))
    assert abs(lhs - rhs) <= 1e-13 * np.linalg.norm(Aug @ x) * np.linalg.norm(y)
    assert np.allclose(o.colsumsq(), (Aug ** 2).sum(0), rtol=1e-14)
    b = rng.standard_normal(o.m_total)
    r = o.lsqr(b, 1000, 1e-14, 1e-14, 1e12)
    xl = np.linalg.lstsq(Aug, b, rcond=None)[0]
    assert np.linalg.norm(r.x - xl) <= 1e-10 * np.linalg.norm(xl)
    p = o.precondition()
    assert np.allclose(p, 1.0 / np.sqrt((Aug ** 2).sum(0)), rtol=1e-14)
    assert np.allclose(o.con_val, val * p[col], rtol=1e-15)
    r = o.lsqr(b, 1000, 1e-14, 1e-14, 1e12)
    assert np.linalg.norm(r.x - xl) <= 1e-10 * np.linalg.norm(xl)


def test_constraints_make_a_rank_deficient_system_unique():
    """The reason the paper gives for them: a column that no observation touches
    is pinned by a constraint row, and LSQR then returns the constrained value."""
    cfg = inputs.micro_config("rankdef", 5, (30, 0, 30), 6, 4)      # star 1 has no observations
    star, att, instr, vals = [t.numpy() for t in inputs.gen_all(cfg)]
    o = make_oracle(cfg, star, att, instr, vals)
    A = csr_from_raw(cfg, star, att, instr, vals)[0].toarray()
    assert np.all(A[:, 5:10] == 0)
    ptr = np.arange(6, dtype=np.int64)
    col = np.arange(5, 10, dtype=np.int32)
    val = np.full(5, 2.0)
    o.set_constraints(ptr, col, val)                                 # 2 * x_j = b_con
    rng = np.random.default_rng(0)
    b = np.concatenate([rng.standard_normal(o.m), [2.0, 4.0, 6.0, 8.0, 10.0]])
    r = o.lsqr(b, 500, 1e-14, 1e-14, 1e12)
    assert np.allclose(r.x[5:10], [1, 2, 3, 4, 5], rtol=0, atol=1e-10)


@pytest.mark.gpu
@pytest.mark.parametrize("fused,n_con,nnz_row", [(1, 7, 200), (0, 7, 200), (1, 700, 30), (0, 3, 100000)])
def test_gpu_constraints_parity(fused, n_con, nnz_row):
    import torch
    from paper_2212_11675_b200 import binding as g
    cfg = inputs.scaled(inputs.named_config("cfg1"), 10, "cfg1/10")
    star, att, instr, vals = inputs.gen_all(cfg)
    from oracle import gsr_oracle
    o = gsr_oracle.from_torch(cfg, star, att, instr, vals)
    C, ptr, col, val = _constraints(o.n, n_con, nnz_row, 9)     # few / many (> grid) / dense rows
    o.set_constraints(ptr, col, val)
    A = g.GsrMatrix.create(cfg, star.cuda(), att.cuda(), instr.cuda(), vals.cuda())
    try:
        g.gsr_matrix_set_constraints(A.h, n_con, ptr, torch.from_numpy(col).cuda(), val)    # host and device arrays
        rng = np.random.default_rng(2)
        x, y = rng.standard_normal(o.n), rng.standard_normal(o.m_total)
        y0, x0 = rng.standard_normal(o.m_total), rng.standard_normal(o.n)
        yd, xd = torch.from_numpy(y0).cuda(), torch.from_numpy(x0).cuda()
        g.gsr_aprod1(A.h, torch.from_numpy(x).cuda(), yd)
        g.gsr_aprod2(A.h, torch.from_numpy(y).cuda(), xd)
        yr, s1 = o.aprod1(x, y0, want_scale=True)
        xr, s2 = o.aprod2(y, x0, want_scale=True)
        assert np.all(np.abs(yd.cpu().numpy() - yr) <= 1e-12 * s1)
        assert np.all(np.abs(xd.cpu().numpy() - xr) <= 1e-12 * s2)
        b = o.aprod1(inputs.x_true(cfg).numpy(), 1e-3 * rng.standard_normal(o.m_total))
        p_ref = o.precondition()
        p = torch.empty(o.n, dtype=torch.float64, device="cuda")
        g.gsr_precondition(A.h, p)
        assert np.allclose(p.cpu().numpy(), p_ref, rtol=1e-13)
        g.gsr_set_option(A.h, g.GSR_OPT_FUSED, fused)
        g.gsr_set_option(A.h, g.GSR_OPT_FORCE_ITNLIM, 1)
        xs = torch.empty(o.n, dtype=torch.float64, device="cuda")
        for k in (1, 8):
            r = g.gsr_lsqr_solve(A.h, torch.from_numpy(b).cuda(), xs, k)
            ro = o.lsqr(b, k, force_itnlim=True, want_se=True)
            assert (r.istop, r.itn) == (ro.istop, ro.itn) == (7, k)
            assert np.linalg.norm(xs.cpu().numpy() - ro.x) <= 1e-9 * np.linalg.norm(ro.x)
            assert abs(r.rnorm - ro.rnorm) <= 1e-9 * ro.rnorm and abs(r.bnorm - ro.bnorm) <= 1e-12 * ro.bnorm
            se = np.empty(o.n)
            g.gsr_lsqr_standard_errors(A.h, se)
            assert np.linalg.norm(se - ro.se) <= 1e-8 * np.linalg.norm(ro.se)
        g.gsr_set_option(A.h, g.GSR_OPT_FORCE_ITNLIM, 0)
        r = g.gsr_lsqr_solve(A.h, b, xs, 500, 1e-10, 1e-10, 1e8)          # host b
        ro = o.lsqr(b, 500, 1e-10, 1e-10, 1e8)
        assert r.istop == ro.istop and abs(r.itn - ro.itn) <= 1
        assert np.linalg.norm(xs.cpu().numpy() - ro.x) <= 1e-9 * np.linalg.norm(ro.x)
    finally:
        A.close()


@pytest.mark.gpu
def test_gpu_constraints_on_a_row_shard_world_1_nccl():
    """Rows e + f3 together: constraint rows on a handle that carries a communicator (one rank:
    the all-reduces are the identity, the sharded kernel sequence with the constraint launches
    inside the graph is what runs).  The N > 1 algebra is tests/test_sharding_gloo.py's."""
    import torch
    from paper_2212_11675_b200 import binding as g
    cfg = inputs.scaled(inputs.named_config("cfg1"), 10, "cfg1/10")
    star, att, instr, vals = inputs.gen_all(cfg)
    from oracle import gsr_oracle
    o = gsr_oracle.from_torch(cfg, star, att, instr, vals)
    n_con = 9
    C, ptr, col, val = _constraints(o.n, n_con, 60, 5)
    o.set_constraints(ptr, col, val)
    A = g.GsrMatrix.create(cfg, star.cuda(), att.cuda(), instr.cuda(), vals.cuda())
    try:
        comm = g.gsr_comm_create(0, 1, g.gsr_comm_unique_id())
        g.gsr_matrix_set_comm(A.h, comm, cfg.n_rows + n_con, cfg.n_cols)
        g.gsr_matrix_set_constraints(A.h, n_con, ptr, col, val)       # after set_comm: both orders are legal
        rng = np.random.default_rng(3)
        b = o.aprod1(inputs.x_true(cfg).numpy(), 1e-3 * rng.standard_normal(o.m_total))
        p_ref = o.precondition()
        p = torch.empty(o.n, dtype=torch.float64, device="cuda")
        g.gsr_precondition(A.h, p)
        assert np.allclose(p.cpu().numpy(), p_ref, rtol=1e-13)
        g.gsr_set_option(A.h, g.GSR_OPT_FORCE_ITNLIM, 1)
        xs = torch.empty(o.n, dtype=torch.float64, device="cuda")
        for k in (1, 10):
            r = g.gsr_lsqr_solve(A.h, torch.from_numpy(b).cuda(), xs, k)
            ro = o.lsqr(b, k, force_itnlim=True, want_se=True)
            assert (r.istop, r.itn) == (ro.istop, ro.itn) == (7, k)
            assert np.linalg.norm(xs.cpu().numpy() - ro.x) <= 1e-9 * np.linalg.norm(ro.x)
            assert abs(r.rnorm - ro.rnorm) <= 1e-9 * ro.rnorm and abs(r.bnorm - ro.bnorm) <= 1e-12 * ro.bnorm
            se = np.empty(o.n)
            g.gsr_lsqr_standard_errors(A.h, se)
            assert np.linalg.norm(se - ro.se) <= 1e-8 * np.linalg.norm(ro.se)
    finally:
        A.close()


@pytest.mark.gpu
def test_gpu_constraints_argument_errors():
    import torch
    from paper_2212_11675_b200 import binding as g
    cfg = inputs.micro_config("c", 3, (20, 20), 8, 4)
    star, att, instr, vals = inputs.gen_all(cfg)
    A = g.GsrMatrix.create(cfg, star.cuda(), att.cuda(), instr.cuda(), vals.cuda())
    try:
        n = cfg.n_cols
        with pytest.raises(g.GsrError) as ei:                  # column out of range
            g.gsr_matrix_set_constraints(A.h, 1, np.array([0, 1], dtype=np.int64), np.array([n], dtype=np.int32), np.ones(1))
        assert ei.value.code == g.GSR_EINVAL
        with pytest.raises(g.GsrError) as ei:                  # row_ptr decreasing
            g.gsr_matrix_set_constraints(A.h, 2, np.array([0, 2, 1], dtype=np.int64), np.zeros(2, dtype=np.int32), np.ones(2))
        assert ei.value.code == g.GSR_EINVAL
        g.gsr_matrix_set_constraints(A.h, 1, np.array([0, 1], dtype=np.int64), np.array([0], dtype=np.int32), np.ones(1))
        g.gsr_matrix_set_constraints(A.h, 0, None, None, None)             # removes them
        g.gsr_precondition(A.h)
        with pytest.raises(g.GsrError) as ei:                  # too late
            g.gsr_matrix_set_constraints(A.h, 1, np.array([0, 1], dtype=np.int64), np.array([0], dtype=np.int32), np.ones(1))
        assert ei.value.code == g.GSR_ESTATE
    finally:
        A.close()
