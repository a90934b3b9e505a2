"""Pins for the oracle's LSQR (CPU only): dense least squares, normal equations, the Krylov
minimiser at a fixed iteration count, consistent-system recovery, the block-diagonal special
case (per-star 5x5 solves), LSQR's own norm estimates, scaling invariances, stop rules 0/3/7
and scipy.sparse.linalg.lsqr used as a black box."""
import numpy as np
import pytest
import scipy.sparse.linalg as spla

from paper_2212_11675_b200 import inputs
from tests.helpers import csr_from_raw, make_oracle, small_system


def _sys(seed=7, **kw):
    cfg, star, att, instr, vals = small_system(seed=seed, **kw)
    o = make_oracle(cfg, star, att, instr, vals)
    A, _ = csr_from_raw(cfg, star, att, instr, vals)
    return cfg, o, A


def _rhs(A, seed, sigma=1e-3):
    rng = np.random.default_rng(seed)
    xt = rng.standard_normal(A.shape[1])
    return xt, A @ xt + sigma * rng.standard_normal(A.shape[0])


def test_matches_dense_lstsq_and_normal_equations():
    cfg, o, A = _sys()
    _, b = _rhs(A, 1)
    r = o.lsqr(b, 500, 1e-14, 1e-14, 1e12)
    Ad = A.toarray()
    x_ls = np.linalg.lstsq(Ad, b, rcond=None)[0]
    x_ne = np.linalg.solve(Ad.T @ Ad, Ad.T @ b)
    assert r.istop in (1, 2, 4, 5)
    assert np.linalg.norm(r.x - x_ls) <= 1e-10 * np.linalg.norm(x_ls)
    assert np.linalg.norm(r.x - x_ne) <= 1e-9 * np.linalg.norm(x_ne)


def test_preconditioned_solve_matches_lstsq_after_unscaling():
    """PC-LSQR: solve on A diag(p), return p (.) z."""
    cfg, o, A = _sys(seed=9)
    _, b = _rhs(A, 2)
    o.precondition()
    r = o.lsqr(b, 500, 1e-14, 1e-14, 1e12)
    x_ls = np.linalg.lstsq(A.toarray(), b, rcond=None)[0]
    assert np.linalg.norm(r.x - x_ls) <= 1e-10 * np.linalg.norm(x_ls)


def test_consistent_system_recovers_x_true():
    cfg, o, A = _sys(seed=3)
    xt, b = _rhs(A, 3, sigma=0.0)
    r = o.lsqr(b, 500, 1e-14, 1e-14, 1e12)
    assert r.istop in (1, 4)
    assert r.rnorm <= 1e-12 * r.bnorm
    assert np.linalg.norm(r.x - xt) <= 1e-10 * np.linalg.norm(xt)


@pytest.mark.parametrize("k", [1, 2, 3, 4, 5, 6])
def test_iterate_k_is_the_krylov_minimiser(k):
    """In exact arithmetic x_k minimises ||b - A x|| over span{A^T b, (A^T A) A^T b, ...}."""
    cfg, o, A = _sys(seed=5)
    _, b = _rhs(A, 4, sigma=0.1)
    Ad = A.toarray()
    K = np.empty((Ad.shape[1], k))
    v = Ad.T @ b
    for j in range(k):
        K[:, j] = v / np.linalg.norm(v)
        v = Ad.T @ (Ad @ K[:, j])
    Q, _ = np.linalg.qr(K)
    c = np.linalg.lstsq(Ad @ Q, b, rcond=None)[0]
    xk = Q @ c
    r = o.lsqr(b, k, force_itnlim=True)
    assert r.istop == 7 and r.itn == k
    assert np.linalg.norm(r.x - xk) <= 1e-8 * np.linalg.norm(xk)


def test_finite_termination_small_n():
    """n = 5*1+3*4+2+1 = 20 columns: LSQR terminates in at most n steps (exact arithmetic)."""
    cfg, o, A = _sys(seed=6, counts=(60,), n_dfa=4, n_instr=2)
    _, b = _rhs(A, 5, sigma=0.05)
    r = o.lsqr(b, 200, 1e-13, 1e-13, 1e12)
    rank = np.linalg.matrix_rank(A.toarray())
    assert r.itn <= rank + 2
    x_ls = np.linalg.lstsq(A.toarray(), b, rcond=None)[0]   # minimum norm
    assert np.linalg.norm(r.x - x_ls) <= 1e-9 * np.linalg.norm(x_ls)


def test_own_estimates_against_direct_norms():
    cfg, o, A = _sys(seed=8)
    _, b = _rhs(A, 6, sigma=0.05)
    fro = np.sqrt((A.toarray() ** 2).sum())
    prev = None
    for k in (1, 2, 4, 8, 16, 32):
        r = o.lsqr(b, k, force_itnlim=True, want_hist=True)
        res = b - A @ r.x
        assert abs(r.rnorm - np.linalg.norm(res)) <= 1e-8 * np.linalg.norm(res)
        assert abs(r.arnorm - np.linalg.norm(A.T @ res)) <= 1e-7 * r.anorm * r.rnorm + 1e-12
        assert abs(r.xnorm - np.linalg.norm(r.x)) <= 1e-8 * np.linalg.norm(r.x)
        assert r.anorm <= fro * (1 + 1e-12)
        h = r.hist
        assert (np.diff(h[:, 0]) <= 1e-12 * h[0, 0]).all()   # rnorm non-increasing
        assert (np.diff(h[:, 2]) >= 0).all()                 # anorm non-decreasing
        assert (np.diff(h[:, 4]) >= -1e-12).all()            # xnorm non-decreasing
        if prev is not None:
            assert np.allclose(h[:len(prev)], prev, rtol=1e-12, atol=0)   # deterministic prefix
        prev = h


def test_block_diagonal_special_case_is_per_star_5x5():
    """With attitude/instrumental/global coefficients zero, A is block diagonal by star."""
    cfg, star, att, instr, vals = small_system(seed=12, counts=(15, 30, 7, 22))
    vals = vals.copy(); vals[:, 5:] = 0.0
    o = make_oracle(cfg, star, att, instr, vals)
    rng = np.random.default_rng(7)
    b = rng.standard_normal(o.m)
    r = o.lsqr(b, 300, 1e-14, 1e-14, 1e12)
    for s in range(cfg.n_stars):
        rows = star == s
        As, bs = vals[rows, :5], b[rows]
        xs = np.linalg.solve(As.T @ As, As.T @ bs)
        assert np.linalg.norm(r.x[5 * s:5 * s + 5] - xs) <= 1e-10 * np.linalg.norm(xs)
    assert np.all(r.x[5 * cfg.n_stars:] == 0.0)    # untouched columns stay exactly zero (A16)


def test_scaling_invariance_and_empty_columns():
    cfg, star, att, instr, vals = small_system(seed=13, counts=(25, 0, 25, 40, 0, 30))
    o = make_oracle(cfg, star, att, instr, vals)
    A, _ = csr_from_raw(cfg, star, att, instr, vals)
    _, b = _rhs(A, 8)
    r1 = o.lsqr(b, 400, 1e-13, 1e-13, 1e12)
    r2 = o.lsqr(8.0 * b, 400, 1e-13, 1e-13, 1e12)       # power of two: exact scaling
    assert r1.itn == r2.itn and r1.istop == r2.istop
    assert np.array_equal(8.0 * r1.x, r2.x)
    for s in (1, 4):
        assert np.all(r1.x[5 * s:5 * s + 5] == 0.0)
    x_ls = np.linalg.lstsq(A.toarray(), b, rcond=None)[0]
    assert np.linalg.norm(r1.x - x_ls) <= 1e-9 * np.linalg.norm(x_ls)


def test_stop_rules_0_3_7():
    cfg, o, A = _sys(seed=14)
    r = o.lsqr(np.zeros(o.m), 10, 1e-8, 1e-8, 1e8)
    assert (r.istop, r.itn) == (0, 0) and np.all(r.x == 0)
    # b orthogonal to range(A): A^T b = 0 up to rounding -> solution x = 0
    Ad = A.toarray()
    Q, _ = np.linalg.qr(Ad, mode="complete")
    b = Q[:, -1]
    r = o.lsqr(b, 10, 1e-8, 1e-8, 1e8)
    assert r.istop in (0, 2) and np.linalg.norm(r.x) <= 1e-12
    _, b = _rhs(A, 9)
    r = o.lsqr(b, 50, 0.0, 0.0, 0.5)              # conlim below 1: rule 3 at iteration 1
    assert (r.istop, r.itn) == (3, 1)
    # closed form: after one step anorm^2 = alpha1^2 + beta2^2 = rho1^2 and ||w1|| = 1, so acond = 1
    assert abs(r.acond - 1.0) <= 1e-14
    r = o.lsqr(b, 50, 0.0, 0.0, 1.5)              # first iteration with acond >= 1.5
    assert r.istop == 3 and r.itn >= 2 and r.acond >= 1.5
    r = o.lsqr(b, 3, 0.0, 0.0, 0.0)
    assert (r.istop, r.itn) == (7, 3)
    # forced mode records when a natural rule would have fired
    rs = o.lsqr(b, 500, 1e-10, 1e-10, 1e8)
    rf = o.lsqr(b, rs.itn + 5, 1e-10, 1e-10, 1e8, force_itnlim=True)
    assert rf.istop == 7 and rf.itn == rs.itn + 5
    assert (rf.istop_natural, rf.itn_natural) == (rs.istop, rs.itn)


@pytest.mark.parametrize("precond", [False, True])
def test_scipy_lsqr_black_box(precond):
    """Independent implementation of the same published algorithm (black-box use)."""
    cfg = inputs.scaled(inputs.named_config("cfg1"), 10, "cfg1/10")   # 20k rows, 1361 cols
    s, a, i, v = inputs.gen_all(cfg)
    o = make_oracle(cfg, s.numpy(), a.numpy(), i.numpy(), v.numpy())
    A, _ = csr_from_raw(cfg, s.numpy(), a.numpy(), i.numpy(), v.numpy())
    xt = inputs.x_true(cfg).numpy()
    b = A @ xt + inputs.noise(cfg, 0, cfg.n_rows).numpy()
    if precond:
        p = o.precondition()
        A = A @ __import__("scipy.sparse").sparse.diags(p)
    ref = spla.lsqr(A, b, damp=0.0, atol=1e-10, btol=1e-10, conlim=1e8, iter_lim=500)
    x_ref, istop, itn, r1norm, _, anorm, acond, arnorm, xnorm = ref[:9]
    if precond:
        x_ref = p * x_ref
    r = o.lsqr(b, 500, 1e-10, 1e-10, 1e8)
    assert r.istop == istop and abs(r.itn - itn) <= 1
    assert np.linalg.norm(r.x - x_ref) <= 1e-9 * np.linalg.norm(x_ref)
    if r.itn == itn:
        # The Lanczos coefficients alpha_k, beta_k (hence anorm, acond) are not forward stable
        # once Ritz values converge: two correct implementations drift apart by ~1e-7 while x
        # and rnorm agree (reading A18).
        assert abs(r.rnorm - r1norm) <= 1e-8 * r1norm
        assert abs(r.anorm - anorm) <= 1e-5 * anorm
        assert abs(r.acond - acond) <= 1e-5 * acond
        assert abs(r.arnorm - arnorm) <= 1e-6 * arnorm + 1e-12 * anorm * r1norm
    # fixed-count mode against scipy with an unreachable tolerance
    # Without column scaling the global column (norm ~141 vs ~10) gives an outlier singular
    # value; once its Ritz value converges (k ~ 8) orthogonality is lost and two correct
    # implementations may differ by one "ghost" step until both converge (measured: 1e-2 at
    # k = 12, back to 1e-9 at k = 16).  Compare before that point (reading A20).
    k = 12 if precond else 4
    ref = spla.lsqr(A, b, damp=0.0, atol=0.0, btol=0.0, conlim=0.0, iter_lim=k)
    xk = p * ref[0] if precond else ref[0]
    rk = o.lsqr(b, k, force_itnlim=True)
    assert ref[2] == k and rk.itn == k and rk.istop == 7 and ref[1] == 7
    assert np.linalg.norm(rk.x - xk) <= 1e-10 * np.linalg.norm(xk)


# ---- row f1: variances / standard errors (Paige & Saunders; Algorithm 3 line 17)

def _krylov_basis(A, b, k):
    """Orthonormal basis of span{A^T b, (A^T A) A^T b, ...} by dense Gram-Schmidt (twice)."""
    n = A.shape[1]
    Q = np.zeros((n, k))
    v = A.T @ b
    for i in range(k):
        for _ in range(2):
            v = v - Q[:, :i] @ (Q[:, :i].T @ v)
        v = v / np.linalg.norm(v)
        Q[:, i] = v
        v = A.T @ (A @ v)
    return Q


@pytest.mark.parametrize("k", [1, 2, 3, 5, 8, 10])
def test_variance_is_diag_of_projected_inverse_normal_matrix(k):
    """After k steps LSQR's var_j = sum (w_j/rho)^2 equals diag(Q (Q^T A^T A Q)^-1 Q^T) with Q an
    orthonormal basis of the k-th Krylov space (D_k D_k^T = V_k (B_k^T B_k)^-1 V_k^T): a dense,
    independent computation.  The standard error follows with the residual computed directly."""
    cfg, star, att, instr, vals = small_system()
    o = make_oracle(cfg, star, att, instr, vals)
    A = csr_from_raw(cfg, star, att, instr, vals)[0].toarray()
    b = np.random.default_rng(5).standard_normal(o.m)
    r = o.lsqr(b, k, force_itnlim=True, want_se=True)
    Q = _krylov_basis(A, b, k)
    T = Q.T @ (A.T @ (A @ Q))
    var_ref = np.einsum("ij,jk,ik->i", Q, np.linalg.inv(T), Q)
    assert np.max(np.abs(r.var - var_ref)) <= 1e-11 * np.max(var_ref)
    res = np.linalg.norm(b - A @ r.x)
    se_ref = res * np.sqrt(var_ref / (o.m - o.n))
    assert np.allclose(r.se, se_ref, rtol=1e-9, atol=1e-12 * se_ref.max())


def test_variance_monotone_and_scaled_by_p():
    """var never decreases with k; with column scaling se is multiplied by p like the solution
    (PAPER.md:43): se(x) = p * rnorm * sqrt(var_z/dof)."""
    cfg, star, att, instr, vals = small_system()
    o = make_oracle(cfg, star, att, instr, vals)
    b = np.random.default_rng(6).standard_normal(o.m)
    prev = np.zeros(o.n)
    for k in (1, 3, 6, 12):
        r = o.lsqr(b, k, force_itnlim=True, want_se=True)
        assert np.all(r.var >= prev)
        prev = r.var
    p = o.precondition()
    r = o.lsqr(b, 6, force_itnlim=True, want_se=True)
    assert np.allclose(r.se, p * r.rnorm * np.sqrt(r.var / (o.m - o.n)), rtol=1e-14)
    # and the projected-inverse identity holds for the scaled matrix too
    A = csr_from_raw(cfg, star, att, instr, vals)[0].toarray() * p[None, :]
    Q = _krylov_basis(A, b, 6)
    var_ref = np.einsum("ij,jk,ik->i", Q, np.linalg.inv(Q.T @ (A.T @ (A @ Q))), Q)
    assert np.max(np.abs(r.var - var_ref)) <= 1e-11 * np.max(var_ref)


def test_standard_errors_of_an_underdetermined_system_use_one_degree_of_freedom():
    """m <= n: there are no residual degrees of freedom, and Paige & Saunders then divide by 1
    (the `dof = 1` branch of orc_standard_errors): se_j = rnorm * sqrt(var_j), with var from the
    dense projected inverse normal matrix as above."""
    cfg, star, att, instr, vals = small_system(seed=9, counts=(3, 2, 4), n_dfa=6, n_instr=8)
    o = make_oracle(cfg, star, att, instr, vals)
    assert o.m == 9 and o.m < o.n
    A = csr_from_raw(cfg, star, att, instr, vals)[0].toarray()
    b = np.random.default_rng(8).standard_normal(o.m)
    k = 4
    r = o.lsqr(b, k, force_itnlim=True, want_se=True)
    Q = _krylov_basis(A, b, k)
    var_ref = np.einsum("ij,jk,ik->i", Q, np.linalg.inv(Q.T @ (A.T @ (A @ Q))), Q)
    res = np.linalg.norm(b - A @ r.x)
    assert np.allclose(r.se, res * np.sqrt(var_ref / 1.0), rtol=1e-9, atol=1e-12 * r.se.max())


# ---- row f4: damping (Paige & Saunders' damp; the paper's solver is undamped)

@pytest.mark.parametrize("damp", [0.3, 2.5])
def test_damped_lsqr_solves_the_augmented_problem(damp):
    """min ||[A; damp I] x - [b; 0]||: dense lstsq on the augmented matrix; rnorm is the norm of
    the augmented residual, computed directly."""
    cfg, star, att, instr, vals = small_system()
    o = make_oracle(cfg, star, att, instr, vals)
    A = csr_from_raw(cfg, star, att, instr, vals)[0].toarray()
    b = np.random.default_rng(8).standard_normal(o.m)
    r = o.lsqr(b, 2000, 1e-15, 1e-15, 1e12, damp=damp)
    aug = np.vstack([A, damp * np.eye(o.n)])
    xl = np.linalg.lstsq(aug, np.concatenate([b, np.zeros(o.n)]), rcond=None)[0]
    assert np.linalg.norm(r.x - xl) <= 1e-11 * np.linalg.norm(xl)
    direct = np.sqrt(np.linalg.norm(b - A @ r.x) ** 2 + damp ** 2 * np.linalg.norm(r.x) ** 2)
    assert abs(r.rnorm - direct) <= 1e-11 * direct
    r0 = o.lsqr(b, 2000, 1e-15, 1e-15, 1e12)
    assert np.linalg.norm(r.x) < np.linalg.norm(r0.x)          # damping shrinks the solution


@pytest.mark.parametrize("damp", [0.3, 2.5])
@pytest.mark.parametrize("precond", [False, True])
def test_damped_scipy_black_box(damp, precond):
    """anorm, acond, xnorm, istop and itn under damping (the line anorm = hyp(anorm, damp), the
    extra rotation, rnorm with the damping rows' share) against scipy.sparse.linalg.lsqr(damp=...)
    used as a black box: an independent implementation of the same published algorithm."""
    cfg = inputs.scaled(inputs.named_config("cfg1"), 10, "cfg1/10")
    s, a, i, v = inputs.gen_all(cfg)
    o = make_oracle(cfg, s.numpy(), a.numpy(), i.numpy(), v.numpy())
    A, _ = csr_from_raw(cfg, s.numpy(), a.numpy(), i.numpy(), v.numpy())
    b = A @ inputs.x_true(cfg).numpy() + inputs.noise(cfg, 0, cfg.n_rows).numpy()
    p = None
    if precond:
        p = o.precondition()
        A = A @ __import__("scipy.sparse").sparse.diags(p)
    # fixed count, before any Ritz value has converged (reading A18): everything to 1e-10
    k = 6
    ref = spla.lsqr(A, b, damp=damp, atol=0.0, btol=0.0, conlim=0.0, iter_lim=k)
    xk, istop, itn, r1norm, r2norm, anorm, acond, arnorm, xnorm = ref[:9]
    r = o.lsqr(b, k, damp=damp, force_itnlim=True)
    assert (r.istop, r.itn) == (7, k) and (istop, itn) == (7, k)
    xs = p * xk if precond else xk
    assert np.linalg.norm(r.x - xs) <= 1e-10 * np.linalg.norm(xs)
    assert abs(r.rnorm - r2norm) <= 1e-10 * r2norm          # residual of the augmented system
    assert abs(r.anorm - anorm) <= 1e-10 * anorm
    assert abs(r.acond - acond) <= 1e-10 * acond
    assert abs(r.xnorm - xnorm) <= 1e-10 * xnorm
    assert abs(r.arnorm - arnorm) <= 1e-9 * arnorm
    # natural stop: same rule, same iteration (+-1), estimates at the level reading A18 allows
    ref = spla.lsqr(A, b, damp=damp, atol=1e-10, btol=1e-10, conlim=1e8, iter_lim=500)
    r = o.lsqr(b, 500, 1e-10, 1e-10, 1e8, damp=damp)
    assert r.istop == ref[1] and abs(r.itn - ref[2]) <= 1
    xs = p * ref[0] if precond else ref[0]
    assert np.linalg.norm(r.x - xs) <= 1e-9 * np.linalg.norm(xs)
    if r.itn == ref[2]:
        assert abs(r.rnorm - ref[4]) <= 1e-8 * ref[4]
        assert abs(r.anorm - ref[5]) <= 1e-5 * ref[5]
        assert abs(r.acond - ref[6]) <= 1e-5 * ref[6]
        assert abs(r.xnorm - ref[8]) <= 1e-8 * ref[8]


def test_stop_rules_4_and_5_are_told_apart():
    """atol = btol = conlim = 0 leaves only the machine-precision rules.  A consistent system
    drives rnorm to rounding level, so 1 + test1/(1 + anorm xnorm/bnorm) <= 1 fires (rule 4, which
    wins over 5); with noise in b the residual stays O(1) and only test2 = ||A^T r||/(||A|| ||r||)
    can reach rounding level (rule 5).  scipy's lsqr, as a black box, names the same rule."""
    cfg, o, A = _sys(seed=7)
    rng = np.random.default_rng(1)
    xt = rng.standard_normal(A.shape[1])
    for noise, rule in ((0.0, 4), (1e-3, 5)):
        b = A @ xt + noise * rng.standard_normal(A.shape[0])
        r = o.lsqr(b, 400, 0.0, 0.0, 0.0)
        ref = spla.lsqr(A, b, atol=0.0, btol=0.0, conlim=0.0, iter_lim=400)
        assert r.istop == rule == ref[1]
        assert abs(r.itn - ref[2]) <= 2          # rounding-level quantities decide the exact step
        assert r.itn < 400


def test_stop_rule_6_is_shadowed_and_test3_underflow_gives_rule_3():
    """Rule 6 (1 + 1/acond <= 1) is evaluated first and loses to every later rule.  With a finite
    acond >= 1/eps the iterate has resolved a singular value below eps ||A||, and then either the
    residual is at rounding level (rule 4) or A^T r is (rule 5); the one reachable state in which
    test3 itself decides is acond = inf: rho^2 underflows to 0 on a matrix scaled by 1e-160,
    ddnorm = ||w||^2 / 0 = inf, test3 = 0 <= ctol = 0, which is rule 3 -- at iteration 1, in the
    oracle and in scipy alike.  (reading A25.)"""
    cfg, star, att, instr, vals = small_system(seed=7)
    o = make_oracle(cfg, star, att, instr, vals * 1e-160)
    A, _ = csr_from_raw(cfg, star, att, instr, vals * 1e-160)
    b = np.random.default_rng(1).standard_normal(A.shape[0])
    r = o.lsqr(b, 50, 0.0, 0.0, 0.0)
    with np.errstate(all="ignore"):
        import warnings
        with warnings.catch_warnings():
            warnings.simplefilter("ignore")
            ref = spla.lsqr(A, b, atol=0.0, btol=0.0, conlim=0.0, iter_lim=50)
    assert (r.istop, r.itn) == (3, 1) == (ref[1], ref[2])
    assert np.isinf(r.acond) and np.isinf(ref[6])
    # in forced mode the same state is recorded as the natural stop and the loop goes on
    rf = o.lsqr(b, 3, 0.0, 0.0, 0.0, force_itnlim=True)
    assert (rf.istop, rf.itn, rf.istop_natural, rf.itn_natural) == (7, 3, 3, 1)
