"""GPU parity tests: the CUDA path (through the C ABI binding) against the CPU oracle on the
same seeded inputs.  Bars: index construction bit-exact; aprod
outputs within 1e-12 of the component-wise scale (reading A13); LSQR x within 1e-9 relative
2-norm after a fixed iteration count, identical istop."""
import numpy as np
import pytest
import torch

from paper_2212_11675_b200 import inputs
from tests.helpers import make_oracle

pytestmark = pytest.mark.gpu

APROD_TOL = 1e-12
X_TOL = 1e-9
X_TOL_CAP = 1e-4      # upper bound of the sensitivity-relaxed tolerance (reading A20): 20 x the
                      # oracle's own one-ulp sensitivity, whose maximum over all cases is 1.6e-6
                      # (skew_hot, k = 60: measured 4e-16 at k = 20, 5e-12 at 40, 1e-8 at 50,
                      # 1.6e-6 at 60, 5e-11 at 70, 2e-15 at 200)
SENS_LOG = []         # (case, fused, k, one-ulp sensitivity of the oracle's x): written to
                      # gpurun_out/lsqr_sensitivity.json at the end of the module (A20)


def _binding():
    from paper_2212_11675_b200 import binding
    return binding


def _cases():
    mc = inputs.micro_config
    return {
        "cfg1": inputs.named_config("cfg1"),
        "one_row": mc("one_row", 21, [1], 4, 1),
        "one_star_many_tiles": mc("one_star", 22, [1000], 9, 7),
        "single_obs_stars": mc("single_obs", 23, [1] * 300 + [0] * 5 + [2] * 17, 12, 6),
        "ragged_empty_stars": mc("ragged", 24, [0, 37, 1, 250, 0, 64, 3, 0, 700, 0], 40, 17),
        "one_instr_col": mc("one_instr", 25, [130, 129, 300], 16, 1),
        "skew_hot": inputs.GsrConfig("cfg4s", 3, 400, 400, 60, n_rows_total=50_000,
                                     powerlaw=(10, 10_000, 1.36), att_hot=(0.9, 0.40, 0.45),
                                     col_scales=True),
    }


CASES = _cases()
# fixed iteration counts compared per case; STABLE ones must meet the plain 1e-9 bar
FIXED_COUNTS = {"cfg1": (1, 3, 200), "ragged_empty_stars": (1, 3, 60), "one_instr_col": (1, 3, 60),
                "skew_hot": (1, 3, 20, 60, 200, 400)}
STABLE_COUNTS = {"cfg1": (1, 3, 200), "ragged_empty_stars": (1, 3, 60), "one_instr_col": (1, 3, 60),
                 "skew_hot": (1, 3, 20, 200, 400)}


class Sys:
    def __init__(self, cfg, edge_att=False):
        self.cfg = cfg
        star, att, instr, vals = inputs.gen_all(cfg)
        if edge_att and cfg.n_rows >= 2:      # attitude start at both ends of the range
            att[0] = 0
            att[-1] = cfg.n_dfa - 4
        self.host = (star, att, instr, vals)
        self.o = make_oracle(cfg, star.numpy(), att.numpy(), instr.numpy(), vals.numpy())
        b = _binding()
        dev = [t.cuda() for t in self.host]
        self.A = b.GsrMatrix.create(cfg, *dev)
        self.m, self.n = cfg.n_rows, cfg.n_cols


@pytest.fixture(scope="module", params=list(CASES))
def sysm(request):
    s = Sys(CASES[request.param], edge_att=True)
    yield s
    s.A.close()


def test_index_construction_bit_exact(sysm):
    b = _binding()
    cols, vals = b.gsr_debug_expand_rows(sysm.A.h, 0, sysm.m)
    oc, ov = sysm.o.expand_rows()
    assert np.array_equal(cols, oc)
    assert np.array_equal(vals, ov)
    d, n = b.gsr_matrix_dims(sysm.A.h)
    assert (d.n_rows, n) == (sysm.m, sysm.n)


def test_aprod1_parity(sysm):
    b = _binding()
    x = inputs.random_vector(sysm.cfg, 1, sysm.n)
    y0 = inputs.random_vector(sysm.cfg, 2, sysm.m)
    y_ref, scale = sysm.o.aprod1(x.numpy(), y0.numpy(), want_scale=True)
    yd = y0.cuda()
    b.gsr_aprod1(sysm.A.h, x.cuda(), yd)
    err = np.abs(yd.cpu().numpy() - y_ref)
    assert np.all(err <= APROD_TOL * scale), float((err / scale).max())


@pytest.mark.parametrize("split", [1, 0, -1])
def test_aprod2_parity(sysm, split):
    """Algorithm 2 through the C ABI: as two launches (GSR_OPT_APROD2_SPLIT = 1:
    the instrumental block in a pass of its own), as one sweep over all four blocks (0), and in
    the default setting (-1 = the split)."""
    b = _binding()
    y = inputs.random_vector(sysm.cfg, 3, sysm.m)
    x0 = inputs.random_vector(sysm.cfg, 4, sysm.n)
    x_ref, scale = sysm.o.aprod2(y.numpy(), x0.numpy(), want_scale=True)
    xd = x0.cuda()
    b.gsr_set_option(sysm.A.h, b.GSR_OPT_APROD2_SPLIT, split)
    try:
        n0 = b.gsr_launch_count()
        b.gsr_aprod2(sysm.A.h, y.cuda(), xd)
        launches = b.gsr_launch_count() - n0
    finally:
        b.gsr_set_option(sysm.A.h, b.GSR_OPT_APROD2_SPLIT, -1)
    two = split != 0                                                  # -1 (default) = the split
    assert launches == (2 if two else 1) or sysm.m == 0, launches     # the form asked for really ran
    err = np.abs(xd.cpu().numpy() - x_ref)
    assert np.all(err <= APROD_TOL * np.maximum(scale, 1e-300)), float((err / scale).max())
    # untouched columns (empty stars, unused instrumental columns) keep x0 exactly
    untouched = scale == np.abs(x0.numpy())
    assert np.array_equal(xd.cpu().numpy()[untouched], x0.numpy()[untouched])


def test_adjoint_identity_on_gpu(sysm):
    b = _binding()
    x = inputs.random_vector(sysm.cfg, 5, sysm.n).cuda()
    y = inputs.random_vector(sysm.cfg, 6, sysm.m).cuda()
    Ax = torch.zeros(sysm.m, dtype=torch.float64, device="cuda")
    ATy = torch.zeros(sysm.n, dtype=torch.float64, device="cuda")
    b.gsr_aprod1(sysm.A.h, x, Ax)
    b.gsr_aprod2(sysm.A.h, y, ATy)
    lhs, rhs = float(Ax @ y), float(x @ ATy)
    assert abs(lhs - rhs) <= 1e-12 * max(float(Ax.norm() * y.norm()), 1e-300)


def _rhs(s):
    xt = inputs.x_true(s.cfg).numpy()
    return s.o.aprod1(xt, inputs.noise(s.cfg, 0, s.m).numpy())


@pytest.mark.parametrize("fused", [1, 0])
@pytest.mark.parametrize("name", ["cfg1", "ragged_empty_stars", "skew_hot", "one_instr_col"])
def test_precondition_and_lsqr_parity(name, fused):
    """Column scaling then fixed-count and standard-mode PC-LSQR, with the fused
    one-pass iteration (GSR_OPT_FUSED = 1, default) and with aprod1 + aprod2 per iteration."""
    b = _binding()
    s = Sys(CASES[name])
    try:
        b.gsr_set_option(s.A.h, b.GSR_OPT_FUSED, fused)
        rhs = _rhs(s)                       # b formed with the oracle's aprod1 on the unscaled A
        p_ref = s.o.precondition()
        p = torch.empty(s.n, dtype=torch.float64, device="cuda")
        b.gsr_precondition(s.A.h, p)
        assert np.allclose(p.cpu().numpy(), p_ref, rtol=1e-13, atol=0)
        with pytest.raises(b.GsrError) as ei:
            b.gsr_precondition(s.A.h, p)
        assert ei.value.code == b.GSR_ESTATE
        _, vals = b.gsr_debug_expand_rows(s.A.h, 0, s.m)
        assert np.allclose(vals, s.o.values, rtol=1e-13, atol=0)
        bd = torch.from_numpy(rhs).cuda()
        x = torch.empty(s.n, dtype=torch.float64, device="cuda")
        # fixed-count mode (reading A9): exactly itnlim iterations, istop 7
        b.gsr_set_option(s.A.h, b.GSR_OPT_FORCE_ITNLIM, 1)
        rng = np.random.default_rng(0)
        rhs_ulp = rhs + np.spacing(rhs) * rng.integers(-1, 2, rhs.shape)
        for k in FIXED_COUNTS[name]:
            r = b.gsr_lsqr_solve(s.A.h, bd, x, k)
            ro = s.o.lsqr(rhs, k, force_itnlim=True, want_se=True)
            assert (r.istop, r.itn) == (ro.istop, ro.itn) == (7, k)
            xg = x.cpu().numpy()
            se = torch.empty(s.n, dtype=torch.float64, device="cuda")
            b.gsr_lsqr_standard_errors(s.A.h, se)      # row f1: p * rnorm * sqrt(var / dof)
            se_host = np.empty(s.n)
            b.gsr_lsqr_standard_errors(s.A.h, se_host)
            assert np.array_equal(se.cpu().numpy(), se_host)
            # Reading A20: at some intermediate k the Lanczos process is unstable (the oracle
            # itself moves by far more than 1e-9 when b changes by one ulp).  The bar is 1e-9
            # wherever the oracle is that stable, else 20x the oracle's own one-ulp sensitivity.
            ru = s.o.lsqr(rhs_ulp, k, force_itnlim=True, want_se=True)
            sens = np.linalg.norm(ru.x - ro.x) / np.linalg.norm(ro.x)
            sens_se = np.linalg.norm(ru.se - ro.se) / np.linalg.norm(ro.se)
            # capped: no assert of this test has an unbounded tolerance (A20 lists the
            # measured sensitivities; the largest, skew_hot k = 60, is far below the cap)
            tol = min(max(X_TOL, 20.0 * sens), X_TOL_CAP)
            SENS_LOG.append((name, fused, k, float(sens)))
            if k in STABLE_COUNTS[name]:
                assert sens < 1e-10 and tol == X_TOL, (name, k, sens)
            assert np.linalg.norm(xg - ro.x) <= tol * np.linalg.norm(ro.x), (name, k, sens)
            # the scaled iterate z = x / p as well (x spans 8 decades at cfg4-like
            # column scales, so the 2-norm of x alone is blind to the small-scale unknowns)
            zg, zo = xg / p_ref, ro.x / p_ref
            assert np.linalg.norm(zg - zo) <= tol * np.linalg.norm(zo), (name, k, sens)
            assert abs(r.rnorm - ro.rnorm) <= tol * ro.rnorm
            # var is a sum of squares of the w vectors.  Before the first natural stop rule fires
            # it is as stable as x; past convergence the Lanczos vectors are rounding noise
            # (reading A18) and the terms (w_j/rho)^2 added from then on are arbitrary on both
            # sides (measured: oracle and GPU differ by O(1) at k = 60 on a system that
            # converged at k = 38), so var is compared only up to convergence.
            converged = ro.itn_natural != 0 and k >= ro.itn_natural
            nz = ro.se > 0
            assert np.all(np.isfinite(se_host)) and np.all(se_host[~nz] == 0.0)
            if not converged:
                # same rule as for x (A20): 20 x the oracle's own one-ulp sensitivity, never above 1e-2.
                # var is a RUNNING sum, so at skew_hot k = 200 it still carries the unstable stage around
                # k = 60: the oracle itself moves by 3.4e-4 there when b changes by one ulp (7.1e-4 at
                # k = 60).  FINDING (round 3): a flat 1e-3 cap does not hold for the kernels in the tree.
                # The order of the floating-point atomics differs from run to run, and three B200 runs of
                # the same library landed 2e-5, < 1e-3 and 1.9e-3 (two-pass form) from the oracle at
                # skew_hot k = 200 -- up to 5.7 x the oracle's own sensitivity, inside the 20 x rule
                # (6.8e-3), outside 1e-3.  The cap stays at 1e-2 and binds only at skew_hot k = 60.
                se_tol = min(max(2 * tol, 20.0 * sens_se), 1e-2)
                assert np.linalg.norm(se_host - ro.se) <= se_tol * np.linalg.norm(ro.se), (name, k, sens_se)
                # element-wise where the oracle's own se is stable too (var is a running sum: at
                # skew_hot k = 200 it still carries the terms of the unstable stage around k = 60)
                if tol == X_TOL and sens_se < 1e-10:
                    assert np.all(np.abs(se_host[nz] - ro.se[nz]) <= 1e-7 * ro.se[nz])
            assert abs(r.xnorm - ro.xnorm) <= tol * ro.xnorm
            assert abs(r.bnorm - ro.bnorm) <= 1e-12 * ro.bnorm
            if tol == X_TOL and (ro.itn_natural == 0 or k < ro.itn_natural):      # reading A18
                # anorm and acond are RUNNING sums over alpha_k, beta_k and ||w_k||/rho_k: like var
                # they keep the terms of an unstable stage the iterate itself has left behind
                # (skew_hot: around k = 60, still in the sums at k = 200), so they get the same rule
                # as x -- 1e-9 where the oracle is that stable under a one-ulp change of b, else
                # 20x its own sensitivity, capped at reading A18's post-convergence bound
                sens_an = abs(ru.anorm - ro.anorm) / ro.anorm
                sens_ac = abs(ru.acond - ro.acond) / ro.acond
                assert abs(r.anorm - ro.anorm) <= min(max(1e-9, 20.0 * sens_an), 1e-2) * ro.anorm, (name, k, sens_an)
                assert abs(r.acond - ro.acond) <= min(max(1e-9, 20.0 * sens_ac), 1e-2) * ro.acond, (name, k, sens_ac)
            else:   # past convergence alpha_k, beta_k are rounding noise: anorm loosely, acond not at all
                assert abs(r.anorm - ro.anorm) <= 1e-2 * ro.anorm
            if ro.itn_natural:
                assert abs(r.itn_natural - ro.itn_natural) <= 1 and r.itn_natural > 0
                assert r.istop_natural == ro.istop_natural, (name, k, r.istop_natural, ro.istop_natural)
            else:
                assert (r.istop_natural, r.itn_natural) == (0, 0)
        # standard mode
        b.gsr_set_option(s.A.h, b.GSR_OPT_FORCE_ITNLIM, 0)
        r = b.gsr_lsqr_solve(s.A.h, bd, x, 500, 1e-10, 1e-10, 1e8)
        ro = s.o.lsqr(rhs, 500, 1e-10, 1e-10, 1e8)
        assert r.istop == ro.istop and abs(r.itn - ro.itn) <= 1
        assert np.linalg.norm(x.cpu().numpy() - ro.x) <= X_TOL * np.linalg.norm(ro.x)
        if r.itn == ro.itn:     # standard errors at the natural stop (row f1)
            ro = s.o.lsqr(rhs, 500, 1e-10, 1e-10, 1e8, want_se=True)
            se_host = np.empty(s.n)
            b.gsr_lsqr_standard_errors(s.A.h, se_host)
            # the last terms before the stop already come from nearly converged Lanczos vectors
            # (measured 4e-4 on ragged_empty_stars): an estimate-level agreement, like anorm
            assert np.linalg.norm(se_host - ro.se) <= 1e-2 * np.linalg.norm(ro.se), name
    finally:
        s.A.close()


def test_stop_rules_3_4_5_against_the_oracle():
    """Device stop rules 3, 4 and 5 (k_scalar_main; Paige & Saunders' tests as listed in DESIGN.md
    C3) against the oracle on the three systems tests/test_oracle_lsqr.py builds for the CPU: a tiny
    conlim (rule 3 at iteration 1, acond = 1 in closed form; then the first iteration with
    acond >= 1.5), a consistent system with atol = btol = conlim = 0 (rule 4) and a noisy one
    (rule 5).  Rules 4 and 5 are decided by rounding-level quantities, so the step may differ by
    two (as against scipy on the CPU); the rule may not.  In fixed-count mode the same rule must
    be recorded as the natural stop."""
    b = _binding()
    s = Sys(inputs.micro_config("tiny", 7, (20,) * 6, 6, 8))
    try:
        rng = np.random.default_rng(1)
        xt = rng.standard_normal(s.n)
        clean = s.o.aprod1(xt, np.zeros(s.m))
        noisy = clean + 1e-3 * rng.standard_normal(s.m)
        x = torch.empty(s.n, dtype=torch.float64, device="cuda")
        for rhs, itnlim, conlim, rule, slack in ((noisy, 50, 0.5, 3, 0), (noisy, 50, 1.5, 3, 0),
                                                 (clean, 400, 0.0, 4, 2), (noisy, 400, 0.0, 5, 2)):
            bd = torch.from_numpy(rhs).cuda()
            ro = s.o.lsqr(rhs, itnlim, 0.0, 0.0, conlim)
            b.gsr_set_option(s.A.h, b.GSR_OPT_FORCE_ITNLIM, 0)
            r = b.gsr_lsqr_solve(s.A.h, bd, x, itnlim, 0.0, 0.0, conlim)
            assert r.istop == ro.istop == rule, (rule, r, ro.istop)
            assert r.istop_natural == ro.istop_natural == rule
            assert abs(r.itn - ro.itn) <= slack and r.itn < itnlim, (rule, r.itn, ro.itn)
            assert r.itn_natural == r.itn
            if rule == 3:
                assert abs(r.acond - ro.acond) <= 1e-9 * ro.acond
            # fixed-count mode: the loop runs on, the rule is recorded
            k = ro.itn + 5
            rf_o = s.o.lsqr(rhs, k, 0.0, 0.0, conlim, force_itnlim=True)
            b.gsr_set_option(s.A.h, b.GSR_OPT_FORCE_ITNLIM, 1)
            rf = b.gsr_lsqr_solve(s.A.h, bd, x, k, 0.0, 0.0, conlim)
            assert (rf.istop, rf.itn) == (rf_o.istop, rf_o.itn) == (7, k)
            assert rf.istop_natural == rf_o.istop_natural == rule
            assert abs(rf.itn_natural - rf_o.itn_natural) <= slack
    finally:
        s.A.close()


@pytest.mark.parametrize("name,counts", [("cfg1", (3, 20)), ("skew_hot", (3, 20)),
                                         ("ragged_empty_stars", (3,)), ("one_instr_col", (3,))])
def test_running_sums_agree_between_the_iteration_forms(name, counts):
    """anorm, acond and var are running sums whose parity bar against the oracle is relaxed where
    the oracle itself is unstable.  This check does not lean on that relaxation: at iteration
    counts where the oracle's one-ulp sensitivity of all three is below 1e-12 (measured on the
    CPU: every case at k <= 3, cfg1 and skew_hot up to k = 20) the three forms of the iteration --
    fused (default), aprod1 + aprod2, and the order-independent sums of GSR_OPT_DETERMINISTIC --
    must agree with each other to 1e-9: a term missed in one form's sums (an alpha, a damp, a
    (w/rho)^2) would show here at full size."""
    b = _binding()
    s = Sys(CASES[name])
    try:
        bd = torch.from_numpy(_rhs(s)).cuda()
        b.gsr_precondition(s.A.h)
        b.gsr_set_option(s.A.h, b.GSR_OPT_FORCE_ITNLIM, 1)
        x = torch.empty(s.n, dtype=torch.float64, device="cuda")
        for k in counts:
            got = {}
            for form, opts in (("fused", ((b.GSR_OPT_FUSED, 1), (b.GSR_OPT_DETERMINISTIC, 0))),
                               ("two-pass", ((b.GSR_OPT_FUSED, 0), (b.GSR_OPT_DETERMINISTIC, 0))),
                               ("deterministic", ((b.GSR_OPT_FUSED, 1), (b.GSR_OPT_DETERMINISTIC, 1)))):
                for key, val in opts:
                    b.gsr_set_option(s.A.h, key, val)
                r = b.gsr_lsqr_solve(s.A.h, bd, x, k)
                se = np.empty(s.n)
                b.gsr_lsqr_standard_errors(s.A.h, se)
                got[form] = (r, se, x.cpu().numpy())
            r0, se0, x0 = got["fused"]
            for form in ("two-pass", "deterministic"):
                r, se, xv = got[form]
                assert (r.istop, r.itn) == (7, k)
                for f in ("anorm", "acond", "rnorm", "xnorm", "arnorm"):
                    a, c = getattr(r, f), getattr(r0, f)
                    assert abs(a - c) <= 1e-9 * abs(c), (name, k, form, f, a, c)
                assert np.linalg.norm(se - se0) <= 1e-9 * np.linalg.norm(se0), (name, k, form)
                assert np.linalg.norm(xv - x0) <= 1e-9 * np.linalg.norm(x0), (name, k, form)
        b.gsr_set_option(s.A.h, b.GSR_OPT_DETERMINISTIC, 0)
        b.gsr_set_option(s.A.h, b.GSR_OPT_FUSED, 1)
    finally:
        s.A.close()


def test_lsqr_unpreconditioned_host_buffers():
    """Host b / x buffers (pageable numpy, pinned torch) go through the same C call."""
    b = _binding()
    cfg = inputs.scaled(inputs.named_config("cfg1"), 10, "cfg1/10")
    s = Sys(cfg)
    try:
        rhs = _rhs(s)
        xh = np.empty(s.n)
        b.gsr_set_option(s.A.h, b.GSR_OPT_FORCE_ITNLIM, 1)
        r = b.gsr_lsqr_solve(s.A.h, rhs, xh, 4)           # numpy host arrays
        ro = s.o.lsqr(rhs, 4, force_itnlim=True)
        assert r.itn == 4 and np.linalg.norm(xh - ro.x) <= 1e-11 * np.linalg.norm(ro.x)
        bp = torch.from_numpy(rhs).pin_memory()
        xp = torch.empty(s.n, dtype=torch.float64).pin_memory()
        b.gsr_lsqr_solve(s.A.h, bp, xp, 4)                # pinned host tensors
        assert np.linalg.norm(xp.numpy() - xh) <= 1e-11 * np.linalg.norm(xh)   # atomics: order varies
    finally:
        s.A.close()


def test_standard_errors_need_a_solve():
    b = _binding()
    s = Sys(CASES["cfg1"])
    try:
        se = torch.empty(s.n, dtype=torch.float64, device="cuda")
        with pytest.raises(b.GsrError) as ei:
            b.gsr_lsqr_standard_errors(s.A.h, se)
        assert ei.value.code == b.GSR_ESTATE
    finally:
        s.A.close()


def test_stop_rule_zero_and_errors():
    b = _binding()
    s = Sys(CASES["ragged_empty_stars"])
    try:
        x = torch.full((s.n,), 7.0, dtype=torch.float64, device="cuda")
        r = b.gsr_lsqr_solve(s.A.h, torch.zeros(s.m, dtype=torch.float64, device="cuda"), x, 10,
                             1e-8, 1e-8, 1e8)
        assert (r.istop, r.itn) == (0, 0) and float(x.abs().max()) == 0.0
        with pytest.raises(b.GsrError) as ei:
            b.gsr_lsqr_solve(s.A.h, x, x, 0)
        assert ei.value.code == b.GSR_EINVAL
    finally:
        s.A.close()
    cfg = CASES["ragged_empty_stars"]
    star, att, instr, vals = inputs.gen_all(cfg)
    for mutate, what in ((lambda: star.__setitem__(5, 0), "star decreasing"),
                         (lambda: att.__setitem__(3, cfg.n_dfa - 3), "att out of range"),
                         (lambda: instr.__setitem__((4, 2), cfg.n_instr), "instr out of range"),
                         (lambda: star.__setitem__(-1, cfg.n_stars), "star out of range")):
        st, at, ic = star.clone(), att.clone(), instr.clone()
        star_, att_, instr_ = star, att, instr
        mutate()
        with pytest.raises(b.GsrError) as ei:
            b.GsrMatrix.create(cfg, star.cuda(), att.cuda(), instr.cuda(), vals.cuda())
        assert ei.value.code == b.GSR_EINVAL, what
        star.copy_(st); att.copy_(at); instr.copy_(ic)
    with pytest.raises(b.GsrError):
        b.gsr_matrix_begin(10, 1, 3, 1)          # D < 4


def test_host_arrays_and_chunked_builder_equal_one_shot():
    b = _binding()
    cfg = CASES["ragged_empty_stars"]
    star, att, instr, vals = inputs.gen_all(cfg)
    A1 = b.GsrMatrix.create(cfg, star.cuda(), att.cuda(), instr.cuda(), vals.cuda())
    A2 = b.GsrMatrix.create(cfg, star.numpy(), att.numpy(), instr.numpy(), vals.numpy())
    h = b.gsr_matrix_begin(cfg.n_rows, cfg.n_stars, cfg.n_dfa, cfg.n_instr)
    cuts = [0, 1, 300, 301, 777, cfg.n_rows]
    for r0, r1 in zip(cuts[:-1], cuts[1:]):
        b.gsr_matrix_append_rows(h, r0, r1 - r0, star[r0:r1].cuda(), att[r0:r1].cuda(),
                                 instr[r0:r1].contiguous().cuda(), vals[r0:r1].contiguous().cuda())
    b.gsr_matrix_finalize(h)
    A3 = b.GsrMatrix(h)
    x = inputs.random_vector(cfg, 1, cfg.n_cols).cuda()
    outs = []
    for A in (A1, A2, A3):
        c, v = b.gsr_debug_expand_rows(A.h, 0, cfg.n_rows)
        y = torch.zeros(cfg.n_rows, dtype=torch.float64, device="cuda")
        b.gsr_aprod1(A.h, x, y)
        outs.append((c, v, y.cpu().numpy()))
        A.close()
    for c, v, y in outs[1:]:
        assert np.array_equal(c, outs[0][0]) and np.array_equal(v, outs[0][1])
        assert np.array_equal(y, outs[0][2])


def test_sharded_solve_world_1_nccl_matches_plain_solve():
    """Row e: the sharded iteration (NCCL all-reduces inside the graph, split norm sums) with a
    one-rank communicator must reproduce the plain solve and the oracle.  The N > 1 algebra is
    covered on the CPU by tests/test_sharding_gloo.py."""
    b = _binding()
    s = Sys(CASES["cfg1"])
    try:
        rhs = _rhs(s)
        comm = b.gsr_comm_create(0, 1, b.gsr_comm_unique_id())
        b.gsr_matrix_set_comm(s.A.h, comm, s.m, s.n)
        s.o.precondition()
        b.gsr_precondition(s.A.h)
        b.gsr_set_option(s.A.h, b.GSR_OPT_FORCE_ITNLIM, 1)
        bd = torch.from_numpy(rhs).cuda()
        x = torch.empty(s.n, dtype=torch.float64, device="cuda")
        r = b.gsr_lsqr_solve(s.A.h, bd, x, 12)
        ro = s.o.lsqr(rhs, 12, force_itnlim=True, want_se=True)
        assert (r.istop, r.itn) == (7, 12)
        assert np.linalg.norm(x.cpu().numpy() - ro.x) <= X_TOL * np.linalg.norm(ro.x)
        assert abs(r.rnorm - ro.rnorm) <= X_TOL * ro.rnorm and abs(r.anorm - ro.anorm) <= X_TOL * ro.anorm
        se = np.empty(s.n)
        b.gsr_lsqr_standard_errors(s.A.h, se)
        assert np.linalg.norm(se - ro.se) <= 1e-8 * np.linalg.norm(ro.se)
        b.gsr_set_option(s.A.h, b.GSR_OPT_FUSED, 0)      # two-pass form is not sharded
        with pytest.raises(b.GsrError) as ei:
            b.gsr_lsqr_solve(s.A.h, bd, x, 3)
        assert ei.value.code == b.GSR_EUNSUPPORTED
        b.gsr_set_option(s.A.h, b.GSR_OPT_FUSED, 1)
        b.gsr_set_option(s.A.h, b.GSR_OPT_FORCE_ITNLIM, 0)
        r = b.gsr_lsqr_solve(s.A.h, bd, x, 500, 1e-10, 1e-10, 1e8)
        ro = s.o.lsqr(rhs, 500, 1e-10, 1e-10, 1e8)
        assert r.istop == ro.istop and abs(r.itn - ro.itn) <= 1
        s.A.close()
        b.gsr_comm_destroy(comm)
    finally:
        s.A.close()


@pytest.mark.parametrize("name", ["cfg1", "skew_hot", "one_instr_col"])
def test_fixed_point_instrumental_pass_matches_fp64_atomics(name):
    """GSR_OPT_FIXED_POINT: on a column-scaled matrix the instrumental block of A^T u_hat is
    accumulated in exact 64-bit fixed point (native 32-bit shared atomics); with the option off,
    with fp64 atomics.  Both must match the oracle, and each other far more closely."""
    b = _binding()
    s = Sys(CASES[name])
    try:
        rhs = _rhs(s)
        s.o.precondition()
        b.gsr_precondition(s.A.h)
        b.gsr_set_option(s.A.h, b.GSR_OPT_FORCE_ITNLIM, 1)
        bd = torch.from_numpy(rhs).cuda()
        k = 3
        ro = s.o.lsqr(rhs, k, force_itnlim=True)
        xs = []
        for i, fixed in enumerate((1, 0, 0, 1)):
            b.gsr_set_option(s.A.h, b.GSR_OPT_FIXED_POINT, fixed)
            x = torch.empty(s.n, dtype=torch.float64, device="cuda")
            r = b.gsr_lsqr_solve(s.A.h, bd, x, k)
            assert (r.istop, r.itn) == (7, k)
            xs.append(x.cpu().numpy())
            assert np.linalg.norm(xs[-1] - ro.x) <= X_TOL * np.linalg.norm(ro.x)
            # the variant of the instrumental pass is frozen into the captured graph: toggling
            # the option must re-capture (1 -> 0 -> 0 -> 1: three graphs), or the second leg
            # would replay the first one's kernels
            assert b.gsr_debug_graph_builds(s.A.h) == (1, 2, 2, 3)[i]
        assert np.linalg.norm(xs[0] - xs[1]) <= 1e-12 * np.linalg.norm(ro.x)
    finally:
        s.A.close()


@pytest.mark.parametrize("fused", [1, 0])
def test_damped_lsqr_parity(fused):
    """Row f4: gsr_lsqr_set_damp against the oracle's damped LSQR, fixed count and standard mode."""
    b = _binding()
    s = Sys(CASES["cfg1"])
    try:
        rhs = _rhs(s)
        s.o.precondition()
        b.gsr_precondition(s.A.h)
        b.gsr_set_option(s.A.h, b.GSR_OPT_FUSED, fused)
        with pytest.raises(b.GsrError):
            b.gsr_lsqr_set_damp(s.A.h, -1.0)
        damp = 0.4
        b.gsr_lsqr_set_damp(s.A.h, damp)
        bd = torch.from_numpy(rhs).cuda()
        x = torch.empty(s.n, dtype=torch.float64, device="cuda")
        b.gsr_set_option(s.A.h, b.GSR_OPT_FORCE_ITNLIM, 1)
        for k in (1, 6):
            r = b.gsr_lsqr_solve(s.A.h, bd, x, k)
            ro = s.o.lsqr(rhs, k, force_itnlim=True, damp=damp)
            assert (r.istop, r.itn) == (ro.istop, ro.itn) == (7, k)
            assert np.linalg.norm(x.cpu().numpy() - ro.x) <= X_TOL * np.linalg.norm(ro.x)
            for f in ("rnorm", "anorm", "xnorm", "acond"):
                assert abs(getattr(r, f) - getattr(ro, f)) <= X_TOL * getattr(ro, f), f
        b.gsr_set_option(s.A.h, b.GSR_OPT_FORCE_ITNLIM, 0)
        r = b.gsr_lsqr_solve(s.A.h, bd, x, 500, 1e-10, 1e-10, 1e8)
        ro = s.o.lsqr(rhs, 500, 1e-10, 1e-10, 1e8, damp=damp)
        assert r.istop == ro.istop and abs(r.itn - ro.itn) <= 1
        assert np.linalg.norm(x.cpu().numpy() - ro.x) <= X_TOL * np.linalg.norm(ro.x)
        b.gsr_lsqr_set_damp(s.A.h, 0.0)                       # back to the paper's undamped LSQR
        r = b.gsr_lsqr_solve(s.A.h, bd, x, 500, 1e-10, 1e-10, 1e8)
        ro = s.o.lsqr(rhs, 500, 1e-10, 1e-10, 1e8)
        assert r.istop == ro.istop and np.linalg.norm(x.cpu().numpy() - ro.x) <= X_TOL * np.linalg.norm(ro.x)
    finally:
        s.A.close()


@pytest.mark.parametrize("name", ["cfg1", "skew_hot", "ragged_empty_stars"])
def test_deterministic_mode_is_bit_reproducible(name):
    """GSR_OPT_DETERMINISTIC (SURVEY 8(a) a5/a8, section 4 tier T4; the paper names its atomics
    as a weakness): every sum that leaves a warp is a 64-bit fixed-point
    integer add, so repeated solves on a handle are bit-identical -- x, the norms and the
    standard errors -- and still match the oracle."""
    b = _binding()
    s = Sys(CASES[name])
    try:
        rhs = _rhs(s)
        bd = torch.from_numpy(rhs).cuda()
        b.gsr_set_option(s.A.h, b.GSR_OPT_DETERMINISTIC, 1)
        x = torch.empty(s.n, dtype=torch.float64, device="cuda")
        with pytest.raises(b.GsrError) as ei:      # needs unit column norms
            b.gsr_lsqr_solve(s.A.h, bd, x, 3)
        assert ei.value.code == b.GSR_EUNSUPPORTED
        s.o.precondition()
        b.gsr_precondition(s.A.h)
        b.gsr_set_option(s.A.h, b.GSR_OPT_FORCE_ITNLIM, 1)
        for k in (1, 8, 30):
            ro = s.o.lsqr(rhs, k, force_itnlim=True)
            runs = []
            for rep in range(3):
                x = torch.empty(s.n, dtype=torch.float64, device="cuda")
                r = b.gsr_lsqr_solve(s.A.h, bd, x, k)
                se = torch.empty(s.n, dtype=torch.float64, device="cuda")
                b.gsr_lsqr_standard_errors(s.A.h, se)
                runs.append((x.cpu().numpy(), se.cpu().numpy(), r))
            for xx, se, r in runs[1:]:
                assert np.array_equal(xx, runs[0][0]) and np.array_equal(se, runs[0][1])
                assert r == runs[0][2]
            assert (runs[0][2].istop, runs[0][2].itn) == (ro.istop, ro.itn) == (7, k)
            assert np.linalg.norm(runs[0][0] - ro.x) <= X_TOL * np.linalg.norm(ro.x)
        # standard mode with stopping rules: same stop, still bit-identical
        ro = s.o.lsqr(rhs, 300, atol=1e-10, btol=1e-10, conlim=1e8)
        b.gsr_set_option(s.A.h, b.GSR_OPT_FORCE_ITNLIM, 0)
        xa = torch.empty(s.n, dtype=torch.float64, device="cuda")
        xb = torch.empty(s.n, dtype=torch.float64, device="cuda")
        ra = b.gsr_lsqr_solve(s.A.h, bd, xa, 300, 1e-10, 1e-10, 1e8)
        rb = b.gsr_lsqr_solve(s.A.h, bd, xb, 300, 1e-10, 1e-10, 1e8)
        assert ra == rb and torch.equal(xa, xb)
        assert (ra.istop, ra.itn) == (ro.istop, ro.itn)
        # back to fp64 atomics: same answer within the parity tolerance
        b.gsr_set_option(s.A.h, b.GSR_OPT_DETERMINISTIC, 0)
        rc = b.gsr_lsqr_solve(s.A.h, bd, xb, 300, 1e-10, 1e-10, 1e8)
        assert (rc.istop, rc.itn) == (ro.istop, ro.itn)
        assert float((xa - xb).norm() / xa.norm()) <= 1e-9
    finally:
        s.A.close()


@pytest.mark.parametrize("fused", [1, 0])
def test_while_graph_loop_equals_one_launch_per_iteration(fused):
    """Row a11, second form: the whole loop as one conditional-WHILE graph launch
    (GSR_OPT_WHILE_GRAPH = 1) against one graph launch per iteration with the stop flag polled
    by the host (default).  Same kernels, same stop decision; in deterministic mode bit-identical."""
    b = _binding()
    s = Sys(CASES["cfg1"])
    try:
        rhs = _rhs(s)
        bd = torch.from_numpy(rhs).cuda()
        s.o.precondition()
        b.gsr_precondition(s.A.h)
        b.gsr_set_option(s.A.h, b.GSR_OPT_FUSED, fused)
        if fused:
            b.gsr_set_option(s.A.h, b.GSR_OPT_DETERMINISTIC, 1)
        out = {}
        for loop in (1, 0):
            b.gsr_set_option(s.A.h, b.GSR_OPT_WHILE_GRAPH, loop)
            # fixed count
            b.gsr_set_option(s.A.h, b.GSR_OPT_FORCE_ITNLIM, 1)
            x = torch.empty(s.n, dtype=torch.float64, device="cuda")
            n0 = b.gsr_launch_count()
            r = b.gsr_lsqr_solve(s.A.h, bd, x, 25)
            launches = b.gsr_launch_count() - n0
            assert b.gsr_debug_while_graph(s.A.h) == loop      # the loop form asked for really ran
            assert (r.istop, r.itn) == (7, 25)
            # natural stop
            b.gsr_set_option(s.A.h, b.GSR_OPT_FORCE_ITNLIM, 0)
            x2 = torch.empty(s.n, dtype=torch.float64, device="cuda")
            r2 = b.gsr_lsqr_solve(s.A.h, bd, x2, 500, 1e-10, 1e-10, 1e8)
            assert b.gsr_debug_while_graph(s.A.h) == loop
            out[loop] = (x.cpu().numpy(), r, x2.cpu().numpy(), r2, launches)
        b.gsr_set_option(s.A.h, b.GSR_OPT_WHILE_GRAPH, 0)
        ro = s.o.lsqr(rhs, 25, force_itnlim=True)
        ro2 = s.o.lsqr(rhs, 500, 1e-10, 1e-10, 1e8)
        for loop in (1, 0):
            xx, r, xx2, r2, _ = out[loop]
            assert np.linalg.norm(xx - ro.x) <= X_TOL * np.linalg.norm(ro.x)
            assert r2.istop == ro2.istop and abs(r2.itn - ro2.itn) <= 1
            assert np.linalg.norm(xx2 - ro2.x) <= X_TOL * np.linalg.norm(ro2.x)
        assert out[1][3].itn == out[0][3].itn and out[1][3].istop == out[0][3].istop
        assert out[1][4] == out[0][4], (out[1][4], out[0][4])      # same kernels per iteration
        if fused:      # integer sums: the two loop forms agree to the last bit
            assert np.array_equal(out[1][0], out[0][0]) and np.array_equal(out[1][2], out[0][2])
            assert out[1][1] == out[0][1] and out[1][3] == out[0][3]
    finally:
        s.A.close()


def test_option_values_are_validated():
    b = _binding()
    s = Sys(CASES["one_instr_col"])
    try:
        for v in (-1, 0, 1):
            b.gsr_set_option(s.A.h, b.GSR_OPT_APROD2_SPLIT, v)
        for key, v in ((b.GSR_OPT_APROD2_SPLIT, 2), (b.GSR_OPT_APROD2_SPLIT, -2), (99, 1), (0, 1)):
            with pytest.raises(b.GsrError) as ei:
                b.gsr_set_option(s.A.h, key, v)
            assert ei.value.code == b.GSR_EINVAL
        b.gsr_set_option(s.A.h, b.GSR_OPT_APROD2_SPLIT, -1)
    finally:
        s.A.close()


def test_zz_write_sensitivity_log():
    """Not a check of its own: records the oracle's one-ulp sensitivities that bounded the
    tolerances of test_precondition_and_lsqr_parity (quoted in DESIGN.md, reading A20)."""
    import json
    import os
    assert all(sn < X_TOL_CAP / 20.0 for _, _, _, sn in SENS_LOG), max(SENS_LOG, key=lambda t: t[3])
    out = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "gpurun_out")
    os.makedirs(out, exist_ok=True)
    with open(os.path.join(out, "lsqr_sensitivity.json"), "w") as f:
        json.dump([{"case": c, "fused": fu, "k": k, "sens": sn} for c, fu, k, sn in SENS_LOG], f, indent=1)
