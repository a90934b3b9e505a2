"""tests/golden/tiny_lsqr.txt (written by tests/golden/make_tiny_lsqr.py from oracle/ only):
the oracle must still return it (a change to the oracle's arithmetic shows up here and has to be
justified in its commit message), and the CUDA path must match it."""
import os

import numpy as np
import pytest

from paper_2212_11675_b200 import inputs

HERE = os.path.dirname(os.path.abspath(__file__))


def _load():
    d = {}
    for line in open(os.path.join(HERE, "golden", "tiny_lsqr.txt")):
        if line.startswith("#"):
            continue
        key, *vals = line.split()
        d[key] = np.array([float(v) for v in vals])
    return d


def _module():
    import importlib.util
    spec = importlib.util.spec_from_file_location("make_tiny_lsqr", os.path.join(HERE, "golden", "make_tiny_lsqr.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    return mod


def test_oracle_reproduces_golden_file():
    gold = _load()
    _, now = _module().compute()
    for key, v in gold.items():
        assert np.allclose(now[key], v, rtol=1e-14, atol=1e-300), key


@pytest.mark.gpu
def test_cuda_path_matches_golden_file():
    import torch
    from paper_2212_11675_b200 import binding as g
    mod = _module()
    gold = _load()
    cfg = inputs.micro_config("golden", mod.SEED, mod.COUNTS, mod.N_DFA, mod.N_INSTR)
    star, att, instr, vals = inputs.gen_all(cfg)
    A = g.GsrMatrix.create(cfg, star.cuda(), att.cuda(), instr.cuda(), vals.cuda())
    try:
        yd = torch.zeros(cfg.n_rows, dtype=torch.float64, device="cuda")
        xd = torch.zeros(cfg.n_cols, dtype=torch.float64, device="cuda")
        g.gsr_aprod1(A.h, inputs.random_vector(cfg, 1, cfg.n_cols).cuda(), yd)
        g.gsr_aprod2(A.h, inputs.random_vector(cfg, 2, cfg.n_rows).cuda(), xd)
        assert np.allclose(yd.cpu().numpy(), gold["aprod1"], rtol=0, atol=1e-13)
        assert np.allclose(xd.cpu().numpy(), gold["aprod2"], rtol=0, atol=1e-13)
        b = torch.zeros(cfg.n_rows, dtype=torch.float64, device="cuda")
        b += inputs.noise(cfg, 0, cfg.n_rows).cuda()
        g.gsr_aprod1(A.h, inputs.x_true(cfg).cuda(), b)
        p = torch.empty(cfg.n_cols, dtype=torch.float64, device="cuda")
        g.gsr_precondition(A.h, p)
        assert np.allclose(p.cpu().numpy(), gold["p"], rtol=1e-13)
        g.gsr_set_option(A.h, g.GSR_OPT_FORCE_ITNLIM, 1)
        x = torch.empty(cfg.n_cols, dtype=torch.float64, device="cuda")
        r = g.gsr_lsqr_solve(A.h, b, x, mod.K)
        assert (r.istop, r.itn) == (7, mod.K)
        assert np.linalg.norm(x.cpu().numpy() - gold["x"]) <= 1e-9 * np.linalg.norm(gold["x"])
        got = np.array([r.rnorm, r.arnorm, r.anorm, r.acond, r.xnorm, r.bnorm])
        assert np.allclose(got, gold["scalars"], rtol=1e-9)
        se = np.empty(cfg.n_cols)
        g.gsr_lsqr_standard_errors(A.h, se)
        assert np.linalg.norm(se - gold["se"]) <= 1e-8 * np.linalg.norm(gold["se"])
    finally:
        A.close()
