"""The OpenMP timing build of the oracle (oracle/gsr_oracle.c with -DORC_OPENMP: the paper's
CPU scheme) against the serial build, which is the definition.  It is what
bench.py times on all host cores and what the full-size parity legs run, so it must agree with
the serial oracle far below the parity tolerances (1e-13 here; the two differ only in the
order of the long-double column sums)."""
import numpy as np
import pytest

from oracle import gsr_oracle
from paper_2212_11675_b200 import inputs


def _pair(name, scale):
    cfg = inputs.scaled(inputs.named_config(name), scale, f"{name}/{scale}")
    star, att, instr, vals = inputs.gen_all(cfg)
    return cfg, gsr_oracle.from_torch(cfg, star, att, instr, vals), \
        gsr_oracle.from_torch(cfg, star, att, instr, vals, omp=True)


@pytest.mark.parametrize("name,scale", [("cfg1", 10), ("cfg4", 5000)])
def test_omp_products_match_serial(name, scale, monkeypatch):
    cfg, s, p = _pair(name, scale)
    assert gsr_oracle.omp_threads() >= 1
    x = inputs.random_vector(cfg, 1, cfg.n_cols).numpy()
    y = inputs.random_vector(cfg, 2, cfg.n_rows).numpy()
    y1, sc1 = s.aprod1(x, y, want_scale=True)
    y2, sc2 = p.aprod1(x, y, want_scale=True)
    assert np.array_equal(y1, y2) and np.array_equal(sc1, sc2)        # row sums: same order
    x1, sx1 = s.aprod2(y, x, want_scale=True)
    x2, sx2 = p.aprod2(y, x, want_scale=True)
    assert np.all(np.abs(x1 - x2) <= 1e-13 * sx1)
    assert np.allclose(sx1, sx2, rtol=1e-13, atol=0)
    assert np.allclose(s.colsumsq(), p.colsumsq(), rtol=1e-13, atol=0)


@pytest.mark.parametrize("name,scale", [("cfg1", 10), ("cfg4", 5000)])
def test_omp_lsqr_matches_serial(name, scale):
    cfg, s, p = _pair(name, scale)
    b = s.aprod1(inputs.x_true(cfg).numpy(), inputs.noise(cfg, 0, cfg.n_rows).numpy())
    ps, pp = s.precondition(), p.precondition()
    assert np.allclose(ps, pp, rtol=1e-13, atol=0)
    for k in (1, 5, 12):
        rs = s.lsqr(b, k, force_itnlim=True, want_se=True)
        rp = p.lsqr(b, k, force_itnlim=True, want_se=True)
        assert (rs.istop, rs.itn) == (rp.istop, rp.itn) == (7, k)
        assert np.linalg.norm(rs.x - rp.x) <= 1e-12 * np.linalg.norm(rs.x)
        for f in ("rnorm", "anorm", "xnorm", "acond"):
            assert abs(getattr(rs, f) - getattr(rp, f)) <= 1e-12 * abs(getattr(rs, f))


def test_omp_thread_count_does_not_change_the_partition_semantics(monkeypatch):
    # star-aligned ranges: a star larger than rows/threads must stay with one thread
    cfg = inputs.scaled(inputs.named_config("cfg1"), 100, "cfg1/100")   # 20 stars x 100 rows
    star, att, instr, vals = inputs.gen_all(cfg)
    s = gsr_oracle.from_torch(cfg, star, att, instr, vals)
    p = gsr_oracle.from_torch(cfg, star, att, instr, vals, omp=True)
    y = inputs.random_vector(cfg, 2, cfg.n_rows).numpy()
    x1, sc = s.aprod2(y, np.zeros(cfg.n_cols), want_scale=True)
    x2 = p.aprod2(y, np.zeros(cfg.n_cols))
    assert np.all(np.abs(x1 - x2) <= 1e-13 * np.maximum(sc, 1e-300))
