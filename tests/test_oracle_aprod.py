"""Pins for the oracle's index expansion, aprod1, aprod2 and preconditioner (CPU only).

Everything here checks oracle/ against something other than itself: a scipy CSR rebuilt from
the raw arrays with numpy index arithmetic, unit-vector probes, the adjoint identity,
closed forms (unit column norms, Frobenius norm) and the paper's structural constants
(tests/golden/structure.txt)."""
import os

import numpy as np
import pytest

from paper_2212_11675_b200 import inputs
from tests.helpers import csr_from_raw, make_oracle, small_system

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "structure.txt")


def _golden():
    out = {}
    for line in open(GOLDEN):
        line = line.split("#")[0].strip()
        if line:
            k, v = line.split("=")
            out[k.strip()] = int(v)
    return out


def _mid():
    cfg = inputs.micro_config("mid", 11, [0, 37, 1, 250, 0, 64, 3, 0], 40, 17)
    s, a, i, v = inputs.gen_all(cfg)
    return cfg, s.numpy(), a.numpy(), i.numpy(), v.numpy()


def test_golden_structure_constants():
    """Section 3 of the paper fixes 24 = 5 + 3*4 + 6 + 1 and config 1 fixes n = 13601."""
    g = _golden()
    assert g["N_par"] == g["N_Astro"] + g["N_Axes"] * g["N_ParAxis"] + g["N_Instr"] + g["N_Glob"] == 24
    cfg = inputs.named_config("cfg1")
    assert cfg.n_rows == g["cfg1_rows"] and cfg.n_cols == g["cfg1_cols"]
    cfg, star, att, instr, vals = small_system()
    o = make_oracle(cfg, star, att, instr, vals)
    cols, _ = o.expand_rows()
    assert cols.shape[1] == g["N_par"]
    # section sizes and their order inside a row: 5 | 12 | 6 | 1
    assert (cols[:, :5] < 5 * cfg.n_stars).all()
    assert ((cols[:, 5:17] >= cfg.off_att) & (cols[:, 5:17] < cfg.off_instr)).all()
    assert ((cols[:, 17:23] >= cfg.off_instr) & (cols[:, 17:23] < cfg.off_glob)).all()
    assert (cols[:, 23] == cfg.off_glob).all()


@pytest.mark.parametrize("maker", [small_system, _mid])
def test_expand_rows_equals_numpy_index_arithmetic(maker):
    cfg, star, att, instr, vals = maker()
    o = make_oracle(cfg, star, att, instr, vals)
    assert o.validate() == 0
    _, cols_np = csr_from_raw(cfg, star, att, instr, vals)
    cols, v = o.expand_rows()
    assert np.array_equal(cols, cols_np)
    assert np.array_equal(v, vals)
    # structural invariants
    assert np.array_equal(cols[:, :5], 5 * star[:, None] + np.arange(5))
    for ax in range(3):
        blk = cols[:, 5 + 4 * ax:9 + 4 * ax]
        assert (np.diff(blk, axis=1) == 1).all()
        assert np.array_equal(blk[:, 0], cfg.off_att + ax * cfg.n_dfa + att)
    # partial range
    c2, v2 = o.expand_rows(5, 9)
    assert np.array_equal(c2, cols[5:14]) and np.array_equal(v2, vals[5:14])


def test_validate_rejects_bad_indices():
    cfg, star, att, instr, vals = small_system()
    bad = star.copy(); bad[3] = bad[2] - 1 if bad[2] > 0 else 5
    bad2 = star.copy(); bad2[10], bad2[11] = 3, 2
    assert make_oracle(cfg, bad2, att, instr, vals).validate() == -3
    a = att.copy(); a[0] = cfg.n_dfa - 3
    assert make_oracle(cfg, star, a, instr, vals).validate() == -4
    ic = instr.copy(); ic[4, 2] = cfg.n_instr
    assert make_oracle(cfg, star, att, ic, vals).validate() == -5
    s = star.copy(); s[-1] = cfg.n_stars
    assert make_oracle(cfg, s, att, instr, vals).validate() == -2


@pytest.mark.parametrize("maker", [small_system, _mid])
def test_unit_vector_probes(maker):
    """aprod1(e_j) is column j of A; aprod2(e_i) is row i of A."""
    cfg, star, att, instr, vals = maker()
    o = make_oracle(cfg, star, att, instr, vals)
    A, _ = csr_from_raw(cfg, star, att, instr, vals)
    Ad = A.toarray()
    rng = np.random.default_rng(1)
    for j in rng.choice(o.n, size=min(o.n, 25), replace=False):
        e = np.zeros(o.n); e[j] = 1.0
        assert np.array_equal(o.aprod1(e, np.zeros(o.m)), Ad[:, j])
    for i in rng.choice(o.m, size=15, replace=False):
        e = np.zeros(o.m); e[i] = 1.0
        assert np.allclose(o.aprod2(e, np.zeros(o.n)), Ad[i, :], rtol=0, atol=1e-16)


def test_aprod_matches_csr_and_accumulates():
    cfg, star, att, instr, vals = _mid()
    o = make_oracle(cfg, star, att, instr, vals)
    A, _ = csr_from_raw(cfg, star, att, instr, vals)
    rng = np.random.default_rng(2)
    x, y = rng.standard_normal(o.n), rng.standard_normal(o.m)
    y0, x0 = rng.standard_normal(o.m), rng.standard_normal(o.n)
    y1, sc1 = o.aprod1(x, y0, want_scale=True)
    x1, sc2 = o.aprod2(y, x0, want_scale=True)
    assert np.all(np.abs(y1 - (y0 + A @ x)) <= 1e-13 * sc1)      # accumulating
    assert np.all(np.abs(x1 - (x0 + A.T @ y)) <= 1e-13 * sc2)    # accumulating
    # the scale vectors are |y0| + |A||x| and |x0| + |A^T||y|
    assert np.allclose(sc1, np.abs(y0) + abs(A) @ np.abs(x), rtol=1e-13)
    assert np.allclose(sc2, np.abs(x0) + abs(A).T @ np.abs(y), rtol=1e-13)


def test_adjoint_identity():
    """<A x, y> = <x, A^T y> (north star's first check)."""
    cfg = inputs.scaled(inputs.named_config("cfg1"), 20, "cfg1/20")
    s, a, i, v = inputs.gen_all(cfg)
    o = make_oracle(cfg, s.numpy(), a.numpy(), i.numpy(), v.numpy())
    rng = np.random.default_rng(3)
    x, y = rng.standard_normal(o.n), rng.standard_normal(o.m)
    Ax = o.aprod1(x, np.zeros(o.m))
    ATy = o.aprod2(y, np.zeros(o.n))
    lhs, rhs = float(np.dot(Ax, y)), float(np.dot(x, ATy))
    assert abs(lhs - rhs) <= 1e-13 * np.linalg.norm(Ax) * np.linalg.norm(y)


def test_duplicate_instrumental_columns_add():
    cfg, star, att, instr, vals = small_system()
    instr = instr.copy(); instr[:, 1] = instr[:, 0]
    o = make_oracle(cfg, star, att, instr, vals)
    A, _ = csr_from_raw(cfg, star, att, instr, vals)
    x = np.random.default_rng(4).standard_normal(o.n)
    assert np.allclose(o.aprod1(x, np.zeros(o.m)), A @ x, rtol=0, atol=1e-13)


def test_preconditioner_unit_columns_and_frobenius():
    """After scaling every non-empty column has norm 1, so ||A'||_F^2 = #non-empty columns."""
    cfg, star, att, instr, vals = _mid()
    o = make_oracle(cfg, star, att, instr, vals)
    A, _ = csr_from_raw(cfg, star, att, instr, vals)
    q_np = np.asarray(A.multiply(A).sum(axis=0)).ravel()
    assert np.allclose(o.colsumsq(), q_np, rtol=1e-14)
    p = o.precondition()
    nonempty = q_np > 0
    assert (~nonempty).sum() >= 15          # stars 0, 4, 7 have no rows
    assert np.all(p[~nonempty] == 1.0)
    assert np.allclose(p[nonempty], 1.0 / np.sqrt(q_np[nonempty]), rtol=1e-14)
    q2 = o.colsumsq()
    assert np.allclose(q2[nonempty], 1.0, rtol=0, atol=1e-14)
    assert np.all(q2[~nonempty] == 0.0)
    assert abs((o.values ** 2).sum() - nonempty.sum()) <= 1e-12 * nonempty.sum()
    # scaled matrix equals A diag(p)
    A2, _ = csr_from_raw(cfg, star, att, instr, o.values)
    assert abs(A2 - A @ __import__("scipy.sparse").sparse.diags(p)).max() <= 1e-15


def test_config4_generator_shape():
    """Skew/contention config at 1/1000 scale: power-law counts sum exactly, hot window, scales."""
    cfg = inputs.GsrConfig("cfg4s", 3, 200, 200, 60, n_rows_total=100_000,
                           powerlaw=(10, 10_000, 1.36), att_hot=(0.9, 0.40, 0.45), col_scales=True)
    counts = inputs.star_counts(cfg).numpy()
    assert counts.sum() == cfg.n_rows == 100_000 and counts.min() >= 1
    s, a, i, v = inputs.gen_all(cfg)
    assert (np.diff(s.numpy()) >= 0).all()
    assert np.array_equal(np.bincount(s.numpy(), minlength=200), counts)
    a = a.numpy()
    lo, hi = int(0.40 * 197), int(0.45 * 197)
    frac = ((a >= lo) & (a < hi)).mean()
    assert 0.88 < frac < 0.93
    ic = np.sort(i.numpy(), axis=1)
    assert (np.diff(ic, axis=1) > 0).all()       # six distinct columns
    o = make_oracle(cfg, s.numpy(), a, i.numpy(), v.numpy())
    q = np.sqrt(o.colsumsq())
    q = q[q > 0]
    assert q.max() / q.min() > 1e6               # column norms span many decades
