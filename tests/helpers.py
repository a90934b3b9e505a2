"""Test helpers: a third, independent expression of the matrix structure (numpy/scipy CSR),
used to pin the oracle -- never used by the CUDA path or by the oracle itself."""
import numpy as np
import scipy.sparse as sp

from paper_2212_11675_b200 import inputs


def csr_from_raw(cfg, star, att, instr, vals):
    """scipy CSR of A from the caller-form arrays, by numpy index arithmetic
    (5 astrometric at 5s.., 3x4 attitude N_DFA apart, 6 instrumental, 1 global)."""
    star = np.asarray(star, dtype=np.int64)
    att = np.asarray(att, dtype=np.int64)
    instr = np.asarray(instr, dtype=np.int64).reshape(-1, 6)
    vals = np.asarray(vals, dtype=np.float64).reshape(-1, 24)
    m = star.shape[0]
    S, D, I = cfg.n_stars, cfg.n_dfa, cfg.n_instr
    cols = np.concatenate([
        5 * star[:, None] + np.arange(5)[None, :],
        (5 * S + att)[:, None] + (np.repeat(np.arange(3), 4) * D + np.tile(np.arange(4), 3))[None, :],
        5 * S + 3 * D + instr,
        np.full((m, 1), 5 * S + 3 * D + I),
    ], axis=1)
    rows = np.repeat(np.arange(m), 24)
    n = 5 * S + 3 * D + I + 1
    # duplicates (repeated instrumental columns) are summed by coo->csr, as the definition says
    A = sp.coo_matrix((vals.ravel(), (rows, cols.ravel())), shape=(m, n)).tocsr()
    return A, cols


def small_system(seed=7, counts=(20,) * 6, n_dfa=6, n_instr=8, **kw):
    cfg = inputs.micro_config("tiny", seed, counts, n_dfa, n_instr, **kw)
    star, att, instr, vals = inputs.gen_all(cfg)
    return cfg, star.numpy(), att.numpy(), instr.numpy(), vals.numpy()


def make_oracle(cfg, star, att, instr, vals):
    from oracle.gsr_oracle import OracleSystem
    return OracleSystem(cfg.n_stars, cfg.n_dfa, cfg.n_instr, star, att, instr, vals)
