#!/usr/bin/env python
"""Writes tests/golden/tiny_lsqr.txt: the ORACLE's results on one tiny seeded system (a
regression anchor for the oracle itself and a fixed target for the CUDA path).  Calls only
oracle/ and the shared input generator -- never the CUDA package's kernels.

    python tests/golden/make_tiny_lsqr.py

The values are not the paper's (it prints no worked example); what pins the oracle
to the mathematics is in tests/test_oracle_*.py.  This file only freezes what the pinned oracle
returned when it was written, at 17 significant digits.
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle.gsr_oracle import OracleSystem   # noqa: E402
from paper_2212_11675_b200 import inputs     # noqa: E402  (seeded generator only)

COUNTS, N_DFA, N_INSTR, SEED, K = (9, 0, 14, 6), 7, 5, 20260101, 5


def compute():
    cfg = inputs.micro_config("golden", SEED, COUNTS, N_DFA, N_INSTR)
    star, att, instr, vals = [t.numpy() for t in inputs.gen_all(cfg)]
    o = OracleSystem(cfg.n_stars, cfg.n_dfa, cfg.n_instr, star, att, instr, vals)
    x1 = inputs.random_vector(cfg, 1, cfg.n_cols).numpy()
    y1 = inputs.random_vector(cfg, 2, cfg.n_rows).numpy()
    ax = o.aprod1(x1, np.zeros(o.m))
    aty = o.aprod2(y1, np.zeros(o.n))
    b = o.aprod1(inputs.x_true(cfg).numpy(), inputs.noise(cfg, 0, cfg.n_rows).numpy())
    p = o.precondition()
    r = o.lsqr(b, K, force_itnlim=True, want_se=True)
    return cfg, {"aprod1": ax, "aprod2": aty, "p": p, "x": r.x, "se": r.se,
                 "scalars": np.array([r.rnorm, r.arnorm, r.anorm, r.acond, r.xnorm, r.bnorm])}


def main():
    cfg, d = compute()
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "tiny_lsqr.txt")
    with open(path, "w") as f:
        f.write("# written by tests/golden/make_tiny_lsqr.py from oracle/ only; see its docstring\n")
        f.write(f"# counts={COUNTS} n_dfa={N_DFA} n_instr={N_INSTR} seed={SEED} k={K} "
                f"m={cfg.n_rows} n={cfg.n_cols}\n")
        f.write("# scalars = rnorm arnorm anorm acond xnorm bnorm after k preconditioned iterations\n")
        for key, v in d.items():
            f.write(key + " " + " ".join(f"{t:.17g}" for t in v) + "\n")
    print("wrote", path)


if __name__ == "__main__":
    main()
