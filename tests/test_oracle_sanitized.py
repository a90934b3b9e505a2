"""CPU-only: the oracle under AddressSanitizer and UndefinedBehaviorSanitizer (SURVEY section 5,
tier T1).  The same oracle/gsr_oracle.c is compiled with -fsanitize=address,undefined into a
temporary directory and a fresh interpreter (libasan preloaded) runs products, the
preconditioner, LSQR with variances, constraint rows and the row expansion on ragged systems;
any out-of-bounds access, signed overflow or misaligned load makes that process fail."""
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

SCRIPT = r"""
import numpy as np
import oracle.gsr_oracle as go
go._LIB = {lib!r}
from paper_2212_11675_b200 import inputs
for seed, counts, D, I in ((7, (20,) * 6, 6, 8), (24, (0, 37, 1, 250, 0, 64, 3, 0, 700, 0), 40, 17),
                           (21, (1,), 4, 1)):
    cfg = inputs.micro_config("asan", seed, counts, D, I)
    s, a, i, v = (t.numpy() for t in inputs.gen_all(cfg))
    o = go.OracleSystem(cfg.n_stars, cfg.n_dfa, cfg.n_instr, s, a, i, v)
    rng = np.random.default_rng(seed)
    x, y = rng.standard_normal(o.n), rng.standard_normal(o.m)
    o.aprod1(x, y.copy(), want_scale=True)
    o.aprod2(y, x.copy(), want_scale=True)
    o.expand_rows()
    b = o.aprod1(x, 1e-3 * rng.standard_normal(o.m))
    o.precondition()
    r = o.lsqr(b, 30, 1e-12, 1e-12, 1e8, want_se=True, want_hist=True)
    assert np.all(np.isfinite(r.x)) and np.all(np.isfinite(r.se))
    o.lsqr(b, 5, force_itnlim=True, damp=0.1)
maps = open("/proc/self/maps").read()
assert "libgsr_oracle_san.so" in maps and "libasan" in maps      # the instrumented build is what ran
print("sanitized oracle ok")
"""


def test_oracle_under_asan_and_ubsan(tmp_path):
    lib = str(tmp_path / "libgsr_oracle_san.so")
    subprocess.check_call(["gcc", "-O1", "-g", "-std=c99", "-ffp-contract=off", "-fPIC", "-shared",
                           "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined",
                           "-o", lib, os.path.join(ROOT, "oracle", "gsr_oracle.c"), "-lm"])
    asan = subprocess.run(["gcc", "-print-file-name=libasan.so"], capture_output=True, text=True).stdout.strip()
    env = dict(os.environ, LD_PRELOAD=asan, ASAN_OPTIONS="detect_leaks=0:abort_on_error=1",
               UBSAN_OPTIONS="halt_on_error=1:print_stacktrace=1")
    out = subprocess.run([sys.executable, "-c", SCRIPT.format(lib=lib)], cwd=ROOT, env=env,
                         capture_output=True, text=True, timeout=600)
    assert out.returncode == 0 and "sanitized oracle ok" in out.stdout, out.stderr[-4000:]
