"""Full-size GPU checks at BASELINE.json's sizes, in the configuration bench.py times
(chunked device-side ingest, preconditioned, fixed-count solve).  The oracle cannot run 1e8
to 3e8 rows, so it computes SAMPLED outputs one by one:
  * aprod1: sampled rows (the oracle gets exactly those rows of the generator's arrays);
  * aprod2: every column touched only by a row set that can be collected during ingest --
    the 5 astrometric columns of sampled stars, one attitude column (rows whose 4-knot window
    covers it) and one instrumental column -- for which the oracle sums the collected rows;
plus properties that hold at any size: the adjoint identity (covers the global column) and
LSQR's residual estimate against the directly computed ||b - A x||."""
import numpy as np
import pytest
import torch

from paper_2212_11675_b200 import inputs
from oracle.gsr_oracle import OracleSystem

pytestmark = pytest.mark.gpu
GEN_ROWS = 1 << 23


def _need_gb(gb):
    free, _ = torch.cuda.mem_get_info()
    if free < gb * 1e9:
        pytest.skip(f"needs {gb} GB of free device memory")


def _build_and_collect(cfg, g, probe_knot, probe_instr, probe_rows):
    """Ingest cfg chunk by chunk; keep host copies of the rows the probes need."""
    dev = "cuda"
    sptr = inputs.star_ptr(cfg)
    scales = inputs.col_scales(cfg, dev)
    h = g.gsr_matrix_begin(cfg.n_rows, cfg.n_stars, cfg.n_dfa, cfg.n_instr)
    keep = {"rows": [], "knot": [], "instr": []}
    probe_rows_t = torch.as_tensor(probe_rows, device=dev)
    for r0 in range(0, cfg.n_rows, GEN_ROWS):
        nr = min(GEN_ROWS, cfg.n_rows - r0)
        star, att, instr, vals = inputs.gen_rows(cfg, r0, nr, dev, sptr=sptr, scales=scales)
        g.gsr_matrix_append_rows(h, r0, nr, star, att, instr, vals)
        sel = probe_rows_t[(probe_rows_t >= r0) & (probe_rows_t < r0 + nr)] - r0
        mk = (att <= probe_knot) & (att >= probe_knot - 3)
        mi = (instr == probe_instr).any(dim=1)
        for key, idx in (("rows", sel), ("knot", mk.nonzero().squeeze(1)), ("instr", mi.nonzero().squeeze(1))):
            keep[key].append((idx.cpu() + r0, star[idx].cpu(), att[idx].cpu(), instr[idx].cpu(), vals[idx].cpu()))
        del star, att, instr, vals
    g.gsr_matrix_finalize(h)
    out = {}
    for key, parts in keep.items():
        out[key] = tuple(torch.cat([p[i] for p in parts]).numpy() for i in range(5))
    return h, sptr, out


def _oracle_rows(cfg, part):
    _, star, att, instr, vals = part
    return OracleSystem(cfg.n_stars, cfg.n_dfa, cfg.n_instr, star, att, instr, vals)


@pytest.mark.parametrize("name,gb", [("cfg2", 40), ("cfg4", 40), ("cfg3", 110)])
def test_fullsize_sampled_parity_and_properties(name, gb):
    from paper_2212_11675_b200 import binding as g
    _need_gb(gb)
    cfg = inputs.named_config(name)
    m, n = cfg.n_rows, cfg.n_cols
    rng = np.random.default_rng(cfg.seed)
    probe_rows = np.unique(rng.integers(0, m, 4000))
    probe_knot = int(0.42 * (cfg.n_dfa - 3)) + 5       # inside config 4's hot window
    probe_instr = int(rng.integers(0, cfg.n_instr))
    h, sptr, kept = _build_and_collect(cfg, g, probe_knot, probe_instr, probe_rows)
    try:
        x = inputs.random_vector(cfg, 1, n, "cuda")
        y = inputs.random_vector(cfg, 2, m, "cuda")
        # ---- aprod1 on sampled rows
        y0 = inputs.random_vector(cfg, 3, m, "cuda")
        yd = y0.clone()
        g.gsr_aprod1(h, x, yd)
        rows = kept["rows"][0]
        o = _oracle_rows(cfg, kept["rows"])
        ref, scale = o.aprod1(x.cpu().numpy(), y0[rows].cpu().numpy(), want_scale=True)
        err = np.abs(yd[rows].cpu().numpy() - ref)
        assert np.all(err <= 1e-12 * scale), float((err / scale).max())
        # index construction of the sampled rows, bit-exact, through the device layout
        for r in rows[:50]:
            c, v = g.gsr_debug_expand_rows(h, int(r), 1)
            i = int(np.searchsorted(rows, r))
            oc, ov = o.expand_rows(i, 1)
            assert np.array_equal(c, oc) and np.array_equal(v, ov)
        # ---- aprod2
        x0 = inputs.random_vector(cfg, 4, n, "cuda")
        xd = x0.clone()
        g.gsr_aprod2(h, y, xd)
        xh, x0h = xd.cpu().numpy(), x0.cpu().numpy()
        # attitude column probe_knot of every axis, and one instrumental column
        for key, cols in (("knot", [cfg.off_att + ax * cfg.n_dfa + probe_knot for ax in range(3)]),
                          ("instr", [cfg.off_instr + probe_instr])):
            o2 = _oracle_rows(cfg, kept[key])
            ysub = y[kept[key][0]].cpu().numpy()
            ref, scale = o2.aprod2(ysub, x0h, want_scale=True)
            for c in cols:
                assert abs(xh[c] - ref[c]) <= 1e-12 * scale[c], (key, c, abs(xh[c] - ref[c]) / scale[c])
        # astrometric columns of sampled stars: their rows are one contiguous run
        stars = rng.integers(0, cfg.n_stars, 6)
        for s in stars:
            r0, r1 = int(sptr[s]), int(sptr[s + 1])
            if r1 == r0:
                assert np.array_equal(xh[5 * s:5 * s + 5], x0h[5 * s:5 * s + 5])
                continue
            c0 = (r0 // inputs.CHUNK) * inputs.CHUNK
            st, at, ic, va = inputs.gen_rows(cfg, c0, r1 - c0, "cuda", sptr=sptr)
            sl = slice(r0 - c0, r1 - c0)
            o3 = OracleSystem(cfg.n_stars, cfg.n_dfa, cfg.n_instr, st[sl].cpu().numpy(), at[sl].cpu().numpy(),
                              ic[sl].cpu().numpy(), va[sl].cpu().numpy())
            ref, scale = o3.aprod2(y[r0:r1].cpu().numpy(), x0h, want_scale=True)
            seg = slice(5 * int(s), 5 * int(s) + 5)
            assert np.all(np.abs(xh[seg] - ref[seg]) <= 1e-12 * scale[seg])
        # ---- adjoint identity <A x, y> = <x, A^T y> at full size (covers the global column)
        Ax = torch.zeros(m, dtype=torch.float64, device="cuda")
        ATy = torch.zeros(n, dtype=torch.float64, device="cuda")
        g.gsr_aprod1(h, x, Ax)
        g.gsr_aprod2(h, y, ATy)
        lhs, rhs = float(Ax @ y), float(x @ ATy)
        assert abs(lhs - rhs) <= 1e-11 * float(Ax.norm() * y.norm())
        del Ax, ATy, yd, y0, xd, x0
        # ---- LSQR in bench.py's configuration: estimates against directly computed norms
        xt = inputs.x_true(cfg, "cuda")
        b = torch.empty(m, dtype=torch.float64, device="cuda")
        for r0 in range(0, m, GEN_ROWS):
            nr = min(GEN_ROWS, m - r0)
            b[r0:r0 + nr] = inputs.noise(cfg, r0, nr, "cuda")
        g.gsr_aprod1(h, xt, b)                       # b = A x_true + noise, before scaling
        res0 = b.clone()
        p = torch.empty(n, dtype=torch.float64, device="cuda")
        g.gsr_precondition(h, p)
        g.gsr_set_option(h, g.GSR_OPT_FORCE_ITNLIM, 1)
        xs = torch.empty(n, dtype=torch.float64, device="cuda")
        K = 12
        r = g.gsr_lsqr_solve(h, b, xs, K)
        assert (r.istop, r.itn) == (7, K)
        z = xs / p                                   # iterate of the scaled system
        neg = -z
        g.gsr_aprod1(h, neg, res0)                   # res0 = b - A' z
        rn = float(res0.norm())
        assert abs(r.rnorm - rn) <= 1e-8 * rn
        assert abs(r.xnorm - float(z.norm())) <= 1e-8 * float(z.norm())
        assert abs(r.bnorm - float(b.norm())) <= 1e-12 * float(b.norm())
        at_r = torch.zeros(n, dtype=torch.float64, device="cuda")
        g.gsr_aprod2(h, res0, at_r)
        assert abs(r.arnorm - float(at_r.norm())) <= 1e-6 * r.anorm * r.rnorm
        r2 = g.gsr_lsqr_solve(h, b, xs, K + 6)
        assert r2.rnorm <= r.rnorm * (1 + 1e-12)
    finally:
        g.gsr_matrix_destroy(h)
        torch.cuda.empty_cache()


def _build_with_host_copy(cfg, g):
    """Chunked device-side generation and ingest, keeping the caller-form arrays on the host
    (22 GB at 1e8 rows, 67 GB at 3e8) so that the oracle can run the SAME system whole."""
    dev = "cuda"
    m = cfg.n_rows
    sptr = inputs.star_ptr(cfg)
    scales = inputs.col_scales(cfg, dev)
    star_h = np.empty(m, dtype=np.int32)
    att_h = np.empty(m, dtype=np.int32)
    instr_h = np.empty((m, 6), dtype=np.int32)
    vals_h = np.empty((m, 24), dtype=np.float64)
    h = g.gsr_matrix_begin(cfg.n_rows, cfg.n_stars, cfg.n_dfa, cfg.n_instr)
    for r0 in range(0, m, GEN_ROWS):
        nr = min(GEN_ROWS, m - r0)
        star, att, instr, vals = inputs.gen_rows(cfg, r0, nr, dev, sptr=sptr, scales=scales)
        g.gsr_matrix_append_rows(h, r0, nr, star, att, instr, vals)
        star_h[r0:r0 + nr] = star.cpu().numpy()
        att_h[r0:r0 + nr] = att.cpu().numpy()
        instr_h[r0:r0 + nr] = instr.cpu().numpy()
        vals_h[r0:r0 + nr] = vals.cpu().numpy()
        del star, att, instr, vals
    g.gsr_matrix_finalize(h)
    return h, star_h, att_h, instr_h, vals_h


def _host_ram_gb():
    with open("/proc/meminfo") as f:
        for line in f:
            if line.startswith("MemAvailable:"):
                return int(line.split()[1]) / 1e6
    return 0.0


# north_star: "the GPU LSQR matches the oracle within the stated tolerances on all five configs".
# The whole system goes to the host and the oracle (OpenMP timing build, itself checked against
# the serial definition in tests/test_oracle_omp.py) runs the same K = 10 fixed-count solve:
# x and the scaled iterate z = x / p to 1e-9 in the 2-norm (x spans 8 decades at
# cfg4), identical istop, and -- through gsr_debug_fused_pass -- the kernels of the timed loop
# element-wise against the oracle's two products, the instrumental block of A^T u with the
# fixed-point accumulator (reading A22: 1.8e5 terms per column at cfg3) and with fp64 atomics.
@pytest.mark.parametrize("name,gb,ram", [("cfg2", 40, 40), ("cfg4", 40, 40), ("cfg3", 110, 110)])
def test_fullsize_lsqr_matches_oracle(name, gb, ram):
    from paper_2212_11675_b200 import binding as g
    _need_gb(gb)
    if _host_ram_gb() < ram:
        pytest.skip(f"needs {ram} GB of host memory for the oracle's copy of the system")
    cfg = inputs.named_config(name)
    m, n = cfg.n_rows, cfg.n_cols
    h, star_h, att_h, instr_h, vals_h = _build_with_host_copy(cfg, g)
    try:
        o = OracleSystem(cfg.n_stars, cfg.n_dfa, cfg.n_instr, star_h, att_h, instr_h, vals_h,
                         omp=True, copy_values=False)
        # b = A x_true + noise by the caller's own aprod1 (reading A17), shared bit for bit
        xt = inputs.x_true(cfg, "cuda")
        b = torch.empty(m, dtype=torch.float64, device="cuda")
        for r0 in range(0, m, GEN_ROWS):
            nr = min(GEN_ROWS, m - r0)
            b[r0:r0 + nr] = inputs.noise(cfg, r0, nr, "cuda")
        g.gsr_aprod1(h, xt, b)
        b_h = b.cpu().numpy()
        p_o = o.precondition()
        p = torch.empty(n, dtype=torch.float64, device="cuda")
        g.gsr_precondition(h, p)
        assert np.allclose(p.cpu().numpy(), p_o, rtol=1e-12, atol=0)
        # ---- one fused pass, element-wise: y = A' x + ca y0 and t = A'^T y
        x = inputs.random_vector(cfg, 1, n, "cuda")
        y0 = inputs.random_vector(cfg, 3, m, "cuda")
        ca = -0.37
        y_ref, ysc = o.aprod1(x.cpu().numpy(), ca * y0.cpu().numpy(), want_scale=True)
        t_ref, tsc = o.aprod2(y_ref, np.zeros(n), want_scale=True)
        worst = {}
        for fixed in (1, 0):
            g.gsr_set_option(h, g.GSR_OPT_FIXED_POINT, fixed)
            yd = y0.clone()
            td = torch.zeros(n, dtype=torch.float64, device="cuda")
            g.gsr_debug_fused_pass(h, x, ca, yd, td)
            ey = np.abs(yd.cpu().numpy() - y_ref) / ysc
            assert ey.max() <= 1e-12, ("u_hat", fixed, float(ey.max()))
            et = np.abs(td.cpu().numpy() - t_ref)
            blocks = {"astro": slice(0, cfg.off_att), "att": slice(cfg.off_att, cfg.off_instr),
                      "instr": slice(cfg.off_instr, cfg.off_instr + cfg.n_instr), "glob": slice(n - 1, n)}
            for bk, sl in blocks.items():
                rel = float((et[sl] / np.maximum(tsc[sl], 1e-300)).max())
                worst[(bk, fixed)] = rel
                if bk == "instr" and fixed:
                    # reading A22: normwise bound n_j 2^-62 ||u|| per column (here against the
                    # column's own scale, which is the stricter, reported figure)
                    ynorm = float(np.linalg.norm(y_ref))
                    assert np.all(et[sl] <= m * 2.0 ** -62 * ynorm + 1e-12 * tsc[sl]), rel
                else:
                    assert rel <= 1e-12, (bk, fixed, rel)
            del yd, td
        print(f"\n[{name}] fused pass vs oracle, max |err|/scale per block (fixed point, fp64 atomics): "
              + ", ".join(f"{bk} {worst[(bk, 1)]:.1e}/{worst[(bk, 0)]:.1e}" for bk in ("astro", "att", "instr", "glob")))
        g.gsr_set_option(h, g.GSR_OPT_FIXED_POINT, 1)
        # ---- K = 10 fixed-count LSQR against the oracle
        K = 10
        g.gsr_set_option(h, g.GSR_OPT_FORCE_ITNLIM, 1)
        xs = torch.empty(n, dtype=torch.float64, device="cuda")
        r = g.gsr_lsqr_solve(h, b, xs, K)
        ro = o.lsqr(b_h, K, force_itnlim=True)
        assert (r.istop, r.itn) == (ro.istop, ro.itn) == (7, K)
        xg = xs.cpu().numpy()
        ex = float(np.linalg.norm(xg - ro.x) / np.linalg.norm(ro.x))
        zg, zo = xg / p_o, ro.x / p_o
        ez = float(np.linalg.norm(zg - zo) / np.linalg.norm(zo))
        print(f"[{name}] K={K}: |x-x_orc|/|x_orc| = {ex:.2e}, |z-z_orc|/|z_orc| = {ez:.2e}, "
              f"rnorm {r.rnorm:.12e} vs {ro.rnorm:.12e}")
        assert ex <= 1e-9 and ez <= 1e-9, (ex, ez)
        for f in ("rnorm", "xnorm", "anorm", "acond", "bnorm"):
            assert abs(getattr(r, f) - getattr(ro, f)) <= 1e-9 * abs(getattr(ro, f)), f
    finally:
        g.gsr_matrix_destroy(h)
        torch.cuda.empty_cache()


# ---- opt-in (GSR_FULLSIZE_SLOW=1): the configs' OWN iteration counts ------------------------
# BASELINE.json names 100 / 50 / 100 iterations for configs 2 / 3 / 4.  The oracle needs minutes
# per config for that (16 host cores), too long for the default GPU leg, so this test runs only
# when asked for; its printed table is kept as profiles/r3_fullsize_parity.md with the command.
# Same bars as the small cases (tests/test_gpu_parity.py): x and z = x/p within 1e-9 in the
# relative 2-norm wherever the oracle itself is that stable under a one-ulp change of b (reading
# A20), else 20 x the oracle's own sensitivity, never above 1e-4; identical istop; the natural
# stop rule and its iteration compared as recorded in fixed-count mode.  At cfg2 size the OpenMP
# timing build that serves as the full-size checker is also tied to the SERIAL definition
# (products to 1e-13 of the term scale, a K = 3 solve to 1e-13 in the 2-norm).
CONFIG_ITERS = {"cfg2": 100, "cfg3": 50, "cfg4": 100}


@pytest.mark.parametrize("name,gb,ram", [("cfg2", 40, 60), ("cfg4", 40, 40), ("cfg3", 110, 110)])
def test_fullsize_lsqr_at_the_configs_iteration_counts(name, gb, ram):
    import json
    import os
    import time
    if os.environ.get("GSR_FULLSIZE_SLOW") != "1":
        pytest.skip("opt-in: GSR_FULLSIZE_SLOW=1 (minutes of oracle time per config)")
    from paper_2212_11675_b200 import binding as g
    _need_gb(gb)
    if _host_ram_gb() < ram:
        pytest.skip(f"needs {ram} GB of host memory for the oracle's copy of the system")
    cfg = inputs.named_config(name)
    m, n, K = cfg.n_rows, cfg.n_cols, CONFIG_ITERS[name]
    row = {"config": name, "rows": m, "cols": n, "K": K}
    h, star_h, att_h, instr_h, vals_h = _build_with_host_copy(cfg, g)
    try:
        o = OracleSystem(cfg.n_stars, cfg.n_dfa, cfg.n_instr, star_h, att_h, instr_h, vals_h,
                         omp=True, copy_values=False)
        xt = inputs.x_true(cfg, "cuda")
        b = torch.empty(m, dtype=torch.float64, device="cuda")
        for r0 in range(0, m, GEN_ROWS):
            nr = min(GEN_ROWS, m - r0)
            b[r0:r0 + nr] = inputs.noise(cfg, r0, nr, "cuda")
        g.gsr_aprod1(h, xt, b)
        b_h = b.cpu().numpy()
        if name == "cfg2":
            # the checker against the serial definition at full size, on the UNSCALED system
            # (a second copy of the values: the serial object scales its own)
            os_ = OracleSystem(cfg.n_stars, cfg.n_dfa, cfg.n_instr, star_h, att_h, instr_h, vals_h, omp=False)
            xv = inputs.random_vector(cfg, 1, n).numpy()
            yv = inputs.random_vector(cfg, 3, m).numpy()
            t0 = time.perf_counter()
            y_s, ysc = os_.aprod1(xv, 0.5 * yv, want_scale=True)
            y_p = o.aprod1(xv, 0.5 * yv)
            e1 = float((np.abs(y_s - y_p) / ysc).max())
            x_s, xsc = os_.aprod2(yv, np.zeros(n), want_scale=True)
            x_p = o.aprod2(yv, np.zeros(n))
            e2 = float((np.abs(x_s - x_p) / np.maximum(xsc, 1e-300)).max())
            p_s = os_.precondition()
            rs = os_.lsqr(b_h, 3, force_itnlim=True)
            row["serial_vs_omp"] = {"aprod1": e1, "aprod2": e2}
            assert e1 <= 1e-13 and e2 <= 1e-13, (e1, e2)
        p_o = o.precondition()
        if name == "cfg2":
            rp = o.lsqr(b_h, 3, force_itnlim=True)
            e3 = float(np.linalg.norm(rs.x - rp.x) / np.linalg.norm(rs.x))
            row["serial_vs_omp"].update({"p": float(np.abs(p_s / p_o - 1).max()), "lsqr_k3_x": e3,
                                         "seconds": time.perf_counter() - t0})
            assert np.allclose(p_s, p_o, rtol=1e-13, atol=0) and e3 <= 1e-13, e3
            del os_, rs, rp, y_s, y_p, x_s, x_p
        g.gsr_precondition(h)
        g.gsr_set_option(h, g.GSR_OPT_FORCE_ITNLIM, 1)
        xs = torch.empty(n, dtype=torch.float64, device="cuda")
        r = g.gsr_lsqr_solve(h, b, xs, K)
        t0 = time.perf_counter()
        ro = o.lsqr(b_h, K, force_itnlim=True)
        row["oracle_seconds"] = time.perf_counter() - t0
        xg = xs.cpu().numpy()
        ex = float(np.linalg.norm(xg - ro.x) / np.linalg.norm(ro.x))
        ez = float(np.linalg.norm(xg / p_o - ro.x / p_o) / np.linalg.norm(ro.x / p_o))
        tol, sens = 1e-9, None
        if max(ex, ez) > 1e-9:     # reading A20: how far does the oracle itself move under one ulp of b?
            rng = np.random.default_rng(0)
            ru = o.lsqr(b_h + np.spacing(b_h) * rng.integers(-1, 2, b_h.shape), K, force_itnlim=True)
            sens = float(np.linalg.norm(ru.x - ro.x) / np.linalg.norm(ro.x))
            tol = min(max(1e-9, 20.0 * sens), 1e-4)
        # a second GPU solve of the same system: what the order of the atomics alone moves
        xs2 = torch.empty(n, dtype=torch.float64, device="cuda")
        g.gsr_lsqr_solve(h, b, xs2, K)
        row.update({"x_rel": ex, "z_rel": ez, "tol": tol, "oracle_one_ulp_sensitivity": sens,
                    "gpu_run_to_run": float((xs2 - xs).norm() / xs.norm()),
                    "istop": [r.istop, ro.istop], "itn": [r.itn, ro.itn],
                    "istop_natural": [r.istop_natural, ro.istop_natural],
                    "itn_natural": [r.itn_natural, ro.itn_natural],
                    "rnorm": [r.rnorm, ro.rnorm], "anorm": [r.anorm, ro.anorm], "acond": [r.acond, ro.acond]})
        print(f"\n[{name}] K={K}: " + json.dumps(row))
        os.makedirs("gpurun_out", exist_ok=True)
        with open("gpurun_out/r3_fullsize_parity.jsonl", "a") as f:
            f.write(json.dumps(row) + "\n")
        assert (r.istop, r.itn) == (ro.istop, ro.itn) == (7, K)
        assert ex <= tol and ez <= tol, (ex, ez, tol, sens)
        assert r.istop_natural == ro.istop_natural
        assert abs(r.itn_natural - ro.itn_natural) <= 1
        assert abs(r.rnorm - ro.rnorm) <= tol * ro.rnorm
    finally:
        g.gsr_matrix_destroy(h)
        torch.cuda.empty_cache()
