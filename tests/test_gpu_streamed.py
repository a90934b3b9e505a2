"""Row f4(iii): out-of-core systems (gsr_matrix_begin_streamed).  The tiled
matrix lives partly in pinned host memory and is streamed through two device buffers on every
pass.  A streamed handle must reproduce a resident handle of the same system -- the layout bit
for bit, aprod1 bit for bit (no atomics), everything else up to the order of floating-point
atomic adds -- and the oracle to the usual tolerances."""
import numpy as np
import pytest
import torch

from paper_2212_11675_b200 import inputs
from tests.helpers import make_oracle

pytestmark = pytest.mark.gpu
TILE_BYTES = 6784


def _g():
    from paper_2212_11675_b200 import binding
    return binding


def _build(g, cfg, arrays, resident_bytes=None, chunk_bytes=0, pieces=1):
    star, att, instr, vals = arrays
    if resident_bytes is None:
        h = g.gsr_matrix_begin(cfg.n_rows, cfg.n_stars, cfg.n_dfa, cfg.n_instr)
    else:
        h = g.gsr_matrix_begin_streamed(cfg.n_rows, cfg.n_stars, cfg.n_dfa, cfg.n_instr,
                                        resident_bytes, chunk_bytes)
    m = cfg.n_rows
    step = (m + pieces - 1) // pieces
    for r0 in range(0, m, step):
        r1 = min(r0 + step, m)
        g.gsr_matrix_append_rows(h, r0, r1 - r0, star[r0:r1].contiguous(), att[r0:r1].contiguous(),
                                 instr[r0:r1].contiguous(), vals[r0:r1].contiguous())
    g.gsr_matrix_finalize(h)
    return h


CASES = {
    # cfg1: 2e5 rows = 6 300 tiles = 43 MB; a third on the device, chunks of 256 tiles (the minimum)
    "cfg1_third": ("cfg1", 14 << 20, 0),
    # nothing resident: every tile comes from the host, chunks of 4 MB
    "cfg1_none": ("cfg1", 0, 4 << 20),
    # a boundary in the middle of a unit (not a multiple of the tile size either)
    "cfg1_odd": ("cfg1", 10_000_003, 3_000_001),
    "skew_hot": ("skew_hot", 3 << 20, 0),
}


def _cfg(name):
    if name == "skew_hot":
        return inputs.GsrConfig("cfg4s", 3, 400, 400, 60, n_rows_total=50_000,
                                powerlaw=(10, 10_000, 1.36), att_hot=(0.9, 0.40, 0.45), col_scales=True)
    return inputs.named_config(name)


@pytest.mark.parametrize("case", list(CASES))
def test_streamed_handle_equals_resident_handle_and_oracle(case):
    g = _g()
    name, resident, chunk = CASES[case]
    cfg = _cfg(name)
    host = inputs.gen_all(cfg)
    dev = [t.cuda() for t in host]
    o = make_oracle(cfg, *[t.numpy() for t in host])
    m, n = cfg.n_rows, cfg.n_cols
    hr = _build(g, cfg, dev)
    hs = _build(g, cfg, dev, resident, chunk, pieces=3)
    try:
        assert g.gsr_matrix_host_bytes(hr) == 0
        assert g.gsr_matrix_host_bytes(hs) > 0 and g.gsr_matrix_host_bytes(hs) % TILE_BYTES == 0
        assert g.gsr_matrix_device_bytes(hs) < g.gsr_matrix_device_bytes(hr) or resident > 20 << 20
        # layout: bit-exact against the oracle's index construction and the resident handle
        cs, vs = g.gsr_debug_expand_rows(hs, 0, m)
        cr, vr = g.gsr_debug_expand_rows(hr, 0, m)
        oc, ov = o.expand_rows()
        assert np.array_equal(cs, oc) and np.array_equal(vs, ov)
        assert np.array_equal(cs, cr) and np.array_equal(vs, vr)
        # aprod1: no atomics anywhere -> identical bits; against the oracle 1e-12 of the scale
        x = inputs.random_vector(cfg, 1, n).cuda()
        y0 = inputs.random_vector(cfg, 2, m)
        ys, yr = y0.cuda(), y0.cuda()
        before = g.gsr_matrix_streamed_bytes(hs)
        g.gsr_aprod1(hs, x, ys)
        g.gsr_aprod1(hr, x, yr)
        torch.cuda.synchronize()
        assert torch.equal(ys, yr)
        y_ref, ysc = o.aprod1(x.cpu().numpy(), y0.numpy().copy(), want_scale=True)
        assert np.all(np.abs(ys.cpu().numpy() - y_ref) <= 1e-12 * ysc)
        # one pass moved exactly the host part of the matrix across the bus, once
        moved = g.gsr_matrix_streamed_bytes(hs) - before
        assert 0 < moved <= g.gsr_matrix_host_bytes(hs)
        # aprod2 against the oracle
        y = inputs.random_vector(cfg, 3, m).cuda()
        x0 = inputs.random_vector(cfg, 4, n)
        xs = x0.cuda()
        g.gsr_aprod2(hs, y, xs)
        x_ref, xsc = o.aprod2(y.cpu().numpy(), x0.numpy().copy(), want_scale=True)
        assert np.all(np.abs(xs.cpu().numpy() - x_ref) <= 1e-12 * np.maximum(xsc, 1e-300))
        # preconditioner: p and the scaled values, written back to the host part
        rhs = o.aprod1(inputs.x_true(cfg).numpy(), inputs.noise(cfg, 0, m).numpy())
        p_ref = o.precondition()
        ps = torch.empty(n, dtype=torch.float64, device="cuda")
        g.gsr_precondition(hs, ps)
        g.gsr_precondition(hr)
        assert np.allclose(ps.cpu().numpy(), p_ref, rtol=1e-13, atol=0)
        _, vs = g.gsr_debug_expand_rows(hs, 0, m)
        assert np.allclose(vs, o.values, rtol=1e-13, atol=0)
        # PC-LSQR, fixed count and standard mode, against the oracle and the resident solve
        bd = torch.from_numpy(rhs).cuda()
        xs_ = torch.empty(n, dtype=torch.float64, device="cuda")
        xr_ = torch.empty(n, dtype=torch.float64, device="cuda")
        for h in (hs, hr):
            g.gsr_set_option(h, g.GSR_OPT_FORCE_ITNLIM, 1)
        for fused in (1, 0):
            g.gsr_set_option(hs, g.GSR_OPT_FUSED, fused)
            for k in (1, 20):
                before = g.gsr_matrix_streamed_bytes(hs)
                rs = g.gsr_lsqr_solve(hs, bd, xs_, k)
                moved = g.gsr_matrix_streamed_bytes(hs) - before
                rr = g.gsr_lsqr_solve(hr, bd, xr_, k)
                ro = o.lsqr(rhs, k, force_itnlim=True)
                assert (rs.istop, rs.itn) == (ro.istop, ro.itn) == (7, k)
                xg = xs_.cpu().numpy()
                assert np.linalg.norm(xg - ro.x) <= 1e-9 * np.linalg.norm(ro.x)
                assert np.linalg.norm(xg / p_ref - ro.x / p_ref) <= 1e-9 * np.linalg.norm(ro.x / p_ref)
                assert np.linalg.norm(xg - xr_.cpu().numpy()) <= 1e-11 * np.linalg.norm(ro.x)
                for f in ("rnorm", "xnorm", "anorm", "acond"):
                    assert abs(getattr(rs, f) - getattr(ro, f)) <= 1e-9 * abs(getattr(ro, f)), f
                # the host part crosses the bus once per fused iteration (+ once for the initial
                # aprod2), twice per two-pass iteration
                per_pass = g.gsr_matrix_host_bytes(hs)
                passes = (k if fused else 2 * k) + 1
                assert moved <= passes * per_pass and moved > (passes - 1) * per_pass * 0.5
        g.gsr_set_option(hs, g.GSR_OPT_FUSED, 1)
        g.gsr_set_option(hs, g.GSR_OPT_FORCE_ITNLIM, 0)
        rs = g.gsr_lsqr_solve(hs, bd, xs_, 500, 1e-10, 1e-10, 1e8)
        ro = o.lsqr(rhs, 500, 1e-10, 1e-10, 1e8)
        assert rs.istop == ro.istop and abs(rs.itn - ro.itn) <= 1
        assert np.linalg.norm(xs_.cpu().numpy() - ro.x) <= 1e-9 * np.linalg.norm(ro.x)
        # options the streamed form does not take
        g.gsr_set_option(hs, g.GSR_OPT_DETERMINISTIC, 1)
        with pytest.raises(g.GsrError) as ei:
            g.gsr_lsqr_solve(hs, bd, xs_, 3)
        assert ei.value.code == g.GSR_EUNSUPPORTED
    finally:
        g.gsr_matrix_destroy(hs)
        g.gsr_matrix_destroy(hr)


def test_streamed_budget_that_covers_everything_is_a_resident_handle():
    g = _g()
    cfg = inputs.scaled(inputs.named_config("cfg1"), 10, "cfg1/10")
    dev = [t.cuda() for t in inputs.gen_all(cfg)]
    h = _build(g, cfg, dev, 1 << 30, 1 << 20)
    try:
        assert g.gsr_matrix_host_bytes(h) == 0 and g.gsr_matrix_streamed_bytes(h) == 0
    finally:
        g.gsr_matrix_destroy(h)
    with pytest.raises(g.GsrError) as ei:
        g.gsr_matrix_begin_streamed(cfg.n_rows, cfg.n_stars, cfg.n_dfa, cfg.n_instr, -1, 0)
    assert ei.value.code == g.GSR_EINVAL


def test_streamed_multi_segment_ingest_matches_resident_solve():
    """More than one ingest segment (2^22 rows each) on the streamed path: 1.2e7 rows of the
    config-5 structure, a quarter of the tiles resident, 64 MB chunks; K = 10 against the
    resident handle of the same system (which test_gpu_fullsize.py ties to the oracle)."""
    g = _g()
    cfg = inputs.named_config("cfg5_12000000")
    m, n = cfg.n_rows, cfg.n_cols
    handles = []
    try:
        for resident in (None, 640 << 20):
            sptr = inputs.star_ptr(cfg)
            h = (g.gsr_matrix_begin(m, cfg.n_stars, cfg.n_dfa, cfg.n_instr) if resident is None else
                 g.gsr_matrix_begin_streamed(m, cfg.n_stars, cfg.n_dfa, cfg.n_instr, resident, 64 << 20))
            handles.append(h)
            for r0 in range(0, m, 1 << 22):
                nr = min(1 << 22, m - r0)
                star, att, instr, vals = inputs.gen_rows(cfg, r0, nr, "cuda", sptr=sptr)
                g.gsr_matrix_append_rows(h, r0, nr, star, att, instr, vals)
            g.gsr_matrix_finalize(h)
        hr, hs = handles
        assert g.gsr_matrix_host_bytes(hs) > 1.5e9
        xt = inputs.x_true(cfg, "cuda")
        b = inputs.noise(cfg, 0, 1 << 20, "cuda").repeat((m + (1 << 20) - 1) >> 20)[:m].contiguous()
        bs = b.clone()
        g.gsr_aprod1(hr, xt, b)
        g.gsr_aprod1(hs, xt, bs)
        assert torch.equal(b, bs)
        pr = torch.empty(n, dtype=torch.float64, device="cuda")
        ps = torch.empty(n, dtype=torch.float64, device="cuda")
        g.gsr_precondition(hr, pr)
        g.gsr_precondition(hs, ps)
        assert torch.allclose(pr, ps, rtol=1e-13, atol=0)
        xr = torch.empty(n, dtype=torch.float64, device="cuda")
        xs = torch.empty(n, dtype=torch.float64, device="cuda")
        for h in handles:
            g.gsr_set_option(h, g.GSR_OPT_FORCE_ITNLIM, 1)
        rr = g.gsr_lsqr_solve(hr, b, xr, 10)
        rs = g.gsr_lsqr_solve(hs, b, xs, 10)
        assert (rs.istop, rs.itn) == (rr.istop, rr.itn) == (7, 10)
        assert float((xs - xr).norm() / xr.norm()) <= 1e-11
        assert abs(rs.rnorm - rr.rnorm) <= 1e-11 * rr.rnorm
    finally:
        for h in handles:
            g.gsr_matrix_destroy(h)
        torch.cuda.empty_cache()
