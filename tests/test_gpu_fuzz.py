"""Seeded random small systems through the C ABI against the oracle: odd shapes the named
configs do not reach (D = 4, I = 1, empty stars, stars spanning many tiles, thousands of fine
attitude bins with a handful of rows each, I just below / above the private-accumulator limit,
hot attitude windows, badly scaled columns), both iteration forms."""
import numpy as np
import pytest
import torch

from paper_2212_11675_b200 import inputs

pytestmark = pytest.mark.gpu


def _case(rng, it):
    S = int(rng.integers(1, 60))
    counts = rng.integers(0, int(rng.choice([3, 40, 400, 5000])), S)
    if counts.sum() == 0:
        counts[0] = 1
    D = int(rng.choice([4, 5, 7, 64, 300, 1000, 5000, 40000]))
    I = int(rng.choice([1, 2, 6, 60, 700, 768, 769, 3000, 12000]))
    hot = (0.9, 0.4, 0.45) if rng.random() < 0.3 else None
    return inputs.micro_config(f"fuzz{it}", int(rng.integers(1, 1 << 30)), counts, D, I, att_hot=hot,
                               col_scales=bool(rng.random() < 0.3),
                               att_time_ordered=bool(rng.random() < 0.3))   # time-ordered scans (row f4)


@pytest.mark.parametrize("seed", [11, 12, 13])
def test_random_small_systems(seed):
    from oracle import gsr_oracle
    from paper_2212_11675_b200 import binding as g
    rng = np.random.default_rng(seed)
    for it in range(8):
        cfg = _case(rng, it)
        star, att, instr, vals = inputs.gen_all(cfg)
        o = gsr_oracle.from_torch(cfg, star, att, instr, vals)
        A = g.GsrMatrix.create(cfg, star.cuda(), att.cuda(), instr.cuda(), vals.cuda())
        try:
            tag = (seed, it, cfg.n_rows, cfg.n_stars, cfg.n_dfa, cfg.n_instr)
            x = inputs.random_vector(cfg, 1, cfg.n_cols)
            y = inputs.random_vector(cfg, 2, cfg.n_rows)
            y0 = inputs.random_vector(cfg, 3, cfg.n_rows)     # products accumulate
            x0 = inputs.random_vector(cfg, 4, cfg.n_cols)
            yd, xd = y0.cuda(), x0.cuda()
            g.gsr_aprod1(A.h, x.cuda(), yd)
            g.gsr_aprod2(A.h, y.cuda(), xd)
            yr, s1 = o.aprod1(x.numpy(), y0.numpy(), want_scale=True)
            xr, s2 = o.aprod2(y.numpy(), x0.numpy(), want_scale=True)
            assert np.all(np.abs(yd.cpu().numpy() - yr) <= 1e-12 * s1), tag
            assert np.all(np.abs(xd.cpu().numpy() - xr) <= 1e-12 * s2), tag
            b = o.aprod1(inputs.x_true(cfg).numpy(), inputs.noise(cfg, 0, cfg.n_rows).numpy())
            o.precondition()
            g.gsr_precondition(A.h)
            g.gsr_set_option(A.h, g.GSR_OPT_FORCE_ITNLIM, 1)
            ro = o.lsqr(b, 3, force_itnlim=True)
            for fused in (1, 0):
                g.gsr_set_option(A.h, g.GSR_OPT_FUSED, fused)
                xs = torch.empty(cfg.n_cols, dtype=torch.float64, device="cuda")
                r = g.gsr_lsqr_solve(A.h, torch.from_numpy(b).cuda(), xs, 3)
                assert (r.istop, r.itn) == (ro.istop, ro.itn), tag
                assert np.linalg.norm(xs.cpu().numpy() - ro.x) <= 1e-9 * np.linalg.norm(ro.x), tag
        finally:
            A.close()
