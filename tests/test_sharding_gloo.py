"""Multi-rank row sharding: host logic of
paper_2212_11675_b200/sharding.py and the sharded PC-LSQR recurrences on two gloo ranks (CPU).

Each rank holds a star-aligned row block as an ordinary local system (oracle products on the
shard), the astrometric slice of every n-vector is distributed, the attitude + instrumental +
global slice is replicated and summed with all_reduce after every aprod2, and the norms are
all-reduced scalars.  The result must equal the single-process oracle LSQR.
"""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2212_11675_b200 import inputs, sharding
from tests.helpers import make_oracle


def _cfg():
    # 37 stars with uneven row counts (one empty star), 3 x 40 knots, 25 instrumental columns
    counts = [30, 7, 0, 55, 12, 41, 9, 23] * 4 + [17, 64, 5, 33, 21]
    return inputs.micro_config("shard", 11, counts, 40, 25)


def test_shard_rows_partition_is_star_aligned_and_balanced():
    cfg = _cfg()
    sptr = inputs.star_ptr(cfg).numpy()
    for world in (1, 2, 3, 5, 8):
        sh = sharding.shard_rows(sptr, world, cfg.n_dfa, cfg.n_instr)
        assert len(sh) == world
        assert sh[0].star0 == 0 and sh[-1].star1 == cfg.n_stars
        assert sh[0].row0 == 0 and sh[-1].row1 == cfg.n_rows
        for a, b in zip(sh[:-1], sh[1:]):
            assert a.star1 == b.star0 and a.row1 == b.row0
        for s in sh:
            assert s.row0 == sptr[s.star0] and s.row1 == sptr[s.star1]      # star aligned
            assert s.n_cols_local == 5 * s.n_stars_local + 3 * cfg.n_dfa + cfg.n_instr + 1
        ideal = cfg.n_rows / world
        biggest_star = int(np.diff(sptr).max())
        assert max(s.n_rows_local for s in sh) <= ideal + biggest_star      # balanced by rows


def test_scatter_gather_roundtrip():
    cfg = _cfg()
    sptr = inputs.star_ptr(cfg).numpy()
    sh = sharding.shard_rows(sptr, 3, cfg.n_dfa, cfg.n_instr)
    x = np.arange(cfg.n_cols, dtype=np.float64)
    loc = [sharding.scatter_x(x, s) for s in sh]
    assert all(len(v) == s.n_cols_local for v, s in zip(loc, sh))
    assert np.array_equal(sharding.gather_x(loc, sh), x)


def _allsum(a):
    t = torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64).reshape(-1).copy())
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return t.numpy().reshape(np.shape(a))


def _con_rows(cfg, n_con=4, nnz=9, seed=7):
    """Constraint rows (row f3) on the replicated slice only -- attitude, instrumental and global
    columns -- in GLOBAL column numbering: (row_ptr, col, val)."""
    rng = np.random.default_rng(seed)
    rep0 = 5 * cfg.n_stars
    ptr, col, val = [0], [], []
    for _ in range(n_con):
        c = np.sort(rng.choice(cfg.n_cols - rep0, nnz, replace=False)) + rep0
        col.extend(c.tolist())
        val.extend(rng.standard_normal(nnz).tolist())
        ptr.append(len(col))
    return np.array(ptr, dtype=np.int64), np.array(col, dtype=np.int32), np.array(val)


def _sharded_lsqr(rank, world, port, k_fixed, fused, out, with_con=False):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        cfg = _cfg()
        star, att, instr, vals = [t.numpy() for t in inputs.gen_all(cfg)]
        sptr = inputs.star_ptr(cfg).numpy()
        sh = sharding.shard_rows(sptr, world, cfg.n_dfa, cfg.n_instr)[rank]
        rows = slice(sh.row0, sh.row1)
        from oracle.gsr_oracle import OracleSystem
        o = OracleSystem(max(sh.n_stars_local, 1), cfg.n_dfa, cfg.n_instr,
                         sharding.local_star_idx(star, sh), att[rows], instr[rows], vals[rows])
        nl, ro = o.n, 5 * max(sh.n_stars_local, 1)         # local columns, replicated offset
        xt = inputs.x_true(cfg).numpy()
        xt_loc = np.concatenate([xt[sh.astro_offset_global:sh.astro_offset_global + 5 * sh.n_stars_local],
                                 np.zeros(ro - 5 * sh.n_stars_local), xt[sh.replicated_offset_global:]])
        noise = inputs.noise(cfg, 0, cfg.n_rows).numpy()[rows]
        if with_con and rank == 0:
            # rank 0 owns every constraint row (local numbering: replicated columns shift by the
            # difference of the two astrometric blocks); its m-vectors get n_con more entries
            ptr, col, val = _con_rows(cfg)
            o.set_constraints(ptr, (col - 5 * cfg.n_stars + ro).astype(np.int32), val)
            noise = np.concatenate([noise, np.zeros(len(ptr) - 1)])
        b = o.aprod1(xt_loc, noise)
        # preconditioner: column sums of squares, replicated slice summed over the ranks
        q = o.colsumsq()
        q[ro:] = _allsum(q[ro:])
        p = np.where(q > 0, 1.0 / np.sqrt(np.where(q > 0, q, 1.0)), 1.0)
        cols, _ = o.expand_rows()
        o.values[:] = o.values * p[cols]
        if o.n_con:
            o.con_val[:] = o.con_val * p[o.con_col]

        def norm2(v_loc):        # distributed slice summed over ranks + replicated slice once
            return float(_allsum(np.array([np.dot(v_loc[:ro], v_loc[:ro])]))[0] + np.dot(v_loc[ro:], v_loc[ro:]))

        def aprod2_sharded(u, v):   # v = A^T u + v ; replicated part of the old v counted once
            if rank != 0:
                v = v.copy()
                v[ro:] = 0.0
            v = o.aprod2(u, v)
            v[ro:] = _allsum(v[ro:])
            return v

        hyp = lambda a, c: np.sqrt(a * a + c * c)
        x = np.zeros(nl)
        u = b.copy()
        beta = np.sqrt(float(_allsum(np.array([np.dot(u, u)]))[0]))
        u /= beta
        v = aprod2_sharded(u, np.zeros(nl))
        alpha = np.sqrt(norm2(v))
        v /= alpha
        w = v.copy()
        rhobar, phibar = alpha, beta
        for _ in range(k_fixed):
            u = o.aprod1(v, -alpha * u)
            beta = np.sqrt(float(_allsum(np.array([np.dot(u, u)]))[0]))
            if fused:
                # the CUDA path's form: t = A^T u_hat with u_hat unnormalised,
                # replicated slice of t summed over the ranks, then v = t/beta - beta v everywhere
                t = o.aprod2(u, np.zeros(nl))
                t[ro:] = _allsum(t[ro:])
                v = t / beta - beta * v
                u /= beta
            else:
                u /= beta
                v = aprod2_sharded(u, -beta * v)
            alpha = np.sqrt(norm2(v))
            v /= alpha
            rho = hyp(rhobar, beta)
            cs, sn = rhobar / rho, beta / rho
            theta, rhobar = sn * alpha, -cs * alpha
            phi, phibar = cs * phibar, sn * phibar
            x = x + (phi / rho) * w
            w = v + (-theta / rho) * w
        out[rank] = (sh, p * x, phibar)
    finally:
        dist.destroy_process_group()


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


@pytest.mark.timeout(300)
@pytest.mark.parametrize("fused,with_con", [(True, False), (False, False), (True, True)])
def test_sharded_lsqr_two_gloo_ranks_matches_single_process_oracle(fused, with_con):
    k = 12
    world = 2
    mgr = mp.get_context("spawn").Manager()
    out = mgr.dict()
    mp.spawn(_sharded_lsqr, args=(world, _free_port(), k, fused, out, with_con), nprocs=world, join=True)
    cfg = _cfg()
    star, att, instr, vals = [t.numpy() for t in inputs.gen_all(cfg)]
    o = make_oracle(cfg, star, att, instr, vals)
    noise = inputs.noise(cfg, 0, cfg.n_rows).numpy()
    if with_con:      # the same rows below the observations of the unsharded system
        ptr, col, val = _con_rows(cfg)
        o.set_constraints(ptr, col, val)
        noise = np.concatenate([noise, np.zeros(len(ptr) - 1)])
    b = o.aprod1(inputs.x_true(cfg).numpy(), noise)
    o.precondition()
    ref = o.lsqr(b, k, force_itnlim=True)
    shards = [out[r][0] for r in range(world)]
    xs = []
    for r in range(world):
        sh, xl, _ = out[r]
        ro = 5 * max(sh.n_stars_local, 1)
        xs.append(np.concatenate([xl[:5 * sh.n_stars_local], xl[ro:]]))
    # replicated slice identical on every rank (same all_reduce result, same recurrences)
    r0 = 5 * shards[0].n_stars_local
    r1 = 5 * shards[1].n_stars_local
    assert np.array_equal(xs[0][r0:], xs[1][r1:])
    x = sharding.gather_x(xs, shards)
    assert x.shape == ref.x.shape
    err = np.linalg.norm(x - ref.x) / np.linalg.norm(ref.x)
    assert err <= 1e-10, err
    assert abs(out[0][2] - ref.rnorm) <= 1e-10 * ref.rnorm
