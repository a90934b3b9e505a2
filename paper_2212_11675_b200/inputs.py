"""Seeded synthetic inputs for the Gaia AVU-GSR hot path.

This module serves BOTH the CUDA path and the CPU oracle and therefore holds none of the
method's arithmetic: no aprod, no norms, no LSQR.  It only draws the caller-form arrays the
paper calls M_i, I_c and A_d (section 3): per row the star number, the index
of the first attitude element, six instrumental column indices and 24 fp64 coefficients in
the order 5 | 12 | 6 | 1, plus plain random vectors (x_true, noise, probe vectors).  The
right-hand side b = A.x_true + noise is formed by the caller with its own aprod1.

Inputs stand in for the paper's simulated / confidential Gaia systems (PAPER.md:477-491,
648); shapes follow BASELINE.json's five configs.

Generation is chunked (CHUNK rows per torch.Generator seeded from (seed, stream, chunk)), so
any chunk-aligned row range can be produced independently on the host or on the GPU.  CPU
and CUDA torch generators produce different streams: an input set is "what the generator
produced on the device it ran on"; the other side always receives a bit-for-bit copy.
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace
from typing import Optional, Sequence

import torch

CHUNK = 1 << 20  # rows per independently seeded chunk

N_ASTRO, N_ATT_AXES, N_PAR_AXIS, N_INSTR_ROW, N_GLOB = 5, 3, 4, 6, 1
N_PAR = 24


@dataclass(frozen=True)
class GsrConfig:
    name: str
    seed: int
    n_stars: int
    n_dfa: int
    n_instr: int
    rows_per_star: int = 0            # >0: every star has exactly this many rows
    n_rows_total: int = 0             # used with powerlaw / explicit counts
    powerlaw: Optional[tuple] = None  # (lo, hi, exponent) truncated power law of rows per star
    counts: Optional[tuple] = None    # explicit rows per star (micro cases)
    att_hot: Optional[tuple] = None   # (frac_rows, win_lo_frac, win_hi_frac) concentrated knots
    col_scales: bool = False          # per-column scale 10^U(-4,4) (config 4)
    att_time_ordered: bool = False    # rows of a star in time order: att_start non-decreasing
                                      # inside every star (per generation chunk), as in real scans
    noise_sigma: float = 1e-3
    iterations: int = 0

    @property
    def n_rows(self) -> int:
        if self.counts is not None:
            return int(sum(self.counts))
        if self.rows_per_star > 0:
            return self.n_stars * self.rows_per_star
        return self.n_rows_total

    @property
    def n_cols(self) -> int:
        return 5 * self.n_stars + 3 * self.n_dfa + self.n_instr + 1

    @property
    def off_att(self) -> int:
        return 5 * self.n_stars

    @property
    def off_instr(self) -> int:
        return 5 * self.n_stars + 3 * self.n_dfa

    @property
    def off_glob(self) -> int:
        return 5 * self.n_stars + 3 * self.n_dfa + self.n_instr


def named_config(name: str) -> GsrConfig:
    """BASELINE.json configs 1-5 (readings A3, A11 of DESIGN.md)."""
    if name == "cfg1":
        return GsrConfig("cfg1", 0, 2_000, 1_000, 600, rows_per_star=100, iterations=200)
    if name == "cfg2":
        return GsrConfig("cfg2", 1, 100_000, 20_000, 6_000, rows_per_star=1000, iterations=100)
    if name == "cfg3":
        return GsrConfig("cfg3", 2, 300_000, 50_000, 10_000, rows_per_star=1000, iterations=50)
    if name == "cfg4":
        return GsrConfig("cfg4", 3, 200_000, 20_000, 60, n_rows_total=100_000_000,
                         powerlaw=(10, 10_000, 1.36), att_hot=(0.9, 0.40, 0.45),
                         col_scales=True, iterations=100)
    if name.startswith("cfg3x"):
        # K copies of config 3's star population over the same attitude and instrumental unknowns:
        # the out-of-core workload (row f4(iii)); K = 6 is the paper's 1.8e9-row production size
        k = int(name[5:])
        return GsrConfig(name, 2, 300_000 * k, 50_000, 10_000, rows_per_star=1000, iterations=50)
    if name.startswith("cfg5_"):
        m = int(float(name[5:]))
        assert m % 5000 == 0
        return GsrConfig(name, 4, m // 1000, max(m // 5000, 4), 600, rows_per_star=1000)
    raise KeyError(name)


def scaled(cfg: GsrConfig, factor: int, name: Optional[str] = None) -> GsrConfig:
    """Same structure with 1/factor of the stars, knots and instrumental columns (tests)."""
    return replace(cfg, name=name or f"{cfg.name}/{factor}",
                   n_stars=max(cfg.n_stars // factor, 1),
                   n_dfa=max(cfg.n_dfa // factor, 8),
                   n_instr=max(cfg.n_instr // factor, 8) if cfg.n_instr > 100 else cfg.n_instr,
                   n_rows_total=cfg.n_rows_total // factor if cfg.n_rows_total else 0)


def _mix(seed: int, stream: int, index: int) -> int:
    """splitmix64-style finaliser of (seed, stream, index) -> 63-bit generator seed."""
    z = (seed * 0x9E3779B97F4A7C15 + stream * 0xBF58476D1CE4E5B9 + index * 0x94D049BB133111EB
         + 0x2545F4914F6CDD1D) & 0xFFFFFFFFFFFFFFFF
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & 0xFFFFFFFFFFFFFFFF
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & 0xFFFFFFFFFFFFFFFF
    z = z ^ (z >> 31)
    return z & 0x7FFFFFFFFFFFFFFF


def _gen(device, seed: int, stream: int, index: int) -> torch.Generator:
    g = torch.Generator(device=device)
    g.manual_seed(_mix(seed, stream, index))
    return g


# stream ids
_S_COUNTS, _S_ATT, _S_INSTR, _S_VAL, _S_SCALE, _S_XTRUE, _S_NOISE, _S_VEC, _S_HOT = range(9)


def star_counts(cfg: GsrConfig) -> torch.Tensor:
    """Rows per star, int64 [S], host.  Deterministic in cfg.seed."""
    if cfg.counts is not None:
        return torch.tensor(cfg.counts, dtype=torch.int64)
    if cfg.rows_per_star > 0:
        return torch.full((cfg.n_stars,), cfg.rows_per_star, dtype=torch.int64)
    lo, hi, expo = cfg.powerlaw
    g = _gen("cpu", cfg.seed, _S_COUNTS, 0)
    u = torch.rand(cfg.n_stars, dtype=torch.float64, generator=g)
    # inverse CDF of p(c) ~ c^-expo on [lo, hi]
    a = 1.0 - expo
    c = (lo ** a + u * (hi ** a - lo ** a)) ** (1.0 / a)
    counts = c.floor().to(torch.int64).clamp_(lo, hi)
    # deterministic adjustment to the exact total: rescale, then spread the remainder
    target = cfg.n_rows_total
    counts = (counts.to(torch.float64) * (target / float(counts.sum()))).floor().to(torch.int64)
    counts.clamp_(min(lo, target // cfg.n_stars), hi)
    diff = int(target - counts.sum())
    step = 1 if diff > 0 else -1
    idx = 0
    S = cfg.n_stars
    while diff != 0:
        take = min(abs(diff), S)
        sel = (torch.arange(take) + idx) % S
        ok = (counts[sel] + step >= 1)
        counts[sel[ok]] += step
        diff -= step * int(ok.sum())
        idx = (idx + take) % S
    return counts


def star_ptr(cfg: GsrConfig) -> torch.Tensor:
    """int64 [S+1] first row of each star (rows are grouped by star)."""
    c = star_counts(cfg)
    p = torch.zeros(cfg.n_stars + 1, dtype=torch.int64)
    torch.cumsum(c, 0, out=p[1:])
    return p


def col_scales(cfg: GsrConfig, device="cpu") -> Optional[torch.Tensor]:
    """Per-column scale s_j = 10^U(-4,4) (config 4), float64 [n]; None when unused."""
    if not cfg.col_scales:
        return None
    g = _gen("cpu", cfg.seed, _S_SCALE, 0)
    e = torch.rand(cfg.n_cols, dtype=torch.float64, generator=g) * 8.0 - 4.0
    return torch.pow(torch.tensor(10.0, dtype=torch.float64), e).to(device)


def x_true(cfg: GsrConfig, device="cpu") -> torch.Tensor:
    g = _gen("cpu", cfg.seed, _S_XTRUE, 0)
    x = torch.randn(cfg.n_cols, dtype=torch.float64, generator=g)
    s = col_scales(cfg)
    if s is not None:
        x = x / s  # keeps every term of b O(1) (reading A11)
    return x.to(device)


def random_vector(cfg: GsrConfig, tag: int, length: int, device="cpu") -> torch.Tensor:
    """N(0,1) probe vector; generated chunk-wise on `device`."""
    out = torch.empty(length, dtype=torch.float64, device=device)
    for c, r0 in enumerate(range(0, length, CHUNK)):
        r1 = min(r0 + CHUNK, length)
        g = _gen(device, cfg.seed, _S_VEC + 16 * tag, c)
        out[r0:r1] = torch.randn(r1 - r0, dtype=torch.float64, device=device, generator=g)
    return out


def noise(cfg: GsrConfig, row0: int, nrows: int, device="cpu") -> torch.Tensor:
    assert row0 % CHUNK == 0
    out = torch.empty(nrows, dtype=torch.float64, device=device)
    for r0 in range(row0, row0 + nrows, CHUNK):
        r1 = min(r0 + CHUNK, row0 + nrows)
        g = _gen(device, cfg.seed, _S_NOISE, r0 // CHUNK)
        out[r0 - row0:r1 - row0] = cfg.noise_sigma * torch.randn(
            r1 - r0, dtype=torch.float64, device=device, generator=g)
    return out


def _instr_distinct(n: int, n_instr: int, device, g: torch.Generator) -> torch.Tensor:
    """[n,6] int32, six distinct uniform columns per row, draw order kept (reading A12)."""
    k = min(N_INSTR_ROW, n_instr)
    c = torch.randint(0, n_instr, (n, N_INSTR_ROW), device=device, generator=g, dtype=torch.int64)
    if n_instr < N_INSTR_ROW:
        return c.to(torch.int32)  # cannot be distinct; duplicates are legal for the library
    while True:
        s, _ = torch.sort(c, dim=1)
        bad = (s[:, 1:] == s[:, :-1]).any(dim=1)
        nb = int(bad.sum())
        if nb == 0:
            break
        c[bad] = torch.randint(0, n_instr, (nb, N_INSTR_ROW), device=device, generator=g,
                               dtype=torch.int64)
    del k
    return c.to(torch.int32)


def gen_rows(cfg: GsrConfig, row0: int, nrows: int, device="cpu",
             sptr: Optional[torch.Tensor] = None, scales: Optional[torch.Tensor] = None):
    """Caller-form arrays for rows [row0, row0+nrows): (star_idx i32[n], att_start i32[n],
    instr_col i32[n,6], values f64[n,24]).  row0 must be a multiple of CHUNK."""
    assert row0 % CHUNK == 0 and 0 <= row0 and row0 + nrows <= cfg.n_rows
    if sptr is None:
        sptr = star_ptr(cfg)
    sptr_d = sptr.to(device)
    if cfg.col_scales and scales is None:
        scales = col_scales(cfg, device)
    star = torch.empty(nrows, dtype=torch.int32, device=device)
    att = torch.empty(nrows, dtype=torch.int32, device=device)
    instr = torch.empty((nrows, N_INSTR_ROW), dtype=torch.int32, device=device)
    vals = torch.empty((nrows, N_PAR), dtype=torch.float64, device=device)
    n_start = cfg.n_dfa - 3  # a_i in {0..D-4} (reading A3)
    for r0 in range(row0, row0 + nrows, CHUNK):
        r1 = min(r0 + CHUNK, row0 + nrows)
        n = r1 - r0
        c = r0 // CHUNK
        sl = slice(r0 - row0, r1 - row0)
        rows = torch.arange(r0, r1, device=device, dtype=torch.int64)
        st = torch.searchsorted(sptr_d, rows, right=True) - 1
        star[sl] = st.to(torch.int32)
        g = _gen(device, cfg.seed, _S_ATT, c)
        a = torch.randint(0, n_start, (n,), device=device, generator=g, dtype=torch.int64)
        if cfg.att_hot is not None:
            frac, wlo, whi = cfg.att_hot
            lo = int(wlo * n_start)
            hi = max(int(whi * n_start), lo + 1)
            gh = _gen(device, cfg.seed, _S_HOT, c)
            hot = torch.rand(n, device=device, generator=gh, dtype=torch.float64) < frac
            ah = torch.randint(lo, hi, (n,), device=device, generator=gh, dtype=torch.int64)
            a = torch.where(hot, ah, a)
        if cfg.att_time_ordered:   # same multiset of knots per star, visited in increasing order
            a = a[torch.argsort(st * n_start + a)]
        att[sl] = a.to(torch.int32)
        g = _gen(device, cfg.seed, _S_INSTR, c)
        ic = _instr_distinct(n, cfg.n_instr, device, g)
        instr[sl] = ic
        g = _gen(device, cfg.seed, _S_VAL, c)
        v = torch.randn((n, N_PAR), dtype=torch.float64, device=device, generator=g)
        if scales is not None:
            # column of every stored coefficient (structure of section 3)
            cols = torch.empty((n, N_PAR), dtype=torch.int64, device=device)
            cols[:, 0:5] = (5 * st)[:, None] + torch.arange(5, device=device)
            for ax in range(3):
                cols[:, 5 + 4 * ax:9 + 4 * ax] = (cfg.off_att + ax * cfg.n_dfa + a)[:, None] \
                    + torch.arange(4, device=device)
            cols[:, 17:23] = cfg.off_instr + ic.to(torch.int64)
            cols[:, 23] = cfg.off_glob
            v = v * scales[cols]
        vals[sl] = v
    return star, att, instr, vals


def gen_all(cfg: GsrConfig, device="cpu"):
    """Whole system (small configs only)."""
    return gen_rows(cfg, 0, cfg.n_rows, device)


def micro_config(name: str, seed: int, counts: Sequence[int], n_dfa: int, n_instr: int,
                 **kw) -> GsrConfig:
    """Adversarial micro-cases for tests: explicit rows per star (zeros allowed)."""
    return GsrConfig(name, seed, len(counts), n_dfa, n_instr, counts=tuple(int(c) for c in counts),
                     **kw)
