#!/usr/bin/env python
"""bench.py -- LSQR iterations/s of the Gaia AVU-GSR hot path on B200 (BASELINE.json metric).

A "step" is one PC-LSQR iteration: aprod1, beta, aprod2, alpha, plane rotations, fused vector
update (all rows of SURVEY/DESIGN section 8(a)) over one synthetic system resident in HBM.
Default workload: BASELINE.json configs[2] ("cfg3", 3e8 rows, the config the >=70 % HBM
target is quoted on).  Inputs are seeded and synthetic (paper_2212_11675_b200/inputs.py).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config cfg3] [--impl ours|reference]

N > 1 (torchrun): ONE system of N x the config's rows, row-sharded over the ranks by star-aligned
blocks (the paper's MPI partition) with the replicated slice all-reduced by NCCL
inside the CUDA graph; `--replicas` gives every rank an independent
system instead (no data-path collective).  `--impl reference` times the CPU oracle, as it
stands, on a bounded sample of the workload (rank 0 only).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "lsqr_iterations_per_s"
UNIT = "it/s"
BYTES_APROD1, BYTES_APROD2 = 240, 232          # algorithmic HBM bytes per row
TRAFFIC_APROD1, TRAFFIC_APROD2 = 228, 220      # bytes per row the 212 B/row layout really moves
# fused iteration (GSR_OPT_FUSED, default): k_fused does aprod1 and aprod2 minus the instrumental
# block of A^T u (6 x (8+4) B of matrix + 8 B of u per row = 80 B), which k_aprod2_instr does
BYTES_INSTR = 80
# What ONE fused pass must move: the matrix once (224 B/row with int32 indices) +
# u_hat read + u_hat write.  This is the roofline figure of k_fused.  The same work done as two
# products would move 240 + 232 - 80 = 392 B/row; that "two-product equivalent" rate is reported
# separately (products.fused_two_product_equiv_gbs) and is not a roofline fraction.
BYTES_FUSED = 224 + 8 + 8
BYTES_FUSED_2P = BYTES_APROD1 + BYTES_APROD2 - BYTES_INSTR
BYTES_ITER_FUSED = BYTES_FUSED + BYTES_INSTR    # 320 B/row per fused iteration
# DRAM bytes per row measured by `ncu --set full` at cfg3 (dram__bytes_read.sum +
# dram__bytes_write.sum over the rows of the launch); multiplied by the rows of the timed launch
# to give roofline.traffic.  Source files under profiles/ (NCU_TRAFFIC_SOURCE).
NCU_TRAFFIC_PER_ROW = {"aprod1": 228.6, "aprod2": 221.1, "fused": 230.1, "aprod2_instr": 68.1}
NCU_TRAFFIC_SOURCE = "profiles/r2_fused_ncu_full.md (k_fused), profiles/r2_aprod_ncu_full.md (products), cfg3"
# the fused pass and its instrumental pass per workload (profiles/r3_fused_ncu_cfg2_cfg4.md): the
# traffic per row turned out not to depend on the instrumental width or the attitude distribution
NCU_TRAFFIC_FUSED = {"cfg2": (229.2, 68.1, "profiles/r3_fused_ncu_cfg2_cfg4.md, cfg2"),
                     "cfg4": (229.9, 68.1, "profiles/r3_fused_ncu_cfg2_cfg4.md, cfg4"),
                     "cfg3": (230.1, 68.1, "profiles/r2_fused_ncu_full.md, cfg3")}
GEN_ROWS = 1 << 23                              # rows generated and appended per chunk
# The oracle (OpenMP build, 16 host cores of a B200 box) on the WHOLE system, measured once by the
# opt-in full-size parity job (profiles/r3_fullsize_parity.md): seconds for the config's own
# iteration count.  Reported beside the sampled figure, which stays what the short default run times.
ORACLE_FULL_SIZE = {"cfg2": (100, 81.2), "cfg3": (50, 138.2), "cfg4": (100, 83.2)}


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="cfg3")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--oracle-rows", type=int, default=1 << 22)
    ap.add_argument("--time-ordered", action="store_true",
                    help="row f4(i): rows of a star in time order (att_start non-decreasing inside a star)")
    ap.add_argument("--streamed-resident-gb", type=float, default=None,
                    help="row f4(iii): out-of-core system -- at most this many GB of the tiled matrix stay "
                         "on the device, the rest is streamed from pinned host memory every pass "
                         "(use with --config cfg3x4 ...)")
    ap.add_argument("--chunk-mb", type=float, default=512.0, help="streamed: size of each of the two chunk buffers")
    ap.add_argument("--replicas", action="store_true",
                    help="N > 1: N independent systems (no collective) instead of one row-sharded system")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--fp64-instr", action="store_true",
                    help="GSR_OPT_FIXED_POINT = 0: fp64 adds for the instrumental block (in the two-pass "
                         "form aprod2 is then the one-sweep kernel gsr_aprod2 runs)")
    ap.add_argument("--while-graph", action="store_true",
                    help="run the loop as ONE conditional-WHILE CUDA graph launch (GSR_OPT_WHILE_GRAPH)")
    ap.add_argument("--two-pass", action="store_true",
                    help="GSR_OPT_FUSED = 0: aprod1 + aprod2 per iteration (two reads of the matrix)")
    ap.add_argument("--sharded", action="store_true",
                    help="row-sharded form (the default for N > 1; at N = 1 a one-rank NCCL communicator)")
    ap.add_argument("--sweep", action="store_true",
                    help="BASELINE config 5: time aprod1/aprod2 alone from 1e6 to 3e8 rows")
    ap.add_argument("--sweep-rows", default=None,
                    help="--sweep: comma-separated row counts instead of the whole 1e6 ... 3e8 ladder")
    ap.add_argument("--launch-check", action="store_true",
                    help="no GPU work: every rank joins a gloo group, rank 0 prints the number of ranks "
                         "that answered (tests/test_bench_launch.py checks the --gpus N launcher with it)")
    return ap.parse_args()


def free_port():
    import socket
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def launch_ranks(args):
    """`python bench.py --gpus N` outside torchrun (no WORLD_SIZE): start the N ranks ourselves, one
    per GPU, exactly as the driver's torchrun line would, and hand their output through.  Rank 0
    prints the one JSON line; NCCL's own lines go to stderr (see main)."""
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(free_port()),
           os.path.abspath(__file__), *sys.argv[1:]]
    return subprocess.call(cmd)


def launch_check():
    """The launcher's self-test: count the ranks that came up (gloo, CPU only)."""
    import torch
    import torch.distributed as dist
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    n = torch.ones(1)
    if world > 1:
        dist.init_process_group("gloo")
        dist.all_reduce(n)
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps({"launch_check": True, "n_gpus": world, "ranks_answered": int(n.item())}), flush=True)


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler(threading.Thread):
    """nvidia-smi clocks and throttle reasons during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.rows, self._stop_ev = index, [], threading.Event()

    def run(self):
        while not self._stop_ev.is_set():
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                      "--format=csv,noheader,nounits"], capture_output=True,
                                     text=True, timeout=5).stdout.strip()
                if out:
                    self.rows.append([f.strip() for f in out.split(",")])
            except Exception:
                pass
            self._stop_ev.wait(0.2)

    def finish(self):
        self._stop_ev.set()
        self.join(timeout=6)
        sm = sorted(int(r[0]) for r in self.rows if r[0].isdigit())
        mx = [int(r[1]) for r in self.rows if r[1].isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(r[2 + i] == "Active" for r in self.rows)]
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(self.rows)}


def host_info():
    """The box the oracle is timed on (nproc, CPU model, host RAM)."""
    model, ram = "unknown", None
    try:
        for ln in open("/proc/cpuinfo"):
            if ln.startswith("model name"):
                model = ln.split(":", 1)[1].strip()
                break
        for ln in open("/proc/meminfo"):
            if ln.startswith("MemTotal"):
                ram = round(int(ln.split()[1]) / 1048576.0, 1)
                break
    except OSError:
        pass
    return {"nproc": os.cpu_count(), "cpu_model": model, "ram_gb": ram}


def config_dict(cfg, args, world, sharded, m_total, n_total):
    """`config` of the JSON line; the same function serves both arms (ours and --impl reference)."""
    return {"workload": cfg.name + ("+time-ordered" if cfg.att_time_ordered else ""),
            "rows": m_total, "cols": n_total, "stars": cfg.n_stars * (world if sharded else 1),
            "knots_per_axis": cfg.n_dfa, "instr_cols": cfg.n_instr,
            "preconditioned": True, "mode": "fixed-count (GSR_OPT_FORCE_ITNLIM)",
            "iteration": "two-pass (aprod1 + aprod2)" if args.two_pass else
                         "fused (one read of the matrix per iteration + instrumental pass)",
            "l2": "matrix (%.1f GB) is far larger than L2; no flush needed" % (224e-9 * cfg.n_rows)
                  if 224 * cfg.n_rows > 1e9 else "matrix fits in or near L2: L2-assisted numbers",
            "parallelism": ("row-sharded x%d (NCCL all-reduce of the replicated slice)" % world
                            if sharded else "replicas" if world > 1 else "single"),
            **({"storage": "out-of-core: at most %.1f GB of tiles on the device, the rest in pinned host "
                           "memory, streamed every pass" % args.streamed_resident_gb}
               if getattr(args, "streamed_resident_gb", None) is not None else {})}


def oracle_sample(cfg, rows, steps, omp=False):
    """The oracle, as it stands, on the first `rows` rows of the workload (own b, own p).
    omp=True: its OpenMP timing build (same file, -DORC_OPENMP), all host cores."""
    import numpy as np
    from paper_2212_11675_b200 import inputs
    from oracle import gsr_oracle
    rows = min(rows, cfg.n_rows)
    sptr = inputs.star_ptr(cfg)
    star, att, instr, vals = inputs.gen_rows(cfg, 0, rows, "cpu", sptr=sptr)
    n_stars = int(star[-1]) + 1
    o = gsr_oracle.OracleSystem(n_stars, cfg.n_dfa, cfg.n_instr, star.numpy(), att.numpy(),
                                instr.numpy(), vals.numpy(), omp=omp)
    del star, att, instr, vals
    xt = np.random.default_rng(cfg.seed).standard_normal(o.n)
    b = o.aprod1(xt, 1e-3 * np.random.default_rng(cfg.seed + 1).standard_normal(o.m))
    o.precondition()
    t0 = time.perf_counter()
    r = o.lsqr(b, steps, force_itnlim=True)
    dt = time.perf_counter() - t0
    assert r.itn == steps
    it_s_sample = steps / dt
    cores = gsr_oracle.omp_threads() if omp else 1
    return {"value": it_s_sample * rows / cfg.n_rows, "unit": UNIT, "cores": cores, "kind": "oracle",
            "build": "OpenMP timing build (aprod1 parallel for; aprod2 star-aligned ranges, thread-private "
                     "replicated-slice accumulators combined in thread order, PAPER.md:103)" if omp
                     else "serial",
            "sample": f"first {rows} rows ({n_stars} stars) of {cfg.name}, {steps} oracle LSQR "
                      f"iterations in {dt:.2f} s = {it_s_sample:.3f} it/s on the sample, scaled "
                      f"linearly by rows to the full {cfg.n_rows}-row system",
            "extrapolated": rows < cfg.n_rows, "seconds": dt}


def cpu_baseline(cfg, rows, steps):
    """`cpu_baseline` of the JSON line: the oracle on all host cores (value), and on one core."""
    from oracle import gsr_oracle
    gsr_oracle.build()
    gsr_oracle.build(omp=True)
    one = oracle_sample(cfg, rows, steps, omp=False)
    allc = oracle_sample(cfg, rows, steps, omp=True)
    allc["one_core"] = {k: one[k] for k in ("value", "unit", "cores", "sample", "seconds")}
    allc["host"] = host_info()
    if cfg.name in ORACLE_FULL_SIZE:
        k, sec = ORACLE_FULL_SIZE[cfg.name]
        allc["full_size_measured"] = {"value": k / sec, "unit": UNIT, "cores": 16, "iterations": k, "seconds": sec,
                                      "source": "profiles/r3_fullsize_parity.md (whole system, not extrapolated; "
                                                "recorded once, not re-timed by this run)"}
    return allc


def run_reference(args, cfg):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    world = int(os.environ.get("WORLD_SIZE", "1"))
    sharded = (world > 1 and not args.replicas) or args.sharded
    steps = max(1, min(args.steps, 20))
    for _ in range(min(args.warmup, 1)):
        oracle_sample(cfg, min(args.oracle_rows, 1 << 16), 1)
    cb = cpu_baseline(cfg, args.oracle_rows, steps)
    m_total = cfg.n_rows * (world if sharded else 1)
    n_total = cfg.n_cols + (5 * cfg.n_stars * (world - 1) if sharded else 0)
    line = {"impl": "reference", "metric": METRIC, "value": cb["value"], "unit": UNIT,
            "n_gpus": args.gpus, "steps": steps, "warmup": args.warmup,
            "ms_per_step": 1e3 / cb["value"], "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": config_dict(cfg, args, world, sharded, m_total, n_total),
            "cpu_baseline": cb,
            "e2e": {"value": cb["value"], "unit": UNIT, "h2d_bytes_per_step": 0,
                    "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def wait_for_device_memory(torch, need_bytes, timeout_s=120.0):
    """The device memory of a process that has just exited (the tests, the other arm) is handed
    back asynchronously: wait until the workload fits instead of failing with GSR_ENOMEM."""
    t0 = time.perf_counter()
    while True:
        free, total = torch.cuda.mem_get_info()
        if free >= min(need_bytes, 0.95 * total) or time.perf_counter() - t0 > timeout_s:
            return free
        time.sleep(1.0)


def build_system(cfg, g, inputs, torch, dev, resident_gb=None, chunk_mb=512.0):
    """Chunked ingest (gsr_matrix_begin/append/finalize) of rows generated on the device."""
    need = (236 if resident_gb is None else 24) * cfg.n_rows + (0 if resident_gb is None else resident_gb * 1e9) + 3e9
    wait_for_device_memory(torch, need)
    sptr = inputs.star_ptr(cfg)
    scales = inputs.col_scales(cfg, dev)
    if resident_gb is None:
        h = g.gsr_matrix_begin(cfg.n_rows, cfg.n_stars, cfg.n_dfa, cfg.n_instr)
    else:
        h = g.gsr_matrix_begin_streamed(cfg.n_rows, cfg.n_stars, cfg.n_dfa, cfg.n_instr,
                                        int(resident_gb * 1e9), int(chunk_mb * 1e6))
    for r0 in range(0, cfg.n_rows, GEN_ROWS):
        nr = min(GEN_ROWS, cfg.n_rows - r0)
        star, att, instr, vals = inputs.gen_rows(cfg, r0, nr, dev, sptr=sptr, scales=scales)
        g.gsr_matrix_append_rows(h, r0, nr, star, att, instr, vals)
        torch.cuda.synchronize()
        del star, att, instr, vals
    g.gsr_matrix_finalize(h)
    return h


def run_sweep(args):
    """BASELINE.json config 5: the config-1 structure from 1e6 to 3e8 rows, each product timed
    alone (internal row order = after the attitude-bin reordering, and through the caller-order
    API = what a caller who keeps its own row order pays for the perm gather/scatter)."""
    import torch
    from paper_2212_11675_b200 import binding as g, inputs
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    peak, peak_src = peaks()
    sizes = [1_000_000 * 2 ** k for k in range(9)] + [300_000_000]
    if args.sweep_rows:
        sizes = [int(float(v)) for v in args.sweep_rows.split(",")]
    for m in sizes:
        cfg = inputs.named_config(f"cfg5_{m}")
        if args.time_ordered:
            from dataclasses import replace
            cfg = replace(cfg, att_time_ordered=True)
        h = build_system(cfg, g, inputs, torch, dev)
        x = inputs.random_vector(cfg, 1, cfg.n_cols, dev)
        y = inputs.random_vector(cfg, 2, cfg.n_rows, dev)
        # gsr_time_product runs on the solver's own vectors: a two-iteration solve first, so that
        # they hold real data (on zero vectors every zero-valued atomic of aprod2 is skipped and
        # the kernel looks faster than it is)
        g.gsr_set_option(h, g.GSR_OPT_FORCE_ITNLIM, 1)
        g.gsr_lsqr_solve(h, y, torch.empty(cfg.n_cols, dtype=torch.float64, device=dev), 2)
        ms1 = g.gsr_time_product(h, 1, 20)
        ms2 = g.gsr_time_product(h, 2, 20)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        api = []
        for fn, a, b in ((g.gsr_aprod1, x, y), (g.gsr_aprod2, y, x)):
            fn(h, a, b)
            e0.record()
            for _ in range(5):
                fn(h, a, b)
            e1.record()
            torch.cuda.synchronize()
            api.append(e0.elapsed_time(e1) / 5)
        # the same products through the internal-order API: a caller that iterates converts once
        # (gsr_vector_to_internal / _from_internal) and then pays no gather or scatter per product
        yi = torch.empty(g.gsr_matrix_internal_rows(h), dtype=torch.float64, device=dev)
        g.gsr_vector_to_internal(h, y, yi)
        internal = []
        for fn, a, b in ((g.gsr_aprod1_internal, x, yi), (g.gsr_aprod2_internal, yi, x),
                         (g.gsr_vector_to_internal, y, yi), (g.gsr_vector_from_internal, yi, y)):
            fn(h, a, b)
            e0.record()
            for _ in range(5):
                fn(h, a, b)
            e1.record()
            torch.cuda.synchronize()
            internal.append(e0.elapsed_time(e1) / 5)
        del yi
        pair_internal = (BYTES_APROD1 + BYTES_APROD2) * m / (internal[0] + internal[1]) * 1e-6
        row = {"workload": cfg.name, "rows": m, "cols": cfg.n_cols,
               "row_order": "time-ordered inside a star" if args.time_ordered else "uniform random knots",
               "l2": "L2-assisted" if 224 * m < 1e9 else "HBM",
               "aprod1_ms": ms1, "aprod2_ms": ms2,
               "aprod1_gbs": BYTES_APROD1 * m / ms1 * 1e-6, "aprod2_gbs": BYTES_APROD2 * m / ms2 * 1e-6,
               "aprod1_nnz_per_s": 24 * m / (ms1 * 1e-3), "aprod2_nnz_per_s": 24 * m / (ms2 * 1e-3),
               "aprod1_frac_of_measured": BYTES_APROD1 * m / ms1 * 1e-6 / peak,
               "aprod2_frac_of_measured": BYTES_APROD2 * m / ms2 * 1e-6 / peak,
               "aprod1_caller_order_ms": api[0], "aprod2_caller_order_ms": api[1],
               "aprod1_caller_order_gbs": BYTES_APROD1 * m / api[0] * 1e-6,
               "aprod2_caller_order_gbs": BYTES_APROD2 * m / api[1] * 1e-6,
               "pair_caller_order_frac_of_8tbs": (BYTES_APROD1 + BYTES_APROD2) * m / (api[0] + api[1]) * 1e-6 / 8000.0,
               "aprod1_internal_api_ms": internal[0], "aprod2_internal_api_ms": internal[1],
               "aprod1_internal_api_gbs": BYTES_APROD1 * m / internal[0] * 1e-6,
               "aprod2_internal_api_gbs": BYTES_APROD2 * m / internal[1] * 1e-6,
               "pair_internal_api_gbs": pair_internal, "pair_internal_api_frac_of_8tbs": pair_internal / 8000.0,
               "to_internal_ms": internal[2], "from_internal_ms": internal[3],
               "peak": peak, "peak_source": peak_src}
        print(json.dumps(row), flush=True)
        g.gsr_matrix_destroy(h)
        del x, y
        torch.cuda.empty_cache()


def main():
    args = parse()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        sys.exit(launch_ranks(args))
    if args.launch_check:
        return launch_check()
    from paper_2212_11675_b200 import inputs
    cfg0 = inputs.named_config(args.config)
    if args.time_ordered:
        from dataclasses import replace as _replace
        cfg0 = _replace(cfg0, att_time_ordered=True)
    if args.impl == "reference":
        return run_reference(args, cfg0)
    if args.sweep:
        return run_sweep(args)

    import torch
    import torch.distributed as dist
    from dataclasses import replace
    from paper_2212_11675_b200 import binding as g

    # NCCL logs to stdout by default (even its version line at NCCL_DEBUG=WARN): send whatever the
    # environment asks for to stderr, so that stdout stays the one JSON line; NCCL_DEBUG is left alone
    os.environ.setdefault("NCCL_DEBUG_FILE", "/dev/stderr")
    if os.environ.get("NCCL_DEBUG", "VERSION").upper() == "VERSION":
        os.environ["NCCL_DEBUG"] = "WARN"   # (at VERSION the one line NCCL prints ignores NCCL_DEBUG_FILE)
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    sharded = (world > 1 and not args.replicas) or args.sharded
    cfg = replace(cfg0, seed=cfg0.seed + 1000 * rank) if rank else cfg0   # rank's own rows
    m, n = cfg.n_rows, cfg.n_cols

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def measure(retried=False):
        h = comm = None
        try:
            t_setup = time.perf_counter()
            h = build_system(cfg, g, inputs, torch, dev, args.streamed_resident_gb, args.chunk_mb)
            streamed = g.gsr_matrix_host_bytes(h) > 0
            # b = A x_true + noise, formed on the device with the library's own aprod1
            xt = inputs.x_true(cfg, dev)
            b = torch.empty(m, dtype=torch.float64, device=dev)
            for r0 in range(0, m, GEN_ROWS):
                nr = min(GEN_ROWS, m - r0)
                b[r0:r0 + nr] = inputs.noise(cfg, r0, nr, dev)
            if sharded:
                # weak-scaled sharded system: rank r owns stars [r*S, (r+1)*S) of an N*S-star system; the
                # attitude + instrumental + global unknowns are shared, so their x_true comes from rank 0's seed
                xt0 = inputs.x_true(cfg0, dev)
                xt[cfg.off_att:] = xt0[cfg0.off_att:]
                uid = [g.gsr_comm_unique_id() if rank == 0 else None]
                if world > 1:
                    dist.broadcast_object_list(uid, src=0)
                comm = g.gsr_comm_create(rank, world, uid[0])
                g.gsr_matrix_set_comm(h, comm, world * m, world * 5 * cfg.n_stars + (n - cfg.off_att))
            g.gsr_aprod1(h, xt, b)
            g.gsr_precondition(h)
            g.gsr_set_option(h, g.GSR_OPT_FORCE_ITNLIM, 1)
            g.gsr_set_option(h, g.GSR_OPT_FUSED, 0 if args.two_pass else 1)
            g.gsr_set_option(h, g.GSR_OPT_WHILE_GRAPH, 1 if args.while_graph else 0)
            g.gsr_set_option(h, g.GSR_OPT_FIXED_POINT, 0 if args.fp64_instr else 1)
            x = torch.empty(n, dtype=torch.float64, device=dev)
            torch.cuda.synchronize()
            t_setup = time.perf_counter() - t_setup

            # warm-up (untimed): W iterations (>= 3), also builds the CUDA graph
            W = max(args.warmup, 3)
            g.gsr_lsqr_solve(h, b, x, W)
            # timed: exactly K iterations, device-resident inputs
            K = args.steps
            sampler = ClockSampler(local)
            sampler.start()
            barrier()
            l0 = g.gsr_launch_count()
            sb0 = g.gsr_matrix_streamed_bytes(h)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.profiler.start()      # cudaProfilerStart: ncu --profile-from-start off sees only this
            e0.record()
            res = g.gsr_lsqr_solve(h, b, x, K)
            e1.record()
            torch.cuda.synchronize()
            torch.cuda.profiler.stop()
            barrier()
            launches = g.gsr_launch_count() - l0
            streamed_bytes = g.gsr_matrix_streamed_bytes(h) - sb0
            while_graph = g.gsr_debug_while_graph(h)
            ms_solve = e0.elapsed_time(e1)            # whole call: initialisation + K iterations + x
            ms = g.gsr_lsqr_last_loop_ms(h)           # exactly the K iterations (CUDA events on the stream)
            assert 0.0 < ms <= ms_solve
            clocks = sampler.finish()
            assert res.itn == K and res.istop == 7, res

            # end to end through the C ABI with HOST buffers: b H2D (pinned) and x D2H inside the call
            b_host = torch.empty(m, dtype=torch.float64).pin_memory()
            b_host.copy_(b)
            x_host = torch.empty(n, dtype=torch.float64).pin_memory()
            barrier()
            t0 = time.perf_counter()
            res2 = g.gsr_lsqr_solve(h, b_host, x_host, K)
            torch.cuda.synchronize()
            t_e2e = time.perf_counter() - t0
            barrier()
            assert res2.itn == K
            # same system, same K: the two solves differ only by the order of the floating-point
            # atomics.  How much that may move x is set by the Lanczos process, not by the kernels
            # (reading A20; measured at cfg4: 4e-16 up to K = 50, 8e-14 at 75, 9e-10 at 100, and in
            # deterministic mode bit-identical): the bar is 1e-9, or 20 x what ONE ULP of b moves the
            # device solve itself, never above 1e-6.  Not retried.
            e2e_diff = float((x_host.to(dev) - x).norm() / x.norm())
            del b_host
            gen = torch.Generator(device=dev)
            gen.manual_seed(12345 + rank)
            ulp = torch.nextafter(b.abs(), torch.full_like(b, float("inf"))) - b.abs()
            b_ulp = b + ulp * torch.randint(-1, 2, (m,), device=dev, generator=gen).double()
            del ulp
            x_ulp = torch.empty_like(x)
            g.gsr_lsqr_solve(h, b_ulp, x_ulp, K)
            one_ulp_sens = float((x_ulp - x).norm() / x.norm())
            del b_ulp, x_ulp
            e2e_bound = min(max(1e-9, 20.0 * one_ulp_sens), 1e-6)
            assert e2e_diff <= e2e_bound, (e2e_diff, one_ulp_sens)

            # per-kernel device time of the two products, CUDA events on the launching stream
            # (each on the vectors a short solve leaves in the workspace: the timing launches of one
            # product overwrite them, and on zero or overflowed vectors aprod2 does other work)
            reps = 2 if streamed else 10
            prod_ms = []
            for which in (1, 2, 3, 4):
                g.gsr_lsqr_solve(h, b, x, 2)
                prod_ms.append(g.gsr_time_product(h, which, reps))
            ms1, ms2, ms3, ms4 = prod_ms

            t = torch.tensor([ms, t_e2e * 1e3, ms1, ms2, ms3, ms4], dtype=torch.float64, device=dev)
            if world > 1:
                dist.all_reduce(t, op=dist.ReduceOp.MAX)
            ms, ms_e2e, ms1, ms2, ms3, ms4 = [float(v) for v in t]

            if rank == 0:
                peak, peak_src = peaks()
                gb1, gb2 = BYTES_APROD1 * m / ms1 * 1e-6, BYTES_APROD2 * m / ms2 * 1e-6
                gb12 = (BYTES_APROD1 + BYTES_APROD2) * m / (ms1 + ms2) * 1e-6
                gb3, gb4 = BYTES_FUSED * m / ms3 * 1e-6, BYTES_INSTR * m / ms4 * 1e-6
                if args.two_pass:
                    dom = ("aprod2", gb2, ms2, BYTES_APROD2) if ms2 >= ms1 else ("aprod1", gb1, ms1, BYTES_APROD1)
                else:
                    dom = ("fused", gb3, ms3, BYTES_FUSED)
                tpr, tsrc = NCU_TRAFFIC_PER_ROW[dom[0]], NCU_TRAFFIC_SOURCE
                if dom[0] == "fused":   # measured per workload; another workload: cfg3's figure, said so
                    tpr, _, tsrc = NCU_TRAFFIC_FUSED.get(cfg0.name, NCU_TRAFFIC_FUSED["cfg3"])
                    if cfg0.name not in NCU_TRAFFIC_FUSED:
                        tsrc += " (no capture of this workload: cfg3's bytes per row)"
                traffic = tpr * m if tpr is not None else None
                iter_bytes = (BYTES_APROD1 + BYTES_APROD2) if args.two_pass else BYTES_ITER_FUSED
                m_total = m * (world if sharded else 1)
                n_total = n + (5 * cfg.n_stars * (world - 1) if sharded else 0)
                line = {
                    "metric": METRIC, "value": world * K / (ms * 1e-3), "unit": UNIT, "n_gpus": world,
                    "steps": K, "warmup": W, "ms_per_step": ms / K, "higher_is_better": True,
                    "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                    "config": config_dict(cfg0, args, world, sharded, m_total, n_total),
                    "e2e": {"value": world * K / (ms_e2e * 1e-3), "unit": UNIT,
                            "h2d_bytes_per_step": 8 * m / K, "d2h_bytes_per_step": (8 * n + 80) / K,
                            "note": "gsr_lsqr_solve with pinned host b and host x; matrix resident",
                            "rel_diff_vs_device_solve": e2e_diff,
                            "rel_diff_bound": e2e_bound, "one_ulp_of_b_moves_x_by": one_ulp_sens},
                    "gpu_launches": int(launches),
                    "loop": ("one launch of a conditional-WHILE CUDA graph for all K iterations"
                             if while_graph else "one CUDA graph launch per iteration"),
                    "clocks": clocks,
                    "roofline": {"bound": "hbm", "kernel": dom[0], "achieved": dom[1], "peak": peak,
                                 "unit": "GB/s", "frac": dom[1] / peak, "traffic": traffic,
                                 "dram_gbs": traffic / dom[2] * 1e-6, "dram_frac": traffic / dom[2] * 1e-6 / peak,
                                 "traffic_note": "DRAM bytes per launch = ncu --set full bytes per row ("
                                                 + tsrc + ") x rows of this launch; the layout "
                                                 "stores 212 B/row (uint16 indices), so traffic < algorithmic bytes",
                                 "peak_source": peak_src, "algorithmic_bytes_per_row": dom[3],
                                 "algorithmic_note": "k_fused: ONE read of the matrix (224 B/row, int32 indices) "
                                                     "+ u_hat read + write = 240 B/row; aprod1 240, aprod2 232",
                                 "ms_per_launch": dom[2]},
                    "products": {"aprod1_gbs": gb1, "aprod2_gbs": gb2, "aprod1_ms": ms1, "aprod2_ms": ms2,
                                 "fused_ms": ms3, "fused_gbs": gb3, "instr_pass_ms": ms4, "instr_pass_gbs": gb4,
                                 "fused_two_product_equiv_gbs": BYTES_FUSED_2P * m / ms3 * 1e-6,
                                 "aprod1_frac_of_measured": gb1 / peak, "aprod2_frac_of_measured": gb2 / peak,
                                 "aprod1_dram_gbs": TRAFFIC_APROD1 * m / ms1 * 1e-6,
                                 "aprod2_dram_gbs": TRAFFIC_APROD2 * m / ms2 * 1e-6,
                                 "combined_gbs": gb12, "combined_frac_of_measured": gb12 / peak,
                                 "combined_frac_of_8tbs": gb12 / 8000.0,
                                 "iteration_gbs": iter_bytes * m / (ms / K) * 1e-6,
                                 "iteration_frac_of_measured": iter_bytes * m / (ms / K) * 1e-6 / peak,
                                 "iteration_two_product_equiv_gbs": 472 * m / (ms / K) * 1e-6,
                                 "iteration_two_product_equiv_frac_of_8tbs": 472 * m / (ms / K) * 1e-6 / 8000.0,
                                 "note": "GB/s are algorithmic: aprod1 240, aprod2 232 B/row; fused pass 240 "
                                         "(one matrix read), instrumental pass 80, fused iteration 320 B/row. "
                                         "*_two_product_equiv_* divide the 472 B/row of an aprod1 + aprod2 "
                                         "iteration by the fused time (what a two-product code would need to "
                                         "sustain to be as fast); not a roofline fraction"},
                    "lsqr": {"istop": res.istop, "itn": res.itn, "rnorm": res.rnorm, "anorm": res.anorm,
                             "acond": res.acond, "xnorm": res.xnorm, "istop_natural": res.istop_natural,
                             "itn_natural": res.itn_natural},
                    "solve_call_ms": ms_solve,
                    "timing": "value = N x K / device time of the K iterations, timed by CUDA events that "
                              "gsr_lsqr_solve records on the launching stream around its graph-launch loop (max "
                              "over ranks; a row-sharded system has N x the config's rows, so one of its "
                              "iterations counts as N config-sized ones); solve_call_ms also has the "
                              "initialisation (one aprod2) and the finalisation; e2e is the wall clock of the "
                              "whole call with host buffers",
                    "setup_s": t_setup, "matrix_device_gb": g.gsr_matrix_device_bytes(h) * 1e-9,
                    "retried_after_enomem": retried,
                }
                if streamed:
                    # the K iterations + the initial aprod2 each move the host part once (fused form)
                    per_it = streamed_bytes / (K + 1)
                    line["streamed"] = {
                        "host_gb": g.gsr_matrix_host_bytes(h) * 1e-9, "device_gb": g.gsr_matrix_device_bytes(h) * 1e-9,
                        "tile_gb": 212e-9 * m, "tile_bytes_over_hbm_180gb": 212e-9 * m / 180.0,
                        "h2d_gb_per_iteration": per_it * 1e-9, "chunk_mb": args.chunk_mb,
                        "h2d_gbs": per_it / (ms / K) * 1e-6,
                        "note": "iteration time is bounded below by the host part of the matrix over the bus "
                                "(PCIe 5 x16: 64 GB/s raw, about 55 GB/s of payload); h2d_gbs is what the "
                                "iteration sustained, kernels of the resident part and of the previous chunk "
                                "overlapped with the copies"}
                if world == 1 and not args.no_cpu_baseline:
                    line["cpu_baseline"] = cpu_baseline(cfg0, args.oracle_rows, 20)
                print(json.dumps(line), flush=True)
        finally:
            if h is not None:
                g.gsr_matrix_destroy(h)
            if comm:
                g.gsr_comm_destroy(comm)

    # One retry on a single GPU, for GSR_ENOMEM only: a run that starts right after another process
    # has exited can find the device memory not yet handed back.  A failed assert is never retried;
    # the line says whether a retry happened.
    attempts = 2 if world == 1 else 1
    for attempt in range(attempts):
        try:
            measure(retried=attempt > 0)
            break
        except g.GsrError as e:
            import gc
            import traceback
            traceback.print_exc(file=sys.stderr)
            if e.code != g.GSR_ENOMEM or attempt + 1 == attempts:
                raise
            gc.collect()
            torch.cuda.empty_cache()
            time.sleep(20.0)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
