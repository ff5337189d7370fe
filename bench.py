#!/usr/bin/env python
"""bench.py — staggered Dslash + multi-shift CG on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c4|c5|c3|c2] [--impl reference]

One STEP = one pass of the whole hot path over one synthetic
pseudo-fermion source: one multi-shift CG solve of (m^2 - D_eo D_oe + sigma_i) x_i = b with all its
Dslash applications, reductions, scalar recurrences and shift updates.  Row a1 (gauge pack) is
setup, done once and reported as `pack_ms`.  `value` = Dslash GFLOP/s sustained through the solve
(570 flop/site x 2 Dslash/iteration x iterations x Vh / time): the BASELINE metric's first figure
measured over the whole path; the CG time-to-solution and the standalone Dslash sweep are beside it.
Prints ONE JSON line (rank 0).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

WORKLOADS = {"c2": "c2_16x16x16x4", "c3": "c3_24x24x24x6", "c4": "c4_32x32x32x8", "c5": "c5_64x64x64x64",
             "t2b": "t2_32x32x32x32", "t2c": "t2_48x48x48x4"}
# the paper's own Dslash figures (Table 2: Tesla C1060, fp32, 12-real, 576 flop/site by its
# own accounting — BASELINE.md §1): context beside the fp32-12 line of the sweep, another machine's numbers
PAPER_TABLE2 = {"c2": (49.31, 56.84, "PAPER.md:103 (4x16^3)"), "t2b": (55.597, 64.091, "PAPER.md:104 (32x32^3)"),
                "t2c": (60.67, 69.94, "PAPER.md:105 (4x48^3)")}
FLOP_PER_SITE = 570                                   # BASELINE.json:north_star
DSLASH_BYTES = {(0, 18): 1248, (0, 12): 864, (1, 18): 624, (1, 12): 432,
                (2, 18): 1248, (2, 12): 864}                               # N3 split-double: 2 floats per real
PREC_NAME = {0: "f64", 1: "f32", 2: "f64split"}
VARIANTS = ((0, 18), (0, 12), (1, 18), (1, 12), (2, 18), (2, 12))
NOMINAL_HBM_GBS = 8000.0                              # "8 TB/s roofline" of BASELINE.json:metric


def measured_peak_gbs():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"


def committed_traffic(workload, variant, kernel="dslash"):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel`, from the committed `ncu
    --set full` capture (profiles/traffic.csv; text written from the capture, never by this run)."""
    import csv
    path = os.path.join(ROOT, "profiles", "traffic.csv")
    try:
        with open(path, newline="") as f:
            for row in csv.DictReader(f):
                if row["workload"] == workload and row["variant"] == variant and kernel in row["kernel"]:
                    return int(row["dram_bytes_per_launch"])
    except Exception:
        pass
    return None


def cg_bytes_per_site(prec, recon, iters, iters_shift):
    """Algorithmic bytes of one solve per even site: per iteration 2 Dslash +
    p re-read (a3) + r,q,r (a5) + r (a6), plus x_i,p_i read+write for every iteration shift i was live."""
    w = 4 if prec == 1 else 8
    vec = 6 * w
    per_iter = 2 * DSLASH_BYTES[(prec, recon)] + vec + 3 * vec + vec
    return iters * per_iter + sum(iters_shift) * 4 * vec


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.path = index, None, "/tmp/stag_clocks_%d.csv" % os.getpid()

    def start(self):
        try:
            self.f = open(self.path, "w")
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        self.f.close()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in open(self.path):
            c = [x.strip() for x in line.split(",")]
            if len(c) < 9:
                continue
            try:
                sm.append(float(c[1])); mx.append(float(c[2]))
            except ValueError:
                continue
            for n, v in zip(names, c[5:9]):
                if v.lower() == "active":
                    reasons.add(n)
        os.unlink(self.path)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "reasons": sorted(reasons),
                "samples": len(sm)}


def make_inputs(cfg):
    import stag_inputs as si
    t0 = time.time()
    U = si.make_links(cfg)
    srcs = [si.make_source(cfg, k) for k in range(cfg["nsrc"])]
    return U, srcs, time.time() - t0


# ---------------------------------------------------------------------------------------------
# reference arm / cpu_baseline: the oracle, as it stands, on the host cores, on a BOUNDED sample
# ---------------------------------------------------------------------------------------------
def oracle_sample(cfg, U, b, budget_s: float, threads: int = 1):
    """Runs `m` oracle CG iterations of the same solve (maxiter = m; the oracle is otherwise untouched)
    with m sized from one probe iteration so the sample costs about budget_s.  Returns (GFLOP/s in the
    metric's accounting, seconds per iteration, m)."""
    import oracle
    oracle.set_threads(threads)
    L, vh = cfg["L"], int(np.prod(cfg["L"])) // 2
    t0 = time.time()
    oracle.mshift_cg(L, U, b, cfg["mass"], cfg["shifts"], cfg["stops"][0], 1)
    t1 = time.time() - t0
    m = int(max(2, min(200, budget_s / max(t1, 1e-6))))
    t0 = time.time()
    res = oracle.mshift_cg(L, U, b, cfg["mass"], cfg["shifts"], cfg["stops"][0], m)
    dt = time.time() - t0
    iters = max(res["iters"], 1)
    return 2 * FLOP_PER_SITE * vh * iters / dt / 1e9, dt / iters, iters


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import stag_inputs as si
    cfg = si.get_config(WORKLOADS[args.workload])
    U, srcs, _ = make_inputs(cfg)
    steps, warm = args.steps, args.warmup
    per_step = max(0.2, min(20.0, args.ref_seconds / max(1, steps + warm)))
    vals, spi, its = [], [], 0
    for k in range(warm + steps):
        g, s, its = oracle_sample(cfg, U, srcs[k % len(srcs)], per_step)
        if k >= warm:
            vals.append(g); spi.append(s)
    value = float(np.mean(vals))
    ms = float(np.mean(spi)) * its * 1e3
    sample = "%d oracle multi-shift CG iterations (maxiter=%d) of the %s solve per step, 1 thread" % (
        its, its, WORKLOADS[args.workload])
    out = {"impl": "reference", "metric": METRIC, "value": value, "unit": "GFLOP/s", "n_gpus": args.gpus,
           "steps": steps, "warmup": warm, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": workload_config(cfg, args.workload, 0, 18),
           "cpu_baseline": {"value": value, "unit": "GFLOP/s", "cores": 1, "kind": "oracle", "sample": sample},
           "e2e": {"value": value, "unit": "GFLOP/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "oracle_s_per_iteration": float(np.mean(spi))}
    print(json.dumps(out))
    return 0


METRIC = "Dslash GFLOP/s (570 flop/site) sustained through the multi-shift CG solve; CG s/solve beside it"


def workload_config(cfg, name, prec, recon):
    L = cfg["L"]
    return {"workload": "%s: %dx%dx%dx%d lattice, %s links, %d-shift multi-shift CG, m=%g, stop=%g, %d source(s)"
            % (WORKLOADS[name], L[0], L[1], L[2], L[3], cfg["links"][0], len(cfg["shifts"]), cfg["mass"],
               cfg["stops"][0], cfg["nsrc"]),
            "prec": PREC_NAME[prec], "recon": recon, "nshift": len(cfg["shifts"]),
            "parallelism": "replicas (independent sources, replicated gauge; no collective)"}


# ---------------------------------------------------------------------------------------------
# N > 1: replicas only.  The two pieces of host logic the ranks share; covered on
# CPU by tests/test_multirank_gloo.py (world_size 2, gloo).
# ---------------------------------------------------------------------------------------------
def source_for(rank: int, steps: int, k: int, nsrc: int) -> int:
    """Which pseudo-fermion source rank `rank` solves at its step k: the sources are dealt
    round-robin over the global step index, so ranks work on different sources."""
    return (rank * steps + k) % nsrc


def reduce_over_ranks(torch, dist, world: int, secs: float, work, device):
    """Whole-job numbers: time = MAX over ranks, work = SUM over ranks.  No data-path collective."""
    t = torch.tensor([secs], dtype=torch.float64, device=device)
    w = torch.tensor([float(v) for v in work], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(w, op=dist.ReduceOp.SUM)
    return float(t.item()), [float(v) for v in w.tolist()]


# ---------------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------------
def time_launches(torch, body, launches, repeats=5):
    """CUDA events around `launches` back-to-back launches issued by body(launches), median of `repeats`.  The
    launches are captured once in a CUDA graph and replayed, so that on small lattices (one launch is ~8 us of
    Python + ctypes, a 16^3x4 Dslash ~3 us) the events time the device, not the host.  Returns s per launch."""
    run = lambda: body(launches)
    try:
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=side):
            body(launches)
        torch.cuda.synchronize()
        run = graph.replay
        run()
    except Exception:
        torch.cuda.synchronize()
    ts = []
    for _ in range(repeats):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        run()
        e1.record()
        torch.cuda.synchronize()
        ts.append(e0.elapsed_time(e1) * 1e-3 / launches)
    return statistics.median(ts)


def time_dslash(torch, ctx, packed, prec, recon, a, b, launches=100, repeats=5, warm=10):
    """SURVEY.md §8(d) protocol: warm-up launches, then `launches` back-to-back launches ping-ponging
    D_oe / D_eo (outputs consumed), median of `repeats`.  Returns s per launch."""
    def pair(n):
        for _ in range(n // 2):
            ctx.dslash_oe(packed, prec, recon, a, b)
            ctx.dslash_eo(packed, prec, recon, b, a)
    pair(warm)
    return time_launches(torch, pair, launches, repeats)


def measure_block(torch, stag, ctx, cfg, srcs, packed, prec, recon, vh, peak):
    """N1: stag_dslash_block for R = 1, 2, 4 sources (100-launch ping-pong, as time_dslash) and ONE
    stag_mshift_cg_block solve of min(4, nsrc) sources.  Algorithmic bytes per site of a block Dslash =
    8 links (once) + R x (one read of the source + one write)."""
    w = 4 if prec == stag.F32 else 8
    vb = ctx.vector_bytes(prec)
    out = {"dslash": {}, "cg": None}
    for R in (1, 2, 4):
        if R > len(srcs):
            continue
        a, b = ctx.upload_vectors(srcs[:R], prec), ctx.alloc(R * vb)

        def pair(n):
            for _ in range(n // 2):
                ctx.dslash_block(packed, prec, recon, 1, R, a, b)
                ctx.dslash_block(packed, prec, recon, 0, R, b, a)
        pair(10)
        s_per = time_launches(torch, pair, 100)
        bps = 8 * recon * w + 2 * 6 * w * R
        gbs = bps * vh / s_per / 1e9
        out["dslash"]["R%d" % R] = {"us": s_per * 1e6, "us_per_source": s_per * 1e6 / R,
                                    "gflops": FLOP_PER_SITE * vh * R / s_per / 1e9, "bytes_per_site": bps,
                                    "gbs_algorithmic": gbs, "pct_of_measured": 100 * gbs / peak}
        del a, b
    R = min(4, len(srcs))
    n = len(cfg["shifts"])
    stop = cfg["stops"][0] if prec != stag.F32 else max(cfg["stops"][0], 1e-5)
    bdev = ctx.upload_vectors(srcs[:R], prec)
    x = ctx.alloc(R * n * vb)
    ws = ctx.alloc(ctx.cg_block_workspace_bytes(prec, n, R))
    ts = []
    for _ in range(2):                                    # first = warm-up
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        rc, infos = ctx.mshift_cg_block(packed, prec, recon, R, bdev, cfg["mass"], cfg["shifts"], stop, 100000, x, ws)
        e1.record()
        torch.cuda.synchronize()
        ts.append(e0.elapsed_time(e1) * 1e-3)
    its = [i["iters"] for i in infos]
    out["cg"] = {"nrhs": R, "rc": rc, "s_per_block_solve": ts[-1], "s_per_source": ts[-1] / R, "iters": its,
                 "us_per_iter": ts[-1] / max(its) * 1e6, "stop": stop,
                 "gflops": 2 * FLOP_PER_SITE * vh * sum(its) / ts[-1] / 1e9,
                 "call": "stag_mshift_cg_block (one persistent launch, links read once per Dslash for all sources)"}
    return out


def measure_mixed(torch, stag, ctx, cfg, U, srcs, vh, fp64_s_per_solve):
    """N2 + N3: stag_mshift_cg_mixed on ONE resident split-double buffer (fp32 stage reads its b planes, the
    fp64 polish reads b + c), same source, shifts and stop as the fp64 step; second of two runs timed."""
    n = len(cfg["shifts"])
    split = ctx.upload_gauge(U, stag.F64_SPLIT, 18)
    p64 = ctx.upload_gauge(U, stag.F64, 18)
    vb = ctx.vector_bytes(stag.F64)
    b = ctx.upload_vector(srcs[0], stag.F64)
    x = ctx.alloc(n * vb)
    ws = ctx.alloc(ctx.mshift_cg_mixed_workspace_bytes(n))
    out = {}
    for name, hi, prec_hi, lo in (("split_buffer", split, stag.F64_SPLIT, split), ("f64_polish_f32_inner", p64, stag.F64, split)):
        for _ in range(2):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            rc, info = ctx.mshift_cg_mixed(hi, prec_hi, 18, lo, 18, b, cfg["mass"], cfg["shifts"], cfg["stops"][0],
                                           100000, x, ws)
            e1.record()
            torch.cuda.synchronize()
        secs = e0.elapsed_time(e1) * 1e-3
        out[name] = {"rc": rc, "s_per_solve": secs, "vs_fp64_multishift": fp64_s_per_solve / secs,
                     "inner_fp32_iters": info["inner"]["iters"], "polish_iters": info["polish"]["iters"],
                     "polish_passes": info["polish"]["passes"],
                     "true_resid_after_fp32": max(info["polish"]["resid_before"]),
                     "true_resid_final": max(info["polish"]["resid_after"]),
                     "kernel_launches": info["inner"]["kernel_launches"] + info["polish"]["kernel_launches"]}
    # single shift (the lightest): the inner stage is the persistent residual-replacement kernel and stops on the
    # TRUE fp64 residual, nothing is left to polish; the fp64 solver on the same single system beside it
    sh1 = cfg["shifts"][:1]
    cgws = ctx.alloc(ctx.cg_workspace_bytes(stag.F64, 1))
    for _ in range(2):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        rc64, i64 = ctx.mshift_cg(p64, stag.F64, 18, b, cfg["mass"], sh1, cfg["stops"][0], 100000, x, cgws)
        e1.record()
        torch.cuda.synchronize()
    t64 = e0.elapsed_time(e1) * 1e-3
    for _ in range(2):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        # fp32 iterations on the b planes, fp64 residual replacement on b + c of the SAME split-double buffer (N3)
        rc, info = ctx.mshift_cg_mixed(split, stag.F64_SPLIT, 18, split, 18, b, cfg["mass"], sh1, cfg["stops"][0], 100000, x, ws)
        e1.record()
        torch.cuda.synchronize()
    tm = e0.elapsed_time(e1) * 1e-3
    out["single_shift_residual_replacement"] = {
        "rc": rc, "s_per_solve": tm, "fp64_s_per_solve": t64, "vs_fp64": t64 / tm, "iters": info["inner"]["iters"],
        "fp64_iters": i64["iters"], "reliable_updates": info["reliable_updates"],
        "polish_iters": sum(info["polish"]["iters"]), "true_resid_final": info["polish"]["resid_after"][0]}
    return out


def measure_force(torch, stag, ctx, cfg, srcs, packed, prec, recon, vh):
    """N4: stag_fermion_force on nshift even vectors (the x_i of a solve; timing does not depend on their
    values, so the sources stand in), 20 calls between CUDA events after 3 warm-up calls.  Algorithmic bytes:
    D_oe x_i through the multi-source kernel (links once per group of 4, each vector read + written once) +
    per link one matrix, one 144-byte output, and every X_i read once."""
    n = len(cfg["shifts"])
    w = 4 if prec == stag.F32 else 8
    x = ctx.upload_vectors([srcs[k % len(srcs)] for k in range(n)], prec)
    F = torch.empty(2 * vh * 72, dtype=torch.float64, device="cuda")
    ws = ctx.alloc(ctx.force_workspace_bytes(prec, n))
    res = [1.0 / (i + 1) for i in range(n)]
    for _ in range(3):
        ctx.fermion_force(packed, prec, recon, res, x, F, ws)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(20):
        ctx.fermion_force(packed, prec, recon, res, x, F, ws)
    e1.record()
    torch.cuda.synchronize()
    secs = e0.elapsed_time(e1) * 1e-3 / 20
    groups = (n + 3) // 4
    bytes_dslash = vh * (groups * 8 * recon * w + n * 2 * 6 * w)
    bytes_force = 2 * vh * (4 * recon * w + 4 * 144 + n * 6 * w)
    gbs = (bytes_dslash + bytes_force) / secs / 1e9
    return {"us_per_call": secs * 1e6, "nshift": n, "launches_per_call": 1 + groups,
            "algorithmic_bytes_per_call": bytes_dslash + bytes_force, "gbs_algorithmic": gbs}


def dslash_sweep(args, torch, stag, ctx, cfg, U, srcs, packed, prec, recon, vh, pack_ms, gen_s):
    """--dslash-only: the SURVEY.md §8(d) Dslash bandwidth sweep alone (no CG), one JSON line."""
    peak, peak_src = measured_peak_gbs()
    del packed
    canon = ctx.alloc(ctx.gauge_canonical_bytes())
    ctx.gauge_load(U, canon)
    torch.cuda.synchronize()
    out = {"metric": "Dslash GFLOP/s & HBM GB/s", "workload": WORKLOADS[args.workload], "peak_gbs": peak,
           "peak_source": peak_src, "pack_ms": pack_ms, "input_gen_s": gen_s, "dslash": {}}
    for p_, r_ in VARIANTS:
        pk = ctx.alloc(ctx.gauge_packed_bytes(p_, r_))
        ctx.gauge_pack(canon, pk, p_, r_)
        a = ctx.upload_vector(srcs[0], p_)
        b = ctx.alloc(ctx.vector_bytes(p_))
        s_per = time_dslash(torch, ctx, pk, p_, r_, a, b, launches=args.dslash_launches)
        gbs = DSLASH_BYTES[(p_, r_)] * vh / s_per / 1e9
        out["dslash"]["%s-%d" % (PREC_NAME[p_], r_)] = {
            "us": s_per * 1e6, "gflops": FLOP_PER_SITE * vh / s_per / 1e9, "gbs_algorithmic": gbs,
            "pct_of_8tbs": 100 * gbs / NOMINAL_HBM_GBS, "pct_of_measured": 100 * gbs / peak}
        del pk, a, b
    if args.workload in PAPER_TABLE2:
        pg, pb, cite = PAPER_TABLE2[args.workload]
        ours = out["dslash"]["f32-12"]
        out["paper_table2"] = {"hardware": "Tesla C1060", "prec": "f32", "recon": 12, "gflops": pg, "gbs": pb,
                               "cite": cite, "ours_f32_12_gflops": ours["gflops"],
                               "ratio_gflops": ours["gflops"] / pg,
                               "note": "another machine's figure: context, not the target"}
    print(json.dumps(out))
    return 0


def run_ours(args):
    import torch
    import torch.distributed as dist
    import stag_inputs as si
    import paper_1010_5433_b200 as stag

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    prec = {"f64": stag.F64, "f32": stag.F32, "f64split": stag.F64_SPLIT}[args.prec]
    recon = args.recon
    cfg = si.get_config(WORKLOADS[args.workload])
    L = cfg["L"]
    vh = int(np.prod(L)) // 2
    shifts, nshift = cfg["shifts"], len(cfg["shifts"])
    stop, maxiter = cfg["stops"][0], 100000

    # ---- setup (a1): seeded synthetic inputs -> HBM, packed once --------------------------------
    U, srcs, gen_s = make_inputs(cfg)
    ctx = stag.Stag(L)
    for kv in args.opt:                                   # tuning knobs of stag_set_option
        k, v = kv.split("=")
        ctx.set_option(k, int(v))
    canon = ctx.alloc(ctx.gauge_canonical_bytes())
    ctx.gauge_load(U, canon)
    torch.cuda.synchronize()
    packed = ctx.alloc(ctx.gauge_packed_bytes(prec, recon))
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    ctx.gauge_pack(canon, packed, prec, recon)
    e1.record()
    torch.cuda.synchronize()
    pack_ms = e0.elapsed_time(e1)
    del canon
    vb = ctx.vector_bytes(prec)
    if args.dslash_only:
        return dslash_sweep(args, torch, stag, ctx, cfg, U, srcs, packed, prec, recon, vh, pack_ms, gen_s)
    bdev = [ctx.upload_vector(s, prec) for s in srcs]
    x = ctx.alloc(nshift * vb)
    ws = ctx.alloc(ctx.cg_workspace_bytes(prec, nshift))

    def solve(k):
        rc, info = ctx.mshift_cg(packed, prec, recon, bdev[k], cfg["mass"], shifts, stop, maxiter, x, ws)
        if rc != 0:
            raise RuntimeError("stag_mshift_cg rc=%d %r" % (rc, info))
        return info

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- timed region: W warm-up solves, then exactly K solves ------------------------------------
    for k in range(args.warmup):
        solve(source_for(rank, args.steps, k, len(bdev)))
    clocks = ClockSampler(local)
    barrier()
    if rank == 0:
        clocks.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    infos = []
    e0.record()
    for k in range(args.steps):
        infos.append(solve(source_for(rank, args.steps, k, len(bdev))))
    e1.record()
    barrier()
    clk = clocks.stop() if rank == 0 else None
    secs, (tot_iters, tot_bytes_site, launches) = reduce_over_ranks(
        torch, dist, world, e0.elapsed_time(e1) * 1e-3,
        [sum(i["iters"] for i in infos),
         sum(cg_bytes_per_site(prec, recon, i["iters"], i["iters_shift"]) for i in infos),
         sum(i["kernel_launches"] for i in infos)], "cuda")
    value = 2 * FLOP_PER_SITE * vh * tot_iters / secs / 1e9
    nsolves = args.steps * world

    # ---- e2e: the same step through the host-buffer call, H<->D copies inside the timed region ----
    n6 = vh * 6
    hb = [torch.from_numpy(s.view(np.float64).reshape(-1).copy()).pin_memory() for s in srcs]
    hx = torch.empty(nshift * n6, dtype=torch.float64).pin_memory()
    scratch = ctx.alloc(ctx.host_scratch_bytes(prec, nshift))
    e2e_steps = max(1, min(args.steps, 3))
    ctx.mshift_cg_host(packed, prec, recon, hb[0], cfg["mass"], shifts, stop, maxiter, hx, scratch)
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    it_e2e = 0
    for k in range(e2e_steps):
        rc, info = ctx.mshift_cg_host(packed, prec, recon, hb[source_for(rank, e2e_steps, k, len(hb))], cfg["mass"],
                                      shifts, stop, maxiter, hx, scratch)
        it_e2e += info["iters"]
    e1.record()
    barrier()
    te_s, (ie_sum,) = reduce_over_ranks(torch, dist, world, e0.elapsed_time(e1) * 1e-3, [it_e2e], "cuda")
    e2e_value = 2 * FLOP_PER_SITE * vh * ie_sum / te_s / 1e9
    del scratch, hx

    # ---- roofline of the dominant kernel (the Dslash) and the sweep over storage variants ---------
    peak, peak_src = measured_peak_gbs()
    dslash = {}
    roof = roof_dslash = None
    if rank == 0:
        va, vb_ = ctx.alloc(ctx.vector_bytes(stag.F64)), ctx.alloc(ctx.vector_bytes(stag.F64))
        for p_, r_ in VARIANTS:
            pk = packed if (p_, r_) == (prec, recon) else ctx.upload_gauge(U, p_, r_)
            a = ctx.upload_vector(srcs[0], p_)
            s_per = time_dslash(torch, ctx, pk, p_, r_, a, vb_ if p_ != stag.F32 else va)
            gbs = DSLASH_BYTES[(p_, r_)] * vh / s_per / 1e9
            dslash["%s-%d" % (PREC_NAME[p_], r_)] = {
                "us": s_per * 1e6, "gflops": FLOP_PER_SITE * vh / s_per / 1e9, "gbs_algorithmic": gbs,
                "pct_of_8tbs": 100 * gbs / NOMINAL_HBM_GBS, "pct_of_measured": 100 * gbs / peak,
                "bytes_per_site": DSLASH_BYTES[(p_, r_)]}
            if (p_, r_) == (prec, recon):
                roof = {"bound": "hbm", "kernel": "dslash_kernel<%s,%d> (stag_dslash_oe/eo, %d launches ping-pong)"
                        % ("float" if p_ == stag.F32 else "double", r_, 100),
                        "achieved": gbs, "peak": peak, "unit": "GB/s", "frac": gbs / peak,
                        "peak_source": peak_src, "frac_of_8tbs": gbs / NOMINAL_HBM_GBS,
                        "algorithmic_bytes_per_launch": DSLASH_BYTES[(p_, r_)] * vh,
                        "avg_launch_us": s_per * 1e6, "traffic": None}
            if pk is not packed:
                del pk
        roof["traffic"] = committed_traffic(args.workload, "%s-%d" % (args.prec, recon))
        roof_dslash = roof
        if launches == nsolves:
            # the whole solve ran as ONE kernel per step (stag_cg_persist.cu): that kernel is the dominant
            # one.  Algorithmic bytes per launch = SURVEY.md §8(d): (2736 + 192 N_live) per even site and
            # iteration (fp64-18), summed over the iterations of the solve; duration = CUDA events around
            # the K launches of the timed region / K.
            cg_bytes_launch = tot_bytes_site * vh / nsolves
            cg_gbs_ = tot_bytes_site * vh / secs / 1e9 / world        # per GPU: ranks run concurrently
            roof = {"bound": "hbm", "kernel": "cg_persistent_kernel<%s,%d> (one launch = one multi-shift solve)"
                    % ("float" if prec == stag.F32 else "double", recon),
                    "achieved": cg_gbs_, "peak": peak, "unit": "GB/s", "frac": cg_gbs_ / peak,
                    "peak_source": peak_src, "frac_of_8tbs": cg_gbs_ / NOMINAL_HBM_GBS,
                    "algorithmic_bytes_per_launch": cg_bytes_launch, "avg_launch_us": secs / args.steps * 1e6,
                    "traffic": committed_traffic(args.workload, "%s-%d" % (args.prec, recon), "cg_persistent")}

    # ---- N1: the 4 pseudo-fermion sources of the workload through ONE link read ----
    block = None
    if rank == 0 and not args.no_block and len(srcs) >= 2 and prec != stag.F64_SPLIT:
        block = measure_block(torch, stag, ctx, cfg, srcs, packed, prec, recon, vh, peak)

    # ---- N2/N3: fp32 multi-shift + fp64 polish on one split-double buffer -----------------------------
    mixed = None
    if rank == 0 and not args.no_block and prec == stag.F64:
        mixed = measure_mixed(torch, stag, ctx, cfg, U, srcs, vh, secs / args.steps)

    force = None
    if rank == 0 and not args.no_block and prec != stag.F64_SPLIT:
        force = measure_force(torch, stag, ctx, cfg, srcs, packed, prec, recon, vh)
        force["pct_of_measured"] = 100 * force["gbs_algorithmic"] / peak

    # ---- cpu_baseline: the oracle on this box's host cores, bounded sample (rank 0, N = 1 only) ----
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        g, s_it, m = oracle_sample(cfg, U, srcs[0], 12.0)
        cpu = {"value": g, "unit": "GFLOP/s", "cores": 1, "kind": "oracle",
               "sample": "%d oracle multi-shift CG iterations (maxiter=%d) of the same %d-shift solve, %.3f s/iteration"
                         % (m, m, nshift, s_it)}

    if rank == 0:
        iters = [i["iters"] for i in infos]
        cg_gbs = tot_bytes_site * vh / secs / 1e9
        out = {"metric": METRIC, "value": value, "unit": "GFLOP/s", "n_gpus": world, "steps": args.steps,
               "warmup": args.warmup, "ms_per_step": secs * 1e3 / args.steps, "higher_is_better": True,
               "scaling": "weak", "vs_baseline": None, "dtype": "f32" if args.prec == "f32" else "f64", "data": "synthetic",
               "config": dict(workload_config(cfg, args.workload, prec, recon),
                              l2="working set (2 link sets + %d vectors = %.0f MB) larger than the 126 MB L2; no flush"
                                 % (2 * nshift + 4, (ctx.gauge_packed_bytes(prec, recon) + (2 * nshift + 4) * vb) / 1e6)),
               "cg": {"s_per_solve": secs / args.steps, "iters": iters, "us_per_iter": secs / (tot_iters / world) * 1e6,
                      "gbs_algorithmic": cg_gbs, "pct_of_8tbs": 100 * cg_gbs / NOMINAL_HBM_GBS,
                      "pct_of_measured": 100 * cg_gbs / peak, "solves": nsolves,
                      "iters_shift_first_solve": infos[0]["iters_shift"]},
               "dslash": dslash, "block": block, "mixed": mixed, "force": force, "roofline": roof, "roofline_dslash": roof_dslash, "cpu_baseline": cpu,
               "e2e": {"value": e2e_value, "unit": "GFLOP/s", "h2d_bytes_per_step": n6 * 8,
                       "d2h_bytes_per_step": nshift * n6 * 8, "s_per_solve": te_s / e2e_steps,
                       "call": "stag_mshift_cg_host (pinned host source in, host solutions out)"},
               "gpu_launches": int(launches), "options": args.opt, "clocks": clk, "pack_ms": pack_ms, "input_gen_s": gen_s}
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=8)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c4", choices=sorted(WORKLOADS))
    ap.add_argument("--prec", default="f64", choices=["f64", "f32", "f64split"],
                    help="f64split = N3: fp64 vectors on split-double (b + c) links")
    ap.add_argument("--recon", type=int, default=18, choices=[18, 12])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-block", action="store_true", help="skip the N1 multi-source and N2/N3 mixed-precision measurements")
    ap.add_argument("--ref-seconds", type=float, default=150.0,
                    help="--impl reference: total oracle time budget over all steps")
    ap.add_argument("--dslash-only", action="store_true", help="Dslash bandwidth sweep only (no CG)")
    ap.add_argument("--dslash-launches", type=int, default=100)
    ap.add_argument("--opt", action="append", default=[], metavar="KEY=INT",
                    help="stag_set_option knob, e.g. cg_persistent=0 (repeatable)")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3                       # timing rule: W >= 3
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
