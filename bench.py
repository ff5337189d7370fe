#!/usr/bin/env python
"""bench.py — staggered Dslash + multi-shift CG on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c4|c5|c3|c2|t2b|t2c] [--impl reference]

One STEP = one pass of the whole hot path over one synthetic
pseudo-fermion source: one multi-shift CG solve of (m^2 - D_eo D_oe + sigma_i) x_i = b with all its
Dslash applications, reductions, scalar recurrences and shift updates.  Row a1 (gauge pack) is
setup, done once and reported as `pack_ms`.

The BASELINE metric has three figures; all three are first-class keys of the ONE JSON line (rank 0):
  value / dslash_gflops_through_solve   Dslash GFLOP/s (570 flop/site) sustained through the timed solves
  dslash_gflops_standalone              the same kernel timed alone (100-launch ping-pong), fp64-18
  cg_s_per_solve                        multi-shift CG time to solution
`roofline` is the dominant kernel of the step; `roofline.also[]` carries one entry per other kernel this run
timed — the Dslash storage variants, the fp32 / 12-real solves, the block (N1) kernel, the force (N4), and the
64^4 section (config 5: the largest single-GPU configuration, multi-kernel CG path) — each with its own
algorithmic bytes, live CUDA-event duration, and the DRAM traffic of the committed ncu capture of the kernel
of that NAME (profiles/traffic.csv; `traffic_stale` if the run launched a kernel the capture does not know).
"""
from __future__ import annotations

import argparse
import json
import os
import re
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
METRIC = "Dslash GFLOP/s (570 flop/site) sustained through the multi-shift CG solve; CG s/solve beside it"


def measured_peak_gbs():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"


# ---------------------------------------------------------------------------------------------
# committed ncu traffic, looked up by KERNEL NAME
# ---------------------------------------------------------------------------------------------
def norm_kernel(name: str) -> str:
    """One spelling for a kernel name, whether it comes from ncu ("void stag::k<double, (int)18, (bool)0>(stag::Geom,
    ...)") or from abi::__cxa_demangle via stag_kernel_log ("void stag::k<double, 18, false>(stag::Geom, ...)")."""
    n = name.strip()
    n = re.sub(r"^void\s+", "", n)
    depth, cut = 0, len(n)
    for i, ch in enumerate(n):                        # drop the parameter list: the first '(' outside <...>
        if ch == "<":
            depth += 1
        elif ch == ">":
            depth -= 1
        elif ch == "(" and depth == 0:
            cut = i
            break
    n = n[:cut]
    n = re.sub(r"\((?:int|bool|unsigned int|unsigned|long)\)", "", n)
    n = n.replace("stag::", "").replace(" ", "").replace("false", "0").replace("true", "1")
    return n


_CSRC_SHA = None


def csrc_sha() -> str:
    """Fingerprint of the CUDA sources the library is built from (csrc/*.cu, *.cuh, include/stag.h): a traffic.csv
    row is evidence for the kernels of exactly these sources.  (No git on the GPU box: the snapshot has no .git.)"""
    global _CSRC_SHA
    if _CSRC_SHA is None:
        import glob
        import hashlib
        h = hashlib.sha256()
        csrc = os.path.join(ROOT, "paper_1010_5433_b200", "csrc")
        for f in sorted(glob.glob(os.path.join(csrc, "*.cu")) + glob.glob(os.path.join(csrc, "*.cuh"))) + \
                [os.path.join(ROOT, "include", "stag.h")]:
            h.update(os.path.basename(f).encode() + b"\0")
            with open(f, "rb") as fh:
                h.update(fh.read())
        _CSRC_SHA = h.hexdigest()[:12]
    return _CSRC_SHA


def load_traffic():
    import csv
    rows = []
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.csv"), newline="") as f:
            for row in csv.DictReader(f):
                row["_k"] = norm_kernel(row["kernel"])
                rows.append(row)
    except Exception:
        pass
    return rows


_TRAFFIC = None


def committed_traffic(workload: str, kernel: str, variant: str = ""):
    """(dram bytes per launch, stale flag).  The row must be for this workload and for a kernel of exactly the
    name the run launched (`kernel` comes from stag_kernel_log); a capture of another build of the kernel — other
    template arguments — is NOT returned: (None, True).  `variant` disambiguates rows of one kernel name whose
    traffic depends on run-time arguments (e.g. the number of sources of the block kernel).  A row captured from
    other sources than the ones in the tree (its `csrc_sha` differs from csrc_sha(): the kernel may have been
    rewritten under the same name) is returned WITH the stale flag."""
    global _TRAFFIC
    if _TRAFFIC is None:
        _TRAFFIC = load_traffic()
    k = norm_kernel(kernel)
    for row in _TRAFFIC:
        if row["workload"] == workload and row["_k"] == k and (not variant or row.get("variant", "") == variant):
            return int(row["dram_bytes_per_launch"]), row.get("csrc_sha", "") != csrc_sha()
    return None, True


def launched(ctx, pattern: str) -> str:
    """Name (as stag_kernel_log gives it) of the one kernel matching `pattern` launched since the last reset."""
    names = [n for n in ctx.kernel_log() if re.search(pattern, n)]
    return names[0] if names else "?"


_READ_PEAK = None


def read_stream_gbs(torch, nbytes: int = 4 << 30, repeats: int = 10):
    """A second yardstick beside MEASURED_PEAKS.json's copy bandwidth (read-dominated kernels exceed the
    copy figure, which mixes reads and writes): GB/s of a READ-ONLY stream over 4 GiB, best of `repeats`, timed with
    CUDA events.  The probe is a torch reduction (a library kernel used as a ruler only, as the driver's copy_ is);
    nothing of the product path runs in it.  Measured once per process."""
    global _READ_PEAK
    if _READ_PEAK is None:
        a = torch.ones(nbytes // 4, dtype=torch.float32, device="cuda")
        best = float("inf")
        for _ in range(repeats + 2):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            a.sum()
            e1.record()
            torch.cuda.synchronize()
            best = min(best, e0.elapsed_time(e1) * 1e-3)
        del a
        torch.cuda.empty_cache()
        _READ_PEAK = nbytes / best / 1e9
    return _READ_PEAK


def roof_entry(workload, kernel, what, alg_bytes, secs_per_launch, peak, peak_src, variant="", **extra):
    gbs = alg_bytes / secs_per_launch / 1e9
    traffic, stale = committed_traffic(workload, kernel, variant)
    e = {"bound": "hbm", "kernel": norm_kernel(kernel), "what": what, "workload": workload, "achieved": gbs, "peak": peak,
         "unit": "GB/s", "frac": gbs / peak, "peak_source": peak_src, "frac_of_8tbs": gbs / NOMINAL_HBM_GBS,
         "algorithmic_bytes_per_launch": alg_bytes, "avg_launch_us": secs_per_launch * 1e6, "traffic": traffic}
    if _READ_PEAK:
        e["frac_read"] = gbs / _READ_PEAK                  # against the read-only stream (never the headline `frac`)
    if stale:
        e["traffic_stale"] = True
    if traffic:
        e["frac_dram"] = traffic / secs_per_launch / 1e9 / peak     # real HBM traffic of the capture / live time / peak
        if e["frac_dram"] > 1.0:
            e["frac_dram_note"] = ("the capture is cold-cache and serialised; in the live back-to-back run part of these bytes "
                                   "(the vector the previous launch wrote) comes from L2, and a read-only stream exceeds the copy figure")
    e.update(extra)
    return e


# ---------------------------------------------------------------------------------------------
# the ONE line the driver reads: short (< 6 KB), strict JSON, last on stdout.  Everything else the run
# measured goes to the --detail file (round 2's 27 KB line was not parsed by the driver).
# ---------------------------------------------------------------------------------------------
HEADLINE_LIMIT = 6144
# which roofline.also[] entries the headline carries, in this order (at most 10): (workload, tag)
HEADLINE_ALSO = (("c4", "solve:f32-12"), ("c4", "block_cg:f64-18"), ("c4", "force:f64-18"), ("c4", "force:f32-18"),
                 ("c4", "ring4:f64-18"), ("c5", "dslash:f64-18"), ("c5", "a2"), ("c5", "a3"), ("c5", "a5"), ("c5", "a6"))


def _sig(v, n=5):
    """floats to n significant digits (shorter line); non-finite floats to None (strict JSON)."""
    if isinstance(v, float):
        if v != v or v in (float("inf"), float("-inf")):
            return None
        return float("%.*g" % (n, v))
    if isinstance(v, dict):
        return {k: _sig(x, n) for k, x in v.items()}
    if isinstance(v, (list, tuple)):
        return [_sig(x, n) for x in v]
    return v


def compact_entry(e: dict) -> dict:
    out = {k: e.get(k) for k in ("workload", "tag", "kernel", "frac", "frac_read", "avg_launch_us", "traffic", "frac_dram")}
    if e.get("traffic_stale"):
        out["traffic_stale"] = True
    return out


def headline(full: dict) -> dict:
    """The driver-facing line from the full measurement dict of run_ours: the bench contract's keys, the roofline of
    the step's dominant kernel with <= 10 compact also[] entries, the c5 (64^4) summary, cpu_baseline, e2e, clocks."""
    keep = ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
            "vs_baseline", "dtype", "data", "config", "l2", "dslash_gflops_standalone", "cg_s_per_solve", "gpu_launches")
    h = {k: full.get(k) for k in keep}
    roof = full.get("roofline") or {}
    also = roof.get("also") or []
    picked = []
    for wl, tag in HEADLINE_ALSO:
        e = next((e for e in also if e.get("workload") == wl and e.get("tag") == tag), None)
        if e is not None:
            picked.append(compact_entry(e))
    if not picked:                                       # other workloads / precisions: the first entries as they come
        picked = [compact_entry(e) for e in also[:10]]
    h["roofline"] = {k: roof.get(k) for k in ("bound", "kernel", "achieved", "peak", "unit", "frac", "frac_of_8tbs",
                                               "algorithmic_bytes_per_launch", "avg_launch_us", "traffic", "frac_dram",
                                               "equivalent_gbs", "bytes_model", "peak_source", "frac_read")}
    h["roofline"]["read_stream_gbs"] = full.get("read_stream_gbs")
    if roof.get("traffic_stale"):
        h["roofline"]["traffic_stale"] = True
    h["roofline"]["also"] = picked[:10]
    c5 = full.get("c5")
    if c5 and c5.get("cg"):
        cg = c5["cg"]
        h["c5"] = {"workload": c5.get("workload"), "s_per_solve": cg.get("s_per_solve"), "iters": cg.get("iters"),
                   "gbs_algorithmic": cg.get("gbs_algorithmic"),
                   "frac": (cg.get("pct_of_measured") or 0.0) / 100.0, "timed_solves": cg.get("timed_solves"),
                   "gflops_through_solve": cg.get("gflops_through_solve")}
    else:
        h["c5"] = None
    h["cpu_baseline"] = full.get("cpu_baseline")
    e2e = full.get("e2e") or {}
    h["e2e"] = {k: e2e.get(k) for k in ("value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step", "s_per_solve")}
    clk = full.get("clocks")
    if isinstance(clk, dict):
        clk = {k: v for k, v in clk.items() if k in ("sm_mhz", "sm_max_mhz", "reasons", "samples", "power_w_max")}
    h["clocks"] = clk
    h["detail"] = full.get("detail_file")
    return _sig(h)


def headline_line(full: dict) -> str:
    line = json.dumps(headline(full), allow_nan=False, separators=(",", ":"))
    if len(line) >= HEADLINE_LIMIT:                     # never print a line the driver may not read: drop also[] first
        h = headline(full)
        h["roofline"]["also"] = h["roofline"]["also"][:4]
        line = json.dumps(h, allow_nan=False, separators=(",", ":"))
    return line


BYTES_MODEL = {0: "2D + 5 vec + 4 vec N_live", 2: "2D + 4 vec N_live (r, q in shared memory)",
               3: "2D - 2 vec + 4 vec N_live (r, q, p_base in shared memory)"}


def cg_bytes_per_site(prec, recon, iters, iters_shift, resident=0):
    """Algorithmic bytes of one solve per even site.  resident = 0, the multi-kernel path, per
    iteration: 2 Dslash + p re-read (a3) + r,q,r (a5) + r (a6), plus x_i,p_i read+write for every iteration shift i was
    live: 2D + 5 vec + 4 vec N.  resident = 3 (True), the persistent kernel with r, q, p_base in shared memory: q is never
    written to memory, p, r, q are never re-read from it, and the base shift only writes p: 2D - 2 vec + 4 vec N.
    resident = 2, r and q in shared memory but p_base in global memory (e.g. 4 x 48^3): as 3 plus the own-site read of
    p in a3 and in the base shift's update: 2D + 4 vec N."""
    w = 4 if prec == 1 else 8
    vec = 6 * w
    extra = {0: 5 * vec, 2: 0, 3: -2 * vec}[3 if resident is True else int(resident)]
    return iters * (2 * DSLASH_BYTES[(prec, recon)] + extra) + sum(iters_shift) * 4 * vec


def resident_slices(vh, prec, num_sms=148):
    """Mirror of launch_persistent's residency rule (csrc/stag_cg_persist.cuh): how many of r, q, p_base the persistent
    kernel keeps in its 200 KB of shared memory (it runs with 2 or 3; below 2 the multi-kernel path is taken)."""
    w = 4 if prec == 1 else 8
    tiles = (vh + 31) // 32
    grid = min(num_sms, tiles)
    slots = 32 * ((tiles + grid - 1) // grid)
    return min(3, (200 * 1024) // (slots * 6 * w))


def fully_resident(vh, prec, num_sms=148):
    return resident_slices(vh, prec, num_sms) == 3


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


def timed_call(torch, fn, repeats=2):
    """CUDA events around fn(); the LAST of `repeats` calls is the one reported (the others warm up)."""
    out = None
    for _ in range(repeats):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        out = fn()
        e1.record()
        torch.cuda.synchronize()
    return e0.elapsed_time(e1) * 1e-3, out


def dslash_variants(torch, stag, ctx, wl, U, srcs, vh, peak, peak_src, launches, have=None):
    """The Dslash bandwidth sweep over the storage variants; returns (table, roofline entries)."""
    table, entries = {}, []
    canon = None
    for p_, r_ in VARIANTS:
        if have is not None and (p_, r_) in have:
            pk = have[(p_, r_)]
        else:
            if canon is None:
                canon = ctx.alloc(ctx.gauge_canonical_bytes())
                ctx.gauge_load(U, canon)
                torch.cuda.synchronize()
            pk = ctx.alloc(ctx.gauge_packed_bytes(p_, r_))
            ctx.gauge_pack(canon, pk, p_, r_)
        vp = stag.F32 if p_ == stag.F32 else stag.F64
        a, b = ctx.upload_vector(srcs[0], vp), ctx.alloc(ctx.vector_bytes(vp))
        ctx.kernel_log_reset()
        s_per = time_dslash(torch, ctx, pk, p_, r_, a, b, launches=launches)
        kern = launched(ctx, r"dslash_kernel")
        name = "%s-%d" % (PREC_NAME[p_], r_)
        gbs = DSLASH_BYTES[(p_, r_)] * vh / s_per / 1e9
        table[name] = {"us": s_per * 1e6, "gflops": FLOP_PER_SITE * vh / s_per / 1e9, "gbs_algorithmic": gbs,
                       "pct_of_8tbs": 100 * gbs / NOMINAL_HBM_GBS, "pct_of_measured": 100 * gbs / peak,
                       "bytes_per_site": DSLASH_BYTES[(p_, r_)]}
        entries.append(roof_entry(wl, kern, "stag_dslash_oe/eo %s, %d launches ping-pong replayed as a CUDA graph" % (name, launches),
                                  DSLASH_BYTES[(p_, r_)] * vh, s_per, peak, peak_src, variant=name, tag="dslash:" + name,
                                  gflops=FLOP_PER_SITE * vh / s_per / 1e9))
        del pk, a, b
    del canon
    return table, entries


def measure_solve(torch, stag, ctx, wl, cfg, packed, prec, recon, src, vh, peak, peak_src, stop=None, warm=1, opts=()):
    """One timed stag_mshift_cg solve (after `warm` untimed ones) of a storage variant; returns (dict, roofline entry)."""
    shifts, n = cfg["shifts"], len(cfg["shifts"])
    vp = stag.F32 if prec == stag.F32 else stag.F64
    vb = ctx.vector_bytes(vp)
    b = ctx.upload_vector(src, vp)
    x, ws = ctx.alloc(n * vb), ctx.alloc(ctx.cg_workspace_bytes(prec, n))
    stop = cfg["stops"][0] if stop is None else stop
    ctx.kernel_log_reset()
    secs, (rc, info) = timed_call(torch, lambda: ctx.mshift_cg(packed, prec, recon, b, cfg["mass"], shifts, stop, 100000, x, ws),
                                  repeats=warm + 1)
    persistent = info["kernel_launches"] == 1
    name = "%s-%d" % (PREC_NAME[prec], recon)
    resident = resident_slices(vh, prec) if persistent else 0
    resident = resident if resident >= 2 else 0        # (cg_resident_slices < 2 is a test knob: reported with the multi-kernel bytes)
    own = cg_bytes_per_site(prec, recon, info["iters"], info["iters_shift"], resident) * vh
    equiv = cg_bytes_per_site(prec, recon, info["iters"], info["iters_shift"], 0) * vh
    d = {"rc": rc, "s_per_solve": secs, "iters": info["iters"], "us_per_iter": secs / max(info["iters"], 1) * 1e6,
         "converged": info["converged"], "stagnated": info["stagnated"], "path": "persistent" if persistent else "multi-kernel",
         "gflops_through_solve": 2 * FLOP_PER_SITE * vh * info["iters"] / secs / 1e9,
         "gbs_algorithmic": own / secs / 1e9, "pct_of_measured": 100 * own / secs / 1e9 / peak,
         "equivalent_gbs": equiv / secs / 1e9, "sum_iters_shift": sum(info["iters_shift"])}
    if persistent:
        kern = launched(ctx, r"cg_persistent(_sr)?_kernel")
        e = roof_entry(wl, kern, "stag_mshift_cg %s: one launch = one %d-shift solve (%d iterations)" % (name, n, info["iters"]),
                       own, secs, peak, peak_src, variant=name, tag="solve:" + name, iters=info["iters"], us_per_iter=d["us_per_iter"],
                       equivalent_gbs=equiv / secs / 1e9,
                       bytes_model=BYTES_MODEL[resident] + " per site and iteration")
    else:
        e = None
    return d, e


def measure_block(torch, stag, ctx, wl, cfg, srcs, packed, prec, recon, vh, peak, peak_src):
    """N1: stag_dslash_block for R = 1, 2, 4 sources (100-launch ping-pong, as time_dslash) and ONE
    stag_mshift_cg_block solve of min(4, nsrc) sources.  Algorithmic bytes per site of a block Dslash =
    8 links (once) + R x (one read of the source + one write)."""
    w = 4 if prec == stag.F32 else 8
    vb = ctx.vector_bytes(prec)
    out = {"dslash": {}, "cg": None}
    entries = []
    name = "%s-%d" % (PREC_NAME[prec], recon)
    for R in (1, 2, 4):
        if R > len(srcs):
            continue
        a, b = ctx.upload_vectors(srcs[:R], prec), ctx.alloc(R * vb)

        def pair(n):
            for _ in range(n // 2):
                ctx.dslash_block(packed, prec, recon, 1, R, a, b)
                ctx.dslash_block(packed, prec, recon, 0, R, b, a)
        pair(10)
        ctx.kernel_log_reset()
        s_per = time_launches(torch, pair, 100)
        bps = 8 * recon * w + 2 * 6 * w * R
        gbs = bps * vh / s_per / 1e9
        out["dslash"]["R%d" % R] = {"us": s_per * 1e6, "us_per_source": s_per * 1e6 / R,
                                    "gflops": FLOP_PER_SITE * vh * R / s_per / 1e9, "bytes_per_site": bps,
                                    "gbs_algorithmic": gbs, "pct_of_measured": 100 * gbs / peak}
        if R == 4:
            entries.append(roof_entry(wl, launched(ctx, r"dslash_(pipe|block)_kernel"),
                                      "stag_dslash_block %s, 4 sources through one link read" % name, bps * vh, s_per,
                                      peak, peak_src, variant=name + "-R4", tag="ring4:" + name,
                                      gflops=FLOP_PER_SITE * vh * 4 / s_per / 1e9))
        del a, b
    R = min(4, len(srcs))
    n = len(cfg["shifts"])
    stop = cfg["stops"][0] if prec != stag.F32 else max(cfg["stops"][0], 1e-5)
    bdev = ctx.upload_vectors(srcs[:R], prec)
    x = ctx.alloc(R * n * vb)
    ws = ctx.alloc(ctx.cg_block_workspace_bytes(prec, n, R))
    ctx.kernel_log_reset()
    secs, (rc, infos) = timed_call(torch, lambda: ctx.mshift_cg_block(packed, prec, recon, R, bdev, cfg["mass"], cfg["shifts"],
                                                                      stop, 100000, x, ws))
    its = [i["iters"] for i in infos]
    # per source and iteration: links / R twice + the vector traffic of the multi-kernel formula (nothing of q, p
    # is resident at R = 4; r is) — reported with the single-source multi-kernel formula so that it compares
    vec = 6 * w
    alg = vh * sum(i["iters"] * (2 * (8 * recon * w / R + 2 * vec) + 5 * vec) + sum(i["iters_shift"]) * 4 * vec for i in infos)
    out["cg"] = {"nrhs": R, "rc": rc, "s_per_block_solve": secs, "s_per_source": secs / R, "iters": its,
                 "us_per_iter": secs / max(its) * 1e6, "stop": stop,
                 "gflops": 2 * FLOP_PER_SITE * vh * sum(its) / secs / 1e9,
                 "gbs_algorithmic": alg / secs / 1e9, "pct_of_measured": 100 * alg / secs / 1e9 / peak,
                 "call": "stag_mshift_cg_block (one persistent launch, links read once per Dslash for all sources)"}
    entries.append(roof_entry(wl, launched(ctx, r"cg_persistent(_block)?_kernel"),
                              "stag_mshift_cg_block %s: one launch = %d sources x %d shifts" % (name, R, n), alg, secs,
                              peak, peak_src, variant=name + "-R%d" % R, tag="block_cg:" + name,
                              us_per_iter=out["cg"]["us_per_iter"]))
    return out, entries


def measure_mixed(torch, stag, ctx, cfg, U, srcs, vh, fp64_s_per_solve):
    """N2 + N3: stag_mshift_cg_mixed with DEFAULT options (fp64 stages on the native fp64 links, fp32 stages on the b
    planes of a split-double buffer) against stag_mshift_cg in fp64 on the same fp64 links, for the lightest 1, 2, 4,
    8, 16 shifts of the workload, same source and stop; the call picks its route (1 residual replacement | 2 fp32 +
    polish | 3 the fp64 multi-shift solve itself, plus the true-residual check).  Then, for the record, everything on
    ONE resident split-double buffer (N3: its fp64 stages read b + c), and the fp32 + polish route forced at all shifts."""
    n = len(cfg["shifts"])
    split = ctx.upload_gauge(U, stag.F64_SPLIT, 18)
    p64 = ctx.upload_gauge(U, stag.F64, 18)
    vb = ctx.vector_bytes(stag.F64)
    b = ctx.upload_vector(srcs[0], stag.F64)
    x = ctx.alloc(n * vb)
    ws = ctx.alloc(ctx.mshift_cg_mixed_workspace_bytes(n))
    cgws = ctx.alloc(ctx.cg_workspace_bytes(stag.F64, n))
    out = {"by_nshift": {}}
    for k in sorted({1, 2, 4, 8, n} & set(range(1, n + 1))):
        sh = cfg["shifts"][:k]
        t64, (rc64, i64) = timed_call(torch, lambda: ctx.mshift_cg(p64, stag.F64, 18, b, cfg["mass"], sh, cfg["stops"][0], 100000, x, cgws))
        tm, (rc, info) = timed_call(torch, lambda: ctx.mshift_cg_mixed(p64, stag.F64, 18, split, 18, b, cfg["mass"], sh,
                                                                       cfg["stops"][0], 100000, x, ws))
        out["by_nshift"][str(k)] = {
            "rc": rc, "route": info["route"], "s_per_solve": tm, "fp64_s_per_solve": t64, "vs_fp64_multishift": t64 / tm,
            "inner_iters": info["inner"]["iters"], "fp64_iters": i64["iters"], "reliable_updates": info["reliable_updates"],
            "polish_iters": sum(info["polish"]["iters"]), "true_resid_final": max(info["polish"]["resid_after"])}
    secs, (rc, info) = timed_call(torch, lambda: ctx.mshift_cg_mixed(split, stag.F64_SPLIT, 18, split, 18, b, cfg["mass"], cfg["shifts"],
                                                                     cfg["stops"][0], 100000, x, ws))
    out["one_split_buffer_all_shifts"] = {"rc": rc, "route": info["route"], "s_per_solve": secs,
                                          "vs_fp64_multishift_native_links": fp64_s_per_solve / secs,
                                          "true_resid_final": max(info["polish"]["resid_after"])}
    ctx.set_option("cg_mixed_fp64_from", 0)
    secs, (rc, info) = timed_call(torch, lambda: ctx.mshift_cg_mixed(split, stag.F64_SPLIT, 18, split, 18, b, cfg["mass"], cfg["shifts"],
                                                                     cfg["stops"][0], 100000, x, ws))
    ctx.set_option("cg_mixed_fp64_from", 3)
    out["forced_fp32_plus_polish_all_shifts"] = {
        "rc": rc, "route": info["route"], "s_per_solve": secs, "vs_fp64_multishift": fp64_s_per_solve / secs,
        "inner_fp32_iters": info["inner"]["iters"], "polish_iters": sum(info["polish"]["iters"]),
        "polish_passes": info["polish"]["passes"], "true_resid_after_fp32": max(info["polish"]["resid_before"]),
        "true_resid_final": max(info["polish"]["resid_after"]),
        "kernel_launches": info["inner"]["kernel_launches"] + info["polish"]["kernel_launches"]}
    return out


def measure_force(torch, stag, ctx, wl, cfg, srcs, packed, prec, recon, vh, peak, peak_src):
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
    ctx.kernel_log_reset()
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
    # the D_oe launches of the call, timed alone, so that the force kernel proper gets its own figure
    vb = ctx.vector_bytes(prec)

    def dsl(k):
        for _ in range(k):
            ctx.dslash_block(packed, prec, recon, 1, n, x, ws)      # the call stag_fermion_force makes: all groups, one launch
    dsl(2)
    s_dsl = time_launches(torch, dsl, 10)
    s_force = max(secs - s_dsl, 1e-9)
    name = "%s-%d" % (PREC_NAME[prec], recon)
    d = {"us_per_call": secs * 1e6, "nshift": n, "launches_per_call": 2, "us_dslash_launches": s_dsl * 1e6,
         "us_force_kernel": s_force * 1e6, "algorithmic_bytes_per_call": bytes_dslash + bytes_force,
         "gbs_algorithmic": gbs, "pct_of_measured": 100 * gbs / peak}
    e = roof_entry(wl, launched(ctx, r"force_kernel"),
                   "stag_fermion_force %s, %d shifts: the force kernel proper (call minus its D_oe launch of %d groups, timed alone)"
                   % (name, n, groups), bytes_force, s_force, peak, peak_src, variant=name, tag="force:" + name,
                   us_per_call=secs * 1e6,
                   call_gbs_algorithmic=gbs, call_frac=gbs / peak)
    return d, e


def c5_section(torch, stag, args, peak, peak_src):
    """Config 5 (64^4: the largest single-GPU configuration of BASELINE.json:configs; the multi-kernel CG path):
    the Dslash sweep, the MEDIAN of --c5-solves (3) timed 8-shift solves after a 32-iteration warm-up call, and the four kernels of an
    iteration timed one by one with CUDA events (option cg_profile, a separate 48-iteration call)."""
    import stag_inputs as si
    wl = "c5"
    cfg = si.get_config(WORKLOADS[wl])
    L, vh = cfg["L"], int(np.prod(cfg["L"])) // 2
    U, srcs, gen_s = make_inputs(cfg)
    ctx = stag.Stag(L)
    for kv in args.opt:
        k, v = kv.split("=")
        ctx.set_option(k, int(v))
    canon = ctx.alloc(ctx.gauge_canonical_bytes())
    ctx.gauge_load(U, canon)
    torch.cuda.synchronize()
    p64 = ctx.alloc(ctx.gauge_packed_bytes(stag.F64, 18))
    secs_pack, _ = timed_call(torch, lambda: ctx.gauge_pack(canon, p64, stag.F64, 18), repeats=1)
    del canon
    out = {"workload": WORKLOADS[wl], "input_gen_s": gen_s, "pack_ms": secs_pack * 1e3, "vh": vh}
    entries = []
    # ---- CG: fp64-18, 8 shifts, stop 1e-9
    shifts, n = cfg["shifts"], len(cfg["shifts"])
    vb = ctx.vector_bytes(stag.F64)
    b = ctx.upload_vector(srcs[0], stag.F64)
    x, ws = ctx.alloc(n * vb), ctx.alloc(ctx.cg_workspace_bytes(stag.F64, n))
    ctx.kernel_log_reset()            # before the warm-up: it captures the CUDA graph the timed solve only replays
    ctx.mshift_cg(p64, stag.F64, 18, b, cfg["mass"], shifts, cfg["stops"][0], 32, x, ws)          # warm-up: 32 iterations
    runs = [timed_call(torch, lambda: ctx.mshift_cg(p64, stag.F64, 18, b, cfg["mass"], shifts, cfg["stops"][0],
                                                    100000, x, ws), repeats=1) for _ in range(max(1, args.c5_solves))]
    secs, (rc, info) = sorted(runs, key=lambda t: t[0])[len(runs) // 2]          # the median solve
    alg = cg_bytes_per_site(0, 18, info["iters"], info["iters_shift"]) * vh
    out["cg"] = {"rc": rc, "s_per_solve": secs, "iters": info["iters"], "us_per_iter": secs / max(info["iters"], 1) * 1e6,
                 "gflops_through_solve": 2 * FLOP_PER_SITE * vh * info["iters"] / secs / 1e9,
                 "gbs_algorithmic": alg / secs / 1e9, "pct_of_measured": 100 * alg / secs / 1e9 / peak,
                 "timed_solves": len(runs), "s_per_solve_all": [t[0] for t in runs],
                 "kernel_launches": info["kernel_launches"], "iters_shift": info["iters_shift"],
                 "path": "multi-kernel (4 launches per iteration, CUDA-graph replay)"}
    names = ctx.kernel_log()
    pick = lambda pat: next((k for k in names if re.search(pat, k)), "?")
    # dslash_kernel<T, RECON, BLOCK, MODE, RT, SPLIT>: MODE 1 = a2 (D_oe inside the CG), MODE 2 = a3 (fused D_eo)
    k_a2, k_a3 = pick(r"dslash_kernel<[^,]+, ?\d+, ?\d+, ?1,"), pick(r"dslash_kernel<[^,]+, ?\d+, ?\d+, ?2,")
    k_a5, k_a6 = pick(r"cg_update_r_kernel"), pick(r"cg_update_shifts_kernel")
    # the four kernels one by one (first 40 iterations: every shift still live)
    ctx.set_option("cg_profile", 1)
    ctx.mshift_cg(p64, stag.F64, 18, b, cfg["mass"], shifts, cfg["stops"][0], 48, x, ws)
    ctx.set_option("cg_profile", 0)
    us, nit = ctx.cg_profile()
    out["cg"]["profile_us"] = {"a2_dslash_oe": us[0], "a3_dslash_eo_fused": us[1], "a5_update_r": us[2], "a6_update_shifts": us[3],
                               "iterations_averaged": nit, "live_shifts": n}
    if nit > 0:
        vec = 48
        for kern, what, bytes_site, t in ((k_a2, "a2: w = D_oe p", 1248, us[0]), (k_a3, "a3: q = c0 p - D_eo w, <p,q>", 1248 + vec, us[1]),
                                          (k_a5, "a5: r -= alpha q, <r,r>", 3 * vec, us[2]),
                                          (k_a6, "a6: all-shift update, %d live shifts" % n, vec + 4 * vec * n, us[3])):
            entries.append(roof_entry(wl, kern, "stag_mshift_cg f64-18 multi-kernel path, " + what + " (CUDA events around each launch)",
                                      bytes_site * vh, t * 1e-6, peak, peak_src, variant="f64-18", tag=what[:2]))
    del x, ws, b
    # ---- Dslash sweep
    table, ents = dslash_variants(torch, stag, ctx, wl, U, srcs, vh, peak, peak_src, args.dslash_launches,
                                  have={(stag.F64, 18): p64})
    out["dslash"] = table
    return out, ents + entries


def ncu_pass(args, torch, stag, ctx, cfg, U, srcs, vh):
    """--ncu-pass: every kernel the default run reports, launched a FEW times each in the launch configuration the
    timed sections use, so that ONE `ncu --set full -k regex:...` run over this command captures them all (the
    source of profiles/traffic.csv; the command is in profiles/README.md).  Nothing is timed.  Prints one JSON line
    listing the calls made and the kernels each launched (names as stag_kernel_log reports them)."""
    wl, seq = args.workload, []
    n = len(cfg["shifts"])

    def note(what, **kw):
        torch.cuda.synchronize()
        seq.append(dict(call=what, kernels=[norm_kernel(k) for k in ctx.kernel_log()], **kw))
        ctx.kernel_log_reset()

    ctx.kernel_log_reset()
    packs = {}
    for p_, r_ in VARIANTS:
        if wl == "c5" and (p_, r_) != (stag.F64, 18):
            pk = ctx.upload_gauge(U, p_, r_)
        else:
            pk = packs[(p_, r_)] = ctx.upload_gauge(U, p_, r_)
        vp = stag.F32 if p_ == stag.F32 else stag.F64
        a, b = ctx.upload_vector(srcs[0], vp), ctx.alloc(ctx.vector_bytes(vp))
        ctx.kernel_log_reset()
        for _ in range(2):
            ctx.dslash_oe(pk, p_, r_, a, b)
            ctx.dslash_eo(pk, p_, r_, b, a)
        note("stag_dslash_oe/eo x2", variant="%s-%d" % (PREC_NAME[p_], r_))
        del pk, a, b
    # ---- the solves: persistent path = one launch each; multi-kernel path (c5) = --ncu-iters iterations
    maxiter = 100000 if wl != "c5" else args.ncu_iters
    for p_, r_ in ((stag.F64, 18), (stag.F64, 12), (stag.F32, 18), (stag.F32, 12)):
        if (p_, r_) not in packs:
            continue
        vp = stag.F32 if p_ == stag.F32 else stag.F64
        vb = ctx.vector_bytes(vp)
        b = ctx.upload_vector(srcs[0], vp)
        x, ws = ctx.alloc(n * vb), ctx.alloc(ctx.cg_workspace_bytes(p_, n))
        ctx.kernel_log_reset()
        rc, info = ctx.mshift_cg(packs[(p_, r_)], p_, r_, b, cfg["mass"], cfg["shifts"], cfg["stops"][0], maxiter, x, ws)
        note("stag_mshift_cg", variant="%s-%d" % (PREC_NAME[p_], r_), rc=rc, iters=info["iters"],
             sum_iters_shift=sum(info["iters_shift"]), kernel_launches=info["kernel_launches"])
        del b, x, ws
    if wl != "c5" and len(srcs) >= 4:
        # ---- N1 (fp64, and fp32 = the MD precision)
        for p_ in (stag.F64, stag.F32):
            pk = packs[(p_, 18)]
            vb = ctx.vector_bytes(p_)
            var = "%s-18-R4" % PREC_NAME[p_]
            a, b = ctx.upload_vectors(srcs[:4], p_), ctx.alloc(4 * vb)
            ctx.kernel_log_reset()
            ctx.dslash_block(pk, p_, 18, 1, 4, a, b)
            ctx.dslash_block(pk, p_, 18, 0, 4, b, a)
            note("stag_dslash_block R=4 x2", variant=var)
            x, ws = ctx.alloc(4 * n * vb), ctx.alloc(ctx.cg_block_workspace_bytes(p_, n, 4))
            bdev = ctx.upload_vectors(srcs[:4], p_)
            stop = cfg["stops"][0] if p_ == stag.F64 else max(cfg["stops"][0], 1e-5)
            ctx.kernel_log_reset()
            rc, infos = ctx.mshift_cg_block(pk, p_, 18, 4, bdev, cfg["mass"], cfg["shifts"], stop, 100000, x, ws)
            note("stag_mshift_cg_block R=4", variant=var, rc=rc, iters=[i["iters"] for i in infos],
                 sum_iters_shift=[sum(i["iters_shift"]) for i in infos])
            del a, b, x, ws, bdev
        pk = packs[(stag.F64, 18)]
        vb = ctx.vector_bytes(stag.F64)
        # ---- N4
        for p_ in (stag.F64, stag.F32):
            xs = ctx.upload_vectors([srcs[k % len(srcs)] for k in range(n)], p_)
            F = torch.empty(2 * vh * 72, dtype=torch.float64, device="cuda")
            ws = ctx.alloc(ctx.force_workspace_bytes(p_, n))
            ctx.kernel_log_reset()
            ctx.fermion_force(packs[(p_, 18)], p_, 18, [1.0 / (i + 1) for i in range(n)], xs, F, ws)
            note("stag_fermion_force", variant="%s-18" % PREC_NAME[p_], nshift=n)
            del xs, F, ws
        # ---- N2: the single-shift residual-replacement route
        b = ctx.upload_vector(srcs[0], stag.F64)
        x, ws = ctx.alloc(vb), ctx.alloc(ctx.mshift_cg_mixed_workspace_bytes(1))
        ctx.kernel_log_reset()
        rc, info = ctx.mshift_cg_mixed(pk, stag.F64, 18, packs[(stag.F64_SPLIT, 18)], 18, b, cfg["mass"], cfg["shifts"][:1],
                                       cfg["stops"][0], 100000, x, ws)
        note("stag_mshift_cg_mixed 1 shift", variant="f64-18+f32-18", rc=rc, route=info["route"], iters=info["inner"]["iters"])
    print(json.dumps({"ncu_pass": WORKLOADS[wl], "csrc_sha": csrc_sha(), "vh": vh, "nshift": n, "sequence": seq}))
    return 0


def dslash_sweep(args, torch, stag, ctx, cfg, U, srcs, vh, pack_ms, gen_s):
    """--dslash-only: the SURVEY.md §8(d) Dslash bandwidth sweep alone (no CG), one JSON line."""
    peak, peak_src = measured_peak_gbs()
    table, entries = dslash_variants(torch, stag, ctx, args.workload, U, srcs, vh, peak, peak_src, args.dslash_launches)
    out = {"metric": "Dslash GFLOP/s & HBM GB/s", "workload": WORKLOADS[args.workload], "peak_gbs": peak,
           "peak_source": peak_src, "pack_ms": pack_ms, "input_gen_s": gen_s, "dslash": table,
           "roofline": {"also": entries}}
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
    wl = args.workload
    cfg = si.get_config(WORKLOADS[wl])
    L = cfg["L"]
    vh = int(np.prod(L)) // 2
    shifts, nshift = cfg["shifts"], len(cfg["shifts"])
    stop, maxiter = cfg["stops"][0], 100000
    peak, peak_src = measured_peak_gbs()
    vprec = stag.F32 if prec == stag.F32 else stag.F64

    # ---- setup (a1): seeded synthetic inputs -> HBM, packed once --------------------------------
    U, srcs, gen_s = make_inputs(cfg)
    ctx = stag.Stag(L)
    for kv in args.opt:                                   # tuning knobs of stag_set_option
        k, v = kv.split("=")
        ctx.set_option(k, int(v))
    if args.ncu_pass:
        return ncu_pass(args, torch, stag, ctx, cfg, U, srcs, vh)
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
    vb = ctx.vector_bytes(vprec)
    if args.dslash_only:
        del packed
        return dslash_sweep(args, torch, stag, ctx, cfg, U, srcs, vh, pack_ms, gen_s)
    bdev = [ctx.upload_vector(s, vprec) for s in srcs]
    x = ctx.alloc(nshift * vb)
    ws = ctx.alloc(ctx.cg_workspace_bytes(prec, nshift))

    def solve(k):
        rc, info = ctx.mshift_cg(packed, prec, recon, bdev[k], cfg["mass"], shifts, stop, maxiter, x, ws)
        if rc != 0 and not (prec == stag.F32 and rc == stag.ERR_NOTCONV):
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
    ctx.kernel_log_reset()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    infos = []
    e0.record()
    for k in range(args.steps):
        infos.append(solve(source_for(rank, args.steps, k, len(bdev))))
    e1.record()
    barrier()
    clk = clocks.stop() if rank == 0 else None
    step_kernels = ctx.kernel_log()
    persistent = all(i["kernel_launches"] == 1 for i in infos)
    resident = resident_slices(vh, prec) if persistent else 0
    resident = resident if resident >= 2 else 0        # (cg_resident_slices < 2 is a test knob: reported with the multi-kernel bytes)
    secs, (tot_iters, own_bytes_site, equiv_bytes_site, launches) = reduce_over_ranks(
        torch, dist, world, e0.elapsed_time(e1) * 1e-3,
        [sum(i["iters"] for i in infos),
         sum(cg_bytes_per_site(prec, recon, i["iters"], i["iters_shift"], resident) for i in infos),
         sum(cg_bytes_per_site(prec, recon, i["iters"], i["iters_shift"], 0) for i in infos),
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

    out = None
    if rank == 0:
        also = []
        name = "%s-%d" % (PREC_NAME[prec], recon)
        read_gbs = read_stream_gbs(torch)                 # sets the `frac_read` of every roofline entry below
        # ---- roofline of the step's dominant kernel ------------------------------------------------
        if persistent:
            # the whole solve is ONE kernel (stag_cg_persist.cuh): that kernel is the step.  `achieved` uses the
            # bytes THIS kernel has to move (r, q, p_base stay in shared memory); the multi-kernel formula of
            # SURVEY.md §8(d) is beside it as `equivalent_gbs`, and the real DRAM bytes of the ncu capture as `traffic`
            roof = roof_entry(wl, next((k for k in step_kernels if re.search(r"cg_persistent(_sr)?_kernel", k)), "?"),
                              "stag_mshift_cg %s: one launch = one %d-shift solve" % (name, nshift),
                              own_bytes_site * vh / nsolves, secs / args.steps, peak, peak_src, variant=name,
                              equivalent_gbs=equiv_bytes_site * vh / secs / 1e9 / world,
                              bytes_model=BYTES_MODEL[resident]
                              + " per even site and iteration, summed over the iterations of the solve")
        else:
            roof = None                                   # set from the Dslash sweep below (multi-kernel path)
        # ---- Dslash sweep over the storage variants ---------------------------------------------------
        dslash, ents = dslash_variants(torch, stag, ctx, wl, U, srcs, vh, peak, peak_src, args.dslash_launches,
                                       have={(prec, recon): packed})
        also += ents
        if roof is None:
            roof = dict(next(e for e in ents if e.get("workload") == wl and name in e["what"]))   # multi-kernel path: the Dslash
        # ---- the solve in the other storage variants (fp32 / 12-real need driver-visible figures) ----
        solves = {}
        if not args.no_block and prec == stag.F64 and recon == 18:
            for p_, r_ in ((stag.F64, 12), (stag.F32, 18), (stag.F32, 12)):
                pk = ctx.upload_gauge(U, p_, r_)
                d, e = measure_solve(torch, stag, ctx, wl, cfg, pk, p_, r_, srcs[0], vh, peak, peak_src)
                solves["%s-%d" % (PREC_NAME[p_], r_)] = d
                if e:
                    also.append(e)
                del pk
        # ---- N1: the 4 pseudo-fermion sources of the workload through ONE link read ----------------------
        block = mixed = force = None
        if not args.no_block and len(srcs) >= 2 and prec != stag.F64_SPLIT:
            block, ents = measure_block(torch, stag, ctx, wl, cfg, srcs, packed, prec, recon, vh, peak, peak_src)
            also += ents
        # ---- N2/N3: fp32 multi-shift + fp64 polish on one split-double buffer -----------------------------
        if not args.no_block and prec == stag.F64:
            mixed = measure_mixed(torch, stag, ctx, cfg, U, srcs, vh, secs / args.steps)
        # ---- N4 ---------------------------------------------------------------------------------------------
        if not args.no_block and prec != stag.F64_SPLIT:
            force, e = measure_force(torch, stag, ctx, wl, cfg, srcs, packed, prec, recon, vh, peak, peak_src)
            also.append(e)
        # ---- N1 / N4 in the MD precision (the force solves run in fp32): fp32-18 links and vectors -----
        md_f32 = None
        if not args.no_block and prec == stag.F64 and recon == 18 and len(srcs) >= 2:
            pk32 = ctx.upload_gauge(U, stag.F32, 18)
            b32, ents = measure_block(torch, stag, ctx, wl, cfg, srcs, pk32, stag.F32, 18, vh, peak, peak_src)
            also += ents
            f32, e = measure_force(torch, stag, ctx, wl, cfg, srcs, pk32, stag.F32, 18, vh, peak, peak_src)
            also.append(e)
            md_f32 = {"block": b32, "force": f32}
            del pk32
        l2_bytes = torch.cuda.get_device_properties(local).L2_cache_size
        wset = ctx.gauge_packed_bytes(prec, recon) + (2 * nshift + 4) * vb
        iters = [i["iters"] for i in infos]
        cg_gbs = own_bytes_site * vh / secs / 1e9
        out = {"metric": METRIC, "value": value, "unit": "GFLOP/s", "n_gpus": world, "steps": args.steps,
               "warmup": args.warmup, "ms_per_step": secs * 1e3 / args.steps, "higher_is_better": True,
               "scaling": "weak", "vs_baseline": None, "dtype": "f32" if args.prec == "f32" else "f64", "data": "synthetic",
               "config": workload_config(cfg, wl, prec, recon),      # the same keys in both arms (the reference arm's too)
               "l2": "working set (2 link sets + %d vectors) = %.0f MB %s the %.0f MB L2%s"
                     % (2 * nshift + 4, wset / 1e6, "exceeds" if wset > l2_bytes else "FITS in", l2_bytes / 1e6,
                        "; no flush between steps" if wset > l2_bytes else
                        ": an L2-resident run, not held to the HBM roofline"),
               "read_stream_gbs": read_gbs,
               "dslash_gflops_through_solve": value,
               "dslash_gflops_standalone": dslash[name]["gflops"],
               "cg_s_per_solve": secs / args.steps,
               "cg": {"s_per_solve": secs / args.steps, "iters": iters, "us_per_iter": secs / (tot_iters / world) * 1e6,
                      "path": "persistent" if persistent else "multi-kernel",
                      "gbs_algorithmic": cg_gbs, "pct_of_8tbs": 100 * cg_gbs / NOMINAL_HBM_GBS,
                      "pct_of_measured": 100 * cg_gbs / peak, "equivalent_gbs": equiv_bytes_site * vh / secs / 1e9,
                      "solves": nsolves, "iters_shift_first_solve": infos[0]["iters_shift"],
                      "kernels": [norm_kernel(k) for k in step_kernels]},
               "dslash": dslash, "solves_other_variants": solves, "block": block, "mixed": mixed, "force": force, "md_f32": md_f32,
               "e2e": {"value": e2e_value, "unit": "GFLOP/s", "h2d_bytes_per_step": n6 * 8,
                       "d2h_bytes_per_step": nshift * n6 * 8, "s_per_solve": te_s / e2e_steps,
                       "call": "stag_mshift_cg_host (pinned host source in, host solutions out)"},
               "gpu_launches": int(launches), "options": args.opt, "clocks": clk, "pack_ms": pack_ms, "input_gen_s": gen_s}
        # free config-4 device memory before the 64^4 section
        del packed, bdev, x, ws
        torch.cuda.empty_cache()

        # ---- config 5 (64^4) in the default run: the largest single-GPU configuration -----------------
        c5 = None
        if wl == "c4" and world == 1 and not args.no_c5 and prec == stag.F64 and recon == 18:
            c5, ents = c5_section(torch, stag, args, peak, peak_src)
            also += ents
        out["c5"] = c5
        roof["also"] = also
        out["roofline"] = roof

        # ---- cpu_baseline: the oracle on this box's host cores, bounded sample (rank 0, N = 1 only) ----
        cpu = None
        if world == 1 and not args.no_cpu_baseline:
            g, s_it, m = oracle_sample(cfg, U, srcs[0], 10.0)
            cpu = {"value": g, "unit": "GFLOP/s", "cores": 1, "kind": "oracle",
                   "sample": "%d oracle multi-shift CG iterations (maxiter=%d) of the same %d-shift solve, %.3f s/iteration"
                             % (m, m, nshift, s_it)}
            # the same oracle, same sample rule, on every host core (its OpenMP mode: chunk-ordered deterministic
            # reductions, bit-equal to one thread — tests/test_oracle_pins.py), BASELINE.md §5
            ncores = len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)
            if ncores > 1:
                ga, sa, ma = oracle_sample(cfg, U, srcs[0], 6.0, threads=ncores)
                cpu["all_cores"] = {"value": ga, "cores": ncores, "iterations": ma, "s_per_iteration": sa}
        out["cpu_baseline"] = cpu
        # every measurement of the run -> the detail file; stdout carries ONE short line, last
        try:
            os.makedirs(os.path.dirname(os.path.abspath(args.detail)), exist_ok=True)
            with open(args.detail, "w") as f:
                json.dump(_sig(out, 9), f, allow_nan=False)
            out["detail_file"] = os.path.relpath(args.detail, ROOT)
        except OSError:
            out["detail_file"] = None
        sys.stdout.flush()
        print(headline_line(out), flush=True)
    if world > 1:
        dist.barrier()
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
    ap.add_argument("--no-block", action="store_true",
                    help="skip the other storage variants' solves and the N1 multi-source, N2/N3 mixed-precision, N4 force measurements")
    ap.add_argument("--no-c5", action="store_true", help="skip the 64^4 section of the default (c4, f64-18, 1 GPU) run")
    ap.add_argument("--c5-solves", type=int, default=3, help="timed 64^4 solves of that section (the median is reported)")
    ap.add_argument("--detail", default=os.path.join(ROOT, "gpurun_out", "bench_detail.json"),
                    help="file that receives every measurement of the run (stdout carries the one short headline line)")
    ap.add_argument("--ref-seconds", type=float, default=150.0,
                    help="--impl reference: total oracle time budget over all steps")
    ap.add_argument("--dslash-only", action="store_true", help="Dslash bandwidth sweep only (no CG)")
    ap.add_argument("--dslash-launches", type=int, default=100)
    ap.add_argument("--ncu-pass", action="store_true",
                    help="launch every reported kernel a few times, untimed: the target of the ncu --set full capture")
    ap.add_argument("--ncu-iters", type=int, default=3, help="--ncu-pass at c5: CG iterations on the multi-kernel path")
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
