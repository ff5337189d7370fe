"""Performance regression guard at config 4 (32^3 x 8, 16 shifts) — VERDICT r2 item 7(a).

The four persistent CG kernels are near-copies of one design and DESIGN.md §6 records that the stencil's register
schedule inside them flips (22 <-> 31-53 us per phase) with unrelated edits.  This test times one solve per storage
variant, the 4-source block solve and the fermion-force call and holds each to the committed figure below, with a
loose margin (clocks on the pool move by ~8 % under the power cap): a flipped schedule costs 15-40 %, which it
catches, while run-to-run noise passes.  Figures: profiles/README.md (round 3), best of 3 timed calls here.

Collected after the parity tests (test_zy_*): a timing failure must not hide a correctness result under `pytest -x`.
"""
import numpy as np
import pytest

import stag_inputs as si

pytestmark = pytest.mark.gpu
MARGIN = 1.25
# microseconds per CG iteration of one solve (persistent single-reduction kernel), committed figures
US_PER_ITER = {(0, 18): 68.1, (0, 12): 55.6, (1, 18): 35.5, (1, 12): 30.5}
US_PER_BLOCK_ITER_F64 = 183.0            # stag_mshift_cg_block, 4 sources, fp64-18
US_PER_FORCE_CALL = {0: 283.3, 1: 169.2}  # stag_fermion_force, 16 shifts, 18 reals: fp64 / fp32


@pytest.fixture(scope="module")
def stag():
    import paper_1010_5433_b200 as m
    return m


@pytest.fixture(scope="module")
def c4():
    cfg = si.get_config("c4_32x32x32x8")
    return cfg, si.make_links(cfg), [si.make_source(cfg, k) for k in range(cfg["nsrc"])]


def best_of(torch, fn, n=3):
    best, out = float("inf"), None
    for _ in range(n + 1):                      # the first call warms up
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        out = fn()
        e1.record()
        torch.cuda.synchronize()
        best = min(best, e0.elapsed_time(e1) * 1e-3)
    return best, out


@pytest.mark.parametrize("prec,recon", sorted(US_PER_ITER))
def test_c4_solve_time_per_iteration(stag, c4, prec, recon):
    import torch
    cfg, U, srcs = c4
    ctx = stag.Stag(cfg["L"])
    packed = ctx.upload_gauge(U, prec, recon)
    n, vb = len(cfg["shifts"]), ctx.vector_bytes(prec)
    b, x, ws = ctx.upload_vector(srcs[0], prec), ctx.alloc(n * vb), ctx.alloc(ctx.cg_workspace_bytes(prec, n))
    secs, (rc, info) = best_of(torch, lambda: ctx.mshift_cg(packed, prec, recon, b, cfg["mass"], cfg["shifts"],
                                                             cfg["stops"][0], 100000, x, ws, check=False))
    assert info["kernel_launches"] == 1 and info["iters"] > 1000, info
    us = secs / info["iters"] * 1e6
    assert us <= MARGIN * US_PER_ITER[(prec, recon)], "%.1f us per iteration, committed %.1f" % (us, US_PER_ITER[(prec, recon)])


def test_c4_block_solve_time_per_iteration(stag, c4):
    import torch
    cfg, U, srcs = c4
    ctx = stag.Stag(cfg["L"])
    packed = ctx.upload_gauge(U, 0, 18)
    n, vb, R = len(cfg["shifts"]), ctx.vector_bytes(0), 4
    b, x = ctx.upload_vectors(srcs[:R], 0), ctx.alloc(R * n * vb)
    ws = ctx.alloc(ctx.cg_block_workspace_bytes(0, n, R))
    secs, (rc, infos) = best_of(torch, lambda: ctx.mshift_cg_block(packed, 0, 18, R, b, cfg["mass"], cfg["shifts"],
                                                                   cfg["stops"][0], 100000, x, ws), n=2)
    assert rc == 0
    us = secs / max(i["iters"] for i in infos) * 1e6
    assert us <= MARGIN * US_PER_BLOCK_ITER_F64, "%.1f us per block iteration, committed %.1f" % (us, US_PER_BLOCK_ITER_F64)


@pytest.mark.parametrize("prec", [0, 1])
def test_c4_force_call_time(stag, c4, prec):
    import torch
    cfg, U, srcs = c4
    ctx = stag.Stag(cfg["L"])
    packed = ctx.upload_gauge(U, prec, 18)
    n = len(cfg["shifts"])
    x = ctx.upload_vectors([srcs[k % len(srcs)] for k in range(n)], prec)
    F = torch.empty(ctx.V * 72, dtype=torch.float64, device="cuda")
    ws = ctx.alloc(ctx.force_workspace_bytes(prec, n))
    res = [1.0 / (i + 1) for i in range(n)]

    def twenty():
        for _ in range(20):
            ctx.fermion_force(packed, prec, 18, res, x, F, ws)
    secs, _ = best_of(torch, twenty)
    us = secs / 20 * 1e6
    assert np.isfinite(F.sum().item())
    assert us <= MARGIN * US_PER_FORCE_CALL[prec], "%.1f us per call, committed %.1f" % (us, US_PER_FORCE_CALL[prec])
