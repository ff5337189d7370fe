"""Run-to-run reproducibility (one partial per CTA, summed in index order): for a fixed launch
configuration every solver returns the same BITS — iteration counts, residual norms and solutions — on every run.
Also a soak of the persistent kernel's sync machinery (neighbour flags, deferred items): many back-to-back solves on
lattices whose CTA ranges have different shapes, each checked against the first."""
import numpy as np
import pytest
import torch

import stag_inputs as si

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def stag():
    import paper_1010_5433_b200 as m
    return m


def solve_bits(stag, ctx, packed, prec, recon, b, m, shifts, stop, opts=()):
    n = len(shifts)
    vb = ctx.vector_bytes(prec)
    x = ctx.alloc(n * vb)
    x.zero_()
    ws = ctx.alloc(ctx.cg_workspace_bytes(prec, n))
    for k, v in opts:
        ctx.set_option(k, v)
    rc, info = ctx.mshift_cg(packed, prec, recon, b, m, shifts, stop, 20000, x, ws)
    return rc, info["iters"], info["rnorm2"], tuple(info["iters_shift"]), x.clone()


@pytest.mark.parametrize("L", [(8, 8, 8, 8), (16, 16, 16, 4), (12, 6, 10, 4), (24, 24, 24, 6)])
@pytest.mark.parametrize("prec,recon", [(0, 18), (0, 12), (1, 18), (2, 18)])
@pytest.mark.parametrize("persistent", [1, 0])
def test_repeated_solves_are_bit_identical(stag, L, prec, recon, persistent):
    U = si.links_haar(L, 301)
    b = si.source_gaussian(L, 301, stream=1)
    shifts = [0.002, 0.03, 0.4, 5.0]
    ctx = stag.Stag(L)
    packed = ctx.upload_gauge(U, prec, recon)
    vprec = 1 if prec == 1 else 0
    bd = ctx.upload_vector(b, vprec)
    stop = 1e-9 if prec != 1 else 1e-5
    first = solve_bits(stag, ctx, packed, prec, recon, bd, 0.05, shifts, stop, opts=(("cg_persistent", persistent),))
    assert first[0] == 0
    for _ in range(12):
        again = solve_bits(stag, ctx, packed, prec, recon, bd, 0.05, shifts, stop)
        assert again[:4] == first[:4]
        assert torch.equal(again[4], first[4])


def test_block_and_force_are_bit_identical_run_to_run(stag):
    L = (16, 16, 16, 4)
    U = si.links_haar(L, 302)
    srcs = [si.source_gaussian(L, 302, stream=1 + k) for k in range(4)]
    shifts = [0.01, 0.1, 1.0]
    ctx = stag.Stag(L)
    packed = ctx.upload_gauge(U, 0, 18)
    n, vb = len(shifts), ctx.vector_bytes(0)
    bdev = ctx.upload_vectors(srcs, 0)
    outs = []
    for _ in range(6):
        x = ctx.alloc(4 * n * vb)
        rc, infos = ctx.mshift_cg_block(packed, 0, 18, 4, bdev, 0.05, shifts, 1e-9, 20000, x,
                                        ctx.alloc(ctx.cg_block_workspace_bytes(0, n, 4)))
        assert rc == 0
        F = torch.empty(ctx.V * 72, dtype=torch.float64, device="cuda")
        ctx.fermion_force(packed, 0, 18, [1.0, 0.5, 0.25], x[:n * vb], F, ctx.alloc(ctx.force_workspace_bytes(0, n)))
        torch.cuda.synchronize()
        outs.append(([i["iters"] for i in infos], x.clone(), F.clone()))
    for o in outs[1:]:
        assert o[0] == outs[0][0] and torch.equal(o[1], outs[0][1]) and torch.equal(o[2], outs[0][2])
