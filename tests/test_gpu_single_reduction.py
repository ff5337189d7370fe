"""The persistent CG with ONE grid-wide reduction per iteration (csrc/stag_cg_persist_sr.cuh; option
cg_single_reduction, default 1) against the two-reduction kernel and against the oracle:
||r - alpha q||^2 = rr - 2 alpha <r,q> + alpha^2 <q,q> with rr recomputed from r in every iteration."""
import numpy as np
import pytest

import oracle
import stag_inputs as si

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def stag():
    import paper_1010_5433_b200 as m
    return m


def rel(a, b):
    return np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)


def solve(stag, ctx, packed, prec, recon, b, m, shifts, stop, maxiter, sr):
    n = len(shifts)
    vprec = 1 if prec == 1 else 0
    vb = ctx.vector_bytes(vprec)
    x, ws = ctx.alloc(n * vb), ctx.alloc(ctx.cg_workspace_bytes(prec, n))
    ctx.set_option("cg_single_reduction", sr)
    ctx.kernel_log_reset()
    rc, info = ctx.mshift_cg(packed, prec, recon, ctx.upload_vector(b, vprec), m, shifts, stop, maxiter, x, ws)
    kernels = " ".join(ctx.kernel_log())
    ctx.set_option("cg_single_reduction", 1)
    return rc, info, [ctx.download_vector(x, vprec, i * vb) for i in range(n)], kernels


@pytest.mark.parametrize("L", [(4, 4, 4, 4), (8, 8, 8, 8), (12, 6, 10, 4), (16, 16, 16, 4)])
@pytest.mark.parametrize("prec,recon", [(0, 18), (0, 12), (2, 18), (1, 18)])
def test_single_reduction_equals_two_reductions_and_meets_the_oracle(stag, L, prec, recon):
    U = si.links_haar(L, 401)
    b = si.source_gaussian(L, 401, stream=1)
    m, shifts = 0.1, [0.01, 0.04, 0.3, 4.0, 19.0]      # (iteration counts stay below the matrix dimension on 4^4)
    stop = 1e-10 if prec != 1 else 1e-5
    ctx = stag.Stag(L)
    packed = ctx.upload_gauge(U, prec, recon)
    rc1, i1, x1, k1 = solve(stag, ctx, packed, prec, recon, b, m, shifts, stop, 20000, 1)
    rc2, i2, x2, k2 = solve(stag, ctx, packed, prec, recon, b, m, shifts, stop, 20000, 0)
    assert "cg_persistent_sr_kernel" in k1 and "cg_persistent_sr_kernel" not in k2 and "cg_persistent_kernel" in k2
    assert rc1 == 0 and rc2 == 0 and i1["converged"] and i1["kernel_launches"] == 1
    assert abs(i1["iters"] - i2["iters"]) <= 2
    ref = oracle.mshift_cg(L, U, b, m, shifts, stop, 20000)
    assert abs(i1["iters"] - ref["iters"]) <= 2
    nb = np.linalg.norm(b)
    for i, s in enumerate(shifts):
        assert rel(x1[i], x2[i]) <= (1e-8 if prec != 1 else 1e-3)
        tr = np.linalg.norm(b - oracle.apply_A(L, U, m, s, x1[i])) / nb
        assert tr <= (stop if prec != 1 else 2e-4), (i, tr)
        assert abs(i1["iters_shift"][i] - i2["iters_shift"][i]) <= 2


def test_drop_below_the_formulas_resolution_is_certified_one_iteration_later(stag):
    """An eigenvector source converges in ONE iteration: r - alpha q = 0 exactly, which rr - 2 alpha <r,q> + alpha^2 <q,q>
    cannot resolve below eps * rr.  The exact <r,r> of the next reduction certifies it before anything of that
    iteration is applied: iters == 1, the closed-form solution to rounding."""
    L, m = (4, 4, 2, 6), 0.2
    shifts = [0.01, 0.04, 0.16, 0.64]
    U = si.links_unit(L)
    b, p = si.source_plane_wave(L, (1, 3, 0, 2), [1.0, 0.5j, -0.25])
    lam = m * m + np.sum(np.sin(p) ** 2)
    ctx = stag.Stag(L)
    packed = ctx.upload_gauge(U, 0, 18)
    rc, info, xs, k = solve(stag, ctx, packed, 0, 18, b, m, shifts, 1e-12, 10, 1)
    assert "cg_persistent_sr_kernel" in k
    assert rc == 0 and info["converged"] and info["iters"] == 1 and not info["breakdown"]
    for i, s in enumerate(shifts):
        assert rel(xs[i], b / (lam + s)) < 1e-14


def test_falls_back_when_r_and_q_cannot_be_resident(stag):
    """The single-reduction kernel needs r and q in shared memory (its extra dot products are a pass over shared
    memory); with cg_resident_slices < 2 the call takes the two-reduction kernel and returns the same answer."""
    L = (8, 8, 8, 8)
    U, b = si.links_haar(L, 402), si.source_gaussian(L, 402, stream=1)
    ctx = stag.Stag(L)
    packed = ctx.upload_gauge(U, 0, 18)
    rc0, i0, x0, _ = solve(stag, ctx, packed, 0, 18, b, 0.05, [0.01, 1.0], 1e-10, 20000, 1)
    ctx.set_option("cg_resident_slices", 1)
    rc1, i1, x1, k1 = solve(stag, ctx, packed, 0, 18, b, 0.05, [0.01, 1.0], 1e-10, 20000, 1)
    ctx.set_option("cg_resident_slices", 3)
    assert "cg_persistent_sr_kernel" not in k1 and "cg_persistent_kernel" in k1
    assert rc0 == 0 and rc1 == 0 and abs(i0["iters"] - i1["iters"]) <= 1 and rel(x0[0], x1[0]) <= 1e-8


def test_maxiter_and_breakdown_on_the_single_reduction_kernel(stag):
    L = (8, 8, 8, 8)
    U, b = si.links_haar(L, 403), si.source_gaussian(L, 403, stream=1)
    ctx = stag.Stag(L)
    packed = ctx.upload_gauge(U, 0, 18)
    rc, info, xs, k = solve(stag, ctx, packed, 0, 18, b, 0.01, [0.0, 0.5], 1e-14, 7, 1)
    assert "cg_persistent_sr_kernel" in k and rc == stag.ERR_NOTCONV and info["iters"] == 7 and not info["converged"]
    ref = oracle.mshift_cg(L, U, b, 0.01, [0.0, 0.5], 1e-14, 7)
    for i in range(2):
        assert rel(xs[i], ref["x"][i]) <= 1e-12              # the same 7 iterates
    bad = b.copy()
    bad[3, 1] = np.nan
    rc, info, _, _ = solve(stag, ctx, packed, 0, 18, bad, 0.01, [0.0, 0.5], 1e-10, 100, 1)
    assert rc == stag.ERR_BREAKDOWN and info["breakdown"]


@pytest.mark.parametrize("fill,nbflags", [(0, 0), (0, 1), (1, 0)])
def test_sync_options_do_not_change_the_arithmetic(stag, fill, nbflags):
    """cg_fill (deferred shift updates worked off in the waits) and cg_nbflags (neighbour flags instead of grid-wide
    waits after the stencil phases) only move work and waits around: the bits of the result stay the same."""
    L = (16, 16, 16, 4)
    U, b = si.links_haar(L, 404), si.source_gaussian(L, 404, stream=1)
    m, shifts = 0.05, [0.002, 0.05, 0.6, 7.0]
    ctx = stag.Stag(L)
    packed = ctx.upload_gauge(U, 0, 18)
    rc0, i0, x0, k0 = solve(stag, ctx, packed, 0, 18, b, m, shifts, 1e-10, 20000, 1)
    ctx.set_option("cg_fill", fill)
    ctx.set_option("cg_nbflags", nbflags)
    rc1, i1, x1, k1 = solve(stag, ctx, packed, 0, 18, b, m, shifts, 1e-10, 20000, 1)
    ctx.set_option("cg_fill", 1)
    ctx.set_option("cg_nbflags", 1)
    assert "cg_persistent_sr_kernel" in k0 and "cg_persistent_sr_kernel" in k1
    assert rc0 == 0 and rc1 == 0 and i0["iters"] == i1["iters"] and i0["rnorm2"] == i1["rnorm2"]
    for a, c in zip(x0, x1):
        assert np.array_equal(a, c)
