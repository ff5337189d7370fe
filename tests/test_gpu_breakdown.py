"""Failure detection ("CG breakdown detection (pAp <= 0, NaN) -> error code"; PAPER.md:129 is the
shifted solver it guards).  A = m^2 - D_eo D_oe + sigma is positive definite for ANY links (D_oe = -D_eo^dagger
holds by construction), so <p,Ap> <= 0 can only come from non-finite data: a NaN in the source or in a link must
end every solver with STAG_ERR_BREAKDOWN and info.breakdown == 1 — never a hang, never a silent "converged"."""
import numpy as np
import pytest

import oracle
import stag_inputs as si

pytestmark = pytest.mark.gpu

L = (4, 4, 4, 4)
SHIFTS = [0.01, 0.04, 0.16, 0.64]
M = 0.1


@pytest.fixture(scope="module")
def stag():
    import paper_1010_5433_b200 as m
    return m


def poisoned(b, where=5):
    v = b.copy()
    v[where, 1] = complex(float("nan"), 0.0)
    return v


@pytest.mark.parametrize("path", ["persistent", "multikernel"])
@pytest.mark.parametrize("prec", [0, 1, 2])
def test_nan_source_is_a_breakdown(stag, path, prec):
    U, b = si.links_haar(L, 61), si.source_gaussian(L, 61)
    ctx = stag.Stag(L)
    ctx.set_option("cg_persistent", 1 if path == "persistent" else 0)
    packed = ctx.upload_gauge(U, prec, 18)
    vp = stag.F32 if prec == stag.F32 else stag.F64
    vb = ctx.vector_bytes(vp)
    x, ws = ctx.alloc(4 * vb), ctx.alloc(ctx.cg_workspace_bytes(prec, 4))
    rc, info = ctx.mshift_cg(packed, prec, 18, ctx.upload_vector(poisoned(b), vp), M, SHIFTS, 1e-8, 500, x, ws)
    assert rc == stag.ERR_BREAKDOWN and info["breakdown"] and not info["converged"]
    assert info["iters"] == 0                      # <b,b> is NaN: caught before the first iteration
    # the context is still usable: the clean source converges right after
    rc, info = ctx.mshift_cg(packed, prec, 18, ctx.upload_vector(b, vp), M, SHIFTS, 1e-4, 500, x, ws)
    assert rc == 0 and info["converged"] and not info["breakdown"]


@pytest.mark.parametrize("path", ["persistent", "multikernel"])
def test_nan_link_is_a_breakdown_at_the_first_pAp(stag, path):
    """<b,b> is finite, the first <p,Ap> is NaN: the alpha = rr / <p,Ap> branch (stag_cg.cuh) must catch it
    and leave x untouched (no update on breakdown: x stays the zero start vector)."""
    U, b = si.links_haar(L, 62), si.source_gaussian(L, 62)
    U = U.copy()
    U[17, 2, 1, 1] = complex(float("nan"), 0.0)
    ctx = stag.Stag(L)
    ctx.set_option("cg_persistent", 1 if path == "persistent" else 0)
    packed = ctx.upload_gauge(U, 0, 18)
    vb = ctx.vector_bytes(0)
    x, ws = ctx.alloc(4 * vb), ctx.alloc(ctx.cg_workspace_bytes(0, 4))
    rc, info = ctx.mshift_cg(packed, 0, 18, ctx.upload_vector(b, 0), M, SHIFTS, 1e-8, 500, x, ws)
    assert rc == stag.ERR_BREAKDOWN and info["breakdown"] and info["iters"] == 0
    for i in range(4):
        assert not ctx.download_vector(x, 0, i * vb).any()


@pytest.mark.parametrize("nrhs,bad", [(4, 2), (2, 0), (3, 2)])
def test_block_one_poisoned_source_does_not_stop_the_others(stag, nrhs, bad):
    """stag_cg_persist.cuh: "every source has its own scalars, shift list and convergence latch" — the poisoned
    source reports breakdown, the call returns STAG_ERR_BREAKDOWN (the worst), every other source converges to
    the ORACLE's residual bound in the oracle's iteration count."""
    U = si.links_haar(L, 63)
    bs = [si.source_gaussian(L, 63, stream=1 + k) for k in range(nrhs)]
    bs_in = list(bs)
    bs_in[bad] = poisoned(bs[bad])
    ctx = stag.Stag(L)
    packed = ctx.upload_gauge(U, 0, 18)
    vb, n = ctx.vector_bytes(0), len(SHIFTS)
    x, ws = ctx.alloc(nrhs * n * vb), ctx.alloc(ctx.cg_block_workspace_bytes(0, n, nrhs))
    rc, infos = ctx.mshift_cg_block(packed, 0, 18, nrhs, ctx.upload_vectors(bs_in, 0), M, SHIFTS, 1e-10, 2000, x, ws)
    assert rc == stag.ERR_BREAKDOWN
    for s in range(nrhs):
        if s == bad:
            assert infos[s]["breakdown"] and not infos[s]["converged"] and infos[s]["iters"] == 0
            continue
        ref = oracle.mshift_cg(L, U, bs[s], M, SHIFTS, 1e-10, 2000)
        assert infos[s]["converged"] and not infos[s]["breakdown"]
        assert abs(infos[s]["iters"] - ref["iters"]) <= 2
        nb = np.linalg.norm(bs[s])
        for i, sg in enumerate(SHIFTS):
            xi = ctx.download_vector(x, 0, (s * n + i) * vb)
            assert np.linalg.norm(bs[s] - oracle.apply_A(L, U, M, sg, xi)) / nb <= 1e-10


@pytest.mark.parametrize("prec_name", ["F64", "F64_SPLIT"])
def test_polish_breakdown_on_nan_source_and_on_nan_start(stag, prec_name):
    prec = getattr(stag, prec_name)
    U, b = si.links_haar(L, 64), si.source_gaussian(L, 64)
    ctx = stag.Stag(L)
    packed = ctx.upload_gauge(U, prec, 18)
    vb = ctx.vector_bytes(stag.F64)
    ws = ctx.alloc(ctx.cg_polish_workspace_bytes())
    x = ctx.alloc(4 * vb)
    x.zero_()
    rc, info = ctx.cg_polish(packed, prec, 18, ctx.upload_vector(poisoned(b), stag.F64), M, SHIFTS, 1e-10, 500, x, ws)
    assert rc == stag.ERR_BREAKDOWN
    # NaN in ONE start vector: its defect is NaN -> breakdown; nothing may hang or be reported as converged
    x0 = [np.zeros_like(b) for _ in SHIFTS]
    x0[1] = poisoned(x0[1])
    x = ctx.upload_vectors(x0, stag.F64)
    rc, info = ctx.cg_polish(packed, prec, 18, ctx.upload_vector(b, stag.F64), M, SHIFTS, 1e-10, 500, x, ws)
    assert rc == stag.ERR_BREAKDOWN
    # and the clean problem still polishes from zero afterwards (ordinary CG)
    x = ctx.alloc(4 * vb)
    x.zero_()
    rc, info = ctx.cg_polish(packed, prec, 18, ctx.upload_vector(b, stag.F64), M, SHIFTS, 1e-10, 2000, x, ws)
    assert rc == 0
    for i, sg in enumerate(SHIFTS):
        xi = ctx.download_vector(x, stag.F64, i * vb)
        assert np.linalg.norm(b - oracle.apply_A(L, U, M, sg, xi)) / np.linalg.norm(b) <= 1e-10


@pytest.mark.parametrize("nshift", [1, 4])
def test_mixed_breakdown_on_nan_source(stag, nshift):
    """nshift = 1 takes the residual-replacement kernel, nshift = 4 the plain fp32 stage: both must report it."""
    U, b = si.links_haar(L, 65), si.source_gaussian(L, 65)
    ctx = stag.Stag(L)
    split = ctx.upload_gauge(U, stag.F64_SPLIT, 18)
    vb = ctx.vector_bytes(stag.F64)
    x, ws = ctx.alloc(nshift * vb), ctx.alloc(ctx.mshift_cg_mixed_workspace_bytes(nshift))
    rc, info = ctx.mshift_cg_mixed(split, stag.F64_SPLIT, 18, split, 18, ctx.upload_vector(poisoned(b), stag.F64), M,
                                   SHIFTS[:nshift], 1e-10, 500, x, ws)
    assert rc == stag.ERR_BREAKDOWN
    assert info["inner"]["breakdown"] or not np.isfinite(info["polish"]["resid_after"][0])
