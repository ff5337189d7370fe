"""N4: fermion force of the rational pseudo-fermion action, thread per link
(PAPER.md:25, :87, :93).  The oracle (oracle.fermion_force) is pinned by finite differences of the
action (tests/test_oracle_pins.py P10); here the CUDA kernel is compared with it element by element."""
import numpy as np
import pytest

import oracle
import stag_inputs as si

pytestmark = pytest.mark.gpu
TOL = {0: 1e-13, 1: 1e-5}


def rel(a, b):
    return np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)


@pytest.fixture(scope="module")
def stag():
    import paper_1010_5433_b200 as m
    return m


def gpu_force(stag, ctx, packed, prec, recon, residues, xs, accumulate_onto=None):
    import torch
    V = ctx.V
    F = torch.full((V * 4 * 18,), float("nan"), dtype=torch.float64, device="cuda")
    if accumulate_onto is not None:
        F.copy_(torch.from_numpy(np.ascontiguousarray(accumulate_onto).view(np.float64).reshape(-1)))
    ws = ctx.alloc(ctx.force_workspace_bytes(prec, len(residues)))
    ctx.fermion_force(packed, prec, recon, residues, ctx.upload_vectors(xs, prec), F, ws,
                      accumulate=accumulate_onto is not None)
    return F.cpu().numpy().view(np.complex128).reshape(V, 4, 3, 3)


@pytest.mark.parametrize("L", [(4, 4, 4, 4), (6, 4, 2, 8), (2, 2, 2, 2), (16, 16, 16, 4)])
@pytest.mark.parametrize("prec,recon", [(0, 18), (0, 12), (1, 18), (1, 12)])
@pytest.mark.parametrize("nshift", [1, 5])
def test_force_matches_oracle(stag, L, prec, recon, nshift):
    U = si.links_haar(L, 71)
    xs = [si.source_gaussian(L, 71, stream=1 + k) for k in range(nshift)]
    residues = [0.7, -0.3, 1.9, 0.05, 2.5][:nshift]
    ctx = stag.Stag(L)
    packed = ctx.upload_gauge(U, prec, recon)
    want = oracle.fermion_force(L, U, residues, np.stack(xs))
    got = gpu_force(stag, ctx, packed, prec, recon, residues, xs)
    assert np.isfinite(got.view(np.float64)).all()
    assert rel(got, want) <= TOL[prec]
    # exactly traceless and anti-Hermitian by construction
    assert np.abs(got + got.conj().transpose(0, 1, 3, 2)).max() <= 1e-14 * np.abs(want).max()
    assert np.abs(np.trace(got, axis1=2, axis2=3)).max() <= 1e-13 * np.abs(want).max()


def test_force_accumulates_over_pseudofermions(stag):
    L = (4, 4, 4, 4)
    U = si.links_haar(L, 72)
    ctx = stag.Stag(L)
    packed = ctx.upload_gauge(U, 0, 18)
    x1 = [si.source_gaussian(L, 72, stream=1 + k) for k in range(3)]
    x2 = [si.source_gaussian(L, 72, stream=11 + k) for k in range(3)]
    res = [1.0, 0.5, 0.25]
    F1 = gpu_force(stag, ctx, packed, 0, 18, res, x1)
    F12 = gpu_force(stag, ctx, packed, 0, 18, res, x2, accumulate_onto=F1)
    want = oracle.fermion_force(L, U, res, np.stack(x1)) + oracle.fermion_force(L, U, res, np.stack(x2))
    assert rel(F12, want) <= 1e-13


def test_force_after_the_solve_config1(stag):
    """The chain the RHMC runs: multi-shift solve, then the force from its x_i — against the oracle's own
    chain (its CG, its force).  The two x_i agree to ~stop*kappa, so the forces agree to ~1e-7."""
    cfg = si.get_config("c1_4x4x4x4")
    L, U, b, m, shifts = cfg["L"], si.make_links(cfg), si.make_source(cfg), cfg["mass"], cfg["shifts"]
    residues = [1.0, 0.5, 0.25, 0.125]
    ctx = stag.Stag(L)
    packed = ctx.upload_gauge(U, 0, 18)
    n, vb = len(shifts), ctx.vector_bytes(0)
    x, ws = ctx.alloc(n * vb), ctx.alloc(ctx.cg_workspace_bytes(0, n))
    rc, _ = ctx.mshift_cg(packed, 0, 18, ctx.upload_vector(b, 0), m, shifts, 1e-12, 2000, x, ws)
    assert rc == 0
    import torch
    F = torch.empty(ctx.V * 72, dtype=torch.float64, device="cuda")
    ctx.fermion_force(packed, 0, 18, residues, x, F, ctx.alloc(ctx.force_workspace_bytes(0, n)))
    got = F.cpu().numpy().view(np.complex128).reshape(ctx.V, 4, 3, 3)
    ref = oracle.mshift_cg(L, U, b, m, shifts, 1e-12, 2000)
    assert rel(got, oracle.fermion_force(L, U, residues, ref["x"])) <= 1e-8


def test_force_bad_arguments(stag):
    import torch
    L = (4, 4, 4, 4)
    ctx = stag.Stag(L)
    U = si.links_haar(L, 3)
    F = torch.empty(ctx.V * 72, dtype=torch.float64, device="cuda")
    x = ctx.alloc(ctx.vector_bytes(0))
    ws = ctx.alloc(ctx.force_workspace_bytes(0, 1))
    with pytest.raises(stag.StagError) as e:
        ctx.fermion_force(ctx.upload_gauge(U, 0, 18), 3, 18, [1.0], x, F, ws)        # no such precision
    assert e.value.code == stag.ERR_BADARG
    with pytest.raises(stag.StagError) as e:
        ctx.fermion_force(ctx.upload_gauge(U, 0, 18), 0, 18, [1.0], x, F, None)
    assert e.value.code == stag.ERR_BADARG
    assert ctx.force_workspace_bytes(0, 0) == 0 and ctx.force_workspace_bytes(0, 33) == 0
