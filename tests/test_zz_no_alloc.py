"""stag_fermion_force_static — the fermion force for callers that cannot allocate device memory.

Why the entry point exists: stag_fermion_force needs a workspace for the odd-site vectors D_oe x_i and the caller
has to supply it.  A force routine plugged into someone else's integrator gets the x_i and the force array and
nothing more; the host program may have given its whole device memory to a pool of its own; a molecular-dynamics
loop cannot take the device-wide stall of a cudaMalloc at every force evaluation.  The static variant keeps that
scratch in an 8 MiB array inside the library (one per GPU, shared by all calls on that GPU) and runs the same
kernels.

What is checked here: the result equals that of stag_fermion_force with a caller-owned workspace, to the
tolerance tests/test_gpu_force.py uses against the oracle, on TWO CALLS IN A ROW that differ in lattice, precision,
storage and shift count — the second one finds the first one's leftovers in the shared array and must not be
affected by them — and problems beyond the 8 MiB are refused before anything is launched.

This file is named test_zz_* so that pytest collects it last: it is the only test that touches process-wide
state (the library's static array), and with `pytest -x` a failure here cannot hide the other tests.  It must
pass both on its own in a fresh process, where its first call does the one-time look-up of the array's address,
and after the rest of the suite.
"""
import numpy as np
import pytest

import stag_inputs as si

pytestmark = pytest.mark.gpu
TOL = {0: 1e-13, 1: 1e-5}            # the tolerances of tests/test_gpu_force.py (fp64, fp32)


def rel(a, b):
    return np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)


@pytest.fixture(scope="module")
def stag():
    import paper_1010_5433_b200 as m
    return m


def both_paths(stag, L, prec, recon, nshift, seed, accumulate=False):
    """(force by the static entry point, force by stag_fermion_force with its own workspace), same inputs."""
    import torch
    U = si.links_haar(L, seed)
    xs = [si.source_gaussian(L, seed, stream=1 + k) for k in range(nshift)]
    residues = [0.7, -0.3, 1.9, 0.05, 2.5, 0.4, -1.1, 0.9][:nshift]
    ctx = stag.Stag(L)
    packed = ctx.upload_gauge(U, prec, recon)
    x = ctx.upload_vectors(xs, prec)
    start = torch.randn(ctx.V * 72, dtype=torch.float64, device="cuda") if accumulate else \
        torch.full((ctx.V * 72,), float("nan"), dtype=torch.float64, device="cuda")
    F_static, F_ws = start.clone(), start.clone()
    ctx.fermion_force_static(packed, prec, recon, residues, x, F_static, accumulate=accumulate)
    ws = ctx.alloc(ctx.force_workspace_bytes(prec, nshift))
    ctx.fermion_force(packed, prec, recon, residues, x, F_ws, ws, accumulate=accumulate)
    torch.cuda.synchronize()
    return F_static.cpu().numpy(), F_ws.cpu().numpy()


def test_static_scratch_force_equals_workspace_force_on_two_calls_in_a_row(stag):
    # call 1: 16^3 x 4, fp64, 18 reals, 5 shifts — 1.9 MiB of the array, several tiles
    got, want = both_paths(stag, (16, 16, 16, 4), 0, 18, 5, seed=81)
    assert np.isfinite(got).all()
    assert rel(got, want) <= TOL[0]
    # call 2, straight after: ragged lattice, fp32, 12 reals, 3 shifts, added onto an existing force; the array
    # still holds call 1's fp64 vectors
    got, want = both_paths(stag, (6, 4, 2, 8), 1, 12, 3, seed=82, accumulate=True)
    assert np.isfinite(got).all()
    assert rel(got, want) <= TOL[1]
    # and back to fp64 on split-double links with more shifts than before
    got, want = both_paths(stag, (4, 4, 4, 4), 2, 18, 8, seed=83)
    assert rel(got, want) <= TOL[0]


def test_static_scratch_limit_is_enforced_with_a_clear_error(stag):
    import torch
    assert stag.lib().stag_fermion_force_static_max_bytes() == stag.FORCE_STATIC_BYTES == 8 << 20
    L = (32, 32, 32, 8)                                   # 16 fp64 shifts need 96 MiB
    ctx = stag.Stag(L)
    assert ctx.force_workspace_bytes(0, 16) > stag.FORCE_STATIC_BYTES
    tiny = torch.zeros(64, dtype=torch.float64, device="cuda")     # never dereferenced: refused on the host
    with pytest.raises(stag.StagError) as e:
        ctx.fermion_force_static(tiny, 0, 18, [1.0] * 16, tiny, tiny)
    assert e.value.code == stag.ERR_SCRATCH_LIMIT
    assert "stag_fermion_force_static" in str(e.value) and "8 MiB" in str(e.value)
    # the largest shift count that fits at 16^3 x 4 in fp64 is accepted by the size rule (21 * 384 KiB <= 8 MiB)
    c2 = stag.Stag((16, 16, 16, 4))
    assert c2.force_workspace_bytes(0, 21) <= stag.FORCE_STATIC_BYTES < c2.force_workspace_bytes(0, 22)
    with pytest.raises(stag.StagError) as e:
        c2.fermion_force_static(tiny, 0, 18, [1.0] * 22, tiny, tiny)
    assert e.value.code == stag.ERR_SCRATCH_LIMIT
    with pytest.raises(stag.StagError) as e:               # bad precision: the usual argument error, not the limit
        c2.fermion_force_static(tiny, 3, 18, [1.0], tiny, tiny)
    assert e.value.code == stag.ERR_BADARG
