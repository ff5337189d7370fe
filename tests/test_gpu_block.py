"""N1: multi-RHS Dslash and the block multi-shift CG — the paper's multiple
pseudo-fermions as independent sources sharing one read of the links.  Every source's
result must be what the ORACLE gives for that source alone (there is no coupling between sources)."""
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


@pytest.mark.parametrize("L", [(4, 4, 4, 4), (16, 16, 16, 4), (6, 4, 2, 8), (2, 2, 2, 2)])
@pytest.mark.parametrize("prec,recon", [(0, 18), (0, 12), (1, 18), (1, 12)])
@pytest.mark.parametrize("nrhs", [1, 2, 3, 4])
@pytest.mark.parametrize("pipe", [1, 0])
def test_dslash_block_matches_oracle(stag, L, prec, recon, nrhs, pipe):
    """pipe = 1: the cp.async-ring kernel where the library picks it (fp64 R >= 3, fp32 R >= 2);
    pipe = 0: the register-staged kernel everywhere."""
    U = si.links_haar(L, 21)
    ctx = stag.Stag(L)
    ctx.set_option("dslash_pipe", pipe)
    packed = ctx.upload_gauge(U, prec, recon)
    vb = ctx.vector_bytes(prec)
    for par in (0, 1):
        vs = [si.source_gaussian(L, 21, stream=1 + 10 * par + k) for k in range(nrhs)]
        vin = ctx.upload_vectors(vs, prec)
        vout = ctx.alloc(nrhs * vb)
        vout.fill_(0xFF)
        ctx.dslash_block(packed, prec, recon, par, nrhs, vin, vout)
        for k in range(nrhs):
            assert rel(ctx.download_vector(vout, prec, k * vb), oracle.dslash(L, U, vs[k], par)) <= TOL[prec]


def block_cg(stag, ctx, packed, prec, recon, bs, mass, shifts, stop, maxiter, residues=None, residue0=0.0,
             want_y=False):
    nrhs, n = len(bs), len(shifts)
    vb = ctx.vector_bytes(prec)
    bdev = ctx.upload_vectors(bs, prec)
    x = ctx.alloc(nrhs * n * vb)
    ws = ctx.alloc(ctx.cg_block_workspace_bytes(prec, n, nrhs))
    y = ctx.alloc(nrhs * vb) if want_y else None
    rc, infos = ctx.mshift_cg_block(packed, prec, recon, nrhs, bdev, mass, shifts, stop, maxiter, x, ws,
                                    residues=residues, residue0=residue0, y_even=y)
    xs = np.stack([np.stack([ctx.download_vector(x, prec, (s * n + i) * vb) for i in range(n)])
                   for s in range(nrhs)])
    ys = [ctx.download_vector(y, prec, s * vb) for s in range(nrhs)] if want_y else None
    return rc, infos, xs, ys


@pytest.mark.parametrize("nrhs", [1, 2, 3, 4])
@pytest.mark.parametrize("recon", [18, 12])
def test_block_cg_config1_every_source_matches_its_own_oracle_solve(stag, nrhs, recon):
    cfg = si.get_config("c1_4x4x4x4")
    L, U, m, shifts = cfg["L"], si.make_links(cfg), cfg["mass"], cfg["shifts"]
    bs = [si.source_gaussian(L, 1001, stream=1 + k) for k in range(nrhs)]
    bs[-1] = 3.0 * bs[-1]                        # different norms: convergence is per source, relative
    ctx = stag.Stag(L)
    packed = ctx.upload_gauge(U, 0, recon)
    residues = [1.0, 0.5, 0.25, 0.125]
    rc, infos, xs, ys = block_cg(stag, ctx, packed, 0, recon, bs, m, shifts, 1e-10, 2000, residues, 2.0, True)
    assert rc == 0 and infos[0]["kernel_launches"] == 1
    A = oracle.dense_A(L, U, m)
    for s, b in enumerate(bs):
        ref = oracle.mshift_cg(L, U, b, m, shifts, 1e-10, 2000)
        assert infos[s]["converged"] and abs(infos[s]["iters"] - ref["iters"]) <= 2
        nb = np.linalg.norm(b)
        for i, sg in enumerate(shifts):
            assert np.linalg.norm(b - oracle.apply_A(L, U, m, sg, xs[s, i])) / nb <= 1e-10
            assert rel(xs[s, i].reshape(-1), oracle.dense_solve(A, sg, b)) < 1e-10 * 16.0 / (m * m + sg)
        assert rel(ys[s], oracle.partial_fraction(b, residues, 2.0, xs[s])) < 1e-15


def test_block_cg_sources_converge_independently(stag):
    """One source is an eigenvector (plane wave on unit links: converges in 1 iteration, P8), one is
    zero (0 iterations, P7 vi), two are Gaussian (<= 4 iterations on free 4^4, P7 v): four different
    iteration counts in one launch, each equal to the single-source result."""
    L, m = (4, 4, 4, 4), 0.2
    shifts = [0.01, 0.04, 0.16, 0.64]
    U = si.links_unit(L)
    pw, p = si.source_plane_wave(L, (1, 3, 0, 2), [1.0, 0.5j, -0.25])
    bs = [pw, np.zeros_like(pw), si.source_gaussian(L, 5, 1), si.source_gaussian(L, 5, 2)]
    ctx = stag.Stag(L)
    packed = ctx.upload_gauge(U, 0, 18)
    rc, infos, xs, _ = block_cg(stag, ctx, packed, 0, 18, bs, m, shifts, 1e-12, 50)
    assert rc == 0
    assert infos[0]["iters"] == 1 and infos[1]["iters"] == 0 and 1 < infos[2]["iters"] <= 4
    lam = m * m + np.sum(np.sin(p) ** 2)
    for i, s in enumerate(shifts):
        assert rel(xs[0, i], pw / (lam + s)) < 1e-14
        assert not xs[1, i].any()
    for k in (2, 3):
        ref = oracle.mshift_cg(L, U, bs[k], m, shifts, 1e-12, 50)
        assert infos[k]["iters"] == ref["iters"]
        for i in range(4):
            assert rel(xs[k, i], ref["x"][i]) < 1e-12


def test_block_cg_notconv_and_same_iterates_as_oracle(stag):
    L, m = (4, 4, 4, 4), 0.1
    shifts = [0.01, 0.04, 0.16, 0.64]
    U = si.links_haar(L, 1)
    bs = [si.source_gaussian(L, 3, 1 + k) for k in range(3)]
    ctx = stag.Stag(L)
    packed = ctx.upload_gauge(U, 0, 18)
    rc, infos, xs, _ = block_cg(stag, ctx, packed, 0, 18, bs, m, shifts, 1e-10, 3)
    assert rc == stag.ERR_NOTCONV
    for s, b in enumerate(bs):
        assert infos[s]["iters"] == 3 and not infos[s]["converged"]
        ref = oracle.mshift_cg(L, U, b, m, shifts, 1e-10, 3)
        for i in range(4):
            assert rel(xs[s, i], ref["x"][i]) < 1e-13


@pytest.mark.parametrize("prec", [0, 1])
def test_block_cg_config2_partial_residency(stag, prec):
    """16^3x4 with 4 sources: 4 x 3 slices do not all fit in shared memory for fp64 (partial residency)."""
    cfg = si.get_config("c2_16x16x16x4")
    L, U, m = cfg["L"], si.make_links(cfg), cfg["mass"]
    shifts = [0.0, 0.05, 0.5]
    stop = 1e-10 if prec == 0 else 1e-4
    bs = [si.source_gaussian(L, 1002, 1 + k) for k in range(4)]
    ctx = stag.Stag(L)
    packed = ctx.upload_gauge(U, prec, 18)
    rc, infos, xs, _ = block_cg(stag, ctx, packed, prec, 18, bs, m, shifts, stop, 5000)
    assert rc == 0
    oracle.set_threads(8)
    try:
        for s, b in enumerate(bs):
            ref = oracle.mshift_cg(L, U, b, m, shifts, stop, 5000)
            assert abs(infos[s]["iters"] - ref["iters"]) <= (2 if prec == 0 else max(2, ref["iters"] // 20))
            nb = np.linalg.norm(b)
            for i, sg in enumerate(shifts):
                tr = np.linalg.norm(b - oracle.apply_A(L, U, m, sg, xs[s, i])) / nb
                assert tr <= (stop if prec == 0 else 2 * stop)
    finally:
        oracle.set_threads(1)


def test_block_badargs(stag):
    L = (4, 4, 4, 4)
    ctx = stag.Stag(L)
    packed = ctx.upload_gauge(si.links_unit(L), 0, 18)
    v = ctx.alloc(5 * ctx.vector_bytes(0))
    w = ctx.alloc(5 * ctx.vector_bytes(0))
    for nrhs in (0, stag.MAX_SHIFTS + 1):
        with pytest.raises(stag.StagError) as ei:
            ctx.dslash_block(packed, 0, 18, 0, nrhs, v, w)
        assert ei.value.code == stag.ERR_BADARG
    assert ctx.cg_block_workspace_bytes(0, 4, 5) == 0


@pytest.mark.parametrize("L", [(4, 4, 4, 4), (16, 16, 16, 4), (6, 4, 2, 8)])
@pytest.mark.parametrize("prec,recon", [(0, 18), (1, 12)])
@pytest.mark.parametrize("nvec", [5, 8, 11])
@pytest.mark.parametrize("pipe", [1, 0])
def test_dslash_block_more_vectors_than_one_link_read_serves(stag, L, prec, recon, nvec, pipe):
    """nrhs > STAG_MAX_RHS: groups of four per read of the links — ONE launch (grid.y = group) where the
    cp.async-ring kernel applies (what stag_fermion_force uses for the D_oe x_i of all its shifts), one launch per
    group otherwise; a short last group included.  Every vector against the oracle."""
    U = si.links_haar(L, 23)
    ctx = stag.Stag(L)
    ctx.set_option("dslash_pipe", pipe)
    packed = ctx.upload_gauge(U, prec, recon)
    vb = ctx.vector_bytes(prec)
    vs = [si.source_gaussian(L, 23, stream=1 + k) for k in range(nvec)]
    vin, vout = ctx.upload_vectors(vs, prec), ctx.alloc(nvec * vb)
    vout.fill_(0xFF)
    ctx.dslash_block(packed, prec, recon, 1, nvec, vin, vout)
    for k in range(nvec):
        assert rel(ctx.download_vector(vout, prec, k * vb), oracle.dslash(L, U, vs[k], 1)) <= TOL[prec]


@pytest.mark.parametrize("slices", [0, 1, 2, 3])
@pytest.mark.parametrize("nrhs", [1, 3])
@pytest.mark.parametrize("prec", [0, 1])
def test_persistent_kernel_with_partial_residency(stag, slices, nrhs, prec):
    """The persistent kernel keeps as many of r, q, p_base in shared memory as fit (all three on small lattices,
    r and q at 4 x 48^3, r only for 4 sources at 32^3 x 8, none at 64^4).  cg_resident_slices forces each of the
    four cases on a lattice the oracle solves in a moment; the result must not depend on it."""
    L = (6, 4, 4, 8)
    U, m, shifts = si.links_haar(L, 91), 0.1, [0.02, 0.3, 0.07, 1.1, 4.0]
    bs = [si.source_gaussian(L, 91, stream=1 + k) for k in range(nrhs)]
    stop = 1e-10 if prec == 0 else 1e-5
    ctx = stag.Stag(L)
    ctx.set_option("cg_resident_slices", slices)
    packed = ctx.upload_gauge(U, prec, 18)
    rc, infos, xs, _ = block_cg(stag, ctx, packed, prec, 18, bs, m, shifts, stop, 5000)
    assert rc == 0
    for s, b in enumerate(bs):
        ref = oracle.mshift_cg(L, U, b, m, shifts, stop, 5000)
        assert abs(infos[s]["iters"] - ref["iters"]) <= 2
        nb = np.linalg.norm(b)
        for i, sg in enumerate(shifts):
            tr = np.linalg.norm(b - oracle.apply_A(L, U, m, sg, xs[s, i])) / nb
            assert tr <= (stop if prec == 0 else 2e-4), (s, i, tr)
    if nrhs == 1:
        vb = ctx.vector_bytes(prec)
        x, ws = ctx.alloc(len(shifts) * vb), ctx.alloc(ctx.cg_workspace_bytes(prec, len(shifts)))
        # the single-source ABI call with the two-reduction kernel is the same arithmetic: bit-equal
        ctx.set_option("cg_single_reduction", 0)
        rc, info = ctx.mshift_cg(packed, prec, 18, ctx.upload_vector(bs[0], prec), m, shifts, stop, 5000, x, ws)
        assert rc == 0 and info["kernel_launches"] == 1 and info["iters"] == infos[0]["iters"]
        assert np.array_equal(ctx.download_vector(x, prec, 2 * vb), xs[0, 2])
        # its default, the single-reduction kernel (needs r and q resident, else it falls back): alpha and beta differ
        # in the last bits, the solutions by rounding
        ctx.set_option("cg_single_reduction", 1)
        rc, info = ctx.mshift_cg(packed, prec, 18, ctx.upload_vector(bs[0], prec), m, shifts, stop, 5000, x, ws)
        assert rc == 0 and info["kernel_launches"] == 1 and abs(info["iters"] - infos[0]["iters"]) <= 1
        got = ctx.download_vector(x, prec, 2 * vb)
        assert np.linalg.norm(got - xs[0, 2]) / np.linalg.norm(xs[0, 2]) <= (1e-9 if prec == 0 else 1e-3)
