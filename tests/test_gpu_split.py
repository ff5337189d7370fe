"""N3: split-double gauge storage.  One resident buffer serves
fp32 (its b planes ARE the fp32 packed format) and ~fp64 (b + c, 48 significant bits).  The oracle side
is oracle.split_double (the paper's two formulas, numpy) + the oracle's own Dslash / operator.

fp64 bound re-derived for b + c: every link real carries a relative error <= 2^-48 = 3.6e-15, a site
sums 72 products of links and O(1) vector entries, so the result is within ~3.6e-15 (rel-L2) of the
unsplit operator — inside the north_star's 1e-13.  Against the oracle applied to the SPLIT links the
difference is rounding only (~3e-16)."""
import numpy as np
import pytest

import oracle
import stag_inputs as si

pytestmark = pytest.mark.gpu


def rel(a, b):
    return np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)


@pytest.fixture(scope="module")
def stag():
    import paper_1010_5433_b200 as m
    return m


@pytest.mark.parametrize("L", [(4, 4, 4, 4), (16, 16, 16, 4), (6, 4, 2, 8), (2, 2, 2, 2), (10, 6, 4, 4)])
@pytest.mark.parametrize("recon", [18, 12])
def test_split_dslash_matches_oracle_on_split_links(stag, L, recon):
    U = si.links_haar(L, 31)
    Us = oracle.split_double(U)
    ctx = stag.Stag(L)
    packed = ctx.upload_gauge(U, stag.F64_SPLIT, recon)
    assert ctx.gauge_packed_bytes(stag.F64_SPLIT, recon) == 2 * ctx.gauge_packed_bytes(stag.F32, recon)
    for par in (0, 1):
        v = si.source_gaussian(L, 31, stream=1 + par)
        vin = ctx.upload_vector(v, stag.F64_SPLIT)
        out = ctx.alloc(ctx.vector_bytes(stag.F64_SPLIT))
        out.fill_(0xFF)
        (ctx.dslash_oe if par else ctx.dslash_eo)(packed, stag.F64_SPLIT, recon, vin, out)
        got = ctx.download_vector(out, stag.F64_SPLIT)
        if recon == 18:
            assert rel(got, oracle.dslash(L, Us, v, par)) <= 2e-15          # rounding only
        assert rel(got, oracle.dslash(L, U, v, par)) <= 1e-13               # the north_star bound still holds


@pytest.mark.parametrize("recon", [18, 12])
def test_split_buffer_serves_fp32_bit_exactly(stag, recon):
    """The first half of the split buffer is the fp32 packed format: an fp32 Dslash on it gives the
    same bits as on a buffer packed with prec = F32."""
    import torch
    L = (8, 8, 4, 6)
    U = si.links_haar(L, 32)
    v = si.source_gaussian(L, 32, stream=3)
    ctx = stag.Stag(L)
    split = ctx.upload_gauge(U, stag.F64_SPLIT, recon)
    p32 = ctx.upload_gauge(U, stag.F32, recon)
    n32 = ctx.gauge_packed_bytes(stag.F32, recon)
    assert torch.equal(split[:n32], p32)
    vin = ctx.upload_vector(v, stag.F32)
    a, b = ctx.alloc(ctx.vector_bytes(stag.F32)), ctx.alloc(ctx.vector_bytes(stag.F32))
    ctx.dslash_oe(split, stag.F32, recon, vin, a)
    ctx.dslash_oe(p32, stag.F32, recon, vin, b)
    assert torch.equal(a, b)
    assert rel(ctx.download_vector(a, stag.F32), oracle.dslash_oe(L, U, v)) <= 1e-5


def test_split_c_planes_are_the_papers_formula(stag):
    """c = (float)(a - (double)b) on the packed hopping matrices: b + c == split_double(W) where W = +-1/2 U
    — checked through the result: with unit-modulus diagonal links exp(i t) the Dslash of a constant
    vector is a sum of split numbers, exactly representable, so the comparison is bit-exact."""
    L = (4, 4, 4, 4)
    V = int(np.prod(L))
    rng = np.random.default_rng(7)
    t = rng.uniform(0, 2 * np.pi, (V, 4, 3))
    U = np.zeros((V, 4, 3, 3), dtype=np.complex128)
    for c in range(3):
        U[:, :, c, c] = np.exp(1j * t[:, :, c])
    ctx = stag.Stag(L)
    packed = ctx.upload_gauge(U, stag.F64_SPLIT, 18)           # recon 18: no SU(3) requirement
    v = np.zeros((V // 2, 3), dtype=np.complex128)
    v[5, 1] = 1.0                                                # delta source: every output is ONE product
    out = ctx.alloc(ctx.vector_bytes(stag.F64_SPLIT))
    ctx.dslash_oe(packed, stag.F64_SPLIT, 18, ctx.upload_vector(v, stag.F64_SPLIT), out)
    got = ctx.download_vector(out, stag.F64_SPLIT)
    want = oracle.dslash_oe(L, oracle.split_double(U), v)
    assert np.count_nonzero(want) == 8
    assert np.array_equal(got, want)
    assert not np.array_equal(got, oracle.dslash_oe(L, U, v))


@pytest.mark.parametrize("path", ["persistent", "multikernel"])
@pytest.mark.parametrize("recon", [18, 12])
def test_split_cg_config1(stag, path, recon):
    cfg = si.get_config("c1_4x4x4x4")
    L, U, b, m, shifts = cfg["L"], si.make_links(cfg), si.make_source(cfg), cfg["mass"], cfg["shifts"]
    ctx = stag.Stag(L)
    ctx.set_option("cg_persistent", 1 if path == "persistent" else 0)
    P = stag.F64_SPLIT
    packed = ctx.upload_gauge(U, P, recon)
    n, vb = len(shifts), ctx.vector_bytes(P)
    x, ws = ctx.alloc(n * vb), ctx.alloc(ctx.cg_workspace_bytes(P, n))
    rc, info = ctx.mshift_cg(packed, P, recon, ctx.upload_vector(b, P), m, shifts, 1e-10, 2000, x, ws)
    ref = oracle.mshift_cg(L, U, b, m, shifts, 1e-10, 2000)
    assert rc == 0 and abs(info["iters"] - ref["iters"]) <= 2
    assert info["kernel_launches"] == 1 if path == "persistent" else info["kernel_launches"] > 1
    A = oracle.dense_A(L, U, m)
    for i, s in enumerate(shifts):
        xi = ctx.download_vector(x, P, i * vb)
        assert np.linalg.norm(b - oracle.apply_A(L, U, m, s, xi)) / np.linalg.norm(b) <= 1e-10
        xd = oracle.dense_solve(A, s, b).reshape(-1, 3)
        assert rel(xi, xd) <= 1e-8


def test_split_cg_config2_single_shift(stag):
    cfg = si.get_config("c2_16x16x16x4")
    L, U, b, m, shifts = cfg["L"], si.make_links(cfg), si.make_source(cfg), cfg["mass"], cfg["shifts"]
    ctx = stag.Stag(L)
    P = stag.F64_SPLIT
    packed = ctx.upload_gauge(U, P, 18)
    vb = ctx.vector_bytes(P)
    x, ws = ctx.alloc(vb), ctx.alloc(ctx.cg_workspace_bytes(P, 1))
    rc, info = ctx.mshift_cg(packed, P, 18, ctx.upload_vector(b, P), m, shifts, 1e-10, 20000, x, ws)
    ref = oracle.mshift_cg(L, U, b, m, shifts, 1e-10, 20000)
    assert rc == 0 and abs(info["iters"] - ref["iters"]) <= 2
    xi = ctx.download_vector(x, P)
    assert np.linalg.norm(b - oracle.apply_A(L, U, m, shifts[0], xi)) / np.linalg.norm(b) <= 1e-10


@pytest.mark.parametrize("L", [(4, 4, 4, 4), (6, 4, 2, 8), (16, 16, 16, 4)])
@pytest.mark.parametrize("recon", [18, 12])
@pytest.mark.parametrize("nrhs", [1, 2, 3, 4, 7])
def test_split_block_dslash_matches_oracle_on_split_links(stag, L, recon, nrhs):
    """N3 x N1: stag_dslash_block on a split-double buffer = the oracle's D applied with oracle.split_double(U),
    every source, both parities, up to rounding; within the north_star's 1e-13 of the unsplit operator."""
    U = si.links_haar(L, 91)
    Us = oracle.split_double(U)
    ctx = stag.Stag(L)
    packed = ctx.upload_gauge(U, stag.F64_SPLIT, recon)
    vb = ctx.vector_bytes(stag.F64)
    srcs = [si.source_gaussian(L, 91, stream=1 + k) for k in range(nrhs)]
    vin, vout = ctx.upload_vectors(srcs, stag.F64), ctx.alloc(nrhs * vb)
    for par, ofun in ((1, oracle.dslash_oe), (0, oracle.dslash_eo)):
        ctx.dslash_block(packed, stag.F64_SPLIT, recon, par, nrhs, vin, vout)
        for k in range(nrhs):
            got = ctx.download_vector(vout, stag.F64, k * vb)
            assert rel(got, ofun(L, Us, srcs[k])) <= 5e-15
            assert rel(got, ofun(L, U, srcs[k])) <= 1e-13


def test_split_block_cg_equals_single_solves(stag):
    """N3 x N1: stag_mshift_cg_block on split-double links: per source the iteration count of the single solve on
    the same buffer and true residuals <= stop by the oracle's operator."""
    cfg = si.get_config("c1_4x4x4x4")
    L, U, m, shifts = cfg["L"], si.make_links(cfg), cfg["mass"], cfg["shifts"]
    ctx = stag.Stag(L)
    P = stag.F64_SPLIT
    packed = ctx.upload_gauge(U, P, 18)
    n, vb = len(shifts), ctx.vector_bytes(P)
    srcs = [si.source_gaussian(L, 92, stream=1 + k) for k in range(3)]
    x = ctx.alloc(3 * n * vb)
    ws = ctx.alloc(ctx.cg_block_workspace_bytes(P, n, 3))
    rc, infos = ctx.mshift_cg_block(packed, P, 18, 3, ctx.upload_vectors(srcs, P), m, shifts, 1e-10, 2000, x, ws)
    assert rc == 0
    x1, ws1 = ctx.alloc(n * vb), ctx.alloc(ctx.cg_workspace_bytes(P, n))
    for s, b in enumerate(srcs):
        rc1, i1 = ctx.mshift_cg(packed, P, 18, ctx.upload_vector(b, P), m, shifts, 1e-10, 2000, x1, ws1)
        assert rc1 == 0 and abs(infos[s]["iters"] - i1["iters"]) <= 1 and infos[s]["converged"]
        for i, sig in enumerate(shifts):
            xi = ctx.download_vector(x, P, (s * n + i) * vb)
            assert np.linalg.norm(b - oracle.apply_A(L, U, m, sig, xi)) / np.linalg.norm(b) <= 1e-10
            assert rel(xi, ctx.download_vector(x1, P, i * vb)) <= 1e-8      # two converged solves: ~ stop * kappa apart


@pytest.mark.parametrize("L", [(4, 4, 4, 4), (6, 4, 2, 8), (16, 16, 16, 4)])
@pytest.mark.parametrize("recon", [18, 12])
def test_split_force_matches_oracle_on_split_links(stag, L, recon):
    """N3 x N4: the fermion force read from a split-double buffer = the oracle's force with split_double(U)."""
    import torch
    U = si.links_haar(L, 93)
    xs = [si.source_gaussian(L, 93, stream=1 + k) for k in range(5)]
    residues = [0.7, -0.3, 1.9, 0.05, 2.5]
    ctx = stag.Stag(L)
    packed = ctx.upload_gauge(U, stag.F64_SPLIT, recon)
    F = torch.full((ctx.V * 72,), float("nan"), dtype=torch.float64, device="cuda")
    ws = ctx.alloc(ctx.force_workspace_bytes(stag.F64_SPLIT, 5))
    ctx.fermion_force(packed, stag.F64_SPLIT, recon, residues, ctx.upload_vectors(xs, stag.F64), F, ws)
    got = F.cpu().numpy().view(np.complex128).reshape(ctx.V, 4, 3, 3)
    assert np.isfinite(got.view(np.float64)).all()
    assert rel(got, oracle.fermion_force(L, oracle.split_double(U), residues, np.stack(xs))) <= 2e-14
    assert rel(got, oracle.fermion_force(L, U, residues, np.stack(xs))) <= 1e-13
