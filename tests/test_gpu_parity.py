"""GPU parity: the CUDA path (through the C ABI) against the oracle, element by element on the same
seeded inputs (SURVEY.md §8(c) acceptance): fp64 Dslash rel-L2 <= 1e-13, fp32 <= 1e-5, CG true
residual (by the ORACLE's operator) <= stop for every shift, iterations within +-2."""
import numpy as np
import pytest

import oracle
import stag_inputs as si

pytestmark = pytest.mark.gpu

TOL = {0: 1e-13, 1: 1e-5}     # north_star tolerances, keyed by prec (F64, F32)


def rel(a, b):
    return np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)


@pytest.fixture(scope="module")
def stag():
    import paper_1010_5433_b200 as m
    return m


_cache = {}


def setup(stag, L, kind, seed, eps=None):
    key = (tuple(L), kind, seed, eps)
    if key not in _cache:
        if kind == "haar":
            U = si.links_haar(L, seed)
        elif kind == "smooth":
            U = si.links_smooth(L, seed, eps)
        else:
            U = si.links_unit(L)
        _cache[key] = (stag.Stag(L), U, {})
    return _cache[key]


def packed_for(stag, entry, prec, recon):
    ctx, U, packs = entry
    if (prec, recon) not in packs:
        packs[(prec, recon)] = ctx.upload_gauge(U, prec, recon)
    return packs[(prec, recon)]


def gpu_dslash(stag, entry, prec, recon, v, out_parity):
    ctx = entry[0]
    packed = packed_for(stag, entry, prec, recon)
    vin = ctx.upload_vector(v, prec)
    vout = ctx.alloc(ctx.vector_bytes(prec))
    (ctx.dslash_eo if out_parity == 0 else ctx.dslash_oe)(packed, prec, recon, vin, vout)
    return ctx.download_vector(vout, prec)


# lattices: config 1, config 2, ragged extents (several CTAs + a tail), the degenerate L=2 cases
LATTICES = [((4, 4, 4, 4), "haar", 1001, None), ((16, 16, 16, 4), "smooth", 1002, 0.3),
            ((6, 4, 2, 8), "haar", 11, None), ((2, 2, 2, 2), "haar", 12, None),
            ((10, 6, 4, 2), "haar", 13, None), ((2, 6, 2, 4), "haar", 14, None)]


@pytest.mark.parametrize("L,kind,seed,eps", LATTICES)
@pytest.mark.parametrize("prec", [0, 1])
@pytest.mark.parametrize("recon", [18, 12])
def test_dslash_matches_oracle(stag, L, kind, seed, eps, prec, recon):
    entry = setup(stag, L, kind, seed, eps)
    U = entry[1]
    for out_parity in (0, 1):
        v = si.source_gaussian(L, seed, stream=1 + out_parity)
        want = oracle.dslash(L, U, v, out_parity)
        got = gpu_dslash(stag, entry, prec, recon, v, out_parity)
        assert rel(got, want) <= TOL[prec], (L, prec, recon, out_parity)


@pytest.mark.parametrize("block", [64, 128, 256])
@pytest.mark.parametrize("ctas", [0, 1, 3])
def test_dslash_launch_configs(stag, block, ctas):
    L = (16, 16, 16, 4)
    entry = setup(stag, L, "smooth", 1002, 0.3)
    ctx = entry[0]
    ctx.set_option("dslash_block", block)
    ctx.set_option("dslash_ctas_per_sm", ctas)
    try:
        v = si.source_gaussian(L, 5, 1)
        assert rel(gpu_dslash(stag, entry, 0, 18, v, 1), oracle.dslash(L, entry[1], v, 1)) <= 1e-13
    finally:
        ctx.set_option("dslash_block", 128)
        ctx.set_option("dslash_ctas_per_sm", 0)


def test_P1_free_spectrum_on_gpu(stag):
    L = (4, 4, 2, 6)
    entry = setup(stag, L, "unit", 0)
    for n, col in [((1, 3, 0, 2), [1.0, 0.5j, -0.25]), ((0, 0, 1, 5), [0, 1, 0]), ((3, 2, 1, 0), [1j, 1, 1])]:
        v, p = si.source_plane_wave(L, n, col)
        for recon in (18, 12):
            w = gpu_dslash(stag, entry, 0, recon, gpu_dslash(stag, entry, 0, recon, v, 1), 0)
            assert rel(w, -np.sum(np.sin(p) ** 2) * v) < 1e-14


def test_P2_antihermitian_on_gpu(stag):
    L = (6, 4, 2, 8)
    entry = setup(stag, L, "haar", 11)
    psi, chi = si.source_gaussian(L, 77, 1), si.source_gaussian(L, 77, 2)
    lhs = np.vdot(chi, gpu_dslash(stag, entry, 0, 18, psi, 1))
    rhs = -np.vdot(gpu_dslash(stag, entry, 0, 18, chi, 0), psi)
    assert abs(lhs - rhs) / abs(lhs) < 1e-14


def test_P3_gauge_covariance_on_gpu(stag):
    L = (4, 4, 4, 4)
    U = si.links_haar(L, 31)
    g = si.gauge_transform_field(L, 31)
    Ug = si.apply_gauge_transform(L, U, g)
    psi = si.source_gaussian(L, 31, 3)
    ctx = stag.Stag(L)
    outs = []
    for links, vec in ((Ug, np.einsum("xij,xj->xi", g[si.parity_sites(L, 1)], psi)), (U, psi)):
        packed = ctx.upload_gauge(links, 0, 18)
        vin = ctx.upload_vector(vec, 0)
        vout = ctx.alloc(ctx.vector_bytes(0))
        ctx.dslash_eo(packed, 0, 18, vin, vout)
        outs.append(ctx.download_vector(vout, 0))
    assert rel(outs[0], np.einsum("xij,xj->xi", g[si.parity_sites(L, 0)], outs[1])) < 1e-14


def test_P6_recon12_equals_recon18_and_rejects_non_su3(stag):
    L = (6, 4, 2, 8)
    entry = setup(stag, L, "haar", 11)
    v = si.source_gaussian(L, 3, 1)
    for par in (0, 1):
        a = gpu_dslash(stag, entry, 0, 18, v, par)
        b = gpu_dslash(stag, entry, 0, 12, v, par)
        assert rel(b, a) < 1e-14
    bad = entry[1].copy()
    bad[7, 2] *= 1.0 + 1e-9                       # not unitary any more
    ctx = entry[0]
    with pytest.raises(stag.StagError) as ei:
        ctx.upload_gauge(bad, 0, 12)
    assert ei.value.code == stag.ERR_NOT_SU3
    ctx.upload_gauge(bad, 0, 18)                  # 18-real storage takes any matrix
    bad2 = entry[1].copy()
    bad2[5, 1] *= np.exp(0.3j)                    # unitary, det != 1
    with pytest.raises(stag.StagError):
        ctx.upload_gauge(bad2, 1, 12)


def test_host_variant_equals_device_variant(stag):
    L = (16, 16, 16, 4)
    entry = setup(stag, L, "smooth", 1002, 0.3)
    ctx = entry[0]
    v = si.source_gaussian(L, 8, 1)
    for prec in (0, 1):
        packed = packed_for(stag, entry, prec, 18)
        scratch = ctx.alloc(ctx.host_scratch_bytes(prec, 0))
        out = np.empty_like(v)
        ctx.dslash_host(packed, prec, 18, 1, v, out, scratch)
        assert np.array_equal(out, gpu_dslash(stag, entry, prec, 18, v, 1))
