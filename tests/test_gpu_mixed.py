"""N2: mixed precision the way the paper uses it: an fp32
multi-shift run, then a per-shift fp64 defect-correction polish = ordinary CG with a non-zero start.

Parity: the polished x_i is a solution of (A + sigma_i) x_i = b, so the bar is the north_star's —
TRUE residual <= stop for every shift by the ORACLE's operator (several x_i are correct, reading A14) —
plus, where the start vector is an input both sides share (stag_cg_polish), the polish iteration count
within +-2 of oracle.cg_polish from the same start, and agreement with the dense solve on 4^4."""
import numpy as np
import pytest

import oracle
import stag_inputs as si

pytestmark = pytest.mark.gpu


def rel(a, b):
    return np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)


def true_res(L, U, m, s, b, x):
    return np.linalg.norm(b - oracle.apply_A(L, U, m, s, x)) / np.linalg.norm(b)


def fp32_like(x, seed):
    """a start vector of fp32 quality, made on the ORACLE side: the solution rounded to fp32 + 1e-6 noise"""
    rng = np.random.default_rng(seed)
    x32 = x.astype(np.complex64).astype(np.complex128)
    return x32 + 1e-6 * np.linalg.norm(x) / np.sqrt(x.size) * (rng.standard_normal(x.shape) + 1j * rng.standard_normal(x.shape))


@pytest.fixture(scope="module")
def stag():
    import paper_1010_5433_b200 as m
    return m


@pytest.mark.parametrize("L", [(4, 4, 4, 4), (6, 4, 2, 8)])
@pytest.mark.parametrize("nvec", [1, 3])
def test_vector_convert_roundtrip(stag, L, nvec):
    ctx = stag.Stag(L)
    vs = [si.source_gaussian(L, 51, stream=1 + k) for k in range(nvec)]
    d64 = ctx.upload_vectors(vs, stag.F64)
    d32 = ctx.alloc(nvec * ctx.vector_bytes(stag.F32))
    ctx.vector_convert(d64, stag.F64, d32, stag.F32, nvec)
    back = ctx.alloc(nvec * ctx.vector_bytes(stag.F64))
    ctx.vector_convert(d32, stag.F32, back, stag.F64, nvec)
    for k, v in enumerate(vs):
        want32 = v.astype(np.complex64).astype(np.complex128)          # b = (float)a
        assert np.array_equal(ctx.download_vector(d32, stag.F32, k * ctx.vector_bytes(stag.F32)), want32)
        assert np.array_equal(ctx.download_vector(back, stag.F64, k * ctx.vector_bytes(stag.F64)), want32)


@pytest.mark.parametrize("prec_name,recon", [("F64", 18), ("F64", 12), ("F64_SPLIT", 18)])
@pytest.mark.parametrize("nshift", [1, 4, 6])
def test_polish_from_shared_start_matches_oracle_polish(stag, prec_name, recon, nshift):
    prec = getattr(stag, prec_name)
    L = (4, 4, 4, 4)
    U, b, m = si.links_haar(L, 52), si.source_gaussian(L, 52), 0.1
    shifts = [0.01, 0.04, 0.16, 0.64, 1.5, 0.0][:nshift]
    stop = 1e-11
    A = oracle.dense_A(L, U, m)
    xd = [oracle.dense_solve(A, s, b).reshape(-1, 3) for s in shifts]
    x0 = [fp32_like(x, 7 + i) for i, x in enumerate(xd)]
    if nshift >= 4:
        x0[2] = xd[2]                                   # already converged: must be left untouched, 0 iterations
    ctx = stag.Stag(L)
    packed = ctx.upload_gauge(U, prec, recon)
    vb = ctx.vector_bytes(stag.F64)
    x = ctx.upload_vectors(x0, stag.F64)
    ws = ctx.alloc(ctx.cg_polish_workspace_bytes())
    rc, info = ctx.cg_polish(packed, prec, recon, ctx.upload_vector(b, stag.F64), m, shifts, stop, 2000, x, ws)
    assert rc == 0, info
    assert 1 <= info["passes"] <= 2
    for i, s in enumerate(shifts):
        xi = ctx.download_vector(x, stag.F64, i * vb)
        ref = oracle.cg_polish(L, U, b, m, s, x0[i], stop, 2000)
        assert abs(info["resid_before"][i] - ref["res0"]) <= 1e-3 * ref["res0"] + 1e-14
        assert true_res(L, U, m, s, b, xi) <= stop
        assert abs(info["resid_after"][i] - true_res(L, U, m, s, b, xi)) <= 0.05 * stop + 1e-13
        assert rel(xi, xd[i]) <= 1e-9
        if nshift >= 4 and i == 2:
            assert info["iters"][i] == 0 and ref["iters"] == 0 and np.array_equal(xi, x0[i])
        elif info["passes"] == 1:
            assert abs(info["iters"][i] - ref["iters"]) <= 2, (i, info["iters"], ref["iters"])
        else:
            assert ref["iters"] - 2 <= info["iters"][i] <= ref["iters"] + 12      # a second pass adds a few


@pytest.mark.parametrize("hi,recon_hi,recon_lo,reliable", [("F64", 18, 18, 2), ("F64", 12, 12, 2), ("F64", 18, 18, 1),
                                                           ("F64", 18, 12, 2), ("F64_SPLIT", 18, 18, 2)])
def test_mixed_config1(stag, hi, recon_hi, recon_lo, reliable):
    """reliable = 2 (forced; the default 1 uses it for single-shift solves only) with fp64 or split-double matrices of the same recon: the inner stage is the persistent kernel with
    residual replacement (fp32 matrices, fp64 x_i, convergence on the TRUE fp64 residual of the base system);
    otherwise (option at its default with several shifts, different recon) the plain fp32 stage + polish."""
    cfg = si.get_config("c1_4x4x4x4")
    L, U, b, m, shifts = cfg["L"], si.make_links(cfg), si.make_source(cfg), cfg["mass"], cfg["shifts"]
    ctx = stag.Stag(L)
    ctx.set_option("cg_mixed_reliable", reliable)
    ctx.set_option("cg_mixed_fp64_from", 0)          # the fp32 routes are what is tested here (default: 4 shifts -> fp64)
    replaced = reliable == 2 and recon_hi == recon_lo
    prec_hi = getattr(stag, hi)
    p_hi = ctx.upload_gauge(U, prec_hi, recon_hi)
    p_lo = p_hi if hi == "F64_SPLIT" else ctx.upload_gauge(U, stag.F32, recon_lo)   # N3: one buffer, both precisions
    n, vb = len(shifts), ctx.vector_bytes(stag.F64)
    x, y = ctx.alloc(n * vb), ctx.alloc(vb)
    ws = ctx.alloc(ctx.mshift_cg_mixed_workspace_bytes(n))
    residues = [1.0, 0.5, 0.25, 0.125]
    rc, info = ctx.mshift_cg_mixed(p_hi, prec_hi, recon_hi, p_lo, recon_lo, ctx.upload_vector(b, stag.F64), m,
                                   shifts, 1e-10, 2000, x, ws, residues=residues, residue0=2.0, y_even=y)
    assert rc == 0, info
    ref = oracle.mshift_cg(L, U, b, m, shifts, 1e-10, 2000)
    if replaced:
        assert info["reliable_updates"] >= 2 and info["inner"]["converged"] and info["inner"]["kernel_launches"] == 1
        assert info["polish"]["resid_before"][shifts.index(min(shifts))] <= 1e-10     # converged on the true residual
        # the shifted systems ride along: their floor is the fp32 rounding of the matrices times ||x_i|| / ||b||
        assert max(info["polish"]["resid_before"]) <= 1e-5
        assert abs(info["inner"]["iters"] - ref["iters"]) <= max(10, ref["iters"] // 5)
    else:
        assert info["reliable_updates"] == 0
        assert info["inner"]["iters"] > 0 and max(info["polish"]["iters"]) > 0
    A = oracle.dense_A(L, U, m)
    xs = []
    for i, s in enumerate(shifts):
        xi = ctx.download_vector(x, stag.F64, i * vb)
        xs.append(xi)
        if not replaced:
            assert 1e-9 < info["polish"]["resid_before"][i] < 1e-2      # what fp32 alone reached
        assert true_res(L, U, m, s, b, xi) <= 1e-10
        assert rel(xi, oracle.dense_solve(A, s, b).reshape(-1, 3)) <= 1e-8
    assert rel(ctx.download_vector(y, stag.F64), oracle.partial_fraction(b, residues, 2.0, np.stack(xs))) <= 1e-14


@pytest.mark.parametrize("slices", [3, 1, 0])
@pytest.mark.parametrize("recon", [18, 12])
@pytest.mark.parametrize("hi", ["F64", "F64_SPLIT"])
def test_mixed_single_shift_residual_replacement(stag, slices, recon, hi):
    """Single shift, default options: the inner stage is the persistent residual-replacement kernel; it must stop
    on the TRUE residual (nothing left to polish), in about as many iterations as the fp64 oracle, in every
    shared-memory residency case."""
    cfg = si.get_config("c2_16x16x16x4")
    L, U, b, m, shifts = cfg["L"], si.make_links(cfg), si.make_source(cfg), cfg["mass"], cfg["shifts"]
    ctx = stag.Stag(L)
    ctx.set_option("cg_resident_slices", slices)
    prec_hi = getattr(stag, hi)
    p64 = ctx.upload_gauge(U, prec_hi, recon)
    p32 = p64 if hi == "F64_SPLIT" else ctx.upload_gauge(U, stag.F32, recon)      # N3: one buffer, both precisions
    vb = ctx.vector_bytes(stag.F64)
    x, ws = ctx.alloc(vb), ctx.alloc(ctx.mshift_cg_mixed_workspace_bytes(1))
    x.fill_(0xFF)
    rc, info = ctx.mshift_cg_mixed(p64, prec_hi, recon, p32, recon, ctx.upload_vector(b, stag.F64), m, shifts,
                                   1e-10, 20000, x, ws)
    ref = oracle.mshift_cg(L, U, b, m, shifts, 1e-10, 20000)
    assert rc == 0 and info["inner"]["converged"] and info["inner"]["kernel_launches"] == 1, info
    assert info["reliable_updates"] >= 5 and sum(info["polish"]["iters"]) == 0 and info["polish"]["passes"] == 0
    assert abs(info["inner"]["iters"] - ref["iters"]) <= max(3, ref["iters"] // 10)
    assert true_res(L, U, m, shifts[0], b, ctx.download_vector(x, stag.F64)) <= 1e-10
    # maxiter reached: reports NOTCONV with the true residual it got to
    rc, info = ctx.mshift_cg_mixed(p64, prec_hi, recon, p32, recon, ctx.upload_vector(b, stag.F64), m, shifts,
                                   1e-10, 5, x, ws)
    assert rc == stag.ERR_NOTCONV and info["inner"]["iters"] == 5 and info["polish"]["resid_after"][0] > 1e-10


def test_mixed_config2_single_shift(stag):
    cfg = si.get_config("c2_16x16x16x4")
    L, U, b, m, shifts = cfg["L"], si.make_links(cfg), si.make_source(cfg), cfg["mass"], cfg["shifts"]
    ctx = stag.Stag(L)
    split = ctx.upload_gauge(U, stag.F64_SPLIT, 18)
    vb = ctx.vector_bytes(stag.F64)
    x, ws = ctx.alloc(vb), ctx.alloc(ctx.mshift_cg_mixed_workspace_bytes(1))
    rc, info = ctx.mshift_cg_mixed(split, stag.F64_SPLIT, 18, split, 18, ctx.upload_vector(b, stag.F64), m, shifts,
                                   1e-10, 20000, x, ws)
    ref = oracle.mshift_cg(L, U, b, m, shifts, 1e-10, 20000)
    assert rc == 0, info
    assert true_res(L, U, m, shifts[0], b, ctx.download_vector(x, stag.F64)) <= 1e-10
    # the fp64 polish is a fraction of a full fp64 solve
    assert info["polish"]["iters"][0] < 0.8 * ref["iters"]


def test_mixed_config3_metropolis_stop_1e12(stag):
    """Reading A8: at stop 1e-12 the fp64 multi-shift run alone ends with true residuals up to ~1.5 stop;
    the polish brings every shift to <= stop."""
    cfg = si.get_config("c3_24x24x24x6")
    L, U, b, m, shifts = cfg["L"], si.make_links(cfg), si.make_source(cfg), cfg["mass"], cfg["shifts"]
    oracle.set_threads(8)
    try:
        ctx = stag.Stag(L)
        p64 = ctx.upload_gauge(U, stag.F64, 18)
        p32 = ctx.upload_gauge(U, stag.F32, 18)
        n, vb = len(shifts), ctx.vector_bytes(stag.F64)
        x, ws = ctx.alloc(n * vb), ctx.alloc(ctx.mshift_cg_mixed_workspace_bytes(n))
        bdev = ctx.upload_vector(b, stag.F64)
        rc, info = ctx.mshift_cg_mixed(p64, stag.F64, 18, p32, 18, bdev, m, shifts, 1e-12, 100000, x, ws)
        assert rc == 0, info
        for i, s in enumerate(shifts):
            assert true_res(L, U, m, s, b, ctx.download_vector(x, stag.F64, i * vb)) <= 1e-12
        # A8 remedy on an fp64 multi-shift result
        cgws = ctx.alloc(ctx.cg_workspace_bytes(stag.F64, n))
        rc, _ = ctx.mshift_cg(p64, stag.F64, 18, bdev, m, shifts, 1e-12, 100000, x, cgws)
        assert rc == 0
        pws = ctx.alloc(ctx.cg_polish_workspace_bytes())
        rc, pinfo = ctx.cg_polish(p64, stag.F64, 18, bdev, m, shifts, 1e-12, 100000, x, pws)
        assert rc == 0, pinfo
        assert max(pinfo["resid_before"]) <= 3e-12                       # the A8 band
        for i, s in enumerate(shifts):
            assert true_res(L, U, m, s, b, ctx.download_vector(x, stag.F64, i * vb)) <= 1e-12
            if pinfo["resid_before"][i] <= 1e-12:
                assert pinfo["iters"][i] == 0
    finally:
        oracle.set_threads(1)


@pytest.mark.parametrize("hi", ["F64", "F64_SPLIT"])
def test_mixed_default_route_is_the_fastest_one(stag, hi):
    """Default options: 1 shift -> route 1 (residual replacement), 2 shifts -> route 2 (fp32 + polish), from 3 shifts
    on -> route 3, the fp64 multi-shift solve itself (the paper's choice for the Metropolis solves):
    then the iteration count is the oracle's +-2 and the polish finds nothing to do.  With a stop fp32 can reach the
    fp32 routes are kept.  Every x_i must meet the stop by the oracle's operator on every route."""
    cfg = si.get_config("c1_4x4x4x4")
    L, U, b, m = cfg["L"], si.make_links(cfg), si.make_source(cfg), cfg["mass"]
    all_shifts = [0.01, 0.04, 0.16, 0.64, 1.5]
    ctx = stag.Stag(L)
    prec_hi = getattr(stag, hi)
    p_hi = ctx.upload_gauge(U, prec_hi, 18)
    p_lo = p_hi if hi == "F64_SPLIT" else ctx.upload_gauge(U, stag.F32, 18)
    vb = ctx.vector_bytes(stag.F64)
    bdev = ctx.upload_vector(b, stag.F64)
    for n, want in ((1, 1), (2, 2), (3, 3), (5, 3)):
        shifts = all_shifts[:n]
        x, ws = ctx.alloc(n * vb), ctx.alloc(ctx.mshift_cg_mixed_workspace_bytes(n))
        rc, info = ctx.mshift_cg_mixed(p_hi, prec_hi, 18, p_lo, 18, bdev, m, shifts, 1e-10, 2000, x, ws)
        assert rc == 0 and info["route"] == want, (n, info["route"])
        for i, s in enumerate(shifts):
            assert true_res(L, U, m, s, b, ctx.download_vector(x, stag.F64, i * vb)) <= 1e-10
        if want == 3:
            ref = oracle.mshift_cg(L, U, b, m, shifts, 1e-10, 2000)
            assert abs(info["inner"]["iters"] - ref["iters"]) <= 2 and info["reliable_updates"] == 0
            assert sum(info["polish"]["iters"]) == 0 and max(info["polish"]["resid_before"]) <= 1e-10
    # a stop fp32 reaches: stays on the fp32 routes whatever the number of shifts
    x, ws = ctx.alloc(5 * vb), ctx.alloc(ctx.mshift_cg_mixed_workspace_bytes(5))
    rc, info = ctx.mshift_cg_mixed(p_hi, prec_hi, 18, p_lo, 18, bdev, m, all_shifts, 1e-5, 2000, x, ws)
    assert rc == 0 and info["route"] == 2
    ctx.set_option("cg_mixed_fp64_from", 0)
    rc, info = ctx.mshift_cg_mixed(p_hi, prec_hi, 18, p_lo, 18, bdev, m, all_shifts, 1e-10, 2000, x, ws)
    assert rc == 0 and info["route"] == 2 and max(info["polish"]["iters"]) > 0


def test_mixed_residual_replacement_stagnation_latch(stag):
    """A stop the true residual cannot reach (1e-18): the residual-replacement kernel must not run to maxiter — three
    replacements in a row that gain less than 10 % latch stagnated = 1 — and the call reports NOTCONV with the
    true residuals it reached (far below fp32's floor, since x and the replacements are fp64)."""
    cfg = si.get_config("c1_4x4x4x4")
    L, U, b, m = cfg["L"], si.make_links(cfg), si.make_source(cfg), cfg["mass"]
    ctx = stag.Stag(L)
    split = ctx.upload_gauge(U, stag.F64_SPLIT, 18)
    vb = ctx.vector_bytes(stag.F64)
    x, ws = ctx.alloc(vb), ctx.alloc(ctx.mshift_cg_mixed_workspace_bytes(1))
    rc, info = ctx.mshift_cg_mixed(split, stag.F64_SPLIT, 18, split, 18, ctx.upload_vector(b, stag.F64), m, [0.01],
                                   1e-18, 20000, x, ws)
    assert rc == stag.ERR_NOTCONV and info["route"] == 1
    assert info["inner"]["stagnated"] and not info["inner"]["converged"] and not info["inner"]["breakdown"]
    assert info["inner"]["iters"] < 2000 and info["reliable_updates"] >= 3
    assert info["polish"]["resid_after"][0] < 1e-12
    assert true_res(L, U, m, 0.01, b, ctx.download_vector(x, stag.F64)) < 1e-12


def test_mixed_bad_arguments(stag):
    L = (4, 4, 4, 4)
    ctx = stag.Stag(L)
    U = si.links_haar(L, 3)
    p64, p32 = ctx.upload_gauge(U, stag.F64, 18), ctx.upload_gauge(U, stag.F32, 18)
    vb = ctx.vector_bytes(stag.F64)
    b, x, ws = ctx.alloc(vb), ctx.alloc(vb), ctx.alloc(ctx.mshift_cg_mixed_workspace_bytes(1))
    b.zero_()
    for kw in (dict(stop=0.0), dict(shifts=[-1.0]), dict(prec_hi=stag.F32)):
        with pytest.raises(stag.StagError) as e:
            ctx.mshift_cg_mixed(p64, kw.get("prec_hi", stag.F64), 18, p32, 18, b, 0.1, kw.get("shifts", [0.1]),
                                kw.get("stop", 1e-10), 100, x, ws)
        assert e.value.code == stag.ERR_BADARG
    rc, info = ctx.mshift_cg_mixed(p64, stag.F64, 18, p32, 18, b, 0.1, [0.1], 1e-10, 100, x, ws)   # b = 0
    assert rc == 0 and info["polish"]["passes"] == 0
    assert not ctx.download_vector(x, stag.F64).any()
