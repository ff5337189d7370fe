"""GPU parity of stag_mshift_cg against the oracle (SURVEY.md §8(c) acceptance, pins P7/P8 on the GPU).
x_i is any vector meeting the residual bound (reading A14): compare by TRUE residual computed with
the ORACLE's operator, iteration counts within +-2, and element-wise only up to stop*kappa."""
import numpy as np
import pytest

import oracle
import stag_inputs as si

pytestmark = pytest.mark.gpu


def rel(a, b):
    return np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)


@pytest.fixture(scope="module", params=["persistent", "multikernel"])
def stag(request):
    """The binding, with Stag(L) pinned to one of the two CG paths: the single cooperative launch
    (stag_cg_persist.cu) or four launches per iteration (stag_cg.cu).  Both must pass every test."""
    import types

    import paper_1010_5433_b200 as m

    def make(L):
        ctx = m.Stag(L)
        ctx.set_option("cg_persistent", 1 if request.param == "persistent" else 0)
        return ctx

    ns = types.SimpleNamespace(**{k: getattr(m, k) for k in dir(m) if not k.startswith("__")})
    ns.Stag, ns.cg_path = make, request.param
    return ns


def gpu_cg(stag, ctx, packed, prec, recon, b, mass, shifts, stop, maxiter, residues=None, residue0=0.0,
           want_y=False):
    n = len(shifts)
    vb = ctx.vector_bytes(prec)
    bdev = ctx.upload_vector(b, prec)
    x = ctx.alloc(n * vb)
    ws = ctx.alloc(ctx.cg_workspace_bytes(prec, n))
    y = ctx.alloc(vb) if want_y else None
    rc, info = ctx.mshift_cg(packed, prec, recon, bdev, mass, shifts, stop, maxiter, x, ws,
                             residues=residues, residue0=residue0, y_even=y)
    if getattr(stag, "cg_path", None) == "persistent":
        assert info["kernel_launches"] == 1
    elif maxiter > 0:
        assert info["kernel_launches"] > 1
    xs = np.stack([ctx.download_vector(x, prec, i * vb) for i in range(n)])
    return rc, info, xs, (ctx.download_vector(y, prec) if want_y else None)


def true_residuals(L, U, b, mass, shifts, xs):
    nb = np.linalg.norm(b)
    return [np.linalg.norm(b - oracle.apply_A(L, U, mass, s, xs[i])) / nb for i, s in enumerate(shifts)]


@pytest.mark.parametrize("recon", [18, 12])
@pytest.mark.parametrize("graph", [1, 0])
def test_config1_fp64(stag, recon, graph):
    cfg = si.get_config("c1_4x4x4x4")
    L, U, b = cfg["L"], si.make_links(cfg), si.make_source(cfg)
    ctx = stag.Stag(L)
    ctx.set_option("cg_graph", graph)
    packed = ctx.upload_gauge(U, 0, recon)
    ref = oracle.mshift_cg(L, U, b, cfg["mass"], cfg["shifts"], 1e-10, 2000)
    rc, info, xs, _ = gpu_cg(stag, ctx, packed, 0, recon, b, cfg["mass"], cfg["shifts"], 1e-10, 2000)
    assert rc == 0 and info["converged"]
    assert abs(info["iters"] - ref["iters"]) <= 2
    assert max(true_residuals(L, U, b, cfg["mass"], cfg["shifts"], xs)) <= 1e-10
    A = oracle.dense_A(L, U, cfg["mass"])
    for i, s in enumerate(cfg["shifts"]):                                  # P7 (i) on the GPU
        xd = oracle.dense_solve(A, s, b)
        assert rel(xs[i].reshape(-1), xd) < 1e-10 * 16.0 / (cfg["mass"] ** 2 + s)


@pytest.mark.parametrize("freeze", [1, 0])
def test_wide_shifts_4x4_fp64(stag, freeze):
    """16 shifts 1e-5..20 (config-4 shifts) on 4^4: zeta underflow (A15) and freezing (A10)."""
    L, m, stop = (4, 4, 4, 4), 0.01, 1e-10
    shifts = [1e-5 * (2e6) ** (i / 15) for i in range(16)]
    U, b = si.links_haar(L, 1004), si.source_gaussian(L, 1004, 1)
    ctx = stag.Stag(L)
    ctx.set_option("cg_freeze", freeze)
    packed = ctx.upload_gauge(U, 0, 18)
    ref = oracle.mshift_cg(L, U, b, m, shifts, stop, 5000)
    rc, info, xs, _ = gpu_cg(stag, ctx, packed, 0, 18, b, m, shifts, stop, 5000)
    assert rc == 0 and np.all(np.isfinite(xs))
    assert abs(info["iters"] - ref["iters"]) <= 2
    assert max(true_residuals(L, U, b, m, shifts, xs)) <= stop
    if freeze:
        assert info["iters_shift"][-1] < info["iters"] // 2      # the sigma=20 system froze early
    else:
        assert all(k == info["iters"] for k in info["iters_shift"])
        for i in range(16):
            assert rel(xs[i], ref["x"][i]) < stop * 16.0 / (m * m + shifts[i])


@pytest.mark.parametrize("recon", [18, 12])
def test_config2_single_shift_fp64(stag, recon):
    cfg = si.get_config("c2_16x16x16x4")
    L, U, b = cfg["L"], si.make_links(cfg), si.make_source(cfg)
    ctx = stag.Stag(L)
    packed = ctx.upload_gauge(U, 0, recon)
    oracle.set_threads(8)
    try:
        ref = oracle.mshift_cg(L, U, b, cfg["mass"], [0.0], 1e-10, 5000)
    finally:
        oracle.set_threads(1)
    rc, info, xs, _ = gpu_cg(stag, ctx, packed, 0, recon, b, cfg["mass"], [0.0], 1e-10, 5000)
    assert rc == 0 and ref["rc"] == 0
    assert abs(info["iters"] - ref["iters"]) <= 2
    assert true_residuals(L, U, b, cfg["mass"], [0.0], xs)[0] <= 1e-10


def test_config2_fp32_reading_A9(stag):
    """fp32 CG cannot reach 1e-10 (floor 1e-2..1e-3 in the paper's setting): it must stop
    by stagnation or maxiter without breakdown, with a true residual far below the start, and report it."""
    cfg = si.get_config("c2_16x16x16x4")
    L, U, b = cfg["L"], si.make_links(cfg), si.make_source(cfg)
    ctx = stag.Stag(L)
    packed = ctx.upload_gauge(U, 1, 18)
    rc, info, xs, _ = gpu_cg(stag, ctx, packed, 1, 18, b, cfg["mass"], [0.0], 1e-10, 5000)
    assert rc in (stag.OK, stag.ERR_NOTCONV) and not info["breakdown"]
    tr = true_residuals(L, U, b, cfg["mass"], [0.0], xs)[0]
    assert tr < 1e-3
    # and a stop fp32 can meet is met, in about as many iterations as the fp64 oracle needs
    ref = oracle.mshift_cg(L, U, b, cfg["mass"], [0.0], 1e-4, 5000)
    rc, info, xs, _ = gpu_cg(stag, ctx, packed, 1, 18, b, cfg["mass"], [0.0], 1e-4, 5000)
    assert rc == 0 and abs(info["iters"] - ref["iters"]) <= max(2, ref["iters"] // 20)
    assert true_residuals(L, U, b, cfg["mass"], [0.0], xs)[0] <= 2e-4


def test_P8_plane_wave_and_partial_fraction(stag):
    L, m = (4, 4, 2, 6), 0.2
    shifts = [0.01, 0.04, 0.16, 0.64]
    residues = [0.7, -0.2, 1.3, 0.05]
    U = si.links_unit(L)
    b, p = si.source_plane_wave(L, (1, 3, 0, 2), [1.0, 0.5j, -0.25])
    lam = m * m + np.sum(np.sin(p) ** 2)
    ctx = stag.Stag(L)
    packed = ctx.upload_gauge(U, 0, 18)
    rc, info, xs, y = gpu_cg(stag, ctx, packed, 0, 18, b, m, shifts, 1e-12, 10, residues, 0.3, True)
    assert rc == 0 and info["iters"] == 1
    for i, s in enumerate(shifts):
        assert rel(xs[i], b / (lam + s)) < 1e-14
    assert rel(y, b * (0.3 + sum(a / (lam + s) for a, s in zip(residues, shifts)))) < 1e-14
    assert rel(y, oracle.partial_fraction(b, residues, 0.3, xs)) < 1e-15


def test_finite_termination_zero_source_notconv_badargs(stag):
    L = (4, 4, 4, 4)
    shifts = [0.01, 0.04, 0.16, 0.64]
    ctx = stag.Stag(L)
    free = ctx.upload_gauge(si.links_unit(L), 0, 18)
    b = si.source_gaussian(L, 3, 1)
    rc, info, xs, _ = gpu_cg(stag, ctx, free, 0, 18, b, 0.1, shifts, 1e-10, 50)
    assert rc == 0 and info["iters"] <= 4                                   # P7 (v)
    assert max(true_residuals(L, si.links_unit(L), b, 0.1, shifts, xs)) < 1e-13
    rc, info, xs, _ = gpu_cg(stag, ctx, free, 0, 18, np.zeros_like(b), 0.1, shifts, 1e-10, 50)
    assert rc == 0 and info["iters"] == 0 and not xs.any()                  # P7 (vi)
    U = si.links_haar(L, 1)
    rough = ctx.upload_gauge(U, 0, 18)
    rc, info, xs, _ = gpu_cg(stag, ctx, rough, 0, 18, b, 0.1, shifts, 1e-10, 3)
    assert rc == stag.ERR_NOTCONV and info["iters"] == 3 and not info["converged"]
    ref = oracle.mshift_cg(L, U, b, 0.1, shifts, 1e-10, 3)                  # same 3 iterates
    for i in range(4):
        assert rel(xs[i], ref["x"][i]) < 1e-13
    x = ctx.alloc(4 * ctx.vector_bytes(0))
    ws = ctx.alloc(ctx.cg_workspace_bytes(0, 4))
    bd = ctx.upload_vector(b, 0)
    for bad in (dict(stop=-1.0), dict(shifts=[-0.5, 0.1]), dict(mass=0.0, shifts=[0.0]), dict(shifts=[])):
        kw = dict(mass=0.1, shifts=shifts, stop=1e-10)
        kw.update(bad)
        with pytest.raises(stag.StagError) as ei:
            ctx.mshift_cg(rough, 0, 18, bd, kw["mass"], kw["shifts"], kw["stop"], 10, x, ws)
        assert ei.value.code == stag.ERR_BADARG


def test_midrun_residual_identity_on_gpu(stag):
    """P7 (iii): after k iterations b - (A+sigma_i) x_i = zeta_i r, checked via the oracle's zeta_i r."""
    L, m = (4, 4, 4, 4), 0.1
    shifts = [0.01, 0.04, 0.16, 0.64]
    U, b = si.links_haar(L, 1001), si.source_gaussian(L, 1001, 1)
    ctx = stag.Stag(L)
    ctx.set_option("cg_freeze", 0)
    packed = ctx.upload_gauge(U, 0, 18)
    for k in (1, 3, 17):
        ref = oracle.mshift_cg(L, U, b, m, shifts, 1e-30, k)
        rc, info, xs, _ = gpu_cg(stag, ctx, packed, 0, 18, b, m, shifts, 1e-30, k)
        assert rc == stag.ERR_NOTCONV and info["iters"] == k
        for i, s in enumerate(shifts):
            tr = b - oracle.apply_A(L, U, m, s, xs[i])
            assert np.linalg.norm(tr - ref["zeta"][i] * ref["r"]) / np.linalg.norm(b) < 1e-13
            assert abs(info["resid_iter"][i] - ref["zeta"][i] * np.linalg.norm(ref["r"]) / np.linalg.norm(b)) \
                < 1e-12 * info["resid_iter"][i] + 1e-300


def test_cg_host_variant(stag):
    cfg = si.get_config("c1_4x4x4x4")
    L, U, b = cfg["L"], si.make_links(cfg), si.make_source(cfg)
    ctx = stag.Stag(L)
    packed = ctx.upload_gauge(U, 0, 18)
    n = len(cfg["shifts"])
    hx = np.empty((n,) + b.shape, dtype=np.complex128)
    hy = np.empty_like(b)
    scratch = ctx.alloc(ctx.host_scratch_bytes(0, n))
    rc, info = ctx.mshift_cg_host(packed, 0, 18, b, cfg["mass"], cfg["shifts"], 1e-10, 2000, hx, scratch,
                                  residues=[1.0, 0.5, 0.25, 0.125], residue0=2.0, host_y=hy)
    assert rc == 0
    assert max(true_residuals(L, U, b, cfg["mass"], cfg["shifts"], hx)) <= 1e-10
    assert rel(hy, oracle.partial_fraction(b, [1.0, 0.5, 0.25, 0.125], 2.0, hx)) < 1e-15


@pytest.mark.slow
@pytest.mark.parametrize("stop", [1e-10, 1e-12])
def test_config3_multishift_fp64(stag, stop):
    cfg = si.get_config("c3_24x24x24x6")
    L, U, b = cfg["L"], si.make_links(cfg), si.make_source(cfg)
    ctx = stag.Stag(L)
    packed = ctx.upload_gauge(U, 0, 18)
    oracle.set_threads(8)
    try:
        ref = oracle.mshift_cg(L, U, b, cfg["mass"], cfg["shifts"], stop, 20000)
        rc, info, xs, y = gpu_cg(stag, ctx, packed, 0, 18, b, cfg["mass"], cfg["shifts"], stop, 20000,
                                 cfg["residues"], cfg["residue0"], True)
        tr = true_residuals(L, U, b, cfg["mass"], cfg["shifts"], xs)
        tr_ref = true_residuals(L, U, b, cfg["mass"], cfg["shifts"], ref["x"])
    finally:
        oracle.set_threads(1)
    assert rc == 0 and ref["rc"] == 0
    assert abs(info["iters"] - ref["iters"]) <= 2, (info["iters"], ref["iters"])
    # reading A8: at 1e-12 the true residual may drift from the iterated one by ~eps*kappa; the GPU
    # must be no worse than the oracle's own drift (x1.5) and never above 3*stop
    bound = stop if stop >= 1e-10 else max(stop, 1.5 * max(tr_ref))
    assert max(tr) <= bound and max(tr) <= 3 * stop, (max(tr), max(tr_ref))
    assert rel(y, oracle.partial_fraction(b, cfg["residues"], cfg["residue0"], xs)) < 1e-14


@pytest.mark.parametrize("L", [(6, 6, 2, 2), (10, 6, 4, 4), (2, 2, 2, 2)])
def test_max_shifts_on_ragged_lattices(stag, L):
    """Edge cases: STAG_MAX_SHIFTS = 32 shifts (unsorted, with a duplicate), on lattices whose Vh (72, 480, 8)
    is not a multiple of the warp, the CTA tile or the per-SM slice — empty CTAs and ragged tails everywhere."""
    U, b, m = si.links_haar(L, 81), si.source_gaussian(L, 81), 0.2
    shifts = [float(0.003 * 1.35 ** i) for i in range(stag.MAX_SHIFTS)]
    shifts[5], shifts[20] = shifts[20], shifts[5]
    shifts[7] = shifts[8]
    ctx = stag.Stag(L)
    packed = ctx.upload_gauge(U, 0, 18)
    rc, info, xs, _ = gpu_cg(stag, ctx, packed, 0, 18, b, m, shifts, 1e-10, 5000)
    ref = oracle.mshift_cg(L, U, b, m, shifts, 1e-10, 5000)
    assert rc == 0 and abs(info["iters"] - ref["iters"]) <= 2
    assert max(true_residuals(L, U, b, m, shifts, xs)) <= 1e-10
    assert rel(xs[7], xs[8]) <= 1e-12
    vb = ctx.vector_bytes(0)
    assert ctx.cg_workspace_bytes(0, stag.MAX_SHIFTS + 1) == 0
    with pytest.raises(stag.StagError):
        ctx.mshift_cg(packed, 0, 18, ctx.upload_vector(b, 0), m, shifts + [1.0], 1e-10, 10, ctx.alloc(33 * vb),
                      ctx.alloc(ctx.cg_workspace_bytes(0, 32)))
