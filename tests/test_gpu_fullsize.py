"""Full-size GPU parity, in the launch configuration bench.py times.

The C++ oracle applies one Dslash at 32^3x8 in well under a second and at 64^4 in a few seconds, so
the stencil is compared element by element even at full size.  The multi-shift solve at 32^3x8 is
checked by what holds at any size: the TRUE residual of every shift by the ORACLE's operator, the
residual identity b - (A+sigma_i)x_i = zeta_i r via the reported iterated residuals, and agreement of
the two CUDA paths; the iteration count is compared with the oracle's own full solve."""
import os

import numpy as np
import pytest

import oracle
import stag_inputs as si

pytestmark = [pytest.mark.gpu, pytest.mark.slow]

TOL = {0: 1e-13, 1: 1e-5}


def rel(a, b):
    return np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)


@pytest.fixture(scope="module")
def stag():
    import paper_1010_5433_b200 as m
    return m


@pytest.fixture(scope="module")
def threads():
    n = max(1, min(32, os.cpu_count() or 1))
    oracle.set_threads(n)          # OpenMP over sites only: same arithmetic per site
    yield n
    oracle.set_threads(1)


@pytest.fixture(scope="module")
def c4(stag, threads):
    cfg = si.get_config("c4_32x32x32x8")
    return cfg, si.make_links(cfg), [si.make_source(cfg, k) for k in range(cfg["nsrc"])]


@pytest.mark.parametrize("prec,recon", [(0, 18), (0, 12), (1, 18), (1, 12)])
@pytest.mark.parametrize("regs", [64, 128])
def test_c4_dslash_all_variants(stag, c4, prec, recon, regs):
    cfg, U, srcs = c4
    L = cfg["L"]
    ctx = stag.Stag(L)
    ctx.set_option("dslash_regs", regs)
    packed = ctx.upload_gauge(U, prec, recon)
    v = srcs[0]
    want_w = oracle.dslash_oe(L, U, v)
    vin, w, q = ctx.upload_vector(v, prec), ctx.alloc(ctx.vector_bytes(prec)), ctx.alloc(ctx.vector_bytes(prec))
    ctx.dslash_oe(packed, prec, recon, vin, w)
    got_w = ctx.download_vector(w, prec)
    assert rel(got_w, want_w) <= TOL[prec]
    ctx.dslash_eo(packed, prec, recon, w, q)
    assert rel(ctx.download_vector(q, prec), oracle.dslash_eo(L, U, got_w)) <= TOL[prec]


@pytest.mark.parametrize("recon", [18, 12])
def test_c4_dslash_split_double(stag, c4, recon):
    """N3 at full size: split-double links (b + c), fp64 vectors; within the
    north_star's 1e-13 of the unsplit oracle (bound re-derived in tests/test_gpu_split.py)."""
    cfg, U, srcs = c4
    L, P = cfg["L"], stag.F64_SPLIT
    ctx = stag.Stag(L)
    packed = ctx.upload_gauge(U, P, recon)
    v = srcs[1]
    vin, w, q = ctx.upload_vector(v, P), ctx.alloc(ctx.vector_bytes(P)), ctx.alloc(ctx.vector_bytes(P))
    ctx.dslash_oe(packed, P, recon, vin, w)
    got_w = ctx.download_vector(w, P)
    assert rel(got_w, oracle.dslash_oe(L, U, v)) <= 1e-13
    ctx.dslash_eo(packed, P, recon, w, q)
    assert rel(ctx.download_vector(q, P), oracle.dslash_eo(L, U, got_w)) <= 1e-13


@pytest.mark.parametrize("prec,recon", [(0, 18), (0, 12), (1, 18), (1, 12)])
@pytest.mark.parametrize("pipe", [1, 0])
def test_c4_dslash_block_four_sources(stag, c4, prec, recon, pipe):
    """N1 at full size, in the configuration bench.py times: the 4 pseudo-fermion sources of config 4
    through one read of the links; every source compared element by element with the oracle."""
    cfg, U, srcs = c4
    L = cfg["L"]
    ctx = stag.Stag(L)
    ctx.set_option("dslash_pipe", pipe)
    packed = ctx.upload_gauge(U, prec, recon)
    vb = ctx.vector_bytes(prec)
    vin, vout = ctx.upload_vectors(srcs, prec), ctx.alloc(4 * vb)
    ctx.dslash_block(packed, prec, recon, 1, 4, vin, vout)
    for k in range(4):
        assert rel(ctx.download_vector(vout, prec, k * vb), oracle.dslash_oe(L, U, srcs[k])) <= TOL[prec]


def test_c4_mixed_precision_on_one_split_buffer(stag, c4):
    """N2 + N3 at full size, as bench.py times it: fp32 multi-shift on the b planes, fp64 polish on b + c of
    the SAME buffer; true residual of every shift by the oracle's operator on the unsplit links."""
    cfg, U, srcs = c4
    L, m, shifts, stop = cfg["L"], cfg["mass"], cfg["shifts"], cfg["stops"][0]
    ctx = stag.Stag(L)
    ctx.set_option("cg_mixed_fp64_from", 0)      # the fp32 + polish route (16 shifts would default to the fp64 solve)
    split = ctx.upload_gauge(U, stag.F64_SPLIT, 18)
    n, vb = len(shifts), ctx.vector_bytes(stag.F64)
    x, ws = ctx.alloc(n * vb), ctx.alloc(ctx.mshift_cg_mixed_workspace_bytes(n))
    b = srcs[2]
    rc, info = ctx.mshift_cg_mixed(split, stag.F64_SPLIT, 18, split, 18, ctx.upload_vector(b, stag.F64), m, shifts,
                                   stop, 100000, x, ws)
    assert rc == 0 and info["route"] == 2, info
    nb = np.linalg.norm(b)
    for i, s in enumerate(shifts):
        xi = ctx.download_vector(x, stag.F64, i * vb)
        tr = np.linalg.norm(b - oracle.apply_A(L, U, m, s, xi)) / nb
        assert tr <= stop, (i, tr)
        assert abs(tr - info["polish"]["resid_after"][i]) <= 0.1 * stop


@pytest.fixture(scope="module")
def c4_force_reference(c4):
    cfg, U, srcs = c4
    n = len(cfg["shifts"])
    xs = [srcs[k % 4] * (1.0 + 0.1 * k) for k in range(n)]
    res = [1.0 / (i + 1) for i in range(n)]
    return xs, res, oracle.fermion_force(cfg["L"], U, res, np.stack(xs))


@pytest.mark.parametrize("prec,recon", [(0, 18), (0, 12), (1, 18), (1, 12), (2, 18)])
def test_c4_fermion_force(stag, c4, c4_force_reference, prec, recon):
    """N4 at full size, as bench.py times it: 16 vectors, every link of the 32^3 x 8 lattice against the oracle —
    fp64 (one link per thread), fp32 (two links per thread), split-double links (N3)."""
    import torch
    cfg, U, srcs = c4
    L, n = cfg["L"], len(cfg["shifts"])
    xs, res, want = c4_force_reference
    ctx = stag.Stag(L)
    packed = ctx.upload_gauge(U, prec, recon)
    vprec = 1 if prec == 1 else 0
    F = torch.empty(ctx.V * 72, dtype=torch.float64, device="cuda")
    ctx.fermion_force(packed, prec, recon, res, ctx.upload_vectors(xs, vprec), F, ctx.alloc(ctx.force_workspace_bytes(prec, n)))
    got = F.cpu().numpy().view(np.complex128).reshape(ctx.V, 4, 3, 3)
    assert rel(got, want) <= TOL[vprec]


@pytest.mark.parametrize("recon", [18, 12])
def test_c4_split_double_block_dslash(stag, c4, recon):
    """N3 x N1 at full size: four sources through one read of the split-double links, both parities, every site."""
    cfg, U, srcs = c4
    L = cfg["L"]
    ctx = stag.Stag(L)
    packed = ctx.upload_gauge(U, stag.F64_SPLIT, recon)
    vb = ctx.vector_bytes(0)
    vin, vout = ctx.upload_vectors(srcs, 0), ctx.alloc(4 * vb)
    for par, ofun in ((1, oracle.dslash_oe), (0, oracle.dslash_eo)):
        ctx.dslash_block(packed, stag.F64_SPLIT, recon, par, 4, vin, vout)
        for k in range(4):
            assert rel(ctx.download_vector(vout, 0, k * vb), ofun(L, U, srcs[k])) <= 1e-13


def test_c4_fp32_block_cg_four_sources(stag, c4):
    """N1 in the MD precision at full size, as bench.py times it (stop 1e-5): every source converges,
    iteration counts equal the single fp32 solves', true residual by the oracle's operator < 1e-2 (what fp32 storage reaches: reading A9)."""
    cfg, U, srcs = c4
    L, m, shifts = cfg["L"], cfg["mass"], cfg["shifts"]
    n = len(shifts)
    ctx = stag.Stag(L)
    packed = ctx.upload_gauge(U, 1, 18)
    vb = ctx.vector_bytes(1)
    x = ctx.alloc(4 * n * vb)
    rc, infos = ctx.mshift_cg_block(packed, 1, 18, 4, ctx.upload_vectors(srcs, 1), m, shifts, 1e-5, 100000, x,
                                    ctx.alloc(ctx.cg_block_workspace_bytes(1, n, 4)))
    assert rc == 0 and all(i["converged"] and not i["breakdown"] for i in infos)
    x1, ws1 = ctx.alloc(n * vb), ctx.alloc(ctx.cg_workspace_bytes(1, n))
    for s in range(4):
        rc1, i1 = ctx.mshift_cg(packed, 1, 18, ctx.upload_vector(srcs[s], 1), m, shifts, 1e-5, 100000, x1, ws1)
        assert rc1 == 0 and abs(infos[s]["iters"] - i1["iters"]) <= 2
        for i in (0, n // 2, n - 1) if s else range(n):
            xi = ctx.download_vector(x, 1, (s * n + i) * vb)
            tr = np.linalg.norm(srcs[s] - oracle.apply_A(L, U, m, shifts[i], xi)) / np.linalg.norm(srcs[s])
            assert tr < 1e-2, (s, i, tr)      # fp32 storage: the paper's "10^-2 - 10^-3" (reading A9)


def test_c4_block_cg_four_sources(stag, c4):
    """The block solve bench.py reports: 4 sources x 16 shifts in one persistent launch; true residual of
    every (source, shift) by the oracle's operator, iteration counts equal to the single-source path's."""
    cfg, U, srcs = c4
    L, shifts, m, stop = cfg["L"], cfg["shifts"], cfg["mass"], cfg["stops"][0]
    n = len(shifts)
    ctx = stag.Stag(L)
    packed = ctx.upload_gauge(U, 0, 18)
    vb = ctx.vector_bytes(0)
    x, ws = ctx.alloc(4 * n * vb), ctx.alloc(ctx.cg_block_workspace_bytes(0, n, 4))
    rc, infos = ctx.mshift_cg_block(packed, 0, 18, 4, ctx.upload_vectors(srcs, 0), m, shifts, stop, 100000, x, ws)
    assert rc == 0 and infos[0]["kernel_launches"] == 1
    x1, ws1 = ctx.alloc(n * vb), ctx.alloc(ctx.cg_workspace_bytes(0, n))
    for s, b in enumerate(srcs):
        nb = np.linalg.norm(b)
        for i in range(n):                                   # north_star: "for every shift"
            xi = ctx.download_vector(x, 0, (s * n + i) * vb)
            assert np.linalg.norm(b - oracle.apply_A(L, U, m, shifts[i], xi)) / nb <= stop, (s, i)
        rc1, info1 = ctx.mshift_cg(packed, 0, 18, ctx.upload_vector(b, 0), m, shifts, stop, 100000, x1, ws1)
        assert rc1 == 0 and abs(info1["iters"] - infos[s]["iters"]) <= 2


@pytest.mark.parametrize("path", ["persistent", "multikernel"])
def test_c4_multishift_cg_bench_configuration(stag, c4, path):
    """The solve bench.py times: 32^3x8, 16 shifts 1e-5..20, m = 0.01, stop 1e-10, fp64 18-real."""
    cfg, U, srcs = c4
    L, b, shifts, m, stop = cfg["L"], srcs[1], cfg["shifts"], cfg["mass"], cfg["stops"][0]
    n = len(shifts)
    ctx = stag.Stag(L)
    ctx.set_option("cg_persistent", 1 if path == "persistent" else 0)
    packed = ctx.upload_gauge(U, 0, 18)
    vb = ctx.vector_bytes(0)
    x, ws = ctx.alloc(n * vb), ctx.alloc(ctx.cg_workspace_bytes(0, n))
    rc, info = ctx.mshift_cg(packed, 0, 18, ctx.upload_vector(b, 0), m, shifts, stop, 100000, x, ws)
    assert rc == 0 and info["converged"]
    assert info["kernel_launches"] == 1 if path == "persistent" else info["kernel_launches"] > 1
    nb = np.linalg.norm(b)
    for i, s in enumerate(shifts):
        xi = ctx.download_vector(x, 0, i * vb)
        tr = np.linalg.norm(b - oracle.apply_A(L, U, m, s, xi)) / nb
        assert tr <= stop, (i, tr)
        # frozen shifts (A10) were frozen at <= 0.1 stop; the iterated value reported must be honest
        assert tr <= 2.0 * info["resid_iter"][i] + 1e-12, (i, tr, info["resid_iter"][i])
    test_c4_multishift_cg_bench_configuration.iters[path] = info["iters"]


test_c4_multishift_cg_bench_configuration.iters = {}


@pytest.mark.parametrize("path", ["persistent", "multikernel"])
@pytest.mark.parametrize("recon", [18, 12])
def test_c4_fp32_multishift_cg_reading_A9(stag, c4, path, recon):
    """The solve `bench.py --prec f32` times (32^3x8, 16 shifts, fp32 vectors and links, fp64 reductions), reading
    A9 / PAPER.md:127: stop 1e-10 is out of reach, so the run must end on stagnation (or stop), without breakdown,
    with a TRUE residual of every shift — by the oracle's fp64 operator — below 1e-2 (the paper's "10^-2 - 10^-3"
    floor for this conditioning) and an honest report of where it stopped."""
    cfg, U, srcs = c4
    L, b, shifts, m = cfg["L"], srcs[0], cfg["shifts"], cfg["mass"]
    n = len(shifts)
    ctx = stag.Stag(L)
    ctx.set_option("cg_persistent", 1 if path == "persistent" else 0)
    packed = ctx.upload_gauge(U, 1, recon)
    vb = ctx.vector_bytes(1)
    x, ws = ctx.alloc(n * vb), ctx.alloc(ctx.cg_workspace_bytes(1, n))
    rc, info = ctx.mshift_cg(packed, 1, recon, ctx.upload_vector(b, 1), m, shifts, cfg["stops"][0], 100000, x, ws)
    assert rc in (stag.OK, stag.ERR_NOTCONV) and not info["breakdown"]
    assert info["converged"] or info["stagnated"]
    assert (info["kernel_launches"] == 1) == (path == "persistent")
    assert 1000 < info["iters"] < 6000, info["iters"]          # the fp64 solve needs 2988
    nb = np.linalg.norm(b)
    worst = 0.0
    for i, s in enumerate(shifts):
        xi = ctx.download_vector(x, 1, i * vb)
        assert np.all(np.isfinite(xi))
        worst = max(worst, np.linalg.norm(b - oracle.apply_A(L, U, m, s, xi)) / nb)
    assert worst < 1e-2, worst


def test_c4_iteration_count_matches_oracle(stag, c4, threads):
    """Iterations within +-2 of the oracle's own full solve (3000 iterations of the plain C++ CG)."""
    cfg, U, srcs = c4
    got = test_c4_multishift_cg_bench_configuration.iters
    if not got:
        pytest.skip("solve test did not run")
    ref = oracle.mshift_cg(cfg["L"], U, srcs[1], cfg["mass"], cfg["shifts"], cfg["stops"][0], 100000)
    assert ref["rc"] == 0
    for path, it in got.items():
        assert abs(it - ref["iters"]) <= 2, (path, it, ref["iters"])


def test_c5_dslash_fp64_and_fp32_full_compare(stag, threads):
    """64^4 (8.4M even sites, 9.7 GB of canonical links): every output element against the oracle."""
    cfg = si.get_config("c5_64x64x64x64")
    L, U, v = cfg["L"], si.make_links(cfg), si.make_source(cfg)
    want = oracle.dslash_oe(L, U, v)
    v_odd = si.source_gaussian(L, cfg["seed"], stream=7)          # an independent vector on the odd sites
    want_eo = oracle.dslash_eo(L, U, v_odd)                       # D_eo reads the OTHER eight packed link sets
    ctx = stag.Stag(L)
    canon = ctx.alloc(ctx.gauge_canonical_bytes())
    ctx.gauge_load(U, canon)
    for prec, recon in ((0, 18), (0, 12), (1, 18), (1, 12), (2, 18)):      # 2 = split-double (N3)
        packed = ctx.alloc(ctx.gauge_packed_bytes(prec, recon))
        ctx.gauge_pack(canon, packed, prec, recon)
        vin, w = ctx.upload_vector(v, prec), ctx.alloc(ctx.vector_bytes(prec))
        ctx.dslash_oe(packed, prec, recon, vin, w)
        assert rel(ctx.download_vector(w, prec), want) <= (1e-5 if prec == 1 else 1e-13), (prec, recon)
        vin = ctx.upload_vector(v_odd, prec)
        ctx.dslash_eo(packed, prec, recon, vin, w)
        assert rel(ctx.download_vector(w, prec), want_eo) <= (1e-5 if prec == 1 else 1e-13), ("eo", prec, recon)
        del packed, vin, w


def test_c5_multishift_cg_true_residuals(stag, threads):
    """Config 5 as bench.py --workload c5 runs it (64^4, 8 shifts, stop 1e-9, multi-kernel path replayed as CUDA
    graphs): the TRUE residual of EVERY shift by the oracle's operator.  The oracle's own
    solve at this size is hours on one core, so the iteration count is not compared."""
    cfg = si.get_config("c5_64x64x64x64")
    L, U, b, m, shifts, stop = cfg["L"], si.make_links(cfg), si.make_source(cfg), cfg["mass"], cfg["shifts"], cfg["stops"][0]
    ctx = stag.Stag(L)
    packed = ctx.upload_gauge(U, 0, 18)
    n, vb = len(shifts), ctx.vector_bytes(0)
    x, ws = ctx.alloc(n * vb), ctx.alloc(ctx.cg_workspace_bytes(0, n))
    rc, info = ctx.mshift_cg(packed, 0, 18, ctx.upload_vector(b, 0), m, shifts, stop, 100000, x, ws)
    assert rc == 0 and info["converged"] and info["kernel_launches"] > 1
    assert info["iters_shift"][0] == info["iters"] and info["iters_shift"][-1] < info["iters"]   # heavy shifts freeze early
    nb = np.linalg.norm(b)
    for i in range(n):
        xi = ctx.download_vector(x, 0, i * vb)
        tr = np.linalg.norm(b - oracle.apply_A(L, U, m, shifts[i], xi)) / nb
        assert tr <= stop, (i, tr)
        assert info["resid_iter"][i] <= stop


@pytest.mark.parametrize("path", ["persistent", "multikernel"])
def test_paper_shape_4x48cubed_cg_and_dslash(stag, threads, path):
    """The paper's largest Table-2 lattice, 4 x 48^3: fp32 12-real Dslash (the paper's storage)
    against the oracle, and the 8-shift fp64 solve on both CUDA paths — the persistent kernel runs here with
    r and q resident and p_base in global memory (partial residency)."""
    cfg = si.get_config("t2_48x48x48x4")
    L, U, b, m, shifts, stop = cfg["L"], si.make_links(cfg), si.make_source(cfg), cfg["mass"], cfg["shifts"], cfg["stops"][0]
    ctx = stag.Stag(L)
    ctx.set_option("cg_persistent", 1 if path == "persistent" else 0)
    if path == "persistent":
        p32 = ctx.upload_gauge(U, 1, 12)
        w = ctx.alloc(ctx.vector_bytes(1))
        ctx.dslash_oe(p32, 1, 12, ctx.upload_vector(b, 1), w)
        assert rel(ctx.download_vector(w, 1), oracle.dslash_oe(L, U, b)) <= 1e-5
        del p32
    packed = ctx.upload_gauge(U, 0, 18)
    n, vb = len(shifts), ctx.vector_bytes(0)
    x, ws = ctx.alloc(n * vb), ctx.alloc(ctx.cg_workspace_bytes(0, n))
    rc, info = ctx.mshift_cg(packed, 0, 18, ctx.upload_vector(b, 0), m, shifts, stop, 100000, x, ws)
    assert rc == 0, info
    assert (info["kernel_launches"] == 1) == (path == "persistent")
    nb = np.linalg.norm(b)
    for i in range(n):
        xi = ctx.download_vector(x, 0, i * vb)
        assert np.linalg.norm(b - oracle.apply_A(L, U, m, shifts[i], xi)) / nb <= stop, i
    test_paper_shape_4x48cubed_cg_and_dslash.iters = getattr(test_paper_shape_4x48cubed_cg_and_dslash, "iters", {})
    test_paper_shape_4x48cubed_cg_and_dslash.iters[path] = info["iters"]
    it = test_paper_shape_4x48cubed_cg_and_dslash.iters
    if len(it) == 2:
        assert abs(it["persistent"] - it["multikernel"]) <= 2


def test_32x32cubed_block_cg_nothing_resident(stag, threads):
    """The paper's 32 x 32^3 lattice, two sources in one persistent launch: at this size no slice
    of r, q, p fits in shared memory (every vector goes through the global workspace) and the single-source call
    takes the multi-kernel path; both must give the oracle's residuals and the same iteration count +-2."""
    cfg = si.get_config("t2_32x32x32x32")
    L, U, m, shifts, stop = cfg["L"], si.make_links(cfg), cfg["mass"], cfg["shifts"], cfg["stops"][0]
    bs = [si.source_gaussian(L, cfg["seed"], stream=1 + k) for k in range(2)]
    ctx = stag.Stag(L)
    packed = ctx.upload_gauge(U, 0, 18)
    n, vb = len(shifts), ctx.vector_bytes(0)
    x, ws = ctx.alloc(2 * n * vb), ctx.alloc(ctx.cg_block_workspace_bytes(0, n, 2))
    rc, infos = ctx.mshift_cg_block(packed, 0, 18, 2, ctx.upload_vectors(bs, 0), m, shifts, stop, 100000, x, ws)
    assert rc == 0 and infos[0]["kernel_launches"] == 1
    x1, ws1 = ctx.alloc(n * vb), ctx.alloc(ctx.cg_workspace_bytes(0, n))
    rc, info = ctx.mshift_cg(packed, 0, 18, ctx.upload_vector(bs[0], 0), m, shifts, stop, 100000, x1, ws1)
    assert rc == 0 and info["kernel_launches"] > 1 and abs(info["iters"] - infos[0]["iters"]) <= 2
    for s, i in ((0, 0), (1, 0), (1, n - 1)):
        xi = ctx.download_vector(x, 0, (s * n + i) * vb)
        assert np.linalg.norm(bs[s] - oracle.apply_A(L, U, m, shifts[i], xi)) / np.linalg.norm(bs[s]) <= stop
    xi = ctx.download_vector(x1, 0, 0)
    assert np.linalg.norm(bs[0] - oracle.apply_A(L, U, m, shifts[0], xi)) / np.linalg.norm(bs[0]) <= stop
