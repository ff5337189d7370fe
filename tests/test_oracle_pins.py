"""Pins for the oracle — nothing here touches the CUDA path.

Each test checks oracle/ against something the paper's statement of the problem or the
mathematics fixes: closed forms, invariants, hand-evaluated special cases, dense brute force.
"""
import itertools
import os

import numpy as np
import pytest

import oracle
import stag_inputs as si

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
RNG_SEED = 4242


def rel(a, b):
    return np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)


def load_spectra():
    out = {}
    with open(os.path.join(GOLDEN, "free_spectrum.txt")) as f:
        for line in f:
            if line.startswith("#"):
                continue
            Ls, rest = line.split("|")
            L = tuple(int(v) for v in Ls.split())
            out[L] = [(float(a.split(":")[0]), int(a.split(":")[1])) for a in rest.split(";")]
    return out


SPECTRA = load_spectra()


# ---------------------------------------------------------------- P1 free-field spectrum
@pytest.mark.parametrize("L", [(2, 2, 2, 2), (4, 4, 4, 4), (4, 4, 2, 6), (6, 4, 4, 2)])
def test_P1_plane_waves_are_eigenvectors(L):
    """D_eo D_oe v = -(sum_mu sin^2 p_mu) v for every momentum (north_star closed form)."""
    U = si.links_unit(L)
    colours = np.eye(3) + 0.25j
    worst = 0.0
    for k, n in enumerate(itertools.product(*[range(l) for l in L])):
        v, p = si.source_plane_wave(L, n, colours[k % 3])
        w = oracle.dslash_eo(L, U, oracle.dslash_oe(L, U, v))
        lam = -np.sum(np.sin(p) ** 2)
        worst = max(worst, np.linalg.norm(w - lam * v) / np.linalg.norm(v))
    assert worst < 5e-15


@pytest.mark.parametrize("L", [(2, 2, 2, 2), (4, 4, 4, 4), (4, 4, 2, 6)])
def test_P1_full_spectrum_matches_golden(L):
    """Whole multiset of eigenvalues of -D_eo D_oe (dense, mass 0) vs tests/golden."""
    A = oracle.dense_A(L, si.links_unit(L), 0.0)
    ev = np.linalg.eigvalsh(A)
    expect = np.concatenate([[lam] * m for lam, m in SPECTRA[L]])
    assert ev.size == expect.size == 3 * si.half_volume(L)
    assert np.max(np.abs(np.sort(ev) - np.sort(expect))) < 1e-13


def test_P1_phases_matter():
    """With eta == 1 the spectrum differs: the golden file pins the anticommuting phases.
    (Unit links, so dropping eta is the same as making every link +1 with eta -> 1; emulate
    by feeding links that cancel eta: U_mu(x) = eta_mu(x) * 1 is still unitary, det = +-1.)"""
    L = (4, 4, 4, 4)
    x = si.site_coords(L)
    U = si.links_unit(L)
    cum = np.cumsum(x, axis=1)
    for mu in range(1, 4):
        U[:, mu] *= ((-1.0) ** cum[:, mu - 1])[:, None, None]
    ev = np.linalg.eigvalsh(oracle.dense_A(L, U, 0.0))
    distinct = np.unique(np.round(ev, 10))
    assert distinct.size != 4  # golden 4^4 spectrum has exactly 4 distinct values


# ---------------------------------------------------------------- P2 anti-hermiticity
@pytest.mark.parametrize("L", [(4, 4, 4, 4), (6, 2, 4, 8), (2, 2, 2, 2)])
def test_P2_antihermitian(L):
    U = si.links_haar(L, 77)
    psi = si.source_gaussian(L, 77, 1)
    chi = si.source_gaussian(L, 77, 2)
    lhs = np.vdot(chi, oracle.dslash_oe(L, U, psi))          # <chi_o, D_oe psi_e>
    rhs = -np.vdot(oracle.dslash_eo(L, U, chi), psi)         # -<D_eo chi_o, psi_e>
    assert abs(lhs - rhs) / abs(lhs) < 1e-14


# ---------------------------------------------------------------- P3 gauge covariance
@pytest.mark.parametrize("L,parity", [((4, 4, 4, 4), 0), ((4, 4, 4, 4), 1), ((6, 4, 2, 4), 1)])
def test_P3_gauge_covariance(L, parity):
    U = si.links_haar(L, 31)
    g = si.gauge_transform_field(L, 31)
    Ug = si.apply_gauge_transform(L, U, g)
    psi = si.source_gaussian(L, 31, 3)
    g_in = g[si.parity_sites(L, 1 - parity)]
    g_out = g[si.parity_sites(L, parity)]
    psi_g = np.einsum("xij,xj->xi", g_in, psi)
    lhs = oracle.dslash(L, Ug, psi_g, parity)
    rhs = np.einsum("xij,xj->xi", g_out, oracle.dslash(L, U, psi, parity))
    assert rel(lhs, rhs) < 1e-14


# ---------------------------------------------------------------- P4 Hermitian, bounded
def test_P4_hermitian_positive_bounded():
    L, m = (4, 4, 4, 4), 0.1
    A = oracle.dense_A(L, si.links_haar(L, 5), m)
    assert np.max(np.abs(A - A.conj().T)) < 1e-14
    ev = np.linalg.eigvalsh(A)
    assert ev.min() >= m * m - 1e-13
    assert ev.max() <= m * m + 16.0
    ev_free = np.linalg.eigvalsh(oracle.dense_A(L, si.links_unit(L), 0.0))
    assert ev_free.min() >= -1e-13 and ev_free.max() <= 4.0 + 1e-13


# ---------------------------------------------------------------- P5 delta source by hand
@pytest.mark.parametrize("y", [(1, 2, 3, 0), (0, 0, 0, 0), (3, 1, 0, 3), (2, 3, 3, 3)])
def test_P5_delta_source_by_hand(y):
    """Unit links, delta at y (colour c): (D delta_y)(x) is
         +1/2 eta_mu(x) s+  at x = y - mu   (forward hop from x reaches y)
         -1/2 eta_mu(x) s-  at x = y + mu   (backward hop from x reaches y)
       eta_0 = 1, eta_mu(x) = (-1)^(x0+..+x_{mu-1}); s = -1 when the hop crosses t = L3-1 -> 0."""
    L = (4, 4, 4, 4)
    U = si.links_unit(L)
    py = sum(y) & 1
    strides = np.array([1, L[0], L[0] * L[1], L[0] * L[1] * L[2]])
    vh = si.half_volume(L)
    c = 1
    src = np.zeros((vh, 3), dtype=np.complex128)
    src[int(np.dot(y, strides)) // 2, c] = 1.0
    got = oracle.dslash(L, U, src, 1 - py)
    expect = np.zeros_like(got)
    for mu in range(4):
        for sgn in (+1, -1):           # x = y - sgn*mu
            x = list(y)
            x[mu] = (y[mu] - sgn) % L[mu]
            eta = 1.0 if mu == 0 else (-1.0) ** sum(x[:mu])
            if sgn == +1:              # forward hop from x
                s = -1.0 if (mu == 3 and x[3] == L[3] - 1) else 1.0
                val = +0.5 * eta * s
            else:                      # backward hop from x
                s = -1.0 if (mu == 3 and x[3] == 0) else 1.0
                val = -0.5 * eta * s
            expect[int(np.dot(x, strides)) // 2, c] += val
    assert np.max(np.abs(got - expect)) == 0.0
    assert np.count_nonzero(got) == 8


def test_dslash_vs_whole_lattice_roll_formulation():
    """Consistency (not a pin): same operator written with np.roll on the full 4-d array."""
    L = (4, 6, 2, 4)
    U = si.links_haar(L, 9)
    V = si.volume(L)
    x = si.site_coords(L)
    par = x.sum(axis=1) & 1
    full = np.zeros((V, 3), dtype=np.complex128)
    full[si.parity_sites(L, 0)] = si.source_gaussian(L, 9, 1)
    full[si.parity_sites(L, 1)] = si.source_gaussian(L, 9, 2)
    shp = (L[3], L[2], L[1], L[0])
    psi = full.reshape(shp + (3,))
    Ug = U.reshape(shp + (4, 3, 3))
    xs = x.reshape(shp + (4,))
    out = np.zeros_like(psi)
    for mu in range(4):
        ax = 3 - mu
        eta = ((-1.0) ** xs[..., :mu].sum(axis=-1))[..., None]
        sp = np.where((xs[..., mu] == L[mu] - 1) & (mu == 3), -1.0, 1.0)[..., None]
        sm = np.where((xs[..., mu] == 0) & (mu == 3), -1.0, 1.0)[..., None]
        fwd = np.einsum("...ij,...j->...i", Ug[..., mu, :, :], np.roll(psi, -1, axis=ax))
        Ub = np.roll(Ug[..., mu, :, :], 1, axis=ax)
        bwd = np.einsum("...ji,...j->...i", Ub.conj(), np.roll(psi, 1, axis=ax))
        out += 0.5 * eta * (sp * fwd - sm * bwd)
    out = out.reshape(V, 3)
    for parity in (0, 1):
        got = oracle.dslash(L, U, full[si.parity_sites(L, 1 - parity)], parity)
        assert rel(got, out[si.parity_sites(L, parity)]) < 1e-15
    assert par.sum() == V // 2


# ---------------------------------------------------------------- P7 multi-shift CG
SHIFTS = [0.01, 0.04, 0.16, 0.64]


@pytest.mark.parametrize("L", [(2, 2, 2, 2), (4, 4, 4, 4)])
def test_P7_dense_solves_every_shift(L):
    m, stop = 0.1, 1e-10
    U = si.links_haar(L, 1001)
    b = si.source_gaussian(L, 1001, 1)
    A = oracle.dense_A(L, U, m)
    res = oracle.mshift_cg(L, U, b, m, SHIFTS, stop, 2000)
    assert res["rc"] == 0
    kappa = 16.0 / (m * m + min(SHIFTS))
    for i, s in enumerate(SHIFTS):
        xd = oracle.dense_solve(A, s, b)
        xl = np.linalg.solve(A + s * np.eye(A.shape[0]), b.reshape(-1))   # library cross-check
        assert rel(xd, xl) < 1e-12
        assert rel(res["x"][i].reshape(-1), xd) < stop * kappa
        true_res = b - oracle.apply_A(L, U, m, s, res["x"][i])
        assert np.linalg.norm(true_res) / np.linalg.norm(b) <= stop      # (ii)


def test_P7_wide_shift_range_no_underflow():
    """Config-4-like shifts (1e-5..20) on 4^4: zeta_i of the large shifts underflows long before
    the base system converges (~600 iterations); every x_i must still be the dense solution
    (reading A15: the zeta recurrence is carried in ratio form, no 0/0)."""
    L, m, stop = (4, 4, 4, 4), 0.01, 1e-10
    shifts = [1e-5 * (2e6) ** (i / 15) for i in range(16)]
    U = si.links_haar(L, 1004)
    b = si.source_gaussian(L, 1004, 1)
    A = oracle.dense_A(L, U, m)
    res = oracle.mshift_cg(L, U, b, m, shifts, stop, 5000)
    assert res["rc"] == 0 and res["iters"] > 300
    assert np.all(np.isfinite(res["x"])) and np.all(np.isfinite(res["zeta"]))
    assert res["zeta"][-1] < 1e-200
    for i, s in enumerate(shifts):
        xd = oracle.dense_solve(A, s, b)
        assert rel(res["x"][i].reshape(-1), xd) < stop * 16.0 / (m * m + s)
        tr = b - oracle.apply_A(L, U, m, s, res["x"][i])
        assert np.linalg.norm(tr) / np.linalg.norm(b) <= stop


def test_P7_unsorted_shifts_and_base_choice():
    L, m = (4, 4, 4, 4), 0.1
    U = si.links_haar(L, 1001)
    b = si.source_gaussian(L, 1001, 1)
    a = oracle.mshift_cg(L, U, b, m, SHIFTS, 1e-10, 2000)
    perm = [2, 0, 3, 1]
    c = oracle.mshift_cg(L, U, b, m, [SHIFTS[k] for k in perm], 1e-10, 2000)
    assert a["iters"] == c["iters"]
    for j, k in enumerate(perm):
        assert rel(c["x"][j], a["x"][k]) < 1e-13


def test_P7_shifted_residual_is_zeta_r_midrun():
    """(iii) b - (A+sigma_i) x_i = zeta_i r at an intermediate iteration."""
    L, m = (4, 4, 4, 4), 0.1
    U = si.links_haar(L, 1001)
    b = si.source_gaussian(L, 1001, 1)
    for k in (1, 3, 17):
        res = oracle.mshift_cg(L, U, b, m, SHIFTS, 1e-30, k)
        assert res["rc"] == -5 and res["iters"] == k
        assert res["zeta"][0] == 1.0
        assert np.all(res["zeta"] > 0) and np.all(res["zeta"] <= 1.0)
        for i, s in enumerate(SHIFTS):
            true_res = b - oracle.apply_A(L, U, m, s, res["x"][i])
            # rounding of b - (A+sigma)x is ~eps*||b||, so the scale of the check is ||b||
            diff = np.linalg.norm(true_res - res["zeta"][i] * res["r"])
            assert diff / np.linalg.norm(b) < 1e-14


def test_P7_single_shift_is_textbook_cg():
    """(iv) N = 1 equals textbook CG (Hestenes-Stiefel) iterate for iterate."""
    L, m, s = (4, 4, 4, 4), 0.1, 0.04
    U = si.links_haar(L, 1001)
    b = si.source_gaussian(L, 1001, 1)
    x = np.zeros_like(b)
    r = b.copy()
    p = b.copy()
    rr = np.vdot(r, r).real
    for k in range(1, 8):
        q = oracle.apply_A(L, U, m, s, p)
        al = rr / np.vdot(p, q).real
        x = x + al * p
        r = r - al * q
        rr_new = np.vdot(r, r).real
        p = r + (rr_new / rr) * p
        rr = rr_new
        got = oracle.mshift_cg(L, U, b, m, [s], 1e-30, k)
        assert rel(got["x"][0], x) < 1e-13
        assert rel(got["r"], r) < 1e-12


def test_P7_finite_termination_free_field():
    """(v) free 4^4: 4 distinct eigenvalues -> <= 4 iterations for every shift; free 2^4: 1."""
    for L, kmax in (((4, 4, 4, 4), 4), ((2, 2, 2, 2), 1)):
        U = si.links_unit(L)
        b = si.source_gaussian(L, 3, 1)
        res = oracle.mshift_cg(L, U, b, 0.1, SHIFTS, 1e-10, 50)
        assert res["rc"] == 0 and res["iters"] <= kmax
        for i, s in enumerate(SHIFTS):
            tr = b - oracle.apply_A(L, U, 0.1, s, res["x"][i])
            assert np.linalg.norm(tr) / np.linalg.norm(b) < 1e-13


def test_P7_zero_source():
    L = (4, 4, 4, 4)
    U = si.links_haar(L, 1)
    b = np.zeros((si.half_volume(L), 3), dtype=np.complex128)
    res = oracle.mshift_cg(L, U, b, 0.1, SHIFTS, 1e-10, 50)
    assert res["rc"] == 0 and res["iters"] == 0 and not res["x"].any()


def test_P7_not_converged_and_bad_args():
    L = (4, 4, 4, 4)
    U = si.links_haar(L, 1)
    b = si.source_gaussian(L, 1, 1)
    assert oracle.mshift_cg(L, U, b, 0.1, SHIFTS, 1e-10, 3)["rc"] == -5
    with pytest.raises(ValueError):
        oracle.mshift_cg(L, U, b, 0.1, SHIFTS, -1.0, 3)
    with pytest.raises(ValueError):
        oracle.mshift_cg(L, U, b, 0.0, [0.0], 1e-10, 3)
    with pytest.raises(ValueError):
        oracle.dslash((4, 4, 3, 4), U[:192], b[:96], 0)


# ---------------------------------------------------------------- P8 plane-wave closed form
def test_P8_plane_wave_solution_and_partial_fraction():
    L, m = (4, 4, 2, 6), 0.2
    U = si.links_unit(L)
    b, p = si.source_plane_wave(L, (1, 3, 0, 2), [1.0, 0.5j, -0.25])
    lam = m * m + np.sum(np.sin(p) ** 2)
    residues = [0.7, -0.2, 1.3, 0.05]
    res = oracle.mshift_cg(L, U, b, m, SHIFTS, 1e-12, 10)
    assert res["rc"] == 0 and res["iters"] == 1
    for i, s in enumerate(SHIFTS):
        assert rel(res["x"][i], b / (lam + s)) < 1e-14
    y = oracle.partial_fraction(b, residues, 0.3, res["x"])
    expect = b * (0.3 + sum(a / (lam + s) for a, s in zip(residues, SHIFTS)))
    assert rel(y, expect) < 1e-14


# ---- N3: split-double storage, PAPER.md:111-117 ---------------------------------
def test_N3_split_double():
    """b = (float)a, c = (float)(a - (double)b), a' = b + c.  Pinned by (i) a worked value: a = 1/3 has
    b = 0x3EAAAAAB = 1/3 + 2^-25/3 and c = -(1/3 + 2^-25/3) 2^-25 (float of -2^-25/3), so
    a' = 1/3 - 2^-50/3 up to the rounding of 1/3 itself; (ii) numbers with <= 48 significant bits are
    reproduced exactly; (iii) the 2^-48 bound on random data; (iv) a wrong formula (c dropped) fails."""
    a = np.array([1.0 / 3.0])
    got = oracle.split_double(a)[0]
    assert abs(got - (1.0 / 3.0 - 2.0 ** -50 / 3.0)) <= 2.0 ** -54
    assert got != 1.0 / 3.0 and abs(got - 1.0 / 3.0) > 2.0 ** -53
    exact = np.array([1.0 + 2.0 ** -40, -0.5 - 2.0 ** -47, 3.0 * 2.0 ** -20 + 2.0 ** -60, 0.0, -2.0])
    assert np.array_equal(oracle.split_double(exact), exact)
    rng = np.random.default_rng(5)
    r = rng.standard_normal(4096) * 10.0 ** rng.integers(-3, 3, 4096)
    d = np.abs(oracle.split_double(r) - r)
    assert np.all(d <= 2.0 ** -48 * np.abs(r))
    assert np.max(d / np.abs(r)) > 2.0 ** -56                      # it is not the identity
    assert np.max(np.abs(r.astype(np.float32).astype(np.float64) - r) / np.abs(r)) > 2.0 ** -26   # (iv)
    z = oracle.split_double(r[:8] + 1j * r[8:16])
    assert np.array_equal(z.real, oracle.split_double(r[:8])) and np.array_equal(z.imag, oracle.split_double(r[8:16]))


# ---- N2: polish = ordinary CG from a non-zero start, PAPER.md:125-129 -------------
def _fp32_like(x, seed):
    """a start vector of fp32 quality: the solution rounded to fp32 plus 1e-6 relative noise"""
    rng = np.random.default_rng(seed)
    x32 = x.astype(np.complex64).astype(np.complex128)
    return x32 + 1e-6 * np.linalg.norm(x) / np.sqrt(x.size) * (rng.standard_normal(x.shape) + 1j * rng.standard_normal(x.shape))


@pytest.mark.parametrize("L", [(2, 2, 2, 2), (4, 4, 4, 4)])
def test_P9_polish_reaches_the_dense_solution(L):
    U, b, m = si.links_haar(L, 41), si.source_gaussian(L, 41), 0.1
    A = oracle.dense_A(L, U, m)
    for sigma in (0.0, 0.04, 0.64):
        xd = oracle.dense_solve(A, sigma, b).reshape(-1, 3)
        x0 = _fp32_like(xd, 3)
        res = oracle.cg_polish(L, U, b, m, sigma, x0, 1e-12, 2000)
        assert res["rc"] == 0 and res["iters"] > 0
        assert 1e-8 < res["res0"] < 1e-4                       # an fp32-quality start
        assert abs(res["res0"] - np.linalg.norm(b - oracle.apply_A(L, U, m, sigma, x0)) / np.linalg.norm(b)) <= 1e-12
        assert rel(res["x"], xd) <= 1e-10
        assert np.linalg.norm(b - oracle.apply_A(L, U, m, sigma, res["x"])) / np.linalg.norm(b) <= 1e-12
        full = oracle.cg_polish(L, U, b, m, sigma, np.zeros_like(b), 1e-12, 2000)
        assert res["iters"] < full["iters"]                    # a good start saves iterations


def test_P9_polish_from_zero_is_the_single_shift_solver():
    L = (4, 4, 4, 4)
    U, b, m, sigma = si.links_haar(L, 42), si.source_gaussian(L, 42), 0.1, 0.02
    a = oracle.cg_polish(L, U, b, m, sigma, np.zeros_like(b), 1e-10, 2000)
    c = oracle.mshift_cg(L, U, b, m, [sigma], 1e-10, 2000)
    assert a["rc"] == 0 and a["iters"] == c["iters"] and a["res0"] == 1.0
    assert rel(a["x"], c["x"][0]) <= 1e-14


def test_P9_polish_of_the_exact_solution_and_bad_args():
    L = (2, 2, 2, 2)
    U, b, m = si.links_haar(L, 43), si.source_gaussian(L, 43), 0.2
    xd = oracle.dense_solve(oracle.dense_A(L, U, m), 0.3, b).reshape(-1, 3)
    res = oracle.cg_polish(L, U, b, m, 0.3, xd, 1e-10, 100)
    assert res["rc"] == 0 and res["iters"] == 0 and np.array_equal(res["x"], xd)
    assert oracle.cg_polish(L, U, b, m, 0.3, np.zeros_like(b), 1e-30, 3)["rc"] == -5
    with pytest.raises(ValueError):
        oracle.cg_polish(L, U, b, m, 0.3, xd, 0.0, 10)


# ---- N4: fermion force = derivative of the rational pseudo-fermion action ---------
GELL_MANN = np.zeros((8, 3, 3), dtype=np.complex128)
GELL_MANN[0][0, 1] = GELL_MANN[0][1, 0] = 1
GELL_MANN[1][0, 1], GELL_MANN[1][1, 0] = -1j, 1j
GELL_MANN[2][0, 0], GELL_MANN[2][1, 1] = 1, -1
GELL_MANN[3][0, 2] = GELL_MANN[3][2, 0] = 1
GELL_MANN[4][0, 2], GELL_MANN[4][2, 0] = -1j, 1j
GELL_MANN[5][1, 2] = GELL_MANN[5][2, 1] = 1
GELL_MANN[6][1, 2], GELL_MANN[6][2, 1] = -1j, 1j
GELL_MANN[7][0, 0] = GELL_MANN[7][1, 1] = 1 / np.sqrt(3)
GELL_MANN[7][2, 2] = -2 / np.sqrt(3)


def _expi(T, t):
    w, v = np.linalg.eigh(T)
    return (v * np.exp(1j * t * w)) @ v.conj().T


def _action(L, U, b, m, shifts, residues, residue0):
    """S = b^dag (residue0 + sum_i residues_i (A + sigma_i)^-1) b from DENSE solves (oracle_dense_*, pinned by P7)."""
    A = oracle.dense_A(L, U, m)
    bv = b.reshape(-1)
    S = residue0 * np.vdot(bv, bv).real
    for s, a in zip(shifts, residues):
        S += a * np.vdot(bv, oracle.dense_solve(A, s, b)).real
    return S


@pytest.mark.parametrize("L,links", [((2, 2, 2, 2), [(0, 0), (3, 3), (9, 3), (12, 1), (15, 2)]),
                                     ((4, 4, 2, 2), [(0, 0), (5, 1), (13, 2), (35, 3), (62, 3), (63, 0)])])
def test_P10_force_is_the_derivative_of_the_action(L, links):
    """d/dt S[U_mu(z) -> exp(itT) U_mu(z)] = tr(i T F_mu(z)), central differences, all 8 generators, links on
    both parities, in every direction and on the antiperiodic layer (x3 = L3 - 1: sites 9.. of 2^4 / 35, 62 of 4.4.2.2)."""
    U, b, m = si.links_haar(L, 61), si.source_gaussian(L, 61), 0.3
    shifts, residues, residue0 = [0.05, 0.4, 1.7], [0.7, -0.3, 1.9], 0.4
    A = oracle.dense_A(L, U, m)
    x = np.stack([oracle.dense_solve(A, s, b).reshape(-1, 3) for s in shifts])
    F = oracle.fermion_force(L, U, residues, x)
    eps = 1e-4
    for z, mu in links:
        for T in GELL_MANN:
            Up, Um = U.copy(), U.copy()
            Up[z, mu] = _expi(T, eps) @ U[z, mu]
            Um[z, mu] = _expi(T, -eps) @ U[z, mu]
            fd = (_action(L, Up, b, m, shifts, residues, residue0) - _action(L, Um, b, m, shifts, residues, residue0)) / (2 * eps)
            an = np.trace(1j * T @ F[z, mu])
            assert abs(an.imag) <= 1e-12 * max(1.0, abs(an.real))
            assert abs(fd - an.real) <= 2e-6 * max(1.0, np.abs(F[z, mu]).max()), (z, mu, fd, an)


def test_P10_force_is_traceless_antihermitian_and_gauge_covariant():
    L = (4, 4, 4, 4)
    U, m = si.links_haar(L, 62), 0.1
    residues = [1.0, 0.5]
    rng = np.random.default_rng(3)
    x = rng.standard_normal((2, 128, 3)) + 1j * rng.standard_normal((2, 128, 3))   # any even-site vectors do
    F = oracle.fermion_force(L, U, residues, x)
    assert np.abs(F + F.conj().transpose(0, 1, 3, 2)).max() <= 1e-14 * np.abs(F).max()
    assert np.abs(np.trace(F, axis1=2, axis2=3)).max() <= 1e-14 * np.abs(F).max()
    assert np.abs(F).max() > 0.1
    # U' = g U g^dag(x+mu), x' = g x  =>  F'_mu(z) = g(z) F_mu(z) g(z)^dag
    g = si.gauge_transform_field(L, 62)
    Ug = si.apply_gauge_transform(L, U, g)
    ge = g[si.parity_sites(L, 0)]
    xg = np.einsum("sab,isb->isa", ge, x)
    Fg = oracle.fermion_force(L, Ug, residues, xg)
    want = np.einsum("zab,zmbc,zdc->zmad", g, F, g.conj())
    assert rel(Fg, want) <= 1e-13
    # linear in the residues, quadratic in x
    assert rel(oracle.fermion_force(L, U, [2.0, 1.0], x), 2 * F) <= 1e-14
    assert rel(oracle.fermion_force(L, U, residues, 3 * x), 9 * F) <= 1e-14


# ---- the threaded mode of the oracle (oracle.set_threads(k > 1)) -----------------------------------------------
# Every full-size GPU parity test runs the oracle on several host cores (tests/test_gpu_fullsize.py and others call
# oracle.set_threads(8..32)).  SURVEY.md §8(d): "no algorithmic change, chunk-ordered deterministic reductions".
# The pin: for any thread count the results are BIT-equal to the one-thread oracle, which pins P1-P10 above hold.
@pytest.mark.parametrize("L", [(4, 4, 4, 4), (6, 4, 2, 8)])
def test_P11_threaded_oracle_is_bit_equal_to_one_thread(L):
    U = si.links_haar(L, 111)
    b = si.source_gaussian(L, 111, stream=1)
    xs = np.stack([si.source_gaussian(L, 111, stream=2 + k) for k in range(3)])
    mass, shifts, residues = 0.25, [0.0, 0.3, 2.0], [0.7, -0.3, 1.9]

    def everything():
        w = oracle.dslash_oe(L, U, b)
        cg = oracle.mshift_cg(L, U, b, mass, shifts, 1e-10, 3000, want_history=True)
        pol = oracle.cg_polish(L, U, b, mass, shifts[1], 0.5 * cg["x"][1], 1e-12, 3000)
        return dict(w=w, q=oracle.dslash_eo(L, U, w), A=oracle.apply_A(L, U, mass, 0.3, b), x=cg["x"], zeta=cg["zeta"],
                    r=cg["r"], hist=cg["rr_hist"], iters=cg["iters"], rc=cg["rc"], px=pol["x"], piters=pol["iters"],
                    pres0=pol["res0"], F=oracle.fermion_force(L, U, residues, xs), n2=oracle.norm2(b))
    try:
        oracle.set_threads(1)
        want = everything()
        assert want["rc"] == 0 and want["iters"] > 10
        for k in (2, 5, 8):
            oracle.set_threads(k)
            got = everything()
            for key, v in want.items():
                if isinstance(v, np.ndarray):
                    assert np.array_equal(got[key], v), (k, key)
                else:
                    assert got[key] == v, (k, key)
    finally:
        oracle.set_threads(1)


def test_P11_norm2_is_the_plain_sum_of_squares():
    # integers: every partial sum is exact, so any summation order must give n(n+1)(2n+1)/6 exactly
    n = 3 * 128
    v = (np.arange(1, 2 * n + 1, 2) + 1j * np.arange(2, 2 * n + 2, 2)).reshape(128, 3)
    m = 2 * n
    assert oracle.norm2(v) == m * (m + 1) * (2 * m + 1) // 6
    b = si.source_gaussian((4, 4, 4, 4), 5)
    assert abs(oracle.norm2(b) - np.vdot(b, b).real) <= 1e-13 * oracle.norm2(b)
    # and it is the <b,b> the CG starts from: rr_hist[0]
    U = si.links_haar((4, 4, 4, 4), 5)
    assert oracle.mshift_cg((4, 4, 4, 4), U, b, 0.1, [0.0], 1e-3, 5, want_history=True)["rr_hist"][0] == oracle.norm2(b)
