"""Counter-based seeded generators (numpy, host side, fp64).

Canonical host formats (the formats at the C-ABI, include/stag.h):
  * site index      lex(x) = x0 + L0*(x1 + L1*(x2 + L2*x3)),  x0 fastest, x3 = time
  * parity          (x0+x1+x2+x3) & 1,  0 = even
  * one-parity idx  e = lex(x) // 2      (bijective on each parity because L0 is even)
  * links           complex128 [V][4][3][3]  == double [V][4][3][3][2]  (row, col)
  * colour vector   complex128 [Vh][3]       == double [Vh][3][2]

Every random number is a pure function of (seed, stream, index, k): generation
order, chunking and threading do not change the values.
"""
from __future__ import annotations

import numpy as np

_U64 = np.uint64
_GAMMA = _U64(0x9E3779B97F4A7C15)
_M1 = _U64(0xBF58476D1CE4E5B9)
_M2 = _U64(0x94D049BB133111EB)


def _mix(z: np.ndarray) -> np.ndarray:
    """splitmix64 finaliser (Steele, Lea, Flood 2014) on uint64 arrays."""
    with np.errstate(over="ignore"):
        z = z + _GAMMA
        z = (z ^ (z >> _U64(30))) * _M1
        z = (z ^ (z >> _U64(27))) * _M2
        return z ^ (z >> _U64(31))


def _key(seed: int, stream: int, idx: np.ndarray) -> np.ndarray:
    h = _mix(np.array([seed], dtype=_U64))
    h = _mix(h ^ _U64(stream))
    return _mix(h ^ idx.astype(_U64))


def _uniform(key: np.ndarray, k: np.ndarray) -> np.ndarray:
    """(0,1) uniforms for every (key, k) pair; result shape key.shape + k.shape."""
    h = _mix(key[..., None] ^ k.astype(_U64))
    return ((h >> _U64(11)).astype(np.float64) + 0.5) * (1.0 / 9007199254740992.0)


def normals(seed: int, stream: int, idx: np.ndarray, nk: int) -> np.ndarray:
    """Standard normals z[i, k], k < nk, for the integer labels idx[i] (Box-Muller)."""
    key = _key(seed, stream, np.asarray(idx))
    k = np.arange(nk, dtype=np.uint64)
    u1 = _uniform(key, 2 * k)
    u2 = _uniform(key, 2 * k + 1)
    return np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)


# ----------------------------------------------------------------------------
# lattice indexing (data layout only)
# ----------------------------------------------------------------------------
def volume(L) -> int:
    return int(L[0]) * int(L[1]) * int(L[2]) * int(L[3])


def half_volume(L) -> int:
    return volume(L) // 2


def site_coords(L) -> np.ndarray:
    """int64 [V][4]: coordinates of every site in lex order."""
    lex = np.arange(volume(L), dtype=np.int64)
    x0 = lex % L[0]
    x1 = (lex // L[0]) % L[1]
    x2 = (lex // (L[0] * L[1])) % L[2]
    x3 = lex // (L[0] * L[1] * L[2])
    return np.stack([x0, x1, x2, x3], axis=1)


def parity_sites(L, parity: int) -> np.ndarray:
    """lex indices of the sites of one parity, ordered by e = lex // 2."""
    x = site_coords(L)
    lex = np.arange(volume(L), dtype=np.int64)
    sel = lex[(x.sum(axis=1) & 1) == parity]
    assert np.array_equal(sel // 2, np.arange(half_volume(L)))
    return sel


# ----------------------------------------------------------------------------
# SU(3) generators
# ----------------------------------------------------------------------------
def su3_project(M: np.ndarray) -> np.ndarray:
    """Gram-Schmidt on rows 1,2; row 3 = conj(row1 x row2)  ->  det = 1 exactly."""
    r1 = M[..., 0, :]
    r1 = r1 / np.linalg.norm(r1, axis=-1, keepdims=True)
    r2 = M[..., 1, :]
    r2 = r2 - np.sum(np.conj(r1) * r2, axis=-1, keepdims=True) * r1
    r2 = r2 / np.linalg.norm(r2, axis=-1, keepdims=True)
    r3 = np.conj(np.cross(r1, r2))
    return np.stack([r1, r2, r3], axis=-2)


def _gaussian_matrices(seed: int, stream: int, idx: np.ndarray) -> np.ndarray:
    z = normals(seed, stream, idx, 18).reshape(-1, 3, 3, 2)
    return z[..., 0] + 1j * z[..., 1]


def links_unit(L) -> np.ndarray:
    U = np.zeros((volume(L), 4, 3, 3), dtype=np.complex128)
    U[..., 0, 0] = U[..., 1, 1] = U[..., 2, 2] = 1.0
    return U


def _chunks(n: int, step: int = 1 << 16):
    for lo in range(0, n, step):
        yield lo, min(n, lo + step)


def _for_chunks(n: int, fn) -> None:
    """fn(lo, hi) over cache-sized chunks, on all host cores (numpy releases the GIL; the values
    are a pure function of the index, so threading does not change them)."""
    import os
    from concurrent.futures import ThreadPoolExecutor
    chunks = list(_chunks(n))
    nt = min(len(chunks), os.cpu_count() or 1)
    if nt <= 1:
        for lo, hi in chunks:
            fn(lo, hi)
        return
    with ThreadPoolExecutor(nt) as ex:
        list(ex.map(lambda c: fn(*c), chunks))


def links_haar(L, seed: int, out: np.ndarray | None = None) -> np.ndarray:
    """'Haar-like' rough links: reunitarised 3x3 iid complex Gaussian matrices."""
    n = 4 * volume(L)
    U = out if out is not None else np.empty((n, 3, 3), dtype=np.complex128)
    U = U.reshape(n, 3, 3)
    def fill(lo, hi):
        U[lo:hi] = su3_project(_gaussian_matrices(seed, 0, np.arange(lo, hi)))

    _for_chunks(n, fill)
    return U.reshape(volume(L), 4, 3, 3)


def _expi(H: np.ndarray, eps: float) -> np.ndarray:
    """exp(i*eps*H) by scaling-and-squaring Taylor series (H Hermitian)."""
    s = 6
    X = (1j * eps / (1 << s)) * H
    E = np.zeros_like(X)
    E[..., 0, 0] = E[..., 1, 1] = E[..., 2, 2] = 1.0
    term = E.copy()
    for n in range(1, 13):
        term = term @ X / n
        E = E + term
    for _ in range(s):
        E = E @ E
    return E


def links_smooth(L, seed: int, eps: float) -> np.ndarray:
    """Smooth links U = exp(i*eps*H), H Gaussian Hermitian traceless, then projected."""
    n = 4 * volume(L)
    U = np.empty((n, 3, 3), dtype=np.complex128)
    eye = np.eye(3)
    def fill(lo, hi):
        G = _gaussian_matrices(seed, 0, np.arange(lo, hi)) * np.sqrt(0.5)
        H = 0.5 * (G + np.conj(np.swapaxes(G, -1, -2)))
        tr = np.trace(H, axis1=-2, axis2=-1).real / 3.0
        H = H - tr[:, None, None] * eye
        U[lo:hi] = su3_project(_expi(H, eps))

    _for_chunks(n, fill)
    return U.reshape(volume(L), 4, 3, 3)


def gauge_transform_field(L, seed: int, stream: int = 99) -> np.ndarray:
    """Random SU(3) g(x) per site, [V][3][3]."""
    return su3_project(_gaussian_matrices(seed, stream, np.arange(volume(L))))


def apply_gauge_transform(L, U: np.ndarray, g: np.ndarray) -> np.ndarray:
    """U'_mu(x) = g(x) U_mu(x) g(x+mu)^dagger  (g periodic; the BC sign is not in U)."""
    x = site_coords(L)
    strides = (1, L[0], L[0] * L[1], L[0] * L[1] * L[2])
    Up = np.empty_like(U)
    for mu in range(4):
        xp = x.copy()
        xp[:, mu] = (xp[:, mu] + 1) % L[mu]
        lexp = xp @ np.array(strides, dtype=np.int64)
        gd = np.conj(np.swapaxes(g[lexp], -1, -2))
        Up[:, mu] = g @ U[:, mu] @ gd
    return Up


# ----------------------------------------------------------------------------
# sources
# ----------------------------------------------------------------------------
def source_gaussian(L, seed: int, stream: int = 1) -> np.ndarray:
    """iid complex normal (re, im each N(0,1)) on one parity, [Vh][3]."""
    out = np.empty((half_volume(L), 3), dtype=np.complex128)

    def fill(lo, hi):
        z = normals(seed, stream, np.arange(lo, hi), 6).reshape(-1, 3, 2)
        out[lo:hi] = z[..., 0] + 1j * z[..., 1]

    _for_chunks(half_volume(L), fill)
    return out


def source_plane_wave(L, n, colour, parity: int = 0) -> np.ndarray:
    """exp(i p.x) * colour on one parity; p_mu = 2 pi n_mu / L_mu (mu<3),
    p_3 = 2 pi (n_3 + 1/2) / L_3 (antiperiodic time).  Returns (v, p)."""
    p = np.array([2 * np.pi * n[0] / L[0], 2 * np.pi * n[1] / L[1],
                  2 * np.pi * n[2] / L[2], 2 * np.pi * (n[3] + 0.5) / L[3]])
    x = site_coords(L)[parity_sites(L, parity)]
    phase = np.exp(1j * (x @ p))
    v = phase[:, None] * np.asarray(colour, dtype=np.complex128)[None, :]
    return np.ascontiguousarray(v), p
