"""ORACLE — TEST INFRASTRUCTURE.  Build + ctypes marshalling for oracle/stag_oracle.cpp.

All arrays are host numpy arrays in the canonical formats of stag_inputs/gen.py:
links complex128 [V][4][3][3], colour vectors complex128 [Vh][3].
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "stag_oracle.cpp")
_SO = os.path.join(_HERE, "libstag_oracle.so")
# STAG_ORACLE_SANITIZE=1: the same source built with -fsanitize=address,undefined; the process
# must then run with libasan preloaded (tests/test_oracle_sanitized.py does that in a subprocess).
_SANITIZE = os.environ.get("STAG_ORACLE_SANITIZE") == "1"
if _SANITIZE:
    _SO = os.path.join(_HERE, "libstag_oracle_san.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (building the checker is not using it)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        tmp = _SO + ".tmp.%d" % os.getpid()
        opt = ["-O2"]
        if _SANITIZE:
            opt = ["-O1", "-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined",
                   "-fno-sanitize-recover=all"]
        subprocess.check_call(["g++"] + opt + ["-fopenmp", "-fPIC", "-shared", "-std=c++14",
                               "-ffp-contract=off", "-o", tmp, _SRC])
        os.replace(tmp, _SO)
    return _SO


_P = C.POINTER
_dp = _P(C.c_double)
_ip = _P(C.c_int)


def lib():
    global _lib
    if _lib is None:
        l = C.CDLL(build())
        l.oracle_set_threads.argtypes = [C.c_int]
        l.oracle_dslash.argtypes = [_ip, _dp, _dp, _dp, C.c_int]
        l.oracle_apply_A.argtypes = [_ip, _dp, C.c_double, C.c_double, _dp, _dp, _dp]
        l.oracle_norm2.argtypes = [_dp, C.c_long]
        l.oracle_norm2.restype = C.c_double
        l.oracle_mshift_cg.argtypes = [_ip, _dp, _dp, C.c_double, C.c_int, _dp, C.c_double,
                                       C.c_int, _dp, _ip, _dp, _dp, _dp]
        l.oracle_partial_fraction.argtypes = [C.c_long, _dp, C.c_int, _dp, C.c_double, _dp, _dp]
        l.oracle_partial_fraction.restype = None
        l.oracle_cg_polish.argtypes = [_ip, _dp, _dp, C.c_double, C.c_double, C.c_double, C.c_int, _dp, _ip, _dp]
        l.oracle_fermion_force.argtypes = [_ip, _dp, C.c_int, _dp, _dp, _dp]
        l.oracle_dense_A.argtypes = [_ip, _dp, C.c_double, _dp]
        l.oracle_dense_solve.argtypes = [C.c_long, _dp, C.c_double, _dp, _dp]
        _lib = l
    return _lib


def _d(a: np.ndarray):
    return a.ctypes.data_as(_dp)


def _L(L):
    return (C.c_int * 4)(*[int(v) for v in L])


def _c128(a, shape=None) -> np.ndarray:
    a = np.ascontiguousarray(a, dtype=np.complex128)
    if shape is not None:
        assert a.shape == tuple(shape), (a.shape, shape)
    return a


def _vh(L) -> int:
    return int(L[0]) * int(L[1]) * int(L[2]) * int(L[3]) // 2


def set_threads(n: int) -> None:
    lib().oracle_set_threads(int(n))


def dslash(L, links, v, out_parity: int) -> np.ndarray:
    vh = _vh(L)
    links = _c128(links, (2 * vh, 4, 3, 3))
    v = _c128(v, (vh, 3))
    out = np.empty((vh, 3), dtype=np.complex128)
    rc = lib().oracle_dslash(_L(L), _d(links), _d(v), _d(out), int(out_parity))
    if rc:
        raise ValueError("oracle_dslash rc=%d" % rc)
    return out


def dslash_eo(L, links, v_odd) -> np.ndarray:
    """even output from odd input"""
    return dslash(L, links, v_odd, 0)


def dslash_oe(L, links, v_even) -> np.ndarray:
    """odd output from even input"""
    return dslash(L, links, v_even, 1)


def apply_A(L, links, mass: float, sigma: float, v_even) -> np.ndarray:
    vh = _vh(L)
    links = _c128(links, (2 * vh, 4, 3, 3))
    v = _c128(v_even, (vh, 3))
    out = np.empty_like(v)
    tmp = np.empty_like(v)
    rc = lib().oracle_apply_A(_L(L), _d(links), float(mass), float(sigma), _d(v), _d(out), _d(tmp))
    if rc:
        raise ValueError("oracle_apply_A rc=%d" % rc)
    return out


def norm2(v) -> float:
    v = _c128(v)
    return float(lib().oracle_norm2(_d(v), v.size * 2))


def mshift_cg(L, links, b, mass: float, shifts, stop: float, maxiter: int,
              want_history: bool = False) -> dict:
    """Returns dict(rc, iters, x [N][Vh][3], zeta [N], r [Vh][3], rr_hist)."""
    vh = _vh(L)
    links = _c128(links, (2 * vh, 4, 3, 3))
    b = _c128(b, (vh, 3))
    sh = np.ascontiguousarray(shifts, dtype=np.float64)
    n = sh.size
    x = np.empty((n, vh, 3), dtype=np.complex128)
    zeta = np.empty(n, dtype=np.float64)
    r = np.empty((vh, 3), dtype=np.complex128)
    hist = np.full(maxiter + 1, np.nan) if want_history else None
    iters = C.c_int(0)
    rc = lib().oracle_mshift_cg(_L(L), _d(links), _d(b), float(mass), n, _d(sh), float(stop),
                                int(maxiter), _d(x), C.byref(iters), _d(zeta), _d(r),
                                _d(hist) if hist is not None else None)
    if rc == -1:
        raise ValueError("oracle_mshift_cg: bad argument")
    return dict(rc=rc, iters=iters.value, x=x, zeta=zeta, r=r,
                rr_hist=hist[: iters.value + 1] if hist is not None else None)


def cg_polish(L, links, b, mass: float, sigma: float, x0, stop: float, maxiter: int) -> dict:
    """N2: ordinary CG on (A + sigma) x = b from the start vector x0.  Returns dict(rc, iters, x, res0)."""
    vh = _vh(L)
    links = _c128(links, (2 * vh, 4, 3, 3))
    b = _c128(b, (vh, 3))
    x = _c128(x0, (vh, 3)).copy()
    iters = C.c_int(0)
    res0 = C.c_double(0.0)
    rc = lib().oracle_cg_polish(_L(L), _d(links), _d(b), float(mass), float(sigma), float(stop), int(maxiter),
                                _d(x), C.byref(iters), C.byref(res0))
    if rc == -1:
        raise ValueError("oracle_cg_polish: bad argument")
    return dict(rc=rc, iters=iters.value, x=x, res0=res0.value)


def fermion_force(L, links, residues, x) -> np.ndarray:
    """N4: F [V][4][3][3] (traceless anti-Hermitian) with d/dt S[exp(itT) U_mu(z)] = tr(i T F_mu(z)) for
    S = b^dag (residue0 + sum_i residues_i (A+sigma_i)^-1) b and x[i] = (A+sigma_i)^-1 b."""
    vh = _vh(L)
    links = _c128(links, (2 * vh, 4, 3, 3))
    res = np.ascontiguousarray(residues, dtype=np.float64)
    x = _c128(x, (res.size, vh, 3))
    F = np.empty((2 * vh, 4, 3, 3), dtype=np.complex128)
    rc = lib().oracle_fermion_force(_L(L), _d(links), res.size, _d(res), _d(x), _d(F))
    if rc:
        raise ValueError("oracle_fermion_force rc=%d" % rc)
    return F


def partial_fraction(b, residues, residue0: float, x) -> np.ndarray:
    b = _c128(b)
    x = _c128(x)
    res = np.ascontiguousarray(residues, dtype=np.float64)
    assert x.shape == (res.size,) + b.shape
    y = np.empty_like(b)
    lib().oracle_partial_fraction(b.size * 2, _d(b), res.size, _d(res), float(residue0), _d(x), _d(y))
    return y


def dense_A(L, links, mass: float) -> np.ndarray:
    vh = _vh(L)
    links = _c128(links, (2 * vh, 4, 3, 3))
    N = 3 * vh
    A = np.empty((N, N), dtype=np.complex128)
    rc = lib().oracle_dense_A(_L(L), _d(links), float(mass), _d(A))
    if rc:
        raise ValueError("oracle_dense_A rc=%d" % rc)
    return A


def dense_solve(A, sigma: float, b) -> np.ndarray:
    A = _c128(A)
    N = A.shape[0]
    b = _c128(b).reshape(-1)
    assert b.size == N
    x = np.empty(N, dtype=np.complex128)
    rc = lib().oracle_dense_solve(N, _d(A), float(sigma), _d(b), _d(x))
    if rc:
        raise ValueError("oracle_dense_solve rc=%d" % rc)
    return x


def split_double(a: np.ndarray) -> np.ndarray:
    """N3: "write a double precision number a by using two single precision numbers b
    and c": b = (float)a, c = (float)(a - (double)b), and "reconstruct the double
    precision number a to be used in calculations" = (double)b + (double)c.  Returns that reconstruction
    a' (same shape; complex arrays are split component-wise).  b + c carries 48 significant bits, so
    |a' - a| <= 2^-48 |a| (pin: tests/test_oracle_pins.py::test_N3_split_double)."""
    a = np.asarray(a)
    if np.iscomplexobj(a):
        return split_double(a.real) + 1j * split_double(a.imag)
    a = a.astype(np.float64)
    b = a.astype(np.float32)
    c = (a - b.astype(np.float64)).astype(np.float32)
    return b.astype(np.float64) + c.astype(np.float64)
