"""ctypes binding of include/stag.h — same names, argument marshalling only."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

HERE = os.path.dirname(os.path.abspath(__file__))
SO = os.path.join(HERE, "libstag_b200.so")
if os.environ.get("STAG_PHASE_TIMERS") == "1":     # per-phase-timer build of the persistent CG (see _build.py)
    SO = os.path.join(HERE, "libstag_b200_timers.so")

F64, F32, F64_SPLIT = 0, 1, 2      # F64_SPLIT (N3): split-double links, fp64 vectors
RECON18, RECON12 = 18, 12
MAX_SHIFTS = 32
MAX_RHS = 4
OK, ERR_BADARG, ERR_UNSUPPORTED, ERR_CUDA, ERR_NOT_SU3, ERR_NOTCONV, ERR_BREAKDOWN = 0, -1, -2, -3, -4, -5, -6
ERR_SCRATCH_LIMIT = -7             # stag_fermion_force_static: problem larger than the built-in scratch
FORCE_STATIC_BYTES = 8 << 20

# every symbol include/stag.h declares
SYMBOLS = [
    "stag_ctx_create", "stag_ctx_destroy", "stag_strerror", "stag_set_option", "stag_get_option",
    "stag_gauge_canonical_bytes", "stag_gauge_packed_bytes", "stag_vector_canonical_bytes",
    "stag_vector_bytes", "stag_cg_workspace_bytes", "stag_host_scratch_bytes",
    "stag_gauge_load", "stag_gauge_pack", "stag_vector_pack", "stag_vector_unpack",
    "stag_dslash_eo", "stag_dslash_oe", "stag_mshift_cg", "stag_dslash_host", "stag_mshift_cg_host",
    "stag_dslash_block", "stag_cg_block_workspace_bytes", "stag_mshift_cg_block",
    "stag_vector_convert", "stag_cg_polish_workspace_bytes", "stag_cg_polish",
    "stag_mshift_cg_mixed_workspace_bytes", "stag_mshift_cg_mixed",
    "stag_force_workspace_bytes", "stag_fermion_force",
    "stag_fermion_force_static_max_bytes", "stag_fermion_force_static",
    "stag_kernel_log_reset", "stag_kernel_log", "stag_cg_profile",
]


class CgInfo(C.Structure):
    _fields_ = [("iters", C.c_int), ("converged", C.c_int), ("breakdown", C.c_int),
                ("stagnated", C.c_int), ("bnorm2", C.c_double), ("rnorm2", C.c_double),
                ("resid_iter", C.c_double * MAX_SHIFTS), ("iters_shift", C.c_int * MAX_SHIFTS),
                ("kernel_launches", C.c_int)]

    def as_dict(self, nshift: int) -> dict:
        return dict(iters=self.iters, converged=bool(self.converged), breakdown=bool(self.breakdown),
                    stagnated=bool(self.stagnated), bnorm2=self.bnorm2, rnorm2=self.rnorm2,
                    resid_iter=list(self.resid_iter[:nshift]), iters_shift=list(self.iters_shift[:nshift]),
                    kernel_launches=self.kernel_launches)


class PolishInfo(C.Structure):
    _fields_ = [("passes", C.c_int), ("iters", C.c_int * MAX_SHIFTS), ("resid_before", C.c_double * MAX_SHIFTS),
                ("resid_after", C.c_double * MAX_SHIFTS), ("kernel_launches", C.c_int)]

    def as_dict(self, nshift: int) -> dict:
        return dict(passes=self.passes, iters=list(self.iters[:nshift]),
                    resid_before=list(self.resid_before[:nshift]), resid_after=list(self.resid_after[:nshift]),
                    kernel_launches=self.kernel_launches)


class MixedInfo(C.Structure):
    _fields_ = [("inner", CgInfo), ("polish", PolishInfo), ("reliable_updates", C.c_int), ("route", C.c_int)]

    def as_dict(self, nshift: int) -> dict:
        return dict(inner=self.inner.as_dict(nshift), polish=self.polish.as_dict(nshift),
                    reliable_updates=self.reliable_updates, route=self.route)


class StagError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        super().__init__("%s: %s (%d)" % (where, strerror(code), code))


_lib = None
_vp, _sz, _dp = C.c_void_p, C.c_size_t, C.POINTER(C.c_double)


def lib() -> C.CDLL:
    """Load libstag_b200.so; there is no fallback if it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(SO):
        raise ImportError("libstag_b200.so is not built: run `python -m paper_1010_5433_b200._build` "
                          "(or __graft_entry__.build()); there is no CPU fallback")
    l = C.CDLL(SO)
    l.stag_ctx_create.argtypes = [C.POINTER(C.c_int), C.POINTER(_vp)]
    l.stag_ctx_destroy.argtypes = [_vp]
    l.stag_ctx_destroy.restype = None
    l.stag_strerror.argtypes = [C.c_int]
    l.stag_strerror.restype = C.c_char_p
    l.stag_set_option.argtypes = [_vp, C.c_char_p, C.c_int]
    l.stag_get_option.argtypes = [_vp, C.c_char_p, C.POINTER(C.c_int)]
    for name, args in [("stag_gauge_canonical_bytes", [_vp]), ("stag_gauge_packed_bytes", [_vp, C.c_int, C.c_int]),
                       ("stag_vector_canonical_bytes", [_vp]), ("stag_vector_bytes", [_vp, C.c_int]),
                       ("stag_cg_workspace_bytes", [_vp, C.c_int, C.c_int]),
                       ("stag_host_scratch_bytes", [_vp, C.c_int, C.c_int])]:
        getattr(l, name).argtypes = args
        getattr(l, name).restype = _sz
    l.stag_gauge_load.argtypes = [_vp, _vp, _vp, _vp]
    l.stag_gauge_pack.argtypes = [_vp, _vp, _vp, C.c_int, C.c_int, _vp]
    l.stag_vector_pack.argtypes = [_vp, _vp, _vp, C.c_int, _vp]
    l.stag_vector_unpack.argtypes = [_vp, _vp, C.c_int, _vp, _vp]
    l.stag_dslash_eo.argtypes = [_vp, _vp, C.c_int, C.c_int, _vp, _vp, _vp]
    l.stag_dslash_oe.argtypes = [_vp, _vp, C.c_int, C.c_int, _vp, _vp, _vp]
    l.stag_dslash_block.argtypes = [_vp, _vp, C.c_int, C.c_int, C.c_int, C.c_int, _vp, _vp, _vp]
    l.stag_cg_block_workspace_bytes.argtypes = [_vp, C.c_int, C.c_int, C.c_int]
    l.stag_cg_block_workspace_bytes.restype = _sz
    l.stag_mshift_cg_block.argtypes = [_vp, _vp, C.c_int, C.c_int, C.c_int, _vp, C.c_double, C.c_int, _dp, _dp,
                                       C.c_double, C.c_double, C.c_int, _vp, _vp, _vp, C.POINTER(CgInfo), _vp]
    l.stag_mshift_cg.argtypes = [_vp, _vp, C.c_int, C.c_int, _vp, C.c_double, C.c_int, _dp, _dp,
                                 C.c_double, C.c_double, C.c_int, _vp, _vp, _vp, C.POINTER(CgInfo), _vp]
    l.stag_vector_convert.argtypes = [_vp, _vp, C.c_int, _vp, C.c_int, C.c_int, _vp]
    l.stag_cg_polish_workspace_bytes.argtypes = [_vp]
    l.stag_cg_polish_workspace_bytes.restype = _sz
    l.stag_cg_polish.argtypes = [_vp, _vp, C.c_int, C.c_int, _vp, C.c_double, C.c_int, _dp, C.c_double, C.c_int,
                                 _vp, _vp, C.POINTER(PolishInfo), _vp]
    l.stag_mshift_cg_mixed_workspace_bytes.argtypes = [_vp, C.c_int]
    l.stag_mshift_cg_mixed_workspace_bytes.restype = _sz
    l.stag_mshift_cg_mixed.argtypes = [_vp, _vp, C.c_int, C.c_int, _vp, C.c_int, _vp, C.c_double, C.c_int, _dp, _dp,
                                       C.c_double, C.c_double, C.c_double, C.c_int, _vp, _vp, _vp,
                                       C.POINTER(MixedInfo), _vp]
    l.stag_force_workspace_bytes.argtypes = [_vp, C.c_int, C.c_int]
    l.stag_force_workspace_bytes.restype = _sz
    l.stag_fermion_force.argtypes = [_vp, _vp, C.c_int, C.c_int, C.c_int, _dp, _vp, _vp, C.c_int, _vp, _vp]
    l.stag_fermion_force_static_max_bytes.argtypes = []
    l.stag_fermion_force_static_max_bytes.restype = _sz
    l.stag_fermion_force_static.argtypes = [_vp, _vp, C.c_int, C.c_int, C.c_int, _dp, _vp, _vp, C.c_int, _vp]
    l.stag_dslash_host.argtypes = [_vp, _vp, C.c_int, C.c_int, C.c_int, _vp, _vp, _vp, _vp]
    l.stag_mshift_cg_host.argtypes = [_vp, _vp, C.c_int, C.c_int, _vp, C.c_double, C.c_int, _dp, _dp,
                                      C.c_double, C.c_double, C.c_int, _vp, _vp, _vp, C.POINTER(CgInfo), _vp]
    l.stag_kernel_log_reset.argtypes = [_vp]
    l.stag_kernel_log.argtypes = [_vp, C.c_char_p, _sz]
    l.stag_cg_profile.argtypes = [_vp, _dp, C.POINTER(C.c_int)]
    _lib = l
    return l


def strerror(code: int) -> str:
    return lib().stag_strerror(int(code)).decode()


def _ptr(t) -> int:
    """Address of a torch tensor / numpy array / raw int."""
    if t is None:
        return None
    if isinstance(t, torch.Tensor):
        return t.data_ptr()
    if isinstance(t, np.ndarray):
        return t.ctypes.data
    return int(t)


def _stream(stream) -> int:
    if stream is None:
        return torch.cuda.current_stream().cuda_stream
    if isinstance(stream, torch.cuda.Stream):
        return stream.cuda_stream
    return int(stream)


def _darr(v):
    if v is None:
        return None
    a = np.ascontiguousarray(v, dtype=np.float64)
    return a.ctypes.data_as(_dp), a


class Stag:
    """One lattice geometry on the current CUDA device.  Methods mirror include/stag.h."""

    def __init__(self, L):
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1010_5433_b200 needs a CUDA device (no CPU fallback)")
        self.L = tuple(int(v) for v in L)
        self._h = _vp()
        rc = lib().stag_ctx_create((C.c_int * 4)(*self.L), C.byref(self._h))
        if rc:
            raise StagError(rc, "stag_ctx_create")
        self.V = self.L[0] * self.L[1] * self.L[2] * self.L[3]
        self.Vh = self.V // 2

    def close(self):
        if getattr(self, "_h", None):
            lib().stag_ctx_destroy(self._h)
            self._h = None

    __del__ = close

    # ---- options / sizes
    def set_option(self, key: str, value: int):
        rc = lib().stag_set_option(self._h, key.encode(), int(value))
        if rc:
            raise StagError(rc, "stag_set_option(%s)" % key)

    def get_option(self, key: str) -> int:
        v = C.c_int()
        rc = lib().stag_get_option(self._h, key.encode(), C.byref(v))
        if rc:
            raise StagError(rc, "stag_get_option(%s)" % key)
        return v.value

    def gauge_canonical_bytes(self): return lib().stag_gauge_canonical_bytes(self._h)
    def gauge_packed_bytes(self, prec, recon): return lib().stag_gauge_packed_bytes(self._h, prec, recon)
    def vector_canonical_bytes(self): return lib().stag_vector_canonical_bytes(self._h)
    def vector_bytes(self, prec): return lib().stag_vector_bytes(self._h, prec)
    def cg_workspace_bytes(self, prec, nshift): return lib().stag_cg_workspace_bytes(self._h, prec, nshift)
    def host_scratch_bytes(self, prec, nshift): return lib().stag_host_scratch_bytes(self._h, prec, nshift)

    @staticmethod
    def alloc(nbytes: int) -> torch.Tensor:
        """Device bytes (torch owns the memory); 256-byte aligned by the caching allocator."""
        return torch.empty(int(nbytes), dtype=torch.uint8, device="cuda")

    # ---- a1
    def gauge_load(self, host_links, dev_canonical, stream=None):
        rc = lib().stag_gauge_load(self._h, _ptr(host_links), _ptr(dev_canonical), _stream(stream))
        if rc:
            raise StagError(rc, "stag_gauge_load")

    def gauge_pack(self, dev_canonical, dev_packed, prec, recon, stream=None):
        rc = lib().stag_gauge_pack(self._h, _ptr(dev_canonical), _ptr(dev_packed), prec, recon, _stream(stream))
        if rc:
            raise StagError(rc, "stag_gauge_pack")

    def vector_pack(self, dev_canonical, dev_vec, prec, stream=None):
        rc = lib().stag_vector_pack(self._h, _ptr(dev_canonical), _ptr(dev_vec), prec, _stream(stream))
        if rc:
            raise StagError(rc, "stag_vector_pack")

    def vector_unpack(self, dev_vec, prec, dev_canonical, stream=None):
        rc = lib().stag_vector_unpack(self._h, _ptr(dev_vec), prec, _ptr(dev_canonical), _stream(stream))
        if rc:
            raise StagError(rc, "stag_vector_unpack")

    # ---- a2 / a3
    def dslash_eo(self, packed, prec, recon, in_odd, out_even, stream=None):
        rc = lib().stag_dslash_eo(self._h, _ptr(packed), prec, recon, _ptr(in_odd), _ptr(out_even), _stream(stream))
        if rc:
            raise StagError(rc, "stag_dslash_eo")

    def dslash_oe(self, packed, prec, recon, in_even, out_odd, stream=None):
        rc = lib().stag_dslash_oe(self._h, _ptr(packed), prec, recon, _ptr(in_even), _ptr(out_odd), _stream(stream))
        if rc:
            raise StagError(rc, "stag_dslash_oe")

    # ---- a3-a7
    def mshift_cg(self, packed, prec, recon, b_even, mass, shifts, stop, maxiter, x_even, workspace,
                  residues=None, residue0=0.0, y_even=None, stream=None, check=True):
        """Returns (rc, info dict).  With check=True anything but OK / NOTCONV / BREAKDOWN raises."""
        sh = _darr(shifts)
        rs = _darr(residues)
        info = CgInfo()
        n = sh[1].size
        rc = lib().stag_mshift_cg(self._h, _ptr(packed), prec, recon, _ptr(b_even), float(mass), n, sh[0],
                                  rs[0] if rs else None, float(residue0), float(stop), int(maxiter),
                                  _ptr(x_even), _ptr(y_even), _ptr(workspace), C.byref(info), _stream(stream))
        if check and rc not in (OK, ERR_NOTCONV, ERR_BREAKDOWN):
            raise StagError(rc, "stag_mshift_cg")
        return rc, info.as_dict(n)

    # ---- N1: nrhs independent sources through one link read
    def cg_block_workspace_bytes(self, prec, nshift, nrhs):
        return lib().stag_cg_block_workspace_bytes(self._h, prec, nshift, nrhs)

    def dslash_block(self, packed, prec, recon, out_parity, nrhs, vin, vout, stream=None):
        rc = lib().stag_dslash_block(self._h, _ptr(packed), prec, recon, int(out_parity), int(nrhs),
                                     _ptr(vin), _ptr(vout), _stream(stream))
        if rc:
            raise StagError(rc, "stag_dslash_block")

    def mshift_cg_block(self, packed, prec, recon, nrhs, b_even, mass, shifts, stop, maxiter, x_even, workspace,
                        residues=None, residue0=0.0, y_even=None, stream=None, check=True):
        """Returns (rc, [info dict per source])."""
        sh = _darr(shifts)
        rs = _darr(residues)
        infos = (CgInfo * int(nrhs))()
        n = sh[1].size
        rc = lib().stag_mshift_cg_block(self._h, _ptr(packed), prec, recon, int(nrhs), _ptr(b_even), float(mass),
                                        n, sh[0], rs[0] if rs else None, float(residue0), float(stop),
                                        int(maxiter), _ptr(x_even), _ptr(y_even), _ptr(workspace), infos,
                                        _stream(stream))
        if check and rc not in (OK, ERR_NOTCONV, ERR_BREAKDOWN):
            raise StagError(rc, "stag_mshift_cg_block")
        return rc, [infos[s].as_dict(n) for s in range(int(nrhs))]

    # ---- N2: mixed precision (fp32 multi-shift + per-shift fp64 polish)
    def vector_convert(self, src, src_prec, dst, dst_prec, nvec=1, stream=None):
        rc = lib().stag_vector_convert(self._h, _ptr(src), src_prec, _ptr(dst), dst_prec, int(nvec), _stream(stream))
        if rc:
            raise StagError(rc, "stag_vector_convert")

    def cg_polish_workspace_bytes(self): return lib().stag_cg_polish_workspace_bytes(self._h)
    def mshift_cg_mixed_workspace_bytes(self, nshift): return lib().stag_mshift_cg_mixed_workspace_bytes(self._h, nshift)

    def cg_polish(self, packed, prec, recon, b_even, mass, shifts, stop, maxiter, x_even, workspace, stream=None,
                  check=True):
        """Returns (rc, info dict); x_even is polished in place."""
        sh = _darr(shifts)
        info = PolishInfo()
        n = sh[1].size
        rc = lib().stag_cg_polish(self._h, _ptr(packed), prec, recon, _ptr(b_even), float(mass), n, sh[0],
                                  float(stop), int(maxiter), _ptr(x_even), _ptr(workspace), C.byref(info),
                                  _stream(stream))
        if check and rc not in (OK, ERR_NOTCONV, ERR_BREAKDOWN):
            raise StagError(rc, "stag_cg_polish")
        return rc, info.as_dict(n)

    def mshift_cg_mixed(self, packed_hi, prec_hi, recon_hi, packed_lo, recon_lo, b_even, mass, shifts, stop,
                        maxiter, x_even, workspace, inner_stop=0.0, residues=None, residue0=0.0, y_even=None,
                        stream=None, check=True):
        sh = _darr(shifts)
        rs = _darr(residues)
        info = MixedInfo()
        n = sh[1].size
        rc = lib().stag_mshift_cg_mixed(self._h, _ptr(packed_hi), prec_hi, recon_hi, _ptr(packed_lo), recon_lo,
                                        _ptr(b_even), float(mass), n, sh[0], rs[0] if rs else None,
                                        float(residue0), float(stop), float(inner_stop), int(maxiter),
                                        _ptr(x_even), _ptr(y_even), _ptr(workspace), C.byref(info),
                                        _stream(stream))
        if check and rc not in (OK, ERR_NOTCONV, ERR_BREAKDOWN):
            raise StagError(rc, "stag_mshift_cg_mixed")
        return rc, info.as_dict(n)

    # ---- N4: fermion force of the rational action
    def force_workspace_bytes(self, prec, nshift): return lib().stag_force_workspace_bytes(self._h, prec, nshift)

    def fermion_force(self, packed, prec, recon, residues, x_even, dev_force, workspace, accumulate=False,
                      stream=None):
        rs = _darr(residues)
        rc = lib().stag_fermion_force(self._h, _ptr(packed), prec, recon, rs[1].size, rs[0], _ptr(x_even),
                                      _ptr(dev_force), int(bool(accumulate)), _ptr(workspace), _stream(stream))
        if rc:
            raise StagError(rc, "stag_fermion_force")

    def fermion_force_static(self, packed, prec, recon, residues, x_even, dev_force, accumulate=False, stream=None):
        """fermion_force for callers that cannot allocate a workspace (a force callback that is handed x and F
        only, a host program whose pool owns all device memory, a loop that must not pay cudaMalloc's device-wide
        stall): the scratch is an 8 MiB array built into the library, one per GPU, shared by every call on that
        GPU — so calls that might overlap on the GPU must be serialised — and problems that need more raise
        StagError(ERR_SCRATCH_LIMIT).  The first call on a GPU also looks that array up; make it at start-up."""
        rs = _darr(residues)
        rc = lib().stag_fermion_force_static(self._h, _ptr(packed), prec, recon, rs[1].size, rs[0], _ptr(x_even),
                                             _ptr(dev_force), int(bool(accumulate)), _stream(stream))
        if rc:
            raise StagError(rc, "stag_fermion_force_static")

    # ---- measurement aids
    def kernel_log_reset(self):
        lib().stag_kernel_log_reset(self._h)

    def kernel_log(self) -> list:
        """Demangled names of the distinct kernels launched on this context since kernel_log_reset()."""
        buf = C.create_string_buffer(1 << 16)
        rc = lib().stag_kernel_log(self._h, buf, len(buf))
        if rc < 0:
            raise StagError(rc, "stag_kernel_log")
        return [n for n in buf.value.decode().split("\n") if n]

    def cg_profile(self):
        """(mean us of the a2, a3, a5, a6 launches, iterations averaged) of the last solve run with cg_profile = 1."""
        us = (C.c_double * 4)()
        n = C.c_int()
        rc = lib().stag_cg_profile(self._h, us, C.byref(n))
        if rc:
            raise StagError(rc, "stag_cg_profile")
        return list(us), n.value

    # ---- host-buffer variants
    def dslash_host(self, packed, prec, recon, out_parity, host_in, host_out, dev_scratch, stream=None):
        rc = lib().stag_dslash_host(self._h, _ptr(packed), prec, recon, int(out_parity), _ptr(host_in),
                                    _ptr(host_out), _ptr(dev_scratch), _stream(stream))
        if rc:
            raise StagError(rc, "stag_dslash_host")

    def mshift_cg_host(self, packed, prec, recon, host_b, mass, shifts, stop, maxiter, host_x, dev_scratch,
                       residues=None, residue0=0.0, host_y=None, stream=None, check=True):
        sh = _darr(shifts)
        rs = _darr(residues)
        info = CgInfo()
        n = sh[1].size
        rc = lib().stag_mshift_cg_host(self._h, _ptr(packed), prec, recon, _ptr(host_b), float(mass), n, sh[0],
                                       rs[0] if rs else None, float(residue0), float(stop), int(maxiter),
                                       _ptr(host_x), _ptr(host_y), _ptr(dev_scratch), C.byref(info),
                                       _stream(stream))
        if check and rc not in (OK, ERR_NOTCONV, ERR_BREAKDOWN):
            raise StagError(rc, "stag_mshift_cg_host")
        return rc, info.as_dict(n)

    # ---- conveniences for tests / bench: torch copies + the calls above, no arithmetic ----------
    def upload_gauge(self, links: np.ndarray, prec: int, recon: int, keep_canonical=None) -> torch.Tensor:
        """host canonical links complex128 [V][4][3][3] -> packed device buffer.  keep_canonical: a caller-owned
        device buffer of gauge_canonical_bytes() that receives the canonical copy (always re-loaded from `links`)."""
        links = np.ascontiguousarray(links, dtype=np.complex128)
        assert links.size == self.V * 36, links.shape
        canon = keep_canonical if keep_canonical is not None else self.alloc(self.gauge_canonical_bytes())
        self.gauge_load(links, canon)
        torch.cuda.current_stream().synchronize()          # pageable source: do not return early
        packed = self.alloc(self.gauge_packed_bytes(prec, recon))
        self.gauge_pack(canon, packed, prec, recon)
        torch.cuda.current_stream().synchronize()
        return packed

    def upload_vectors(self, vs, prec: int) -> torch.Tensor:
        """several host canonical vectors -> contiguous device-format vectors (stride vector_bytes)."""
        vb = self.vector_bytes(prec)
        dev = self.alloc(len(vs) * vb)
        for k, v in enumerate(vs):
            dev[k * vb:(k + 1) * vb].copy_(self.upload_vector(v, prec))
        return dev

    def upload_vector(self, v: np.ndarray, prec: int) -> torch.Tensor:
        """host canonical vector complex128 [Vh][3] -> device-format vector."""
        v = np.ascontiguousarray(v, dtype=np.complex128)
        assert v.size == self.Vh * 3, v.shape
        canon = torch.from_numpy(v.view(np.float64).reshape(-1)).cuda()
        dev = self.alloc(self.vector_bytes(prec))
        self.vector_pack(canon, dev, prec)
        torch.cuda.current_stream().synchronize()
        return dev

    def download_vector(self, dev_vec, prec: int, offset_bytes: int = 0) -> np.ndarray:
        """device-format vector -> host canonical complex128 [Vh][3]."""
        canon = torch.empty(self.Vh * 6, dtype=torch.float64, device="cuda")
        self.vector_unpack(_ptr(dev_vec) + int(offset_bytes), prec, canon)
        return canon.cpu().numpy().view(np.complex128).reshape(self.Vh, 3)
