"""Out-of-bounds writes: every output / workspace buffer of the main calls is carved out of a larger allocation
with 4 KB guard zones on both sides, filled with a pattern; after the call the guards must be untouched and the
*_bytes() sizes the header promises must have been enough.  (compute-sanitizer is closed on the GPU pool: profiles/r3_sanitizer_unavailable.txt holds the command and the pool's refusal.)
Ragged lattices, so that partial warps / CTAs / per-SM slices are exercised."""
import numpy as np
import pytest

import stag_inputs as si

pytestmark = pytest.mark.gpu
GUARD = 4096


@pytest.fixture(scope="module")
def stag():
    import paper_1010_5433_b200 as m
    return m


class Guarded:
    def __init__(self, nbytes):
        import torch
        self.n = int(nbytes)
        pad = (-self.n) % 256
        self.buf = torch.full((GUARD + self.n + pad + GUARD,), 0xA5, dtype=torch.uint8, device="cuda")
        self.view = self.buf[GUARD:GUARD + self.n]
        assert self.view.data_ptr() % 256 == 0

    def intact(self):
        lo, hi = self.buf[:GUARD], self.buf[GUARD + self.n:]
        return bool((lo == 0xA5).all().item()) and bool((hi == 0xA5).all().item())


@pytest.mark.parametrize("L", [(6, 6, 2, 2), (10, 6, 4, 4), (2, 2, 2, 2), (4, 4, 4, 4)])
@pytest.mark.parametrize("prec_name,recon", [("F64", 18), ("F32", 12), ("F64_SPLIT", 18)])
def test_no_call_writes_outside_its_buffers(stag, L, prec_name, recon):
    import torch
    prec = getattr(stag, prec_name)
    vprec = stag.F32 if prec == stag.F32 else stag.F64
    U, b, m = si.links_haar(L, 95), si.source_gaussian(L, 95), 0.3
    shifts = [0.05, 0.4, 1.7, 0.01, 3.0]
    n = len(shifts)
    ctx = stag.Stag(L)
    canon = Guarded(ctx.gauge_canonical_bytes())
    ctx.gauge_load(np.ascontiguousarray(U), canon.view)
    torch.cuda.synchronize()
    packed = Guarded(ctx.gauge_packed_bytes(prec, recon))
    ctx.gauge_pack(canon.view, packed.view, prec, recon)
    vb = ctx.vector_bytes(prec)
    bdev = ctx.upload_vector(b, prec)
    out = Guarded(vb)
    ctx.dslash_oe(packed.view, prec, recon, bdev, out.view)
    guards = [canon, packed, out]
    for path in (1, 0):
        ctx.set_option("cg_persistent", path)
        x, y, ws = Guarded(n * vb), Guarded(vb), Guarded(ctx.cg_workspace_bytes(prec, n))
        rc, _ = ctx.mshift_cg(packed.view, prec, recon, bdev, m, shifts, 1e-9 if vprec == stag.F64 else 1e-4, 500,
                              x.view, ws.view, residues=[1.0] * n, residue0=0.5, y_even=y.view)
        assert rc == 0
        guards += [x, y, ws]
    if prec != stag.F64_SPLIT:
        for R in (2, 3, 4):
            bs = ctx.upload_vectors([b] * R, prec)
            xb, wsb, ob = Guarded(R * n * vb), Guarded(ctx.cg_block_workspace_bytes(prec, n, R)), Guarded(R * vb)
            ctx.dslash_block(packed.view, prec, recon, 0, R, bs, ob.view)
            ctx.mshift_cg_block(packed.view, prec, recon, R, bs, m, shifts, 1e-9 if vprec == stag.F64 else 1e-4, 500,
                                xb.view, wsb.view)
            guards += [xb, wsb, ob]
        F, fws = Guarded(ctx.V * 72 * 8), Guarded(ctx.force_workspace_bytes(prec, n))
        ctx.fermion_force(packed.view, prec, recon, [1.0] * n, guards[3].view, F.view.view(torch.float64), fws.view)
        guards += [F, fws]
    if prec != stag.F32:
        b64 = ctx.upload_vector(b, stag.F64)
        xp, pws = Guarded(n * ctx.vector_bytes(stag.F64)), Guarded(ctx.cg_polish_workspace_bytes())
        xp.view.zero_()
        rc, _ = ctx.cg_polish(packed.view, prec, recon, b64, m, shifts, 1e-9, 500, xp.view, pws.view)
        assert rc == 0
        p32 = Guarded(ctx.gauge_packed_bytes(stag.F32, recon))
        ctx.gauge_pack(canon.view, p32.view, stag.F32, recon)
        xm, mws = Guarded(n * ctx.vector_bytes(stag.F64)), Guarded(ctx.mshift_cg_mixed_workspace_bytes(n))
        rc, _ = ctx.mshift_cg_mixed(packed.view, prec, recon, p32.view, recon, b64, m, shifts, 1e-9, 500, xm.view, mws.view)
        assert rc == 0
        guards += [xp, pws, p32, xm, mws]
    torch.cuda.synchronize()
    for k, gd in enumerate(guards):
        assert gd.intact(), "guard zone %d overwritten" % k
