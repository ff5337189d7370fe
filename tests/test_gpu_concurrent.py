"""Several solves in flight on ONE context (independent pseudo-fermions): every synchronising call
leases its own host staging slot, so two host threads on two streams may solve at the same time, and the
multi-kernel path's CUDA graph is cached per slot and replayed by later solves with the same buffers.  Results must
equal the serial ones bit for bit (reductions are order-deterministic per launch configuration)."""
import threading

import numpy as np
import pytest
import torch

import oracle
import stag_inputs as si

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def stag():
    import paper_1010_5433_b200 as m
    return m


def true_res(L, U, m, s, b, x):
    return np.linalg.norm(b - oracle.apply_A(L, U, m, s, x)) / np.linalg.norm(b)


@pytest.mark.parametrize("path", ["multikernel", "persistent"])
@pytest.mark.parametrize("nthreads", [2, 6])
def test_concurrent_solves_on_one_context(stag, path, nthreads):
    """nthreads > 4 also exercises waiting for a free slot."""
    L, m, stop = (8, 8, 8, 4), 0.1, 1e-10
    shifts = [0.01, 0.04, 0.16, 0.64]
    U = si.links_haar(L, 71)
    bs = [si.source_gaussian(L, 71, stream=1 + k) for k in range(nthreads)]
    ctx = stag.Stag(L)
    ctx.set_option("cg_persistent", 1 if path == "persistent" else 0)
    packed = ctx.upload_gauge(U, 0, 18)
    n, vb = len(shifts), ctx.vector_bytes(0)
    bdev = [ctx.upload_vector(b, 0) for b in bs]
    # serial reference results
    serial = []
    for k in range(nthreads):
        x, ws = ctx.alloc(n * vb), ctx.alloc(ctx.cg_workspace_bytes(0, n))
        rc, info = ctx.mshift_cg(packed, 0, 18, bdev[k], m, shifts, stop, 5000, x, ws)
        assert rc == 0
        serial.append((info["iters"], x.clone()))
    # concurrent: one host thread and one stream per source
    xs = [ctx.alloc(n * vb) for _ in range(nthreads)]
    wss = [ctx.alloc(ctx.cg_workspace_bytes(0, n)) for _ in range(nthreads)]
    streams = [torch.cuda.Stream() for _ in range(nthreads)]
    torch.cuda.synchronize()
    out = [None] * nthreads

    def work(k):
        try:
            out[k] = ctx.mshift_cg(packed, 0, 18, bdev[k], m, shifts, stop, 5000, xs[k], wss[k], stream=streams[k])
        except Exception as e:      # pragma: no cover
            out[k] = e

    for rep in range(3):
        ts = [threading.Thread(target=work, args=(k,)) for k in range(nthreads)]
        for t in ts:
            t.start()
        for t in ts:
            t.join()
        torch.cuda.synchronize()
        for k in range(nthreads):
            assert not isinstance(out[k], Exception), out[k]
            rc, info = out[k]
            assert rc == 0 and info["iters"] == serial[k][0], (k, rc, info["iters"], serial[k][0])
            assert torch.equal(xs[k], serial[k][1]), k
    for i, s in enumerate(shifts):
        assert true_res(L, U, m, s, bs[0], ctx.download_vector(xs[0], 0, i * vb)) <= stop


def test_graph_cache_follows_the_buffers(stag):
    """Multi-kernel path: the cached graph is replayed while packed / workspace / x / storage stay the same and is
    rebuilt when one of them changes; results never depend on which happened."""
    L, m, stop = (8, 8, 8, 4), 0.1, 1e-10
    shifts = [0.02, 0.3, 1.1]
    U, b = si.links_haar(L, 72), si.source_gaussian(L, 72)
    ref = oracle.mshift_cg(L, U, b, m, shifts, stop, 5000)
    ctx = stag.Stag(L)
    ctx.set_option("cg_persistent", 0)
    p18, p12 = ctx.upload_gauge(U, 0, 18), ctx.upload_gauge(U, 0, 12)
    n, vb = len(shifts), ctx.vector_bytes(0)
    bdev = ctx.upload_vector(b, 0)
    xa, xb = ctx.alloc(n * vb), ctx.alloc(n * vb)
    wa, wb = ctx.alloc(ctx.cg_workspace_bytes(0, n)), ctx.alloc(ctx.cg_workspace_bytes(0, n))
    for packed, recon, x, ws in ((p18, 18, xa, wa), (p18, 18, xa, wa), (p18, 18, xb, wa), (p12, 12, xb, wb),
                                 (p18, 18, xa, wa), (p18, 18, xa, wa)):
        x.fill_(0xFF)
        rc, info = ctx.mshift_cg(packed, 0, recon, bdev, m, shifts, stop, 5000, x, ws)
        assert rc == 0 and abs(info["iters"] - ref["iters"]) <= 2 and info["kernel_launches"] > 1
        for i, s in enumerate(shifts):
            assert true_res(L, U, m, s, b, ctx.download_vector(x, 0, i * vb)) <= stop
    # a different number of shifts with the same buffers: the graph must be rebuilt, not replayed
    rc, info = ctx.mshift_cg(p18, 0, 18, bdev, m, shifts[:2], stop, 5000, xa, wa)
    assert rc == 0
    for i, s in enumerate(shifts[:2]):
        assert true_res(L, U, m, s, b, ctx.download_vector(xa, 0, i * vb)) <= stop
