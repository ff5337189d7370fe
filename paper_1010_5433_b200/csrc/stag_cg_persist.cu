// stag_cg_persist.cu — dispatch of the persistent multi-shift CG kernel (stag_cg_persist.cuh):
// the single-source path of stag_mshift_cg on small lattices, and stag_mshift_cg_block (N1: R
// independent sources — the paper's multiple pseudo-fermions, PAPER.md:48 — through one link read).
#include <cstring>

#include "stag_cg_persist.cuh"

namespace stag {

int cg_persistent_sr_launch(const stag_ctx *ctx, int prec, int recon, const PersistArgs &a, cudaStream_t st);

STAG_DEFINE_PERSIST_R(1)

// single source: the persistent kernel is used when at least r and q fit in shared memory (all three of
// r, q, p_base up to Vh ~ 210 K fp64 sites; r and q up to ~ 315 K, e.g. the paper's 4 x 48^3).  Beyond that an
// iteration takes milliseconds, launch ramps and reduction tails no longer matter, and the multi-kernel path
// (which runs at the copy bandwidth at 64^4) is used.
bool cg_persistent_fits(const stag_ctx *ctx, int prec) {
    if (persist_grid(ctx) > kMaxPersistGrid) return false;
    return (size_t)2 * persist_slots(ctx) * vec_bytes_per_site(prec) <= kMaxDynSmem;
}

int cg_persistent_dispatch(const stag_ctx *ctx, const void *packed, int prec, int recon,
                           const void *b, int nshift, const double *host_shifts, void *x, size_t x_stride,
                           void *y, char *ws, const CgLayout &lay, cudaStream_t st) {
    PersistArgs a;
    std::memset(&a, 0, sizeof(a));
    a.W = static_cast<const char *>(packed);
    a.b = static_cast<const char *>(b);
    a.b_stride = 0;
    a.w = ws + lay.w;
    a.r_g = ws + lay.r;
    a.q_g = ws + lay.q;
    a.vec_stride = lay.vec_stride;
    a.p = ws + lay.p;
    a.p_stride = lay.vec_stride;
    a.x = static_cast<char *>(x);
    a.x_stride = x_stride;
    a.y = static_cast<char *>(y);
    a.state = reinterpret_cast<CgState *>(ws + lay.state);
    a.state_stride = align256(sizeof(CgState));
    a.partials = reinterpret_cast<double *>(ws + lay.partials);
    a.flags = reinterpret_cast<unsigned int *>(ws + lay.flags);
    a.nrhs = 1;
    a.keep_mask = persist_keep_mask(ctx, prec, 1, nshift, host_shifts);
    if (ctx->opt.cg_single_reduction) {                  // one grid-wide reduction per iteration (stag_cg_persist_sr.cuh)
        const int rc = cg_persistent_sr_launch(ctx, prec, recon, a, st);
        if (rc != STAG_ERR_UNSUPPORTED) return rc;
    }
    if (prec == STAG_F64_SPLIT) return cg_persistent_launch_split(ctx, recon, 1, a, st);
    return cg_persistent_launch_r<1>(ctx, prec, recon, a, st);
}

// ---- block solve -----------------------------------------------------------------------------------
struct BlockLayout {
    size_t state, partials, flags, r, q, w, p, total;
    size_t vec_stride, state_stride;
};

static BlockLayout block_layout(const stag_ctx *ctx, int prec, int nshift, int nrhs) {
    BlockLayout l;
    const size_t vec = align256((size_t)ctx->g.Vh * vec_bytes_per_site(prec));
    size_t off = 0;
    l.state_stride = align256(sizeof(CgState));
    l.state = off;    off += l.state_stride * (size_t)nrhs;
    l.partials = off; off += align256(sizeof(double) * 2 * STAG_MAX_RHS * (size_t)ctx->num_sms);
    l.flags = off;    off += kPersistFlagBytes;
    l.r = off;        off += vec * (size_t)nrhs;
    l.q = off;        off += vec * (size_t)nrhs;
    l.w = off;        off += vec * (size_t)nrhs;
    l.p = off;        off += vec * (size_t)nrhs * (size_t)nshift;
    l.vec_stride = vec;
    l.total = off;
    return l;
}

}  // namespace stag

using namespace stag;

extern "C" size_t stag_cg_block_workspace_bytes(const stag_ctx *ctx, int prec, int nshift, int nrhs) {
    if (!ctx || !valid_prec(prec) || nshift < 1 || nshift > STAG_MAX_SHIFTS || nrhs < 1 || nrhs > STAG_MAX_RHS)
        return 0;
    return block_layout(ctx, prec, nshift, nrhs).total;
}

extern "C" int stag_mshift_cg_block(const stag_ctx *ctx, const void *packed, int prec, int recon, int nrhs,
                                    const void *b_even, double mass, int nshift, const double *host_shifts,
                                    const double *host_residues, double residue0, double stop,
                                    int maxiter, void *x_even, void *y_even, void *workspace,
                                    stag_cg_info *info, void *stream) {
    if (!ctx || !packed || !b_even || !host_shifts || !x_even || !workspace) return STAG_ERR_BADARG;
    if (!valid_prec(prec) || !valid_recon(recon)) return STAG_ERR_BADARG;
    if (nrhs < 1 || nrhs > STAG_MAX_RHS) return STAG_ERR_BADARG;
    if (nshift < 1 || nshift > STAG_MAX_SHIFTS || !(stop > 0.0) || maxiter < 0) return STAG_ERR_BADARG;
    if (y_even && !host_residues) return STAG_ERR_BADARG;
    double smin = host_shifts[0];
    for (int i = 0; i < nshift; ++i) {
        if (!(host_shifts[i] >= 0.0)) return STAG_ERR_BADARG;
        if (host_shifts[i] < smin) smin = host_shifts[i];
    }
    if (!(mass * mass + smin > 0.0)) return STAG_ERR_BADARG;
    if (((uintptr_t)workspace & 255) != 0) return STAG_ERR_BADARG;
    SlotLease lease(ctx);
    return block_solve(ctx, lease.slot(), packed, prec, recon, nrhs, b_even, mass, nshift, host_shifts, nullptr, nullptr,
                       host_residues, residue0, stop, maxiter, x_even, y_even, workspace, info,
                       static_cast<cudaStream_t>(stream));
}

int stag::block_solve(const stag_ctx *ctx, Slot &slot, const void *packed, int prec, int recon, int nrhs, const void *b_even,
                      double mass, int nshift, const double *host_shifts, const double *src_sigma,
                      const double *src_stop, const double *host_residues, double residue0, double stop,
                      int maxiter, void *x_even, void *y_even, void *workspace, stag_cg_info *info,
                      cudaStream_t st) {
    int base = 0;
    for (int i = 0; i < nshift; ++i)
        if (host_shifts[i] < host_shifts[base]) base = i;
    char *ws = static_cast<char *>(workspace);
    const BlockLayout lay = block_layout(ctx, prec, nshift, nrhs);
    const size_t vbytes = (size_t)ctx->g.Vh * vec_bytes_per_site(prec);

    // initial state: the same for every source, staged through the ctx's pinned buffer
    CgState *h = static_cast<CgState *>(slot.pinned_info);
    std::memset(h, 0, sizeof(*h));
    h->alpha_old = 1.0;
    h->c0 = mass * mass + host_shifts[base];
    h->stop = stop; h->residue0 = residue0;
    for (int i = 0; i < nshift; ++i) {
        h->delta[i] = host_shifts[i] - host_shifts[base];
        h->zeta[i] = 1.0; h->theta[i] = 1.0; h->active[i] = 1;
        h->residues[i] = host_residues ? host_residues[i] : 0.0;
        h->resid_shift[i] = 1.0;
    }
    h->nshift = nshift; h->base = base; h->maxiter = maxiter;
    h->freeze = ctx->opt.cg_freeze; h->fp32 = (prec == STAG_F32);
    for (int s = 0; s < nrhs; ++s) {
        if (src_sigma) {                       // N2 polish: one shift per source
            h->c0 = mass * mass + src_sigma[s];
            h->stop = src_stop[s];
            h->zero_ok = 1;
            // the pinned staging is re-used per source: wait until the previous copy has left it
            if (s > 0) STAG_CUDA_OK(cudaStreamSynchronize(st));
        }
        STAG_CUDA_OK(cudaMemcpyAsync(ws + lay.state + (size_t)s * lay.state_stride, h, sizeof(CgState),
                                     cudaMemcpyHostToDevice, st));
    }
    if (src_sigma) STAG_CUDA_OK(cudaStreamSynchronize(st));

    PersistArgs a;
    std::memset(&a, 0, sizeof(a));
    a.W = static_cast<const char *>(packed);
    a.b = static_cast<const char *>(b_even);
    a.b_stride = vbytes;
    a.w = ws + lay.w; a.r_g = ws + lay.r; a.q_g = ws + lay.q;
    a.vec_stride = lay.vec_stride;
    a.p = ws + lay.p; a.p_stride = lay.vec_stride;
    a.x = static_cast<char *>(x_even); a.x_stride = vbytes;
    a.y = static_cast<char *>(y_even);
    a.state = reinterpret_cast<CgState *>(ws + lay.state);
    a.state_stride = lay.state_stride;
    a.partials = reinterpret_cast<double *>(ws + lay.partials);
    a.flags = reinterpret_cast<unsigned int *>(ws + lay.flags);
    a.nrhs = nrhs;
    // N2 polish (one shift per source): every e_s is live to the end and small enough to stay in L2
    a.keep_mask = persist_keep_mask(ctx, prec, nrhs, nshift, host_shifts);
    int rc = prec == STAG_F64_SPLIT ? cg_persistent_launch_split(ctx, recon, nrhs == 1 ? 1 : nrhs == 2 ? 2 : 4, a, st)
           : nrhs == 1 ? cg_persistent_launch_r<1>(ctx, prec, recon, a, st)
           : nrhs == 2 ? cg_persistent_launch_r<2>(ctx, prec, recon, a, st)
                       : cg_persistent_launch_r<4>(ctx, prec, recon, a, st);
    if (rc) { cudaGetLastError(); return rc; }

    // read-back: the pinned staging holds one state at a time
    int worst = STAG_OK;
    for (int s = 0; s < nrhs; ++s) {
        STAG_CUDA_OK(cudaMemcpyAsync(h, ws + lay.state + (size_t)s * lay.state_stride, sizeof(CgState),
                                     cudaMemcpyDeviceToHost, st));
        STAG_CUDA_OK(cudaStreamSynchronize(st));
        if (info) {
            stag_cg_info *o = info + s;
            std::memset(o, 0, sizeof(*o));
            o->iters = h->iter; o->converged = h->converged; o->breakdown = h->breakdown;
            o->stagnated = h->stagnated; o->bnorm2 = h->bb; o->rnorm2 = h->rr;
            o->kernel_launches = s == 0 ? 1 : 0;
            for (int i = 0; i < nshift; ++i) {
                o->resid_iter[i] = h->bb > 0.0 ? h->resid_shift[i] : 0.0;
                o->iters_shift[i] = h->iters_shift[i];
            }
        }
        if (h->breakdown) worst = STAG_ERR_BREAKDOWN;
        else if (!h->converged && worst == STAG_OK) worst = STAG_ERR_NOTCONV;
    }
    return worst;
}
