// stag_cg.cuh — device-resident state of one multi-shift CG solve and the workspace layout.
// (recurrences = DESIGN.md reading C4 in ratio form, reading A15.)
#pragma once

#include "stag_common.cuh"

namespace stag {

// Everything the iteration needs between kernels lives here, in the caller's workspace: the
// host never sees a scalar until the final read-back.
struct CgState {
    // scalars of the base (smallest-shift) system
    double bb, rr, pq, alpha, alpha_old, beta, beta_old;
    double c0;              // m^2 + sigma_0
    double stop;            // on sqrt(rr/bb)
    double residue0;
    double best_rr;         // fp32 stagnation watch (reading A9)
    // per shift
    double delta[STAG_MAX_SHIFTS];     // sigma_i - sigma_0 >= 0
    double zeta[STAG_MAX_SHIFTS];      // residual of system i is zeta_i * r
    double theta[STAG_MAX_SHIFTS];     // zeta_i / zetaold_i
    double theta_new[STAG_MAX_SHIFTS];
    double alpha_i[STAG_MAX_SHIFTS];
    double beta_i[STAG_MAX_SHIFTS];
    double residues[STAG_MAX_SHIFTS];
    double resid_shift[STAG_MAX_SHIFTS];
    int active[STAG_MAX_SHIFTS];       // 1 updating, 2 last update this iteration, 0 frozen
    int iters_shift[STAG_MAX_SHIFTS];
    int nshift, base, maxiter, freeze, fp32;
    int iter;
    int done;               // 0 running | 1 finishing (x update of this iteration pending) | 2 over
    int converged, breakdown, stagnated, since_best;
    int zero_ok;            // N2 polish: stop >= 1 means "the zero start is good enough": 0 iterations
    int replacements;       // N2 residual-replacement kernel: true-residual replacements done (read-back only)
    unsigned int ticket;    // last-block detection for the grid-wide reductions
};

static constexpr size_t kPersistFlagBytes = 256 * 128;   // kMaxPersistGrid CTAs (stag_cg_persist.cuh)

struct CgLayout {
    size_t state, partials, flags, r, q, w, p;   // byte offsets into the workspace; p = nshift vectors
    size_t vec_stride;                    // bytes between consecutive p_i
    int max_grid;                         // doubles reserved at `partials`
};

inline int cg_max_grid(const stag_ctx *ctx) {
    const int persistent = ctx->num_sms * 32;
    const int one_per_tile = (ctx->g.Vh + 63) / 64;
    return persistent > one_per_tile ? persistent : one_per_tile;
}

inline size_t cg_workspace_layout(const stag_ctx *ctx, int prec, int nshift, CgLayout *out) {
    CgLayout l;
    const size_t vec = align256((size_t)ctx->g.Vh * vec_bytes_per_site(prec));
    size_t off = 0;
    l.state = off;    off += align256(sizeof(CgState));
    l.max_grid = cg_max_grid(ctx);
    l.partials = off; off += align256(sizeof(double) * (size_t)l.max_grid);
    l.flags = off;    off += kPersistFlagBytes;      // persistent kernel: one epoch word per CTA and 128-byte line
    l.r = off;        off += vec;
    l.q = off;        off += vec;
    l.w = off;        off += vec;
    l.p = off;        off += vec * (size_t)nshift;
    l.vec_stride = vec;
    if (out) *out = l;
    return off;
}

#ifdef __CUDACC__
// ---- a4: scalar recurrences, run by warp 0 of the last CTA of the two reducing kernels ----------
// (lane i owns shift i; `total` is the grid-wide sum, valid in every lane of warp 0.)

// after <p,q>:  alpha = rr / <p,q>;  theta_new_i, alpha_i   (C4 / A15)
__device__ __forceinline__ void cg_scalars_after_pq(CgState *s, double pq) {
    const int lane = threadIdx.x & 31;
    const double alpha = s->rr / pq;
    if (!(pq > 0.0) || !isfinite(alpha)) {            // breakdown: no update this iteration
        if (lane == 0) { s->pq = pq; s->breakdown = 1; s->done = 2; }
        return;
    }
    const double k = alpha * s->beta_old / s->alpha_old;
    __syncwarp();
    if (lane < s->nshift) {
        if (s->active[lane] == 2) s->active[lane] = 0;     // frozen at the previous iteration
        const double th = 1.0 / ((1.0 + s->delta[lane] * alpha) + k * (1.0 - s->theta[lane]));
        s->theta_new[lane] = th;
        s->alpha_i[lane] = alpha * th;
    }
    if (lane == 0) { s->pq = pq; s->alpha = alpha; }
}

// after <r,r>:  beta, beta_i, zeta_i; convergence latch, freezing, fp32 stagnation watch
__device__ __forceinline__ void cg_scalars_after_rr(CgState *s, double rr_new) {
    const int lane = threadIdx.x & 31;
    const double beta = rr_new / s->rr;
    const double rel = sqrt(rr_new / s->bb);
    const int iter = s->iter + 1;
    __syncwarp();                                // all lanes hold the old rr/bb/iter before lane 0 writes
    if (lane < s->nshift) {
        const double th = s->theta_new[lane];
        const double z = s->zeta[lane] * th;
        s->beta_i[lane] = beta * th * th;
        s->zeta[lane] = z;
        s->theta[lane] = th;
        if (s->active[lane] == 1) {
            s->resid_shift[lane] = z * rel;
            s->iters_shift[lane] = iter;
            if (s->freeze && lane != s->base && z * rel <= 0.1 * s->stop) s->active[lane] = 2;
        }
    }
    if (lane == 0) {
        s->alpha_old = s->alpha;
        s->beta_old = beta;
        s->beta = beta;
        s->rr = rr_new;
        s->iter = iter;
        int done = 0;
        if (rel <= s->stop) { s->converged = 1; done = 1; }
        else if (iter >= s->maxiter) done = 1;
        else if (!(rr_new == rr_new)) { s->breakdown = 1; done = 1; }
        else if (s->fp32) {                      // reading A9: stop when ||r|| stops falling
            if (rr_new < s->best_rr) { s->best_rr = rr_new; s->since_best = 0; }
            else if (++s->since_best >= 50) { s->stagnated = 1; done = 1; }
        }
        if (done) s->done = 1;                   // this iteration's x/p update still runs
    }
}
#endif

// implemented in stag_dslash.cu
int dslash_dispatch(const stag_ctx *ctx, const void *packed, int prec, int recon, const void *in,
                    void *out, int par, void *stream);
// D_eo fused with q = c0 p - D_eo w and the partial sums of Re<p,q>; last CTA finishes a4.
int dslash_eo_fused_dispatch(const stag_ctx *ctx, const void *packed, int prec, int recon,
                             const void *w_odd, const void *p_even, void *q_even,
                             CgState *state, double *partials, void *stream);
// D_oe inside CG: same kernel as stag_dslash_oe but returns at once when state->done != 0.
int dslash_oe_cg_dispatch(const stag_ctx *ctx, const void *packed, int prec, int recon,
                          const void *p_even, void *w_odd, CgState *state, void *stream);

// implemented in stag_cg_persist.cu: nrhs independent sources in one persistent launch.  src_sigma /
// src_stop (nullable): N2 polish — nshift must be 1 and source s solves (A + src_sigma[s]) e = b_s to
// src_stop[s]; a source whose src_stop[s] >= 1 returns e = 0 after 0 iterations.
int block_solve(const stag_ctx *ctx, Slot &slot, const void *packed, int prec, int recon, int nrhs, const void *b_even,
                double mass, int nshift, const double *host_shifts, const double *src_sigma,
                const double *src_stop, const double *host_residues, double residue0, double stop,
                int maxiter, void *x_even, void *y_even, void *workspace, stag_cg_info *info,
                cudaStream_t st);

// stag_mshift_cg on a staging slot the caller has leased (stag_cg.cu)
int mshift_cg_impl(const stag_ctx *ctx, Slot &slot, const void *packed, int prec, int recon, const void *b_even,
                   double mass, int nshift, const double *host_shifts, const double *host_residues, double residue0,
                   double stop, int maxiter, void *x_even, void *y_even, void *workspace, stag_cg_info *info,
                   void *stream);

// implemented in stag_cg_persist.cu: the whole solve as one cooperative kernel (small lattices)
bool cg_persistent_fits(const stag_ctx *ctx, int prec);
int cg_persistent_dispatch(const stag_ctx *ctx, const void *packed, int prec, int recon,
                           const void *b, int nshift, const double *host_shifts, void *x, size_t x_stride,
                           void *y, char *ws, const CgLayout &lay, cudaStream_t st);

}  // namespace stag
