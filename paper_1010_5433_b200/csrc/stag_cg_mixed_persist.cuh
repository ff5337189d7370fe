// stag_cg_mixed_persist.cuh — N2: the multi-shift CG in MIXED precision with residual replacement, one
// persistent cooperative kernel (single source).
//
//   PAPER.md:127  "the residual replacement strategy: sometimes the true residual is explicitly calculated
//                 in double precision and the algorithm is restarted ... using almost always single precision"
//   PAPER.md:129  a shifted solver cannot be RESTARTED from a non-zero x — but nothing forbids REPLACING
//                 the recursive residual of the base system by the true one while the recurrences run on
//                 (van der Vorst & Ye, the paper's ref [7]): x is never reset, the directions p_i carry on.
//
// Storage: hopping matrices fp32 for every iteration (the 92 % of the stencil's bytes), r, q, w, p_i fp32,
// the solutions x_i fp64 with fp64 coefficients (x_i += alpha_i p_i adds an fp32 vector to an fp64 one, so the
// solutions do not inherit fp32's storage rounding), all reductions and scalars fp64.  Whenever the recursive
// ||r||^2 has fallen by ru_delta^2 since the last replacement, and once more when it reaches stop, the true
// residual r = b - (A + sigma_0) x_base is computed with the fp64 matrices and fp64 vectors (two extra stencil
// phases), written over r, and its norm over rr.  Convergence is declared on that TRUE residual only.  The
// shifted systems ride on the base system (their residuals are taken to be zeta_i r, as in the fp64 solver);
// what accuracy they reach is measured afterwards by stag_mshift_cg_mixed's fp64 polish, which leaves shifts
// that are already at stop untouched.
// One grid-wide reduction per iteration, as in stag_cg_persist_sr.cuh: <p,q>, <r,q>, <q,q> and <r,r> of the current
// r together, ||r - alpha q||^2 by the one-step formula, phases C and D merged (0.1075 -> 0.1024 s for the
// single-shift solve at 32^3 x 8).
#pragma once

#include "stag_cg_persist.cuh"

namespace stag {

struct MixedArgs {
    const char *W_lo, *W_hi;   // packed hopping matrices: fp32 and fp64 or split-double (same recon)
    const char *b64;           // source, fp64 device format
    char *w32, *w64;           // odd-site scratch: fp32 (every iteration), fp64 (residual replacement)
    char *r_g, *q_g;           // global homes of r, q (fp32) when not resident
    char *p;                   // fp32 search directions [nshift], stride p_stride
    size_t p_stride;
    char *x;                   // fp64 solutions [nshift], stride x_stride
    size_t x_stride;
    CgState *state;
    double *partials;          // 2 * gridDim.x doubles
    int S;
    int res_r, res_q, res_p;
    double ru_delta;           // replace when ||r|| has fallen by this factor since the last replacement
};

struct MixedExtra {            // scalars the mixed kernel needs on top of Scalars<float>
    double ca64[STAG_MAX_SHIFTS];   // alpha_i of the live shifts in fp64 (for the fp64 x_i)
    double a_base64, c0_64, rr_ru;
    int ru, verify, nru, last;
    int stall;                      // consecutive replacements whose TRUE residual fell by less than 10 %
};

// SPLIT_HI: W_hi is a split-double buffer (N3) — typically the very buffer whose b planes are W_lo.
template <int RECON, int NT, bool SPLIT_HI>
__global__ void __launch_bounds__(NT, 1)
cg_mixed_kernel(const Geom g, const MixedArgs a) {
    typedef float T;
    extern __shared__ __align__(16) unsigned char dyn[];
    __shared__ Scalars<T> sc1[1];
    __shared__ MixedExtra mx;
    __shared__ double red[(NT / 32) * 4];
    __shared__ double tot[4];                        // <p,q>, <r,q>, <q,q>, <r,r> of the current r
    Scalars<T> &c = sc1[0];

    const int tid = threadIdx.x, G = gridDim.x, Vh = g.Vh, S = a.S;
    const int e0 = min(Vh, (int)blockIdx.x * S), ns = min(Vh, e0 + S) - e0;
    unsigned int *bar = &a.state->ticket;
    unsigned int epoch = 0;
    double *part_pq = a.partials, *part_rr = a.partials + 3 * (size_t)G;    // [4][G]: <p,q>, <r,q>, <q,q>, <r,r>
    const CgState *st = a.state;
    const int nshift = st->nshift, base = st->base, maxiter = st->maxiter, freeze = st->freeze;
    char *p_base = a.p + (size_t)base * a.p_stride;
    char *x_base = a.x + (size_t)base * a.x_stride;

    Slice<T> r_s, q_s, p_s;
    {
        const size_t slice = (size_t)S * 6 * sizeof(T);
        unsigned char *d = dyn;
        r_s.res = a.res_r != 0; r_s.g = a.r_g; r_s.gstride = 0;
        if (r_s.res) { r_s.s.init(d, S); d += slice; }
        q_s.res = a.res_q != 0; q_s.g = a.q_g; q_s.gstride = 0;
        if (q_s.res) { q_s.s.init(d, S); d += slice; }
        p_s.res = a.res_p != 0; p_s.g = p_base; p_s.gstride = 0;
        if (p_s.res) { p_s.s.init(d, S); d += slice; }
    }

    // ---- start: x_i = 0 (fp64), r = p_i = (float) b, bb = <b,b> in fp64 ---------------------------------
    if (tid < 32) {
        const int i = tid;
        const bool on = i < nshift;
        c.delta[i] = on ? st->delta[i] : 0.0;
        c.zeta[i] = 1.0; c.theta[i] = 1.0; c.theta_new[i] = 1.0; c.resid[i] = 1.0;
        c.active[i] = on ? 1 : 0;
        c.iters_shift[i] = 0;
    }
    {
        double acc = 0.0;
        for (int ls = tid; ls < ns; ls += NT) {
            const int e = e0 + ls;
            double bv[6], z[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
            T v[6];
            load_vec<true>(a.b64, Vh, e, bv);
#pragma unroll
            for (int k = 0; k < 6; ++k) { acc += bv[k] * bv[k]; v[k] = (T)bv[k]; }
            r_s.store(ls, 0, Vh, e, v);
            if (p_s.res) p_s.s.store(ls, v);
            for (int i = 0; i < nshift; ++i) {
                if (i == base) store_vec(p_base, Vh, e, v);
                else store_vec_cs(a.p + (size_t)i * a.p_stride, Vh, e, v);
                store_vec_cs(a.x + (size_t)i * a.x_stride, Vh, e, z);
            }
        }
        cta_partials_stream<NT, 1>(acc, red, part_rr + blockIdx.x, G);
    }
    grid_arrive(bar);
    grid_wait(bar, ++epoch * G);
    if (tid < 32) {
        const double bb = grid_total(part_rr, G);
        if (tid == 0) {
            c.c0 = (T)st->c0; c.stop = st->stop;
            c.bb = bb; c.rr = bb; c.best_rr = bb; c.alpha = 0.0; c.alpha_old = 1.0; c.beta_old = 0.0;
            c.pq = 0.0; c.iter = 0; c.done = 0; c.converged = 0; c.breakdown = 0; c.stagnated = 0;
            c.since_best = 0; c.nlive = 0;
            mx.c0_64 = st->c0; mx.rr_ru = bb; mx.ru = 0; mx.verify = 0; mx.nru = 0; mx.last = 0; mx.stall = 0;
            if (!(bb > 0.0)) { c.converged = (bb == 0.0); c.breakdown = !(bb == 0.0); c.done = 2; }
            else if (maxiter <= 0) c.done = 2;
        }
    }
    __syncthreads();

    const char *pin[1] = {p_base};
    const char *win[1] = {a.w32};
    const char *xin64[1] = {x_base};
    const char *win64[1] = {a.w64};

    while (c.done == 0) {
        // ---- residual replacement: r = b - (A + sigma_0) x_base in fp64, rr = <r,r> --------
        if (mx.ru) {
            for (int ls = tid; ls < ns; ls += NT) {
                double acc[1][6];
                dslash_site_multi<double, RECON, 1, false, SPLIT_HI>(g, a.W_hi, xin64, 1u, 1, e0 + ls, acc);
                store_vec(a.w64, Vh, e0 + ls, acc[0]);
            }
            grid_arrive(bar);
            grid_wait(bar, ++epoch * G);
            double acc2 = 0.0;
            const double c0 = mx.c0_64;
            for (int ls = tid; ls < ns; ls += NT) {
                const int e = e0 + ls;
                double t[1][6], xv[6], bv[6];
                T rv[6];
                dslash_site_multi<double, RECON, 1, false, SPLIT_HI>(g, a.W_hi, win64, 1u, 0, e, t);
                load_vec<false>(x_base, Vh, e, xv);
                load_vec<true>(a.b64, Vh, e, bv);
#pragma unroll
                for (int k = 0; k < 6; ++k) {
                    const double r64 = (bv[k] - c0 * xv[k]) + t[0][k];
                    acc2 += r64 * r64;
                    rv[k] = (T)r64;
                }
                r_s.store(ls, 0, Vh, e, rv);
            }
            cta_partials_stream<NT, 1>(acc2, red, part_rr + blockIdx.x, G);
            grid_arrive(bar);
            grid_wait(bar, ++epoch * G);
            if (tid < 32) {
                const double rr_true = grid_total(part_rr, G);
                if (tid == 0) {
                    // stagnation latch (reading A9 for this kernel): the recursive residual keeps falling and keeps
                    // triggering replacements, but if the TRUE one has stopped following it — an unreachable stop, or
                    // the fp32 rounding of the matrices — three replacements in a row that gain less than 10 % end
                    // the run with stagnated = 1 and the polish takes over
                    if (rr_true > 0.81 * mx.rr_ru) ++mx.stall; else mx.stall = 0;
                    c.rr = rr_true; mx.rr_ru = rr_true; mx.ru = 0; ++mx.nru;
                    c.best_rr = rr_true; c.since_best = 0;
                    if (mx.verify) {
                        mx.verify = 0;
                        if (sqrt(rr_true / c.bb) <= c.stop) { c.converged = 1; c.done = 2; }
                    }
                    if (c.done == 0 && mx.stall >= 3) { c.stagnated = 1; c.done = 2; }
                    if (mx.last || !(rr_true == rr_true)) { if (!(rr_true == rr_true)) c.breakdown = 1; c.done = 2; }
                }
            }
            __syncthreads();
            if (c.done != 0) break;
        }

        // ---- phase A (a2): w = D_oe p_base, fp32 matrices ---------------------------------------------------
        for (int ls = tid; ls < ns; ls += NT) {
            T acc[1][6];
            dslash_site_multi<T, RECON, 1, false>(g, a.W_lo, pin, 1u, 1, e0 + ls, acc);
            store_vec(a.w32, Vh, e0 + ls, acc[0]);
        }
        grid_arrive(bar);
        grid_wait(bar, ++epoch * G);

        // ---- phase B (a3): q = c0 p - D_eo w, partial Re<p,q>; then the partials of <r,q>, <q,q> and <r,r> of the
        // current r, so that ONE grid-wide reduction gives alpha AND ||r - alpha q||^2 = rr - 2 alpha <r,q> + alpha^2
        // <q,q> (hence beta): see stag_cg_persist_sr.cuh.  rr is recomputed from the vector r in every iteration.
        {
            double dot[4] = {0.0, 0.0, 0.0, 0.0};
            const T c0 = c.c0;
            for (int ls = tid; ls < ns; ls += NT) {
                const int e = e0 + ls;
                T acc[1][6], pv[6];
                dslash_site_multi<T, RECON, 1, false>(g, a.W_lo, win, 1u, 0, e, acc);
                p_s.load(ls, 0, Vh, e, pv);
#pragma unroll
                for (int k = 0; k < 6; ++k) {
                    acc[0][k] = c0 * pv[k] - acc[0][k];
                    dot[0] += (double)pv[k] * (double)acc[0][k];
                }
                q_s.store(ls, 0, Vh, e, acc[0]);
            }
            for (int ls = tid; ls < ns; ls += NT) {        // a thread re-reads the q it wrote
                const int e = e0 + ls;
                T rv[6], qv[6];
                r_s.load(ls, 0, Vh, e, rv);
                q_s.load(ls, 0, Vh, e, qv);
#pragma unroll
                for (int k = 0; k < 6; ++k) {
                    dot[1] += (double)rv[k] * (double)qv[k];
                    dot[2] += (double)qv[k] * (double)qv[k];
                    dot[3] += (double)rv[k] * (double)rv[k];
                }
            }
            cta_partials_all<NT, 4>(dot, red, part_pq + blockIdx.x, G);
        }
        grid_arrive(bar);
        grid_wait(bar, ++epoch * G);
        if (tid < 128) {
            const double t = grid_total(part_pq + (size_t)(tid >> 5) * G, G);
            if ((tid & 31) == 0) tot[tid >> 5] = t;
        }
        __syncthreads();

        // ---- phase CD (a4, a5, a7, a6): alpha, beta, theta_i, zeta_i, replacement / verification trigger;
        // r -= alpha q;  x_i (fp64), p_i (fp32) --------------------------------------------------------------
        if (tid < 32) {
            const int i = tid;
            const double pq = tot[0], rq = tot[1], qq = tot[2], rr = tot[3];
            const double alpha = rr / pq;
            const bool bad = !(pq > 0.0) || !isfinite(alpha);
            double rr_new = fma(alpha, fma(alpha, qq, -2.0 * rq), rr);     // || r - alpha q ||^2
            if (!bad && !(rr_new > 0.0) && rr_new == rr_new) rr_new = 0.0;
            const double kk = alpha * c.beta_old / c.alpha_old;
            const double beta = rr_new / rr;
            const double rel = sqrt(rr_new / c.bb);
            const int iter = c.iter + 1;
            bool live = false;
            double th = 1.0, z = 1.0;
            __syncwarp();
            if (bad) {
                if (i == 0) { c.pq = pq; c.breakdown = 1; c.done = 2; }
            } else {
            if (i < nshift) {
                if (c.active[i] == 2) c.active[i] = 0;
                th = 1.0 / ((1.0 + c.delta[i] * alpha) + kk * (1.0 - c.theta[i]));
                c.theta_new[i] = th;
                z = c.zeta[i] * th;
                c.zeta[i] = z;
                c.theta[i] = th;
                if (c.active[i] != 0) {
                    live = true;
                    if (c.active[i] == 1) {
                        c.resid[i] = z * rel;
                        c.iters_shift[i] = iter;
                        if (freeze && i != base && z * rel <= 0.1 * c.stop) c.active[i] = 2;
                    }
                }
            }
            const unsigned m = __ballot_sync(0xffffffffu, live && i != base);
            if (live && i != base) {
                const int j = __popc(m & ((1u << i) - 1u));
                c.live[j] = i;
                mx.ca64[j] = alpha * th;
                c.cz[j] = (T)z;
                c.cb[j] = (T)(beta * th * th);
            }
            if (i == base) { mx.a_base64 = alpha * th; c.z_base = (T)z; c.b_base = (T)(beta * th * th); }
            if (i == 0) {
                c.pq = pq;
                c.alpha = alpha;
                c.nlive = __popc(m);
                c.alpha_old = alpha;
                c.beta_old = beta;
                c.rr = rr_new;
                c.iter = iter;
                if (!(rr_new == rr_new)) { c.breakdown = 1; mx.ru = 1; mx.last = 1; }
                else if (rel <= c.stop) { mx.ru = 1; mx.verify = 1; }              // convergence only on the TRUE residual
                else if (rr_new < a.ru_delta * a.ru_delta * mx.rr_ru) mx.ru = 1;
                else if (rr_new < c.best_rr) { c.best_rr = rr_new; c.since_best = 0; }
                else if (++c.since_best >= 50) { mx.ru = 1; c.since_best = 0; }   // reading A9: the recursive residual has
                                                                                 // stopped falling too — look at the true one
                if (iter >= maxiter) { mx.ru = 1; mx.verify = 1; mx.last = 1; }
            }
            }
        }
        __syncthreads();
        if (c.done != 0) break;
        {
            const double ab = mx.a_base64;
            const T na = (T)(-c.alpha), zb = c.z_base, bb_ = c.b_base;
            for (int ls = tid; ls < ns; ls += NT) {
                const int e = e0 + ls;
                T rv[6], qv[6], pv[6];
                double xv[6];
                load_vec_cs(x_base, Vh, e, xv);
                r_s.load(ls, 0, Vh, e, rv);
                q_s.load(ls, 0, Vh, e, qv);
                p_s.load(ls, 0, Vh, e, pv);
#pragma unroll
                for (int k = 0; k < 6; ++k) {
                    rv[k] = fma(na, qv[k], rv[k]);
                    xv[k] = fma(ab, (double)pv[k], xv[k]);
                    pv[k] = fma(zb, rv[k], bb_ * pv[k]);
                }
                r_s.store(ls, 0, Vh, e, rv);
                store_vec(x_base, Vh, e, xv);              // re-read by the residual replacement: keep it cached
                if (p_s.res) p_s.s.store(ls, pv);
                store_vec(p_base, Vh, e, pv);
            }
        }
        grid_arrive(bar);
        {
            const int n = c.nlive;
            for (int ls = tid; ls < ns; ls += NT) {
                const int e = e0 + ls;
                T rv[6];
                r_s.load(ls, 0, Vh, e, rv);
#pragma unroll 2
                for (int j = 0; j < n; ++j) {
                    char *xp = a.x + (size_t)c.live[j] * a.x_stride;
                    char *pp = a.p + (size_t)c.live[j] * a.p_stride;
                    const double aj = mx.ca64[j];
                    const T zj = c.cz[j], bj = c.cb[j];
                    T pv[6];
                    double xv[6];
                    load_vec_cs(pp, Vh, e, pv);
                    load_vec_cs(xp, Vh, e, xv);
#pragma unroll
                    for (int k = 0; k < 6; ++k) {
                        xv[k] = fma(aj, (double)pv[k], xv[k]);
                        pv[k] = fma(zj, rv[k], bj * pv[k]);
                    }
                    store_vec_cs(xp, Vh, e, xv);
                    store_vec_cs(pp, Vh, e, pv);
                }
            }
        }
        grid_wait(bar, ++epoch * G);
    }

    // ---- read-back state ---------------------------------------------------------------------------------
    if (blockIdx.x == 0 && tid < 32) {
        const int i = tid;
        CgState *o = a.state;
        if (i < nshift) {
            o->zeta[i] = c.zeta[i];
            o->theta[i] = c.theta[i];
            o->resid_shift[i] = c.resid[i];
            o->iters_shift[i] = c.iters_shift[i];
            o->active[i] = c.active[i];
        }
        if (i == 0) {
            o->bb = c.bb; o->rr = c.rr; o->pq = c.pq; o->alpha = c.alpha;
            o->iter = c.iter; o->converged = c.converged; o->breakdown = c.breakdown;
            o->stagnated = c.stagnated; o->replacements = mx.nru; o->done = 2;
        }
    }
}

template <int RECON, int NT, bool SPLIT_HI>
int launch_mixed(const stag_ctx *ctx, const MixedArgs &args, cudaStream_t st) {
    const Geom &g = ctx->g;
    int grid = ctx->num_sms;
    const int tiles = (g.Vh + 31) / 32;
    if (grid > tiles) grid = tiles;
    MixedArgs a = args;
    a.S = sites_per_cta(g.Vh, grid);
    const size_t slice = (size_t)a.S * 6 * sizeof(float);
    int fit = (int)(kMaxDynSmem / slice);
    if (fit > ctx->opt.cg_resident_slices) fit = ctx->opt.cg_resident_slices;
    a.res_r = fit >= 1; a.res_q = fit >= 2; a.res_p = fit >= 3;
    const size_t smem = slice * (size_t)(a.res_r + a.res_q + a.res_p);
    auto kern = cg_mixed_kernel<RECON, NT, SPLIT_HI>;
    STAG_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int per_sm = 0;
    STAG_CUDA_OK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, NT, smem));
    if (per_sm < 1) return STAG_ERR_UNSUPPORTED;
    Geom gg = g;
    void *params[] = {(void *)&gg, (void *)&a};
    log_kernel(ctx, (const void *)kern);
    STAG_CUDA_OK(cudaLaunchCooperativeKernel((const void *)kern, dim3(grid), dim3(NT), params, smem, st));
    return STAG_OK;
}

}  // namespace stag
