// stag_cg_persist_block.cuh — the persistent multi-shift CG kernel for R >= 2 independent sources (N1).
//
// This is the round-1 form of the kernel in stag_cg_persist.cuh: grid barriers between the four phases, the shift
// updates of an iteration done at once between the arrive and the wait of the last barrier, x_i / p_i streamed with
// ld.cs / st.cs.  The single-source kernel has since moved on (deferred updates worked off at the sync points,
// neighbour flags, L2 keep set); with four sources per thread those changes were measured and LOSE: the stencil
// phases are register-bound (24 fp64 accumulators + one matrix per thread), every extra live value spills inside
// them, and the extra bookkeeping took 32^3 x 8, 4 sources x 16 shifts from 184 to 203-260 us per block iteration
// (profiles/README.md, round 2, "N1 block kernel").  So the multi-source path keeps this form.
//
// Phases, residency, scalars and per-source latches: see the header of stag_cg_persist.cuh (the description of
// R > 1 there applies unchanged).
#pragma once

#include "stag_cg_persist.cuh"

namespace stag {

template <typename T, int RECON, int NT, int R, bool SPLIT = false>
__global__ void __launch_bounds__(NT, 1)
cg_persistent_block_kernel(const Geom g, const PersistArgs a) {
    extern __shared__ __align__(16) unsigned char dyn[];
    __shared__ Scalars<T> sc[R];
    __shared__ double red[(NT / 32) * R];
    __shared__ int n_running;

    constexpr int LS = NT / R;                       // streaming phases: sites per pass and source
    const int tid = threadIdx.x, G = gridDim.x, Vh = g.Vh, S = a.S;
    const int rhs = tid / LS, l0 = tid % LS;         // streaming phases: this thread's source (warp-uniform)
    // balanced contiguous ranges of 32-site tiles (no idle SM), computed once by thread 0
    __shared__ int s_range[2];
    if (tid == 0) {
        const int tiles = (Vh + 31) >> 5;
        s_range[0] = min(Vh, cta_first_tile(blockIdx.x, tiles, G) << 5);
        s_range[1] = min(Vh, cta_first_tile(blockIdx.x + 1, tiles, G) << 5);
    }
    __syncthreads();
    const int e0 = s_range[0], ns = s_range[1] - e0;
    unsigned int *bar = &a.state->ticket;
    unsigned int epoch = 0;
    double *part_pq = a.partials, *part_rr = a.partials + (size_t)R * G;

    CgState *st = reinterpret_cast<CgState *>(reinterpret_cast<char *>(a.state) + (size_t)rhs * a.state_stride);
    const int nshift = a.state->nshift, base = a.state->base, maxiter = a.state->maxiter;   // same for every source
    const int freeze = a.state->freeze, fp32 = a.state->fp32;

    const char *b_r = a.b + (size_t)rhs * a.b_stride;
    char *p_r = a.p + (size_t)rhs * nshift * a.p_stride;
    char *x_r = a.x + (size_t)rhs * nshift * a.x_stride;
    char *p_base = p_r + (size_t)base * a.p_stride;
    char *x_base = x_r + (size_t)base * a.x_stride;
    const size_t pb_stride = (size_t)nshift * a.p_stride;       // between the sources' p_base
    char *p_base0 = a.p + (size_t)base * a.p_stride;            // p_base of source 0

    Slice<T> r_s, q_s, p_s;
    {
        const size_t slice = (size_t)S * R * 6 * sizeof(T);
        unsigned char *d = dyn;
        r_s.res = a.res_r != 0; r_s.g = a.r_g; r_s.gstride = a.vec_stride;
        if (r_s.res) { r_s.s.init(d, S * R); d += slice; }
        q_s.res = a.res_q != 0; q_s.g = a.q_g; q_s.gstride = a.vec_stride;
        if (q_s.res) { q_s.s.init(d, S * R); d += slice; }
        p_s.res = a.res_p != 0; p_s.g = p_base0; p_s.gstride = pb_stride;
        if (p_s.res) { p_s.s.init(d, S * R); d += slice; }
    }
    const bool present = rhs < a.nrhs;

    // ---- start: x_i = 0, r = p_i = b, bb = <b,b> ---------------------------------------------------
    if (tid < 32 * R && (tid & 31) < STAG_MAX_SHIFTS) {
        const int s = tid >> 5, i = tid & 31;
        const CgState *ss = reinterpret_cast<const CgState *>(reinterpret_cast<const char *>(a.state) + (size_t)s * a.state_stride);
        const bool on = i < nshift && s < a.nrhs;
        sc[s].delta[i] = on ? ss->delta[i] : 0.0;
        sc[s].zeta[i] = 1.0; sc[s].theta[i] = 1.0; sc[s].theta_new[i] = 1.0;
        sc[s].resid[i] = 1.0;
        sc[s].active[i] = on ? 1 : 0;
        sc[s].iters_shift[i] = 0;
    }
    {
        double acc = 0.0;
        if (present)
            for (int ls = l0; ls < ns; ls += LS) {
                const int e = e0 + ls, slot = rhs * S + ls;
                T v[6], z[6] = {T(0), T(0), T(0), T(0), T(0), T(0)};
                load_vec<true>(b_r, Vh, e, v);
#pragma unroll
                for (int k = 0; k < 6; ++k) acc += (double)v[k] * (double)v[k];
                r_s.store(slot, rhs, Vh, e, v);
                if (p_s.res) p_s.s.store(slot, v);
                for (int i = 0; i < nshift; ++i) {
                    if (i == base) store_vec(p_base, Vh, e, v);
                    else store_vec_cs(p_r + (size_t)i * a.p_stride, Vh, e, v);
                    store_vec_cs(x_r + (size_t)i * a.x_stride, Vh, e, z);
                }
            }
        cta_partials_stream<NT, R>(acc, red, part_rr + blockIdx.x, G);
    }
    grid_arrive(bar);
    grid_wait(bar, ++epoch * G);
    if (tid < 32 * R) {
        const int s = tid >> 5;
        const double bb = grid_total(part_rr + (size_t)s * G, G);
        if ((tid & 31) == 0) {
            Scalars<T> &c = sc[s];
            const CgState *ss = reinterpret_cast<const CgState *>(reinterpret_cast<const char *>(a.state) + (size_t)min(s, a.nrhs - 1) * a.state_stride);
            c.c0 = (T)ss->c0; c.stop = ss->stop;
            c.bb = bb; c.rr = bb; c.best_rr = bb; c.alpha = 0.0; c.alpha_old = 1.0; c.beta_old = 0.0;
            c.pq = 0.0; c.iter = 0; c.done = 0; c.converged = 0; c.breakdown = 0; c.stagnated = 0;
            c.since_best = 0; c.nlive = 0;
            if (s >= a.nrhs) c.done = 2;
            else if (!(bb > 0.0)) { c.converged = (bb == 0.0); c.breakdown = !(bb == 0.0); c.done = 2; }
            else if (ss->zero_ok && ss->stop >= 1.0) { c.converged = 1; c.done = 2; }   // polish: x = 0 already meets it
            else if (maxiter <= 0) c.done = 2;
        }
    }
    __syncthreads();
    if (tid == 0) {
        int n = 0;
        for (int s = 0; s < R; ++s) n += sc[s].done == 0;
        n_running = n;
    }
    __syncthreads();

    // stencil phases: the R sources' input / output vectors
    const char *pin[R];
    const char *win[R];
    char *wout[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        pin[r] = p_base0 + (size_t)r * pb_stride;
        win[r] = a.w + (size_t)r * a.vec_stride;
        wout[r] = a.w + (size_t)r * a.vec_stride;
    }

    // ---- iterations -----------------------------------------------------------------------------------
    STAG_T_DECL
    while (n_running > 0) {
        const bool act = sc[rhs].done == 0;          // streaming phases: this thread's source is still iterating
        unsigned mask = 0;                           // stencil phases: the sources still iterating
#pragma unroll
        for (int r = 0; r < R; ++r) mask |= (sc[r].done == 0 ? 1u : 0u) << r;

        // phase A (a2): w = D_oe p_base on this CTA's odd sites
        for (int ls = tid; ls < ns; ls += NT) {
            T acc[R][6];
            dslash_site_multi<T, RECON, R, false, SPLIT>(g, a.W, pin, mask, 1, e0 + ls, acc);
#pragma unroll
            for (int r = 0; r < R; ++r)
                if (R == 1 || ((mask >> r) & 1u)) store_vec(wout[r], Vh, e0 + ls, acc[r]);
        }
        STAG_TICK(0);
        grid_arrive(bar);
        grid_wait(bar, ++epoch * G);
        STAG_TICK(1);

        // phase B (a3): q = c0 p - D_eo w, partial Re<p,q>
        {
            double dot[R];
            T c0[R];
#pragma unroll
            for (int r = 0; r < R; ++r) { dot[r] = 0.0; c0[r] = sc[r].c0; }
            for (int ls = tid; ls < ns; ls += NT) {
                const int e = e0 + ls;
                T acc[R][6];
                dslash_site_multi<T, RECON, R, false, SPLIT>(g, a.W, win, mask, 0, e, acc);
#pragma unroll
                for (int r = 0; r < R; ++r)
                    if (R == 1 || ((mask >> r) & 1u)) {
                        T pv[6];
                        p_s.load(r * S + ls, r, Vh, e, pv);
#pragma unroll
                        for (int k = 0; k < 6; ++k) {
                            acc[r][k] = c0[r] * pv[k] - acc[r][k];
                            dot[r] += (double)pv[k] * (double)acc[r][k];
                        }
                        q_s.store(r * S + ls, r, Vh, e, acc[r]);
                    }
            }
            cta_partials_all<NT, R>(dot, red, part_pq + blockIdx.x, G);
        }
        STAG_TICK(2);
        grid_arrive(bar);
        grid_wait(bar, ++epoch * G);
        STAG_TICK(3);

        // phase C (a4 after <p,q>, then a5): alpha, theta_new_i;  r -= alpha q;  partial <r,r>
        if (tid < 32 * R) {
            const int s = tid >> 5, i = tid & 31;
            Scalars<T> &c = sc[s];
            if (c.done == 0) {
                const double pq = grid_total(part_pq + (size_t)s * G, G);
                const double alpha = c.rr / pq;
                const bool bad = !(pq > 0.0) || !isfinite(alpha);
                const double k = alpha * c.beta_old / c.alpha_old;
                __syncwarp();
                if (!bad && i < nshift) {
                    if (c.active[i] == 2) c.active[i] = 0;            // frozen at the previous iteration
                    c.theta_new[i] = 1.0 / ((1.0 + c.delta[i] * alpha) + k * (1.0 - c.theta[i]));
                }
                if (i == 0) {
                    c.pq = pq;
                    if (bad) { c.breakdown = 1; c.done = 2; } else c.alpha = alpha;   // breakdown: no update
                }
            }
        }
        __syncthreads();
        const bool act2 = act && sc[rhs].done == 0;
        {
            double acc = 0.0;
            if (act2) {
                const T na = (T)(-sc[rhs].alpha);
                for (int ls = l0; ls < ns; ls += LS) {
                    const int e = e0 + ls, slot = rhs * S + ls;
                    T rv[6], qv[6];
                    r_s.load(slot, rhs, Vh, e, rv);
                    q_s.load(slot, rhs, Vh, e, qv);
#pragma unroll
                    for (int k = 0; k < 6; ++k) {
                        rv[k] = fma(na, qv[k], rv[k]);
                        acc += (double)rv[k] * (double)rv[k];
                    }
                    r_s.store(slot, rhs, Vh, e, rv);
                }
            }
            cta_partials_stream<NT, R>(acc, red, part_rr + blockIdx.x, G);
        }
        STAG_TICK(4);
        grid_arrive(bar);
        grid_wait(bar, ++epoch * G);
        STAG_TICK(5);

        // phase D (a4 after <r,r>, a7 latch, a6)
        if (tid < 32 * R) {
            const int s = tid >> 5, i = tid & 31;
            Scalars<T> &c = sc[s];
            if (c.done == 0) {
                const double rr_new = grid_total(part_rr + (size_t)s * G, G);
                const double alpha = c.alpha;
                const double beta = rr_new / c.rr;
                const double rel = sqrt(rr_new / c.bb);
                const int iter = c.iter + 1;
                bool live = false;
                double th = 1.0, z = 1.0;
                __syncwarp();
                if (i < nshift) {
                    th = c.theta_new[i];
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
                    c.ca[j] = (T)(alpha * th);
                    c.cz[j] = (T)z;
                    c.cb[j] = (T)(beta * th * th);
                }
                if (i == base) { c.a_base = (T)(alpha * th); c.z_base = (T)z; c.b_base = (T)(beta * th * th); }
                if (i == 0) {
                    c.nlive = __popc(m);
                    c.alpha_old = alpha;
                    c.beta_old = beta;
                    c.rr = rr_new;
                    c.iter = iter;
                    int done = 0;
                    if (rel <= c.stop) { c.converged = 1; done = 1; }
                    else if (iter >= maxiter) done = 1;
                    else if (!(rr_new == rr_new)) { c.breakdown = 1; done = 1; }
                    else if (fp32) {                                     // reading A9
                        if (rr_new < c.best_rr) { c.best_rr = rr_new; c.since_best = 0; }
                        else if (++c.since_best >= 50) { c.stagnated = 1; done = 1; }
                    }
                    c.done = done;
                }
            }
        }
        __syncthreads();
        if (act2) {   // base shift first: its new p is what phase A of the next iteration gathers
            const T ab = sc[rhs].a_base, zb = sc[rhs].z_base, bb_ = sc[rhs].b_base;
            for (int ls = l0; ls < ns; ls += LS) {
                const int e = e0 + ls, slot = rhs * S + ls;
                T rv[6], pv[6], xv[6];
                load_vec_cs(x_base, Vh, e, xv);
                r_s.load(slot, rhs, Vh, e, rv);
                p_s.load(slot, rhs, Vh, e, pv);
#pragma unroll
                for (int k = 0; k < 6; ++k) {
                    xv[k] = fma(ab, pv[k], xv[k]);
                    pv[k] = fma(zb, rv[k], bb_ * pv[k]);
                }
                store_vec_cs(x_base, Vh, e, xv);
                if (p_s.res) p_s.s.store(slot, pv);
                store_vec(p_base, Vh, e, pv);
            }
        }
        STAG_TICK(6);
        grid_arrive(bar);
        if (act2) {
            const Scalars<T> &c = sc[rhs];
            const int n = c.nlive;
            for (int ls = l0; ls < ns; ls += LS) {
                const int e = e0 + ls, slot = rhs * S + ls;
                T rv[6];
                r_s.load(slot, rhs, Vh, e, rv);
#pragma unroll 2
                for (int j = 0; j < n; ++j) {
                    char *xp = x_r + (size_t)c.live[j] * a.x_stride;
                    char *pp = p_r + (size_t)c.live[j] * a.p_stride;
                    const T aj = c.ca[j], zj = c.cz[j], bj = c.cb[j];
                    T pv[6], xv[6];
                    load_vec_cs(pp, Vh, e, pv);
                    load_vec_cs(xp, Vh, e, xv);
#pragma unroll
                    for (int k = 0; k < 6; ++k) {
                        xv[k] = fma(aj, pv[k], xv[k]);
                        pv[k] = fma(zj, rv[k], bj * pv[k]);
                    }
                    store_vec_cs(xp, Vh, e, xv);
                    store_vec_cs(pp, Vh, e, pv);
                }
            }
        }
        __syncthreads();                               // every thread has read sc[].done / coefficients
        if (tid == 0) {
            int n = 0;
            for (int s = 0; s < R; ++s) {
                if (sc[s].done == 1) sc[s].done = 2;   // its last x/p update has just run
                n += sc[s].done == 0;
            }
            n_running = n;
        }
        STAG_TICK(7);
        grid_wait(bar, ++epoch * G);                   // ends with __syncthreads: n_running, done visible
        STAG_TICK(8);
    }

    STAG_T_REPORT(R, sc[0].iter)

    // ---- a7: y = residue0 b + sum_i residues_i x_i (own sites only: no barrier needed) ---------------
    if (a.y && present) {
        char *y_r = a.y + (size_t)rhs * a.x_stride;
        const T r0 = (T)st->residue0;
        for (int ls = l0; ls < ns; ls += LS) {
            const int e = e0 + ls;
            T bv[6], acc[6];
            load_vec<true>(b_r, Vh, e, bv);
#pragma unroll
            for (int k = 0; k < 6; ++k) acc[k] = r0 * bv[k];
            for (int i = 0; i < nshift; ++i) {
                const T ri = (T)st->residues[i];
                T xv[6];
                load_vec_cs(x_r + (size_t)i * a.x_stride, Vh, e, xv);
#pragma unroll
                for (int k = 0; k < 6; ++k) acc[k] = fma(ri, xv[k], acc[k]);
            }
            store_vec(y_r, Vh, e, acc);
        }
    }

    // ---- read-back state (every CTA holds the same scalars; CTA 0 writes them) -------------------------
    if (blockIdx.x == 0 && tid < 32 * R && (tid >> 5) < a.nrhs) {
        const int s = tid >> 5, i = tid & 31;
        CgState *o = reinterpret_cast<CgState *>(reinterpret_cast<char *>(a.state) + (size_t)s * a.state_stride);
        const Scalars<T> &c = sc[s];
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
            o->stagnated = c.stagnated; o->done = 2;
        }
    }
}

template <typename T, int RECON, int NT, int R, bool SPLIT = false>
int launch_persistent_block(const stag_ctx *ctx, const PersistArgs &args, cudaStream_t st) {
    const Geom &g = ctx->g;
    int grid = ctx->num_sms;
    const int tiles = (g.Vh + 31) / 32;
    if (grid > tiles) grid = tiles;
    PersistArgs a = args;
    a.S = 32 * ((tiles + grid - 1) / grid);            // slots of a resident slice = the largest CTA's sites
    // residency: as many of r, q, p (in that order of bytes saved) as fit
    const size_t slice = (size_t)a.S * R * 6 * sizeof(T);
    // cg_resident_slices (test / tuning knob): cap on how many of r, q, p stay in shared memory (default 3)
    int fit = (int)(kMaxDynSmem / slice);
    if (fit > ctx->opt.cg_resident_slices) fit = ctx->opt.cg_resident_slices;
    a.res_r = fit >= 1; a.res_q = fit >= 2; a.res_p = fit >= 3;
    const size_t smem = slice * (size_t)(a.res_r + a.res_q + a.res_p);
    auto kern = cg_persistent_block_kernel<T, RECON, NT, R, SPLIT>;
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

// one explicit-instantiation translation unit per R (parallel compilation); thread counts as in STAG_DEFINE_PERSIST_R
#define STAG_DEFINE_PERSIST_BLOCK_R(RR)                                                                 \
    template <>                                                                                         \
    int cg_persistent_launch_r<RR>(const stag_ctx *ctx, int prec, int recon, const PersistArgs &a,      \
                                   cudaStream_t st) {                                                   \
        int nt = ctx->opt.cg_persistent_threads;                                                        \
        if (nt == 0) nt = prec == STAG_F64 ? 512 : 1024;                                                \
        if (prec == STAG_F64) {                                                                         \
            if (recon == 12)                                                                            \
                return nt == 256 ? launch_persistent_block<double, 12, 256, RR>(ctx, a, st)             \
                                 : launch_persistent_block<double, 12, 512, RR>(ctx, a, st);            \
            return nt == 1024  ? launch_persistent_block<double, 18, 1024, RR>(ctx, a, st)              \
                   : nt == 256 ? launch_persistent_block<double, 18, 256, RR>(ctx, a, st)               \
                               : launch_persistent_block<double, 18, 512, RR>(ctx, a, st);              \
        }                                                                                               \
        if (recon == 18)                                                                                \
            return nt == 1024 ? launch_persistent_block<float, 18, 1024, RR>(ctx, a, st)                \
                              : launch_persistent_block<float, 18, 512, RR>(ctx, a, st);                \
        return nt == 1024 ? launch_persistent_block<float, 12, 1024, RR>(ctx, a, st)                    \
                          : launch_persistent_block<float, 12, 512, RR>(ctx, a, st);                    \
    }

}  // namespace stag
