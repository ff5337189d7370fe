// stag_cg_persist_sr.cuh — the persistent multi-shift CG kernel with ONE grid-wide reduction per iteration
// (single source; rows a2-a7 of SURVEY.md §8(a)).
//
// The kernel of stag_cg_persist.cuh needs two grid-wide reductions per iteration: <p,q> for alpha, then <r,r> of the
// updated residual for beta.  At 32^3 x 8 a grid-wide sync point costs 2.5-3 us of pure latency, and the fixed cost
// of an iteration (two of them, two neighbour syncs, two scalar sections) is what keeps the fp32 and 12-real solves
// below their roofline (DESIGN.md §6 "Where an iteration goes").  Here the second reduction is gone:
//
//   phase B also forms, in a pass over shared memory (r and q are resident), the partials of <r,q>, <q,q> and of
//   <r,r> of the CURRENT r; after the one reduction every CTA has alpha = rr / <p,q> and
//       rr_new = rr - 2 alpha <r,q> + alpha^2 <q,q>        ( = || r - alpha q ||^2 exactly )
//   hence beta = rr_new / rr at once, and phases C and D merge into one: r -= alpha q, x_base += alpha p_base,
//   p_base = r + beta p_base, the other shifts queued — with no sync between.
//
// This is NOT the recurrence that chains rr_new on itself (measured in round 1: its absolute error never decays):
// rr is recomputed from the vector r every iteration, so an error of the formula lives for one iteration only, and
// the formula's own error is a few ulp of rr (its three terms are all of the size of rr).  alpha and beta differ
// from the two-reduction kernel's in the last bits; the iteration counts are the same (tests: +-2 of the oracle's).
// Everything else — tile ranges, neighbour flags after the stencil phases, deferred shift updates worked off at
// the sync points, the L2 keep set, freezing, the latch — is as in stag_cg_persist.cuh.
#pragma once

#include "stag_cg_persist.cuh"

namespace stag {

template <typename T, int RECON, int NT, bool SPLIT = false>
__global__ void __launch_bounds__(NT, 1)
cg_persistent_sr_kernel(const Geom g, const PersistArgs a) {
    extern __shared__ __align__(16) unsigned char dyn[];
    __shared__ Scalars<T> sc1;
    __shared__ double red[(NT / 32) * 4];
    __shared__ double tot[4];                        // <p,q>, <r,q>, <q,q>, <r,r>
    __shared__ int n_running;
    __shared__ unsigned int nb_mask[kMaxPersistGrid / 32];
    __shared__ int nb_list[kMaxPersistGrid];
    __shared__ int nb_n;
    __shared__ unsigned int sync_seen;

    const int tid = threadIdx.x, G = gridDim.x, Vh = g.Vh, S = a.S;
    const int tiles = (Vh + 31) >> 5;
    const int e0 = min(Vh, cta_first_tile(blockIdx.x, tiles, G) << 5);
    const int ns = min(Vh, cta_first_tile(blockIdx.x + 1, tiles, G) << 5) - e0;
    unsigned int *bar = &a.state->ticket;
    // [2][4][G]: two sets of partials, used alternately by iteration parity.  There is only ONE grid-wide barrier per
    // iteration and the syncs after phases CD and A reach a CTA's neighbours only, so a fast CTA can be in phase B of
    // iteration n+1 while a far one has not yet summed the partials of iteration n: it must not overwrite them.  A set
    // is rewritten two iterations later, i.e. after the next grid-wide barrier, at which every reader has arrived.
    // The start's <b,b> sits in slot 3 of set 0, which phase B first writes in iteration 2 (same argument).
    double *part = a.partials;
    Scalars<T> &c = sc1;

    CgState *st = a.state;
    const int nshift = st->nshift, base = st->base, maxiter = st->maxiter;
    const int freeze = st->freeze, fp32 = st->fp32;
    char *p_base = a.p + (size_t)base * a.p_stride;
    char *x_base = a.x + (size_t)base * a.x_stride;
    auto shift_policy = [&](int i) { return ((a.keep_mask >> i) & 1u) ? policy_evict_last() : policy_evict_first(); };

    Slice<T> r_s, q_s, p_s;                          // r and q are resident (the launcher guarantees it); p_base may be
    {
        const size_t slice = (size_t)S * 6 * sizeof(T);
        unsigned char *d = dyn;
        r_s.res = true; r_s.g = a.r_g; r_s.gstride = a.vec_stride; r_s.s.init(d, S); d += slice;
        q_s.res = true; q_s.g = a.q_g; q_s.gstride = a.vec_stride; q_s.s.init(d, S); d += slice;
        p_s.res = a.res_p != 0; p_s.g = p_base; p_s.gstride = 0;
        if (p_s.res) p_s.s.init(d, S);
    }

    // ---- the CTAs that own a neighbour of one of this CTA's sites (either parity) ---------------------
    if (tid < kMaxPersistGrid / 32) nb_mask[tid] = 0u;
    if (tid == 0) { nb_n = 0; sync_seen = 0u; }
    __syncthreads();
    if (a.nbflags) {
        for (int ls = tid; ls < 2 * ns; ls += NT) {
            const int par = ls >= ns, e = e0 + (par ? ls - ns : ls);
            const Site s = site_of(g, e, par);
            const int x[4] = {s.x0, s.x1, s.x2, s.x3};
            int stride = 1;
#pragma unroll
            for (int mu = 0; mu < 4; ++mu) {
                const int Lmu = g.L[mu];
                const int ef = (s.lex + stride - (x[mu] == Lmu - 1 ? Lmu * stride : 0)) >> 1;
                const int eb = (s.lex - stride + (x[mu] == 0 ? Lmu * stride : 0)) >> 1;
                const int of = tile_owner(ef >> 5, tiles, G), ob = tile_owner(eb >> 5, tiles, G);
                if (of != (int)blockIdx.x) atomicOr(&nb_mask[of >> 5], 1u << (of & 31));
                if (ob != (int)blockIdx.x) atomicOr(&nb_mask[ob >> 5], 1u << (ob & 31));
                stride *= Lmu;
            }
        }
        __syncthreads();
    }
    for (int k = tid; k < G; k += NT)
        if (k != (int)blockIdx.x && (!a.nbflags || ((nb_mask[k >> 5] >> (k & 31)) & 1u))) nb_list[atomicAdd(&nb_n, 1)] = k;
    __syncthreads();
    const int nnb = nb_n;

    // ---- start: x_i = 0, r = p_i = b, bb = <b,b> ---------------------------------------------------
    if (tid < 32 && tid < STAG_MAX_SHIFTS) {
        const int i = tid;
        const bool on = i < nshift;
        c.delta[i] = on ? st->delta[i] : 0.0;
        c.zeta[i] = 1.0; c.theta[i] = 1.0; c.theta_new[i] = 1.0;
        c.resid[i] = 1.0;
        c.active[i] = on ? 1 : 0;
        c.iters_shift[i] = 0;
    }
    {
        double acc = 0.0;
        for (int ls = tid; ls < ns; ls += NT) {
            const int e = e0 + ls;
            T v[6], z[6] = {T(0), T(0), T(0), T(0), T(0), T(0)};
            load_vec<true>(a.b, Vh, e, v);
#pragma unroll
            for (int k = 0; k < 6; ++k) acc += (double)v[k] * (double)v[k];
            r_s.s.store(ls, v);
            if (p_s.res) p_s.s.store(ls, v);
            for (int i = 0; i < nshift; ++i) {
                const uint64_t pol = shift_policy(i);
                if (i == base) store_vec(p_base, Vh, e, v);
                else store_vec_pol(a.p + (size_t)i * a.p_stride, Vh, e, v, pol);
                store_vec_pol(a.x + (size_t)i * a.x_stride, Vh, e, z, pol);
            }
        }
        cta_partials_stream<NT, 1>(acc, red, part + 3 * G + blockIdx.x, G);
    }
    grid_arrive(bar);                                  // grid-wide: bb, and every p_base is in place for phase A
    grid_wait(bar, (unsigned)G);
    if (tid < 32) {
        const double bb = grid_total(part + 3 * G, G);
        if (tid == 0) {
            c.c0 = (T)st->c0; c.stop = st->stop;
            c.bb = bb; c.rr = bb; c.best_rr = bb; c.alpha = 0.0; c.alpha_old = 1.0; c.beta_old = 0.0;
            c.pq = 0.0; c.iter = 0; c.done = 0; c.converged = 0; c.breakdown = 0; c.stagnated = 0;
            c.since_best = 0; c.nlive = 0;
            if (!(bb > 0.0)) { c.converged = (bb == 0.0); c.breakdown = !(bb == 0.0); c.done = 2; }
            else if (st->zero_ok && st->stop >= 1.0) { c.converged = 1; c.done = 2; }
            else if (maxiter <= 0) c.done = 2;
            n_running = c.done == 0;
        }
    }
    __syncthreads();

    const char *pin[1] = {p_base};
    const char *win[1] = {a.w};

    // deferred shift updates (see stag_cg_persist.cuh): pending passes over the CTA's sites, one shift per item
    int pn = 0, pj = 0, ppass = 0, pnpass = 0;
    unsigned int gepoch = 1, nepoch = 0;
    int phase = 0;                                    // 0 A | 1 B | 2 CD
    STAG_T_DECL                                       // (timer build: "C" = the merged phase CD, "D" stays 0)
    while (n_running > 0 || phase != 0) {
        if (phase == 0) {
            // phase A (a2): w = D_oe p_base on this CTA's odd sites
            for (int ls = tid; ls < ns; ls += NT) {
                T acc[1][6];
                dslash_site_multi<T, RECON, 1, false, SPLIT>(g, a.W, pin, 1u, 1, e0 + ls, acc);
                store_vec(a.w, Vh, e0 + ls, acc[0]);
            }
        } else if (phase == 1) {
            // phase B (a3): q = c0 p - D_eo w -> shared memory, partial Re<p,q>; then, over shared memory only,
            // the partials of <r,q>, <q,q> and <r,r>
            double dot[4] = {0.0, 0.0, 0.0, 0.0};
            const T c0 = c.c0;
            for (int ls = tid; ls < ns; ls += NT) {
                const int e = e0 + ls;
                T acc[1][6];
                dslash_site_multi<T, RECON, 1, false, SPLIT>(g, a.W, win, 1u, 0, e, acc);
                T pv[6];
                p_s.load(ls, 0, Vh, e, pv);
#pragma unroll
                for (int k = 0; k < 6; ++k) {
                    acc[0][k] = c0 * pv[k] - acc[0][k];
                    dot[0] += (double)pv[k] * (double)acc[0][k];
                }
                q_s.s.store(ls, acc[0]);
            }
            for (int ls = tid; ls < ns; ls += NT) {        // a thread re-reads the q it wrote: no barrier needed
                T rv[6], qv[6];
                r_s.s.load(ls, rv);
                q_s.s.load(ls, qv);
#pragma unroll
                for (int k = 0; k < 6; ++k) {
                    dot[1] += (double)rv[k] * (double)qv[k];
                    dot[2] += (double)qv[k] * (double)qv[k];
                    dot[3] += (double)rv[k] * (double)rv[k];
                }
            }
            cta_partials_all<NT, 4>(dot, red, part + (size_t)(gepoch & 1u) * 4 * G + blockIdx.x, G);   // gepoch = iteration
        } else {
            // phase CD: the four totals (one warp each, same order in every CTA), then every scalar of the iteration
            if (tid < 128) {
                // the set phase B of this iteration wrote (gepoch has been incremented by the barrier since)
                const double t = grid_total(part + (size_t)((gepoch ^ 1u) & 1u) * 4 * G + (size_t)(tid >> 5) * G, G);
                if ((tid & 31) == 0) tot[tid >> 5] = t;
            }
            __syncthreads();
            if (tid < 32) {
                const int i = tid;
                bool live_skip = false;
                const double pq = tot[0], rq = tot[1], qq = tot[2], rr = tot[3];
                // rr is the exact norm of the residual the previous iteration left: if the formula could not certify
                // its convergence (a drop of more than ~1e8 in ONE iteration — an eigenvector source, the last step
                // of a finite termination — is below the formula's resolution eps * rr_old), it is certified here,
                // before anything of this iteration is applied: the solve ends with the previous iteration's count
                if (c.iter > 0 && sqrt(rr / c.bb) <= c.stop) {
                    if (i == 0) { c.rr = rr; c.converged = 1; c.done = 2; }
                    live_skip = true;
                }
                const double alpha = rr / pq;
                const bool bad = live_skip || !(pq > 0.0) || !isfinite(alpha);
                double rr_new = fma(alpha, fma(alpha, qq, -2.0 * rq), rr);     // || r - alpha q ||^2
                if (!bad && !(rr_new > 0.0) && rr_new == rr_new) rr_new = 0.0; // converged to rounding
                const double kk = alpha * c.beta_old / c.alpha_old;
                const double beta = rr_new / rr;
                // The formula resolves rr_new only down to a few eps * rr (its three terms are all of the size of rr): a
                // smaller value, or the clamped 0, says "below that", not "zero".  Convergence, the per-shift residuals
                // and the freezing therefore use the bound max(rr_new, 16 eps rr); if the stop lies below it the solve
                // goes on and the next reduction certifies the drop with the exact <r,r> (the check above).
                const double rel = sqrt(fmax(rr_new, 16.0 * 2.220446049250313e-16 * rr) / c.bb);
                const int iter = c.iter + 1;
                bool live = false;
                double th = 1.0, z = 1.0;
                __syncwarp();
                if (!bad && i < nshift) {
                    if (c.active[i] == 2) c.active[i] = 0;            // frozen at the previous iteration
                    th = 1.0 / ((1.0 + c.delta[i] * alpha) + kk * (1.0 - c.theta[i]));
                    z = c.zeta[i] * th;
                    c.zeta[i] = z;
                    c.theta[i] = th;
                    c.theta_new[i] = th;
                    if (c.active[i] != 0) {
                        live = true;
                        c.resid[i] = z * rel;
                        c.iters_shift[i] = iter;
                        if (freeze && i != base && z * rel <= 0.1 * c.stop) c.active[i] = 2;
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
                if (!bad && i == base) { c.a_base = (T)(alpha * th); c.z_base = (T)z; c.b_base = (T)(beta * th * th); }
                if (i == 0) {
                    c.pq = pq;
                    if (live_skip) { }                                     // converged already: no update
                    else if (bad) { c.breakdown = 1; c.done = 2; }        // breakdown: no update
                    else {
                        c.nlive = __popc(m);
                        c.alpha = alpha;
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
            if (c.done != 2) {
                // r -= alpha q;  x_base += alpha p_base;  p_base = zeta r + beta p_base (shared memory + global)
                const T na = (T)(-c.alpha), ab = c.a_base, zb = c.z_base, bb_ = c.b_base;
                const uint64_t pol = shift_policy(base);
                for (int ls = tid; ls < ns; ls += NT) {
                    const int e = e0 + ls;
                    T rv[6], qv[6], pv[6], xv[6];
                    load_vec_pol(x_base, Vh, e, xv, pol);
                    r_s.s.load(ls, rv);
                    q_s.s.load(ls, qv);
                    p_s.load(ls, 0, Vh, e, pv);
#pragma unroll
                    for (int k = 0; k < 6; ++k) {
                        rv[k] = fma(na, qv[k], rv[k]);
                        xv[k] = fma(ab, pv[k], xv[k]);
                        pv[k] = fma(zb, rv[k], bb_ * pv[k]);
                    }
                    r_s.s.store(ls, rv);
                    if (p_s.res) p_s.s.store(ls, pv);
                    store_vec(p_base, Vh, e, pv);
                    store_vec_pol(x_base, Vh, e, xv, pol);
                }
                // the other live shifts of this iteration: deferred, worked off at the sync points that follow
                pn = c.nlive; pj = 0; ppass = 0;
                pnpass = pn > 0 ? (ns + NT - 1) / NT : 0;
            }
            __syncthreads();                               // every thread has read c.done / coefficients
            if (tid == 0) {
                if (c.done == 1) c.done = 2;               // its last x/p update is queued
                n_running = c.done == 0;
            }
        }

        STAG_TICK(2 * phase);
        // ---- sync point (see stag_cg_persist.cuh): arrive, work off deferred items while waiting -----------
        {
            const bool global = phase == 1;
            __syncthreads();                               // this phase's writes are issued; n_running is visible
            // pending items must be finished before phase CD rewrites their coefficients and r, and at the end
            const bool force = !a.fill || phase == 1 || (phase == 2 && n_running == 0);
            const unsigned int sync_id = gepoch + nepoch + 1u;
            unsigned int target;
            if (global) {
                target = ++gepoch * (unsigned)G;
                if (tid == 0) asm volatile("red.release.gpu.global.add.u32 [%0], %1;" :: "l"(bar), "r"(1u) : "memory");
            } else {
                target = ++nepoch;
                if (tid == 0)
                    asm volatile("st.release.gpu.global.u32 [%0], %1;" :: "l"(a.flags + (size_t)blockIdx.x * 32), "r"(target) : "memory");
            }
            const bool poll_warp = tid < 32;
            bool released = false;
            while (!released || (force && ppass < pnpass)) {
                unsigned int v = target;
                if (poll_warp && !released) {
                    if (global) {
                        if (tid == 0) asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(bar) : "memory");
                    } else {
                        for (int k = tid; k < nnb; k += 32) {      // wrapped unsigned min over this lane's flags
                            unsigned int f;
                            asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];"
                                         : "=r"(f) : "l"(a.flags + (size_t)nb_list[k] * 32) : "memory");
                            if ((int)(f - v) < 0) v = f;
                        }
                    }
                }
                if (ppass < pnpass) {                      // one item; the poll is in flight meanwhile
                    const int ls = tid + ppass * NT;
                    if (ls < ns) {
                        const int e = e0 + ls;
                        const int i = c.live[pj];
                        const uint64_t pol = shift_policy(i);
                        const T aj = c.ca[pj], zj = c.cz[pj], bj = c.cb[pj];
                        T rv[6], pv[6], xv[6];
                        r_s.s.load(ls, rv);
                        load_vec_pol(a.p + (size_t)i * a.p_stride, Vh, e, pv, pol);
                        load_vec_pol(a.x + (size_t)i * a.x_stride, Vh, e, xv, pol);
#pragma unroll
                        for (int k = 0; k < 6; ++k) {
                            xv[k] = fma(aj, pv[k], xv[k]);
                            pv[k] = fma(zj, rv[k], bj * pv[k]);
                        }
                        store_vec_pol(a.x + (size_t)i * a.x_stride, Vh, e, xv, pol);
                        store_vec_pol(a.p + (size_t)i * a.p_stride, Vh, e, pv, pol);
                    }
                    if (++pj >= pn) { pj = 0; ++ppass; }
                }
                if (poll_warp) {
                    if (!released && __all_sync(0xffffffffu, (int)(v - target) >= 0)) {
                        if (tid == 0) {
                            asm volatile("fence.acquire.gpu;" ::: "memory");
                            *reinterpret_cast<volatile unsigned int *>(&sync_seen) = sync_id;
                        }
                        released = true;
                    }
                } else {
                    released = ppass >= pnpass || *reinterpret_cast<volatile unsigned int *>(&sync_seen) == sync_id;
                }
            }
            __syncthreads();
        }
        STAG_TICK(2 * phase + 1);
        phase = phase == 2 ? 0 : phase + 1;
    }
    STAG_T_REPORT(1, c.iter)

    // ---- a7: y = residue0 b + sum_i residues_i x_i (own sites only: no barrier needed) ---------------
    if (a.y) {
        const T r0 = (T)st->residue0;
        for (int ls = tid; ls < ns; ls += NT) {
            const int e = e0 + ls;
            T bv[6], acc[6];
            load_vec<true>(a.b, Vh, e, bv);
#pragma unroll
            for (int k = 0; k < 6; ++k) acc[k] = r0 * bv[k];
            for (int i = 0; i < nshift; ++i) {
                const T ri = (T)st->residues[i];
                T xv[6];
                load_vec_pol(a.x + (size_t)i * a.x_stride, Vh, e, xv, policy_evict_first());
#pragma unroll
                for (int k = 0; k < 6; ++k) acc[k] = fma(ri, xv[k], acc[k]);
            }
            store_vec(a.y, Vh, e, acc);
        }
    }

    // ---- read-back state (every CTA holds the same scalars; CTA 0 writes them) -------------------------
    if (blockIdx.x == 0 && tid < 32) {
        const int i = tid;
        if (i < nshift) {
            st->zeta[i] = c.zeta[i];
            st->theta[i] = c.theta[i];
            st->resid_shift[i] = c.resid[i];
            st->iters_shift[i] = c.iters_shift[i];
            st->active[i] = c.active[i];
        }
        if (i == 0) {
            st->bb = c.bb; st->rr = c.rr; st->pq = c.pq; st->alpha = c.alpha;
            st->iter = c.iter; st->converged = c.converged; st->breakdown = c.breakdown;
            st->stagnated = c.stagnated; st->done = 2;
        }
    }
}

template <typename T, int RECON, int NT, bool SPLIT = false>
int launch_persistent_sr(const stag_ctx *ctx, const PersistArgs &args, cudaStream_t st) {
    const Geom &g = ctx->g;
    const int grid = persist_grid(ctx);
    if (grid > kMaxPersistGrid) return STAG_ERR_UNSUPPORTED;
    PersistArgs a = args;
    a.S = persist_slots(ctx);
    a.fill = ctx->opt.cg_fill != 0;
    a.nbflags = ctx->opt.cg_nbflags != 0;
    const size_t slice = (size_t)a.S * 6 * sizeof(T);
    int fit = (int)(kMaxDynSmem / slice);
    if (fit > ctx->opt.cg_resident_slices) fit = ctx->opt.cg_resident_slices;
    if (fit < 2) return STAG_ERR_UNSUPPORTED;            // r and q must be resident: the caller falls back
    a.res_r = 1; a.res_q = 1; a.res_p = fit >= 3;
    const size_t smem = slice * (size_t)(2 + a.res_p);
    auto kern = cg_persistent_sr_kernel<T, RECON, NT, SPLIT>;
    STAG_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int per_sm = 0;
    STAG_CUDA_OK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, NT, smem));
    if (per_sm < 1) return STAG_ERR_UNSUPPORTED;
    STAG_CUDA_OK(cudaMemsetAsync(a.flags, 0, (size_t)grid * 128, st));
    Geom gg = g;
    void *params[] = {(void *)&gg, (void *)&a};
    log_kernel(ctx, (const void *)kern);
    STAG_CUDA_OK(cudaLaunchCooperativeKernel((const void *)kern, dim3(grid), dim3(NT), params, smem, st));
    return STAG_OK;
}

// implemented in stag_cg_persist_sr.cu
int cg_persistent_sr_launch(const stag_ctx *ctx, int prec, int recon, const PersistArgs &a, cudaStream_t st);

}  // namespace stag
