// stag_cg_persist.cu — the whole multi-shift CG solve as ONE persistent cooperative kernel
// (DESIGN.md "persistent CG").
//
// For the lattices of the paper's runs (4 x 16^3 ... 8 x 32^3, 4 x 48^3) one
// CG iteration moves only a few hundred MB, so four kernel launches per iteration — each with a
// fill/drain ramp and, twice, a serial "last CTA" reduction tail — cost as much as 15 % of the
// iteration.  Here one CTA per SM owns a fixed, contiguous range of sites for the whole solve:
//
//   phase A  w = D_oe p_base                on the CTA's odd sites   -> global (neighbours read it)
//            grid barrier
//   phase B  q = (m^2+sigma_0) p - D_eo w   on the CTA's even sites  -> q stays in SHARED memory
//            per-CTA partial of Re<p,q>     -> global;  grid barrier
//   phase C  every CTA adds the partials in the same order (bit-identical alpha everywhere),
//            runs the a4 recurrences in its own shared memory, then r -= alpha q with r and q
//            both in shared memory (a5 moves no HBM bytes at all); partial of <r,r>; grid barrier
//   phase D  every CTA: beta, beta_i, zeta_i, convergence latch, freezing (a4, a7); then a6:
//            the base shift first (p_base is what the neighbours need), ARRIVE at the barrier,
//            the other live shifts' x_i, p_i streamed once, then WAIT — the barrier latency hides
//            behind the shift updates.
//
// r, q and the CTA's own slice of p_base live in shared memory for the whole solve (3 x 48 B x
// sites/SM: 129 KB at 32^3 x 8), so per iteration and even site the kernel moves 2 x 1248 (links +
// neighbours) + 48 (p_base store) + 192 x live shifts bytes instead of 2736 + 192 x live.  All
// scalars are fp64 and never leave the SM; the host sees one launch and one read-back.
//
// Lattices whose three resident vectors do not fit in shared memory use the multi-kernel path
// in stag_cg.cu (launch overhead is negligible there).
#include <cooperative_groups.h>

#include "stag_cg.cuh"
#include "stag_dslash.cuh"

namespace stag {

// ---- grid barrier: monotone counter, arrive / wait split ---------------------------------------
// Safe only because the kernel is launched cooperatively (all CTAs co-resident).
__device__ __forceinline__ void grid_arrive(unsigned int *bar) {
    __syncthreads();                       // every thread's writes of this phase are issued
    if (threadIdx.x == 0) {
        __threadfence();                   // ... and ordered before the arrival (cumulative)
        atomicAdd(bar, 1u);
    }
}
__device__ __forceinline__ void grid_wait(unsigned int *bar, unsigned int target) {
    if (threadIdx.x == 0) {
        unsigned int v;
        do {
            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(bar) : "memory");
        } while ((int)(v - target) < 0);
        __threadfence();
    }
    __syncthreads();
}

// ---- a vector slice resident in shared memory: S sites, thread-private slots ---------------------
template <typename T> struct SVec;
template <> struct SVec<double> {
    double2 *a; int S;
    __device__ __forceinline__ void init(unsigned char *base, int S_) { a = reinterpret_cast<double2 *>(base); S = S_; }
    __device__ __forceinline__ void load(int slot, double (&x)[6]) const {
#pragma unroll
        for (int c = 0; c < 3; ++c) { const double2 t = a[c * S + slot]; x[2 * c] = t.x; x[2 * c + 1] = t.y; }
    }
    __device__ __forceinline__ void store(int slot, const double (&x)[6]) {
#pragma unroll
        for (int c = 0; c < 3; ++c) a[c * S + slot] = make_double2(x[2 * c], x[2 * c + 1]);
    }
};
template <> struct SVec<float> {
    float4 *a; float2 *b;
    __device__ __forceinline__ void init(unsigned char *base, int S_) {
        a = reinterpret_cast<float4 *>(base); b = reinterpret_cast<float2 *>(base + (size_t)S_ * 16);
    }
    __device__ __forceinline__ void load(int slot, float (&x)[6]) const {
        const float4 u = a[slot]; const float2 v = b[slot];
        x[0] = u.x; x[1] = u.y; x[2] = u.z; x[3] = u.w; x[4] = v.x; x[5] = v.y;
    }
    __device__ __forceinline__ void store(int slot, const float (&x)[6]) {
        a[slot] = make_float4(x[0], x[1], x[2], x[3]); b[slot] = make_float2(x[4], x[5]);
    }
};

// ---- streaming (evict-first) own-site access to x_i, p_i -----------------------------------------
__device__ __forceinline__ void load_vec_cs(const char *v, int Vh, int e, double (&x)[6]) {
    const double2 *p = reinterpret_cast<const double2 *>(v) + e;
#pragma unroll
    for (int c = 0; c < 3; ++c) { const double2 t = __ldcs(p + (size_t)c * Vh); x[2 * c] = t.x; x[2 * c + 1] = t.y; }
}
__device__ __forceinline__ void load_vec_cs(const char *v, int Vh, int e, float (&x)[6]) {
    const float4 a = __ldcs(reinterpret_cast<const float4 *>(v) + e);
    const float2 b = __ldcs(reinterpret_cast<const float2 *>(v + (size_t)Vh * 16) + e);
    x[0] = a.x; x[1] = a.y; x[2] = a.z; x[3] = a.w; x[4] = b.x; x[5] = b.y;
}
__device__ __forceinline__ void store_vec_cs(char *v, int Vh, int e, const double (&x)[6]) {
    double2 *p = reinterpret_cast<double2 *>(v) + e;
#pragma unroll
    for (int c = 0; c < 3; ++c) __stcs(p + (size_t)c * Vh, make_double2(x[2 * c], x[2 * c + 1]));
}
__device__ __forceinline__ void store_vec_cs(char *v, int Vh, int e, const float (&x)[6]) {
    __stcs(reinterpret_cast<float4 *>(v) + e, make_float4(x[0], x[1], x[2], x[3]));
    __stcs(reinterpret_cast<float2 *>(v + (size_t)Vh * 16) + e, make_float2(x[4], x[5]));
}

// ---- per-CTA copy of the scalar state (every CTA carries the same values) ------------------------
template <typename T>
struct Scalars {
    double delta[STAG_MAX_SHIFTS], zeta[STAG_MAX_SHIFTS], theta[STAG_MAX_SHIFTS], theta_new[STAG_MAX_SHIFTS];
    double resid[STAG_MAX_SHIFTS];
    T ca[STAG_MAX_SHIFTS], cz[STAG_MAX_SHIFTS], cb[STAG_MAX_SHIFTS];   // alpha_i, zeta_i(new), beta_i of live shifts
    int live[STAG_MAX_SHIFTS];                                           // compacted list, base excluded
    int active[STAG_MAX_SHIFTS], iters_shift[STAG_MAX_SHIFTS];
    double bb, rr, alpha, alpha_old, beta_old, best_rr, pq, total;
    T a_base, z_base, b_base;
    int nlive, iter, done, converged, breakdown, stagnated, since_best;
};

// sum of the G per-CTA partials, same order in every CTA => bit-identical result everywhere.
// Valid in every lane of warp 0.
__device__ __forceinline__ double grid_total(const double *part, int G) {
    double t = 0.0;
    for (int i = threadIdx.x & 31; i < G; i += 32) t += __ldcg(part + i);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
    return t;
}

template <int NT>
__device__ __forceinline__ void cta_partial(double v, double *red, double *slot) {
    const double s = block_sum<NT>(v, red);
    if (threadIdx.x == 0) __stcg(slot, s);
}

struct PersistArgs {
    const char *W;        // packed gauge
    const char *b;        // source
    char *w;              // odd-site scratch vector (global)
    char *p;              // nshift search directions (global), stride p_stride
    size_t p_stride;
    char *x;              // nshift solutions, stride x_stride
    size_t x_stride;
    char *y;              // nullable
    CgState *state;
    double *partials;     // 2 * gridDim.x doubles
    int S;                // sites per CTA (multiple of 32)
};

template <typename T, int RECON, int NT>
__global__ void __launch_bounds__(NT, 1)
cg_persistent_kernel(const Geom g, const PersistArgs a) {
    extern __shared__ __align__(16) unsigned char dyn[];
    __shared__ Scalars<T> sc;
    __shared__ double red[NT / 32 + 1];

    const int tid = threadIdx.x, G = gridDim.x, Vh = g.Vh, S = a.S;
    const int e0 = min(Vh, (int)blockIdx.x * S), e1 = min(Vh, e0 + S);
    CgState *st = a.state;
    unsigned int *bar = &st->ticket;
    unsigned int epoch = 0;
    double *part_pq = a.partials, *part_rr = a.partials + G;

    SVec<T> r_s, q_s, p_s;
    r_s.init(dyn, S);
    q_s.init(dyn + (size_t)S * 6 * sizeof(T), S);
    p_s.init(dyn + (size_t)2 * S * 6 * sizeof(T), S);

    const int nshift = st->nshift, base = st->base, maxiter = st->maxiter;
    const int freeze = st->freeze, fp32 = st->fp32;
    const double stop = st->stop;
    const T c0 = (T)st->c0;
    char *p_base = a.p + (size_t)base * a.p_stride;
    char *x_base = a.x + (size_t)base * a.x_stride;

    // ---- start: x_i = 0, r = p_i = b, bb = <b,b> ---------------------------------------------------
    if (tid < STAG_MAX_SHIFTS) {
        const bool on = tid < nshift;
        sc.delta[tid] = on ? st->delta[tid] : 0.0;
        sc.zeta[tid] = 1.0; sc.theta[tid] = 1.0; sc.theta_new[tid] = 1.0;
        sc.resid[tid] = 1.0;
        sc.active[tid] = on ? 1 : 0;
        sc.iters_shift[tid] = 0;
    }
    {
        double acc = 0.0;
        for (int e = e0 + tid; e < e1; e += NT) {
            T v[6], z[6] = {T(0), T(0), T(0), T(0), T(0), T(0)};
            load_vec<true>(a.b, Vh, e, v);
#pragma unroll
            for (int k = 0; k < 6; ++k) acc += (double)v[k] * (double)v[k];
            r_s.store(e - e0, v);
            p_s.store(e - e0, v);
            for (int i = 0; i < nshift; ++i) {
                if (i == base) store_vec(p_base, Vh, e, v);
                else store_vec_cs(a.p + (size_t)i * a.p_stride, Vh, e, v);
                store_vec_cs(a.x + (size_t)i * a.x_stride, Vh, e, z);
            }
        }
        cta_partial<NT>(acc, red, part_rr + blockIdx.x);
    }
    grid_arrive(bar);
    grid_wait(bar, ++epoch * G);
    if (tid < 32) {
        const double bb = grid_total(part_rr, G);
        if (tid == 0) {
            sc.bb = bb; sc.rr = bb; sc.best_rr = bb; sc.alpha = 0.0; sc.alpha_old = 1.0; sc.beta_old = 0.0;
            sc.pq = 0.0; sc.iter = 0; sc.done = 0; sc.converged = 0; sc.breakdown = 0; sc.stagnated = 0;
            sc.since_best = 0;
            if (!(bb > 0.0)) { sc.converged = (bb == 0.0); sc.breakdown = !(bb == 0.0); sc.done = 2; }
            if (maxiter <= 0) sc.done = 2;
        }
    }
    __syncthreads();

    // ---- iterations -----------------------------------------------------------------------------------
    while (sc.done == 0) {
        // phase A (a2): w = D_oe p_base on this CTA's odd sites
        for (int e = e0 + tid; e < e1; e += NT) {
            T acc[6];
            dslash_site<T, RECON, false>(g, a.W, p_base, 1, e, acc);
            store_vec(a.w, Vh, e, acc);
        }
        grid_arrive(bar);
        grid_wait(bar, ++epoch * G);

        // phase B (a3): q = c0 p - D_eo w, partial Re<p,q>
        {
            double dot = 0.0;
            for (int e = e0 + tid; e < e1; e += NT) {
                T acc[6], pv[6];
                dslash_site<T, RECON, false>(g, a.W, a.w, 0, e, acc);
                p_s.load(e - e0, pv);
#pragma unroll
                for (int k = 0; k < 6; ++k) {
                    acc[k] = c0 * pv[k] - acc[k];
                    dot += (double)pv[k] * (double)acc[k];
                }
                q_s.store(e - e0, acc);
            }
            cta_partial<NT>(dot, red, part_pq + blockIdx.x);
        }
        grid_arrive(bar);
        grid_wait(bar, ++epoch * G);

        // phase C (a4 after <p,q>, then a5): alpha, theta_new_i, alpha_i;  r -= alpha q;  partial <r,r>
        if (tid < 32) {
            const double pq = grid_total(part_pq, G);
            const double alpha = sc.rr / pq;
            const bool bad = !(pq > 0.0) || !isfinite(alpha);
            const double k = alpha * sc.beta_old / sc.alpha_old;
            __syncwarp();
            if (!bad && tid < nshift) {
                if (sc.active[tid] == 2) sc.active[tid] = 0;        // frozen at the previous iteration
                sc.theta_new[tid] = 1.0 / ((1.0 + sc.delta[tid] * alpha) + k * (1.0 - sc.theta[tid]));
            }
            if (tid == 0) {
                sc.pq = pq;
                if (bad) { sc.breakdown = 1; sc.done = 2; } else sc.alpha = alpha;
            }
        }
        __syncthreads();
        if (sc.done != 0) break;                                     // breakdown: no update this iteration
        {
            const T na = (T)(-sc.alpha);
            double acc = 0.0;
            for (int e = e0 + tid; e < e1; e += NT) {
                T rv[6], qv[6];
                r_s.load(e - e0, rv);
                q_s.load(e - e0, qv);
#pragma unroll
                for (int k = 0; k < 6; ++k) {
                    rv[k] = fma(na, qv[k], rv[k]);
                    acc += (double)rv[k] * (double)rv[k];
                }
                r_s.store(e - e0, rv);
            }
            cta_partial<NT>(acc, red, part_rr + blockIdx.x);
        }
        grid_arrive(bar);
        grid_wait(bar, ++epoch * G);

        // phase D (a4 after <r,r>, a7 latch, a6)
        if (tid < 32) {
            const double rr_new = grid_total(part_rr, G);
            const double alpha = sc.alpha;
            const double beta = rr_new / sc.rr;
            const double rel = sqrt(rr_new / sc.bb);
            const int iter = sc.iter + 1;
            bool live = false;
            double th = 1.0, z = 1.0;
            __syncwarp();
            if (tid < nshift) {
                th = sc.theta_new[tid];
                z = sc.zeta[tid] * th;
                sc.zeta[tid] = z;
                sc.theta[tid] = th;
                if (sc.active[tid] != 0) {
                    live = true;
                    if (sc.active[tid] == 1) {
                        sc.resid[tid] = z * rel;
                        sc.iters_shift[tid] = iter;
                        if (freeze && tid != base && z * rel <= 0.1 * stop) sc.active[tid] = 2;
                    }
                }
            }
            const unsigned m = __ballot_sync(0xffffffffu, live && tid != base);
            if (live && tid != base) {
                const int j = __popc(m & ((1u << tid) - 1u));
                sc.live[j] = tid;
                sc.ca[j] = (T)(alpha * th);
                sc.cz[j] = (T)z;
                sc.cb[j] = (T)(beta * th * th);
            }
            if (tid == base) { sc.a_base = (T)(alpha * th); sc.z_base = (T)z; sc.b_base = (T)(beta * th * th); }
            if (tid == 0) {
                sc.nlive = __popc(m);
                sc.alpha_old = alpha;
                sc.beta_old = beta;
                sc.rr = rr_new;
                sc.iter = iter;
                int done = 0;
                if (rel <= stop) { sc.converged = 1; done = 1; }
                else if (iter >= maxiter) done = 1;
                else if (!(rr_new == rr_new)) { sc.breakdown = 1; done = 1; }
                else if (fp32) {                                     // reading A9
                    if (rr_new < sc.best_rr) { sc.best_rr = rr_new; sc.since_best = 0; }
                    else if (++sc.since_best >= 50) { sc.stagnated = 1; done = 1; }
                }
                sc.done = done;
            }
        }
        __syncthreads();
        const bool last = sc.done != 0;
        {   // base shift first: its new p is what phase A of the next iteration gathers
            const T ab = sc.a_base, zb = sc.z_base, bb_ = sc.b_base;
            for (int e = e0 + tid; e < e1; e += NT) {
                T rv[6], pv[6], xv[6];
                load_vec_cs(x_base, Vh, e, xv);
                r_s.load(e - e0, rv);
                p_s.load(e - e0, pv);
#pragma unroll
                for (int k = 0; k < 6; ++k) {
                    xv[k] = fma(ab, pv[k], xv[k]);
                    pv[k] = fma(zb, rv[k], bb_ * pv[k]);
                }
                store_vec_cs(x_base, Vh, e, xv);
                p_s.store(e - e0, pv);
                store_vec(p_base, Vh, e, pv);
            }
        }
        if (!last) grid_arrive(bar);
        {
            const int n = sc.nlive;
            for (int e = e0 + tid; e < e1; e += NT) {
                T rv[6];
                r_s.load(e - e0, rv);
#pragma unroll 2
                for (int j = 0; j < n; ++j) {
                    char *xp = a.x + (size_t)sc.live[j] * a.x_stride;
                    char *pp = a.p + (size_t)sc.live[j] * a.p_stride;
                    const T aj = sc.ca[j], zj = sc.cz[j], bj = sc.cb[j];
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
        if (last) break;
        grid_wait(bar, ++epoch * G);
    }

    // ---- a7: y = residue0 b + sum_i residues_i x_i (own sites only: no barrier needed) ---------------
    if (a.y) {
        const T r0 = (T)st->residue0;
        for (int e = e0 + tid; e < e1; e += NT) {
            T bv[6], acc[6];
            load_vec<true>(a.b, Vh, e, bv);
#pragma unroll
            for (int k = 0; k < 6; ++k) acc[k] = r0 * bv[k];
            for (int i = 0; i < nshift; ++i) {
                const T ri = (T)st->residues[i];
                T xv[6];
                load_vec_cs(a.x + (size_t)i * a.x_stride, Vh, e, xv);
#pragma unroll
                for (int k = 0; k < 6; ++k) acc[k] = fma(ri, xv[k], acc[k]);
            }
            store_vec(a.y, Vh, e, acc);
        }
    }

    // ---- read-back state (every CTA holds the same scalars; CTA 0 writes them) -------------------------
    if (blockIdx.x == 0) {
        __syncthreads();
        if (tid < nshift) {
            st->zeta[tid] = sc.zeta[tid];
            st->theta[tid] = sc.theta[tid];
            st->resid_shift[tid] = sc.resid[tid];
            st->iters_shift[tid] = sc.iters_shift[tid];
            st->active[tid] = sc.active[tid];
        }
        if (tid == 0) {
            st->bb = sc.bb; st->rr = sc.rr; st->pq = sc.pq; st->alpha = sc.alpha;
            st->iter = sc.iter; st->converged = sc.converged; st->breakdown = sc.breakdown;
            st->stagnated = sc.stagnated; st->done = 2;
        }
    }
}

// ---- host side ---------------------------------------------------------------------------------------
static constexpr size_t kMaxDynSmem = 200 * 1024;     // of 227 KB; the rest: static scalars + L1

// sites per CTA for a grid of `grid` CTAs (multiple of 32: every CTA's slice starts on a 512-byte line)
static int sites_per_cta(int Vh, int grid) {
    const int s = (Vh + grid - 1) / grid;
    return (s + 31) & ~31;
}

bool cg_persistent_fits(const stag_ctx *ctx, int prec) {
    const int S = sites_per_cta(ctx->g.Vh, ctx->num_sms);
    return (size_t)3 * S * vec_bytes_per_site(prec) <= kMaxDynSmem;
}

template <typename T, int RECON, int NT>
static int launch_persistent(const stag_ctx *ctx, const PersistArgs &args, cudaStream_t st) {
    const Geom &g = ctx->g;
    int grid = ctx->num_sms;
    const int tiles = (g.Vh + 31) / 32;
    if (grid > tiles) grid = tiles;
    PersistArgs a = args;
    a.S = sites_per_cta(g.Vh, grid);
    const size_t smem = (size_t)3 * a.S * 6 * sizeof(T);
    auto kern = cg_persistent_kernel<T, RECON, NT>;
    STAG_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int per_sm = 0;
    STAG_CUDA_OK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, NT, smem));
    if (per_sm < 1) return STAG_ERR_UNSUPPORTED;
    Geom gg = g;
    void *params[] = {(void *)&gg, (void *)&a};
    STAG_CUDA_OK(cudaLaunchCooperativeKernel((const void *)kern, dim3(grid), dim3(NT), params, smem, st));
    return STAG_OK;
}

int cg_persistent_dispatch(const stag_ctx *ctx, const void *packed, int prec, int recon,
                           const void *b, void *x, size_t x_stride, void *y, char *ws,
                           const CgLayout &lay, cudaStream_t st) {
    PersistArgs a;
    a.W = static_cast<const char *>(packed);
    a.b = static_cast<const char *>(b);
    a.w = ws + lay.w;
    a.p = ws + lay.p;
    a.p_stride = lay.vec_stride;
    a.x = static_cast<char *>(x);
    a.x_stride = x_stride;
    a.y = static_cast<char *>(y);
    a.state = reinterpret_cast<CgState *>(ws + lay.state);
    a.partials = reinterpret_cast<double *>(ws + lay.partials);
    a.S = 0;
    // 1024 threads x 64 registers or 512 x 128 per SM (fp64 12-real needs ~100 registers for the row rebuild)
    const bool wide = ctx->opt.cg_persistent_threads != 512;
    if (prec == STAG_F64) {
        if (recon == 12) return launch_persistent<double, 12, 512>(ctx, a, st);
        return wide ? launch_persistent<double, 18, 1024>(ctx, a, st)
                    : launch_persistent<double, 18, 512>(ctx, a, st);
    }
    if (recon == 18)
        return wide ? launch_persistent<float, 18, 1024>(ctx, a, st)
                    : launch_persistent<float, 18, 512>(ctx, a, st);
    return wide ? launch_persistent<float, 12, 1024>(ctx, a, st)
                : launch_persistent<float, 12, 512>(ctx, a, st);
}

}  // namespace stag
