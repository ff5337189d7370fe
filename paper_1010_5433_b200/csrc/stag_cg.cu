// stag_cg.cu — stag_mshift_cg: multi-shift conjugate gradient for (m^2 - D_eo D_oe + sigma_i) x_i = b
// ("Krylov solvers for shifted systems", zero start vector; ref [9]).
//
// One iteration = four launches, no host round trip:
//   a2  w = D_oe p                                   dslash_kernel<MODE 1>
//   a3  q = (m^2+sigma_0) p - D_eo w, <p,q>, then a4 dslash_kernel<MODE 2> (+ last-CTA scalars)
//   a5  r -= alpha q, <r,r>, then a4 + a7 latch      cg_update_r_kernel   (+ last-CTA scalars)
//   a6  x_i += alpha_i p_i ; p_i = zeta_i r + beta_i p_i  for every active shift, one pass
//                                                    cg_update_shifts_kernel
// Vectors are T (fp64 or fp32); every reduction and scalar is fp64.
#include <cstring>

#include "stag_cg.cuh"

namespace stag {

template <typename T> struct Vec16;
template <> struct Vec16<double> { typedef double2 type; static constexpr int n = 2; };
template <> struct Vec16<float> { typedef float4 type; static constexpr int n = 4; };

__device__ __forceinline__ double2 ldcs(const double2 *p) { return __ldcs(p); }
__device__ __forceinline__ float4 ldcs(const float4 *p) { return __ldcs(p); }

// per-component helpers on 16-byte chunks
__device__ __forceinline__ double2 fma2(double a, double2 x, double2 y) {   // a*x + y
    return make_double2(fma(a, x.x, y.x), fma(a, x.y, y.y));
}
__device__ __forceinline__ float4 fma2(float a, float4 x, float4 y) {
    return make_float4(fmaf(a, x.x, y.x), fmaf(a, x.y, y.y), fmaf(a, x.z, y.z), fmaf(a, x.w, y.w));
}
__device__ __forceinline__ double2 axpby(double a, double2 x, double b, double2 y) {   // a*x + b*y
    return make_double2(fma(a, x.x, b * y.x), fma(a, x.y, b * y.y));
}
__device__ __forceinline__ float4 axpby(float a, float4 x, float b, float4 y) {
    return make_float4(fmaf(a, x.x, b * y.x), fmaf(a, x.y, b * y.y), fmaf(a, x.z, b * y.z),
                       fmaf(a, x.w, b * y.w));
}
__device__ __forceinline__ double norm2_of(double2 v) { return v.x * v.x + v.y * v.y; }
__device__ __forceinline__ double norm2_of(float4 v) {
    return (double)v.x * v.x + (double)v.y * v.y + (double)v.z * v.z + (double)v.w * v.w;
}
__device__ __forceinline__ double2 zero_of(double2) { return make_double2(0.0, 0.0); }
__device__ __forceinline__ float4 zero_of(float4) { return make_float4(0.f, 0.f, 0.f, 0.f); }

// ---- start: r = b, p_i = b, x_i = 0, bb = <b,b> ---------------------------------------------------
template <typename T, int BLOCK>
__global__ void __launch_bounds__(BLOCK)
cg_init_kernel(const long nchunk, const char *__restrict__ b, char *__restrict__ r,
               char *__restrict__ p, const size_t p_stride, char *__restrict__ x,
               const size_t x_stride, CgState *__restrict__ state, double *__restrict__ partials) {
    typedef typename Vec16<T>::type V;
    __shared__ double red[BLOCK / 32 + 1];
    const int nshift = state->nshift;
    double acc = 0.0;
    for (long k = (long)blockIdx.x * BLOCK + threadIdx.x; k < nchunk; k += (long)gridDim.x * BLOCK) {
        const V v = reinterpret_cast<const V *>(b)[k];
        acc += norm2_of(v);
        reinterpret_cast<V *>(r)[k] = v;
        for (int i = 0; i < nshift; ++i) {
            reinterpret_cast<V *>(p + (size_t)i * p_stride)[k] = v;
            reinterpret_cast<V *>(x + (size_t)i * x_stride)[k] = zero_of(v);
        }
    }
    double total;
    if (grid_sum_last_cta<BLOCK>(acc, partials, &state->ticket, red, total) && threadIdx.x == 0) {
        state->bb = total;
        state->rr = total;
        state->best_rr = total;
        if (!(total > 0.0)) {                       // b = 0: x = 0 after 0 iterations (pin P7 vi)
            state->converged = (total == 0.0);
            state->breakdown = !(total == 0.0);     // NaN source
            state->done = 2;
        }
    }
}

// ---- a5: r -= alpha q ; <r,r> ; last CTA: beta, beta_i, zeta_i, latch -----------------------------
template <typename T, int BLOCK>
__global__ void __launch_bounds__(BLOCK)
cg_update_r_kernel(const long nchunk, char *__restrict__ r, const char *__restrict__ q,
                   CgState *__restrict__ state, double *__restrict__ partials) {
    typedef typename Vec16<T>::type V;
    __shared__ double red[BLOCK / 32 + 1];
    if (*reinterpret_cast<volatile int *>(&state->done) != 0) return;
    const T na = (T)(-state->alpha);
    double acc = 0.0;
    const long stride = (long)gridDim.x * BLOCK;
    long k = (long)blockIdx.x * BLOCK + threadIdx.x;
    for (; k + 3 * stride < nchunk; k += 4 * stride) {        // 4 independent chunks in flight
        V rv[4], qv[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            rv[u] = reinterpret_cast<const V *>(r)[k + u * stride];
            qv[u] = ldcs(reinterpret_cast<const V *>(q) + k + u * stride);
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            rv[u] = fma2(na, qv[u], rv[u]);
            acc += norm2_of(rv[u]);
            reinterpret_cast<V *>(r)[k + u * stride] = rv[u];
        }
    }
    for (; k < nchunk; k += stride) {
        V rv = reinterpret_cast<const V *>(r)[k];
        rv = fma2(na, ldcs(reinterpret_cast<const V *>(q) + k), rv);
        acc += norm2_of(rv);
        reinterpret_cast<V *>(r)[k] = rv;
    }
    double total;
    if (grid_sum_last_cta<BLOCK>(acc, partials, &state->ticket, red, total) && threadIdx.x < 32)
        cg_scalars_after_rr(state, total);
}

// ---- a6: all-shift update, each x_i and p_i read once and written once ------------------------------
template <typename T, int BLOCK>
__global__ void __launch_bounds__(BLOCK)
cg_update_shifts_kernel(const long nchunk, const char *__restrict__ r, char *__restrict__ p,
                        const size_t p_stride, char *__restrict__ x, const size_t x_stride,
                        const CgState *__restrict__ state) {
    typedef typename Vec16<T>::type V;
    __shared__ T s_alpha[STAG_MAX_SHIFTS], s_zeta[STAG_MAX_SHIFTS], s_beta[STAG_MAX_SHIFTS];
    __shared__ int s_idx[STAG_MAX_SHIFTS];
    __shared__ int s_n;
    if (*reinterpret_cast<const volatile int *>(&state->done) == 2) return;
    if (threadIdx.x < 32) {
        const int i = threadIdx.x;
        const bool on = i < state->nshift && state->active[i] != 0;
        const unsigned m = __ballot_sync(0xffffffffu, on);
        if (on) {
            const int j = __popc(m & ((1u << i) - 1u));
            s_idx[j] = i;
            s_alpha[j] = (T)state->alpha_i[i];
            s_zeta[j] = (T)state->zeta[i];
            s_beta[j] = (T)state->beta_i[i];
        }
        if (i == 0) s_n = __popc(m);
    }
    __syncthreads();
    const int n = s_n;
    for (long k = (long)blockIdx.x * BLOCK + threadIdx.x; k < nchunk; k += (long)gridDim.x * BLOCK) {
        const V rv = reinterpret_cast<const V *>(r)[k];
#pragma unroll 4
        for (int j = 0; j < n; ++j) {
            V *xp = reinterpret_cast<V *>(x + (size_t)s_idx[j] * x_stride) + k;
            V *pp = reinterpret_cast<V *>(p + (size_t)s_idx[j] * p_stride) + k;
            const V pv = ldcs(pp);
            const V xv = ldcs(xp);
            __stcs(xp, fma2(s_alpha[j], pv, xv));
            __stcs(pp, axpby(s_zeta[j], rv, s_beta[j], pv));
        }
    }
}

// ---- a7: y = residue0 b + sum_i residues_i x_i -----------------------------------------------------
template <typename T, int BLOCK>
__global__ void __launch_bounds__(BLOCK)
cg_partial_fraction_kernel(const long nchunk, const char *__restrict__ b, const char *__restrict__ x,
                           const size_t x_stride, char *__restrict__ y,
                           const CgState *__restrict__ state) {
    typedef typename Vec16<T>::type V;
    const int nshift = state->nshift;
    const T r0 = (T)state->residue0;
    for (long k = (long)blockIdx.x * BLOCK + threadIdx.x; k < nchunk; k += (long)gridDim.x * BLOCK) {
        const V bv = reinterpret_cast<const V *>(b)[k];
        V acc = axpby(r0, bv, T(0), bv);
        for (int i = 0; i < nshift; ++i)
            acc = fma2((T)state->residues[i], reinterpret_cast<const V *>(x + (size_t)i * x_stride)[k], acc);
        reinterpret_cast<V *>(y)[k] = acc;
    }
}

// ---- host side --------------------------------------------------------------------------------------
template <typename T>
struct CgLaunch {
    static constexpr int BLOCK = 256;
    const stag_ctx *ctx;
    const void *packed;
    int prec, recon;
    long nchunk;
    int grid;
    char *ws;
    CgLayout lay;
    CgState *state;
    double *partials;
    char *x;
    size_t x_stride;
    int nshift, base;
    cudaStream_t st;

    char *p_base() const { return ws + lay.p + (size_t)base * lay.vec_stride; }

    // ev (nullable): 5 events recorded around the 4 launches (option cg_profile)
    int iteration(cudaEvent_t *ev = nullptr) const {
        if (ev) STAG_CUDA_OK(cudaEventRecord(ev[0], st));
        int rc = dslash_oe_cg_dispatch(ctx, packed, prec, recon, p_base(), ws + lay.w, state, st);
        if (rc) return rc;
        if (ev) STAG_CUDA_OK(cudaEventRecord(ev[1], st));
        rc = dslash_eo_fused_dispatch(ctx, packed, prec, recon, ws + lay.w, p_base(), ws + lay.q,
                                      state, partials, st);
        if (rc) return rc;
        if (ev) STAG_CUDA_OK(cudaEventRecord(ev[2], st));
        STAG_LAUNCH_K(ctx, (cg_update_r_kernel<T, BLOCK>), grid, BLOCK, 0, st, nchunk, ws + lay.r, ws + lay.q, state, partials);
        if (ev) STAG_CUDA_OK(cudaEventRecord(ev[3], st));
        STAG_LAUNCH_K(ctx, (cg_update_shifts_kernel<T, BLOCK>), grid, BLOCK, 0, st, nchunk, ws + lay.r, ws + lay.p,
                      lay.vec_stride, x, x_stride, state);
        if (ev) STAG_CUDA_OK(cudaEventRecord(ev[4], st));
        STAG_CUDA_OK(cudaGetLastError());
        return STAG_OK;
    }
};


// multi-kernel path: four launches per iteration, batches replayed as a CUDA graph, the host
// polls the device-latched `done` word once per batch.
template <typename T>
static int run_multikernel(const CgLaunch<T> &L, Slot &slot, const void *b, void *y, int maxiter, int *launches_out) {
    typedef CgLaunch<T> Lz;
    const stag_ctx *ctx = L.ctx;
    cudaStream_t st = L.st;
    STAG_LAUNCH_K(ctx, (cg_init_kernel<T, Lz::BLOCK>), L.grid, Lz::BLOCK, 0, st, L.nchunk, static_cast<const char *>(b),
                  L.ws + L.lay.r, L.ws + L.lay.p, L.lay.vec_stride, L.x, L.x_stride, L.state, L.partials);
    STAG_CUDA_OK(cudaGetLastError());

    // iterations in batches of cg_check_every; one batch always in flight behind the one polled
    const int batch = ctx->opt.cg_check_every;
    cudaGraphExec_t gexec = nullptr;
    int rc = STAG_OK;
    // option cg_profile (measurement aid, stag_cg_profile): no graph; CUDA events around each of the four kernels
    // of iterations kProfSkip .. kProfSkip + kProfIters - 1, averaged per kernel after the solve
    constexpr int kProfSkip = 8, kProfIters = 32;
    const bool profile = ctx->opt.cg_profile != 0;
    cudaEvent_t pev[kProfIters][5];
    int nprof = 0;
    if (profile) {
        { std::lock_guard<std::mutex> lk(ctx->mu); ctx->prof_iters = 0; }
        for (int i = 0; i < kProfIters && rc == STAG_OK; ++i)
            for (int j = 0; j < 5; ++j)
                if (cudaEventCreate(&pev[i][j]) != cudaSuccess) rc = STAG_ERR_CUDA;
        if (rc) { cudaGetLastError(); return rc; }
    }
    if (ctx->opt.cg_graph && maxiter > 0 && !profile) {
        // the instantiated graph of one batch is kept in the staging slot and replayed by every later solve whose
        // launches would be identical (same buffers, storage and options: an MD trajectory makes hundreds of those)
        GraphKey key;
        std::memset(&key, 0, sizeof(key));
        key.packed = L.packed; key.ws = L.ws; key.x = L.x;
        key.prec = L.prec; key.recon = L.recon; key.nshift = L.nshift; key.base = L.base; key.batch = batch;
        key.dslash_block = ctx->opt.dslash_block; key.dslash_regs = ctx->opt.dslash_regs;
        key.dslash_ctas_per_sm = ctx->opt.dslash_ctas_per_sm; key.cg_ctas_per_sm = ctx->opt.cg_ctas_per_sm;
        if (slot.gexec && std::memcmp(&key, &slot.key, sizeof(key)) != 0) {
            cudaGraphExecDestroy(slot.gexec);
            slot.gexec = nullptr;
        }
        if (!slot.gexec) {
            cudaGraph_t graph = nullptr;
            cudaStream_t cap = nullptr;
            // capture on a private stream so the caller's stream (possibly the legacy default) is untouched
            if (cudaStreamCreateWithFlags(&cap, cudaStreamNonBlocking) != cudaSuccess) return STAG_ERR_CUDA;
            Lz Lc = L;
            Lc.st = cap;
            if (cudaStreamBeginCapture(cap, cudaStreamCaptureModeThreadLocal) != cudaSuccess) rc = STAG_ERR_CUDA;
            for (int j = 0; j < batch && rc == STAG_OK; ++j) rc = Lc.iteration();
            if (cudaStreamEndCapture(cap, &graph) != cudaSuccess) rc = rc ? rc : STAG_ERR_CUDA;
            if (rc == STAG_OK && cudaGraphInstantiate(&slot.gexec, graph, 0) != cudaSuccess) rc = STAG_ERR_CUDA;
            if (graph) cudaGraphDestroy(graph);
            cudaStreamDestroy(cap);
            if (rc) { cudaGetLastError(); slot.gexec = nullptr; return rc; }
            slot.key = key;
        }
        gexec = slot.gexec;
    }
    volatile int *poll = slot.pinned_flags + 8;      // two words: poll[0], poll[1]
    cudaEvent_t *ev = slot.ev;
    const int nbatch = (maxiter + batch - 1) / batch;
    int launches = 1;
    for (int k = 0; k <= nbatch && rc == STAG_OK; ++k) {
        if (k < nbatch) {
            launches += 4 * batch;
            if (gexec) {
                if (cudaGraphLaunch(gexec, st) != cudaSuccess) rc = STAG_ERR_CUDA;
            } else {
                for (int j = 0; j < batch && rc == STAG_OK; ++j) {
                    const int it = k * batch + j;
                    const bool rec = profile && it >= kProfSkip && nprof < kProfIters;
                    rc = L.iteration(rec ? pev[nprof] : nullptr);
                    nprof += rec;
                }
            }
            if (rc == STAG_OK &&
                (cudaMemcpyAsync((void *)(poll + (k & 1)), &L.state->done, sizeof(int),
                                 cudaMemcpyDeviceToHost, st) != cudaSuccess ||
                 cudaEventRecord(ev[k & 1], st) != cudaSuccess))
                rc = STAG_ERR_CUDA;
        }
        if (k > 0 && rc == STAG_OK) {                 // look at the batch before the one just queued
            if (cudaEventSynchronize(ev[(k - 1) & 1]) != cudaSuccess) rc = STAG_ERR_CUDA;
            else if (poll[(k - 1) & 1] != 0) break;
        }
    }
    if (profile) {
        double sum[4] = {0.0, 0.0, 0.0, 0.0};
        if (rc == STAG_OK && nprof > 0 && cudaEventSynchronize(pev[nprof - 1][4]) == cudaSuccess) {
            for (int i = 0; i < nprof; ++i)
                for (int j = 0; j < 4; ++j) {
                    float ms = 0.f;
                    cudaEventElapsedTime(&ms, pev[i][j], pev[i][j + 1]);
                    sum[j] += ms * 1e3;
                }
            std::lock_guard<std::mutex> lk(ctx->mu);         // stag_cg_profile may be called from another thread
            for (int j = 0; j < 4; ++j) ctx->prof_us[j] = sum[j] / nprof;
            ctx->prof_iters = nprof;        // (iterations run after the latch closed would count as ~0: stop is far here)
        }
        for (int i = 0; i < kProfIters; ++i)
            for (int j = 0; j < 5; ++j) cudaEventDestroy(pev[i][j]);
    }
    if (rc) { cudaGetLastError(); return rc; }

    if (y) {
        ++launches;
        STAG_LAUNCH_K(ctx, (cg_partial_fraction_kernel<T, Lz::BLOCK>), L.grid, Lz::BLOCK, 0, st, L.nchunk,
                      static_cast<const char *>(b), L.x, L.x_stride, static_cast<char *>(y), L.state);
        STAG_CUDA_OK(cudaGetLastError());
    }
    *launches_out = launches;
    return STAG_OK;
}

template <typename T>
static int run_cg(const stag_ctx *ctx, Slot &slot, const void *packed, int prec, int recon, const void *b,
                  double mass, int nshift, const double *shifts, const double *residues,
                  double residue0, double stop, int maxiter, void *x, void *y, void *workspace,
                  stag_cg_info *info, cudaStream_t st) {
    typedef CgLaunch<T> Lz;
    Lz L;
    L.ctx = ctx; L.packed = packed; L.prec = prec; L.recon = recon; L.st = st;
    L.ws = static_cast<char *>(workspace);
    cg_workspace_layout(ctx, prec, nshift, &L.lay);
    L.state = reinterpret_cast<CgState *>(L.ws + L.lay.state);
    L.partials = reinterpret_cast<double *>(L.ws + L.lay.partials);
    L.x = static_cast<char *>(x);
    L.x_stride = (size_t)ctx->g.Vh * vec_bytes_per_site(prec);
    L.nshift = nshift;
    L.nchunk = (long)ctx->g.Vh * 6 / Vec16<T>::n;
    {
        const long want = (L.nchunk + Lz::BLOCK - 1) / Lz::BLOCK;
        const long cap = (long)ctx->num_sms * ctx->opt.cg_ctas_per_sm;
        L.grid = (int)(want < cap ? want : cap);
    }
    int base = 0;
    for (int i = 1; i < nshift; ++i)
        if (shifts[i] < shifts[base]) base = i;
    L.base = base;

    // initial state, staged through the ctx's pinned buffer
    CgState *h = static_cast<CgState *>(slot.pinned_info);
    memset(h, 0, sizeof(*h));
    h->alpha_old = 1.0; h->beta_old = 0.0;
    h->c0 = mass * mass + shifts[base];
    h->stop = stop; h->residue0 = residue0;
    for (int i = 0; i < nshift; ++i) {
        h->delta[i] = shifts[i] - shifts[base];
        h->zeta[i] = 1.0; h->theta[i] = 1.0; h->active[i] = 1;
        h->residues[i] = residues ? residues[i] : 0.0;
        h->resid_shift[i] = 1.0;
    }
    h->nshift = nshift; h->base = base; h->maxiter = maxiter;
    h->freeze = ctx->opt.cg_freeze; h->fp32 = (prec == STAG_F32);
    if (maxiter == 0) h->done = 2;
    STAG_CUDA_OK(cudaMemcpyAsync(L.state, h, sizeof(CgState), cudaMemcpyHostToDevice, st));
    int launches = 0;
    bool persistent = ctx->opt.cg_persistent != 0 && cg_persistent_fits(ctx, prec);
    if (persistent) {
        // small lattice: the whole solve is one cooperative launch (stag_cg_persist.cu)
        const int prc = cg_persistent_dispatch(ctx, packed, prec, recon, b, nshift, shifts, x, L.x_stride, y, L.ws,
                                               L.lay, st);
        if (prc == STAG_ERR_UNSUPPORTED) persistent = false;       // cannot be co-resident: multi-kernel path
        else if (prc) { cudaGetLastError(); return prc; }
        else launches = 1;
    }
    if (!persistent) {
        const int mrc = run_multikernel(L, slot, b, y, maxiter, &launches);
        if (mrc) return mrc;
    }
    STAG_CUDA_OK(cudaMemcpyAsync(h, L.state, sizeof(CgState), cudaMemcpyDeviceToHost, st));
    STAG_CUDA_OK(cudaStreamSynchronize(st));
    if (info) {
        memset(info, 0, sizeof(*info));
        info->iters = h->iter;
        info->converged = h->converged;
        info->breakdown = h->breakdown;
        info->stagnated = h->stagnated;
        info->bnorm2 = h->bb;
        info->rnorm2 = h->rr;
        info->kernel_launches = launches;
        for (int i = 0; i < nshift; ++i) {
            info->resid_iter[i] = h->bb > 0.0 ? h->resid_shift[i] : 0.0;
            info->iters_shift[i] = h->iters_shift[i];
        }
    }
    if (h->breakdown) return STAG_ERR_BREAKDOWN;
    if (!h->converged) return STAG_ERR_NOTCONV;
    return STAG_OK;
}

}  // namespace stag

using namespace stag;

int stag::mshift_cg_impl(const stag_ctx *ctx, Slot &slot, const void *packed, int prec, int recon,
                         const void *b_even, double mass, int nshift,
                         const double *host_shifts, const double *host_residues,
                         double residue0, double stop, int maxiter, void *x_even,
                         void *y_even, void *workspace, stag_cg_info *info, void *stream) {
    if (!ctx || !packed || !b_even || !host_shifts || !x_even || !workspace) return STAG_ERR_BADARG;
    if (!valid_prec(prec) || !valid_recon(recon)) return STAG_ERR_BADARG;
    if (nshift < 1 || nshift > STAG_MAX_SHIFTS || !(stop > 0.0) || maxiter < 0) return STAG_ERR_BADARG;
    if (y_even && !host_residues) return STAG_ERR_BADARG;
    double smin = host_shifts[0];
    for (int i = 0; i < nshift; ++i) {
        if (!(host_shifts[i] >= 0.0)) return STAG_ERR_BADARG;
        if (host_shifts[i] < smin) smin = host_shifts[i];
    }
    if (!(mass * mass + smin > 0.0)) return STAG_ERR_BADARG;
    if (((uintptr_t)workspace & 255) != 0) return STAG_ERR_BADARG;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (prec != STAG_F32)
        return run_cg<double>(ctx, slot, packed, prec, recon, b_even, mass, nshift, host_shifts,
                              host_residues, residue0, stop, maxiter, x_even, y_even, workspace,
                              info, st);
    return run_cg<float>(ctx, slot, packed, prec, recon, b_even, mass, nshift, host_shifts, host_residues,
                         residue0, stop, maxiter, x_even, y_even, workspace, info, st);
}

extern "C" int stag_mshift_cg(const stag_ctx *ctx, const void *packed, int prec, int recon,
                              const void *b_even, double mass, int nshift,
                              const double *host_shifts, const double *host_residues,
                              double residue0, double stop, int maxiter, void *x_even,
                              void *y_even, void *workspace, stag_cg_info *info, void *stream) {
    if (!ctx) return STAG_ERR_BADARG;
    SlotLease lease(ctx);
    return mshift_cg_impl(ctx, lease.slot(), packed, prec, recon, b_even, mass, nshift, host_shifts, host_residues,
                          residue0, stop, maxiter, x_even, y_even, workspace, info, stream);
}
