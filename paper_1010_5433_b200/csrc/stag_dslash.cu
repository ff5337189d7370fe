// stag_dslash.cu — stag_dslash_eo / stag_dslash_oe and the two Dslash launches of a CG
// iteration.  One kernel launch per application.  ("Dirac kernel"; SURVEY.md §8(a)
// rows a2, a3.)
//
// MODE 0  out = D in                                            (stag_dslash_eo / _oe)
// MODE 1  the same, but a no-op once the CG has latched `done`  (a2 inside stag_mshift_cg)
// MODE 2  q = c0 p - D w,  partial sums of Re<p,q>, and — in the last CTA to finish — the
//         scalar recurrences that follow <p,q>                  (a3 + a4 inside stag_mshift_cg)
#include "stag_cg.cuh"
#include "stag_dslash.cuh"

namespace stag {

// Register budget: 64 per thread (1024 resident threads / SM, so that the 1024 CTAs of a
// 32^3x8 lattice are one wave), except fp64 12-real whose row-3 rebuild needs ~100.
// RT = resident threads per SM the kernel is compiled for: 1024 (64 registers each), 512 (128) or
// 256 (255): fewer threads, each with a deeper queue of independent loads.
template <int BLOCK, int RT>
constexpr int min_ctas() { return RT / BLOCK > 0 ? RT / BLOCK : 1; }

template <typename T, int RECON, int BLOCK, int MODE, int RT, bool SPLIT = false>
__global__ void __launch_bounds__(BLOCK, (min_ctas<BLOCK, RT>()))
dslash_kernel(const Geom g, const char *__restrict__ W, const char *__restrict__ in,
              char *__restrict__ out, const int par, const char *__restrict__ p,
              CgState *__restrict__ state, double *__restrict__ partials) {
    __shared__ double red[BLOCK / 32 + 1];
    if (MODE != 0) {
        const int done = *reinterpret_cast<volatile int *>(&state->done);
        if (done != 0) {
            // the x/p update of the converged iteration has run by now: close the latch
            if (MODE == 1 && done == 1 && blockIdx.x == 0 && threadIdx.x == 0) state->done = 2;
            return;
        }
    }
    double dot = 0.0;
    T c0 = T(0);
    if (MODE == 2) c0 = (T)state->c0;
    for (int e = blockIdx.x * BLOCK + threadIdx.x; e < g.Vh; e += gridDim.x * BLOCK) {
        T acc[6];
        dslash_site<T, RECON, true, SPLIT>(g, W, in, par, e, acc);
        if (MODE == 2) {
            T pv[6];
            load_vec(p, g.Vh, e, pv);
#pragma unroll
            for (int k = 0; k < 6; ++k) {
                acc[k] = c0 * pv[k] - acc[k];
                dot += (double)pv[k] * (double)acc[k];
            }
        }
        store_vec(out, g.Vh, e, acc);
    }
    if (MODE == 2) {
        double total;
        if (grid_sum_last_cta<BLOCK>(dot, partials, &state->ticket, red, total) && threadIdx.x < 32)
            cg_scalars_after_pq(state, total);
    }
}

// N1: R sources through one link read.  thread = one output site, ALL R sources: the 8 hopping
// matrices are loaded into registers once and applied to the R gathered neighbours in turn, so both
// the HBM bytes and the load-instruction count of the links are paid once per site, not per source.
template <typename T, int RECON, int BLOCK, int RT, int R, bool SPLIT = false>
__global__ void __launch_bounds__(BLOCK, (min_ctas<BLOCK, RT>()))
dslash_block_kernel(const Geom g, const char *__restrict__ W, const char *__restrict__ in,
                    char *__restrict__ out, const int par, const size_t stride, const int nrhs) {
    const int e = blockIdx.x * BLOCK + threadIdx.x;
    if (e >= g.Vh) return;
    const char *ins[R];
#pragma unroll
    for (int r = 0; r < R; ++r) ins[r] = in + (size_t)(r < nrhs ? r : 0) * stride;
    T acc[R][6];
    dslash_site_multi<T, RECON, R, true, SPLIT>(g, W, ins, (1u << nrhs) - 1u, par, e, acc);
#pragma unroll
    for (int r = 0; r < R; ++r)
        if (r < nrhs) store_vec(out + (size_t)r * stride, g.Vh, e, acc[r]);
}

template <typename T, int RECON, int R, bool SPLIT = false>
static int launch_dslash_block(const stag_ctx *ctx, const void *packed, const void *in, void *out, int par,
                               int nrhs, cudaStream_t st) {
    const Geom &g = ctx->g;
    constexpr int BLOCK = 128;
    const size_t stride = (size_t)g.Vh * 6 * sizeof(T);
    const int grid = (g.Vh + BLOCK - 1) / BLOCK;
    const char *W = static_cast<const char *>(packed);
    // registers: R accumulators + one matrix + one neighbour.  fp64: 128 per thread up to R = 2, 255 at
    // R = 4 (24 fp64 accumulators alone are 48 registers); fp32: 64 / 128.
    constexpr int RT = sizeof(T) == 8 ? (R >= 4 ? 256 : 512) : (R >= 2 ? 512 : 1024);
    STAG_LAUNCH_K(ctx, (dslash_block_kernel<T, RECON, BLOCK, RT, R, SPLIT>), grid, BLOCK, 0, st, g, W,
                  static_cast<const char *>(in), static_cast<char *>(out), par, stride, nrhs);
    STAG_CUDA_OK(cudaGetLastError());
    return STAG_OK;
}

template <typename T, int RECON, bool SPLIT = false>
static int dslash_block_r(const stag_ctx *ctx, const void *packed, const void *in, void *out, int par,
                          int nrhs, cudaStream_t st) {
    if (nrhs == 1) return launch_dslash_block<T, RECON, 1, SPLIT>(ctx, packed, in, out, par, nrhs, st);
    if (nrhs == 2) return launch_dslash_block<T, RECON, 2, SPLIT>(ctx, packed, in, out, par, nrhs, st);
    return launch_dslash_block<T, RECON, 4, SPLIT>(ctx, packed, in, out, par, nrhs, st);
}

static int dslash_grid(const stag_ctx *ctx, int block, bool persistent_default) {
    const int tiles = (ctx->g.Vh + block - 1) / block;
    int per_sm = ctx->opt.dslash_ctas_per_sm;
    if (per_sm == 0 && persistent_default) per_sm = 1024 / block;   // fused kernel: one fence per CTA
    if (per_sm == 0) return tiles;
    const int grid = ctx->num_sms * per_sm;
    return grid < tiles ? grid : tiles;
}

template <typename T, int RECON, int MODE>
static int launch_dslash(const stag_ctx *ctx, const void *packed, const void *in, void *out,
                         int par, const void *p, CgState *state, double *partials,
                         cudaStream_t st) {
    const Geom &g = ctx->g;
    const char *W = static_cast<const char *>(packed);
    const char *i = static_cast<const char *>(in);
    const char *pp = static_cast<const char *>(p);
    char *o = static_cast<char *>(out);
    const int block = ctx->opt.dslash_block;
    const int grid = dslash_grid(ctx, block, MODE == 2);
    // dslash_regs = 0 (auto): measured best at 32^3x8 and 64^4 (profiles/README.md) — fp64 wants 128
    // registers (18-real: no spills, deeper load queue; 12-real: the row-3 rebuild needs ~100),
    // fp32 wants 64 and twice the threads.
    int regs = ctx->opt.dslash_regs;
    if (regs == 0) regs = sizeof(T) == 8 ? 128 : 64;
    if (regs == 64 && sizeof(T) == 8 && RECON == 12) regs = 128;
#define STAG_LAUNCH(B)                                                                                            \
    if (regs == 64) STAG_LAUNCH_K(ctx, (dslash_kernel<T, RECON, B, MODE, 1024>), grid, B, 0, st, g, W, i, o, par, pp, state, partials);      \
    else if (regs == 128) STAG_LAUNCH_K(ctx, (dslash_kernel<T, RECON, B, MODE, 512>), grid, B, 0, st, g, W, i, o, par, pp, state, partials); \
    else STAG_LAUNCH_K(ctx, (dslash_kernel<T, RECON, B, MODE, 256>), grid, B, 0, st, g, W, i, o, par, pp, state, partials)
    switch (block) {
        case 64: STAG_LAUNCH(64); break;
        case 256: STAG_LAUNCH(256); break;
        default: STAG_LAUNCH(128); break;
    }
#undef STAG_LAUNCH
    STAG_CUDA_OK(cudaGetLastError());
    return STAG_OK;
}

// N3: split-double links, fp64 vectors.  One configuration: 128 threads, 128 registers (the fp64 default).
template <int RECON, int MODE>
static int launch_dslash_split(const stag_ctx *ctx, const void *packed, const void *in, void *out, int par,
                               const void *p, CgState *state, double *partials, cudaStream_t st) {
    const Geom &g = ctx->g;
    const int grid = dslash_grid(ctx, 128, MODE == 2);
    STAG_LAUNCH_K(ctx, (dslash_kernel<double, RECON, 128, MODE, 512, true>), grid, 128, 0, st, g,
                  static_cast<const char *>(packed), static_cast<const char *>(in), static_cast<char *>(out), par,
                  static_cast<const char *>(p), state, partials);
    STAG_CUDA_OK(cudaGetLastError());
    return STAG_OK;
}

template <int MODE>
static int dispatch(const stag_ctx *ctx, const void *packed, int prec, int recon, const void *in,
                    void *out, int par, const void *p, CgState *state, double *partials,
                    void *stream) {
    if (!ctx || !packed || !in || !out || in == out) return STAG_ERR_BADARG;
    if (!valid_prec(prec) || !valid_recon(recon)) return STAG_ERR_BADARG;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (prec == STAG_F64_SPLIT)
        return recon == 18 ? launch_dslash_split<18, MODE>(ctx, packed, in, out, par, p, state, partials, st)
                           : launch_dslash_split<12, MODE>(ctx, packed, in, out, par, p, state, partials, st);
    if (prec == STAG_F64)
        return recon == 18
                   ? launch_dslash<double, 18, MODE>(ctx, packed, in, out, par, p, state, partials, st)
                   : launch_dslash<double, 12, MODE>(ctx, packed, in, out, par, p, state, partials, st);
    return recon == 18
               ? launch_dslash<float, 18, MODE>(ctx, packed, in, out, par, p, state, partials, st)
               : launch_dslash<float, 12, MODE>(ctx, packed, in, out, par, p, state, partials, st);
}

int dslash_dispatch(const stag_ctx *ctx, const void *packed, int prec, int recon, const void *in,
                    void *out, int par, void *stream) {
    return dispatch<0>(ctx, packed, prec, recon, in, out, par, nullptr, nullptr, nullptr, stream);
}

int dslash_oe_cg_dispatch(const stag_ctx *ctx, const void *packed, int prec, int recon,
                          const void *p_even, void *w_odd, CgState *state, void *stream) {
    return dispatch<1>(ctx, packed, prec, recon, p_even, w_odd, 1, nullptr, state, nullptr, stream);
}

int dslash_eo_fused_dispatch(const stag_ctx *ctx, const void *packed, int prec, int recon,
                             const void *w_odd, const void *p_even, void *q_even, CgState *state,
                             double *partials, void *stream) {
    return dispatch<2>(ctx, packed, prec, recon, w_odd, q_even, 0, p_even, state, partials, stream);
}

// implemented in stag_dslash_pipe.cu
int dslash_pipe_dispatch(const stag_ctx *ctx, const void *packed, int prec, int recon, int par, int nrhs,
                         const void *in, void *out, cudaStream_t st);

}  // namespace stag

extern "C" int stag_dslash_block(const stag_ctx *ctx, const void *packed, int prec, int recon,
                                 int out_parity, int nrhs, const void *in, void *out, void *stream) {
    using namespace stag;
    if (!ctx || !packed || !in || !out || in == out) return STAG_ERR_BADARG;
    if (!valid_prec(prec) || !valid_recon(recon) || (out_parity != 0 && out_parity != 1)) return STAG_ERR_BADARG;
    if (nrhs < 1 || nrhs > STAG_MAX_SHIFTS) return STAG_ERR_BADARG;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    // split-double links (N3): the register-staged kernel rebuilds a = b + c as it loads; the cp.async ring copies
    // raw bytes into its slots and has no such variant
    if (ctx->opt.dslash_pipe != 0 && prec != STAG_F64_SPLIT) {
        const int rc = dslash_pipe_dispatch(ctx, packed, prec, recon, out_parity, nrhs, in, out, st);
        if (rc != STAG_ERR_UNSUPPORTED) return rc;
    }
    if (nrhs > STAG_MAX_RHS) {                       // groups of STAG_MAX_RHS, one launch each
        const size_t vb = (size_t)ctx->g.Vh * vec_bytes_per_site(prec);
        for (int i0 = 0; i0 < nrhs; i0 += STAG_MAX_RHS) {
            const int n = nrhs - i0 < STAG_MAX_RHS ? nrhs - i0 : STAG_MAX_RHS;
            const int rc = stag_dslash_block(ctx, packed, prec, recon, out_parity, n, static_cast<const char *>(in) + i0 * vb,
                                             static_cast<char *>(out) + i0 * vb, stream);
            if (rc) return rc;
        }
        return STAG_OK;
    }
    if (prec == STAG_F64_SPLIT)
        return recon == 18 ? dslash_block_r<double, 18, true>(ctx, packed, in, out, out_parity, nrhs, st)
                           : dslash_block_r<double, 12, true>(ctx, packed, in, out, out_parity, nrhs, st);
    if (prec == STAG_F64)
        return recon == 18 ? dslash_block_r<double, 18>(ctx, packed, in, out, out_parity, nrhs, st)
                           : dslash_block_r<double, 12>(ctx, packed, in, out, out_parity, nrhs, st);
    return recon == 18 ? dslash_block_r<float, 18>(ctx, packed, in, out, out_parity, nrhs, st)
                       : dslash_block_r<float, 12>(ctx, packed, in, out, out_parity, nrhs, st);
}

extern "C" int stag_dslash_eo(const stag_ctx *ctx, const void *packed, int prec, int recon,
                              const void *in_odd, void *out_even, void *stream) {
    return stag::dslash_dispatch(ctx, packed, prec, recon, in_odd, out_even, 0, stream);
}

extern "C" int stag_dslash_oe(const stag_ctx *ctx, const void *packed, int prec, int recon,
                              const void *in_even, void *out_odd, void *stream) {
    return stag::dslash_dispatch(ctx, packed, prec, recon, in_even, out_odd, 1, stream);
}
