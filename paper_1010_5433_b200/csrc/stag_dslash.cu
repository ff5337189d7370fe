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
template <typename T, int RECON, int BLOCK>
constexpr int min_ctas() { return (sizeof(T) == 8 && RECON == 12 ? 512 : 1024) / BLOCK; }

template <typename T, int RECON, int BLOCK, int MODE>
__global__ void __launch_bounds__(BLOCK, (min_ctas<T, RECON, BLOCK>()))
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
        dslash_site<T, RECON>(g, W, in, par, e, acc);
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
    switch (block) {
        case 64:
            dslash_kernel<T, RECON, 64, MODE><<<grid, 64, 0, st>>>(g, W, i, o, par, pp, state, partials);
            break;
        case 256:
            dslash_kernel<T, RECON, 256, MODE><<<grid, 256, 0, st>>>(g, W, i, o, par, pp, state, partials);
            break;
        default:
            dslash_kernel<T, RECON, 128, MODE><<<grid, 128, 0, st>>>(g, W, i, o, par, pp, state, partials);
            break;
    }
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

}  // namespace stag

extern "C" int stag_dslash_eo(const stag_ctx *ctx, const void *packed, int prec, int recon,
                              const void *in_odd, void *out_even, void *stream) {
    return stag::dslash_dispatch(ctx, packed, prec, recon, in_odd, out_even, 0, stream);
}

extern "C" int stag_dslash_oe(const stag_ctx *ctx, const void *packed, int prec, int recon,
                              const void *in_even, void *out_odd, void *stream) {
    return stag::dslash_dispatch(ctx, packed, prec, recon, in_even, out_odd, 1, stream);
}
