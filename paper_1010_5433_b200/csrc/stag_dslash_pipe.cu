// stag_dslash_pipe.cu — launches of the cp.async-ring Dslash (stag_dslash_pipe.cuh) for
// stag_dslash_block: R sources per link read, matrices (and optionally the gathered neighbours)
// staged through shared memory so that the loads in flight are bounded by the 227 KB of shared
// memory per SM instead of by the register file.
#include "stag_dslash_pipe.cuh"

namespace stag {

template <typename T, int RECON, int R, int BLOCK, int STAGES, bool VA>
constexpr int pipe_ctas_per_sm() {
    constexpr int smem = STAGES * pipe_stage_bytes<T, RECON, R, BLOCK, VA>() + 1024;
    constexpr int by_smem = (227 * 1024) / smem;
    constexpr int by_threads = 1024 / BLOCK;          // never fewer than 64 registers per thread
    return by_smem < 1 ? 1 : (by_smem < by_threads ? by_smem : by_threads);
}

template <typename T, int RECON, int R, int BLOCK, int STAGES, bool VA>
__global__ void __launch_bounds__(BLOCK, (pipe_ctas_per_sm<T, RECON, R, BLOCK, STAGES, VA>()))
dslash_pipe_kernel(const Geom g, const char *__restrict__ W, const char *__restrict__ in_all,
                   char *__restrict__ out_all, const int par, const size_t stride, const int nvec) {
    extern __shared__ __align__(16) unsigned char ring[];
    // blockIdx.y = group of R vectors (stag_fermion_force: the D_oe x_i of all shifts in ONE launch, so that the
    // groups' fill / drain ramps overlap); the last group may be short
    const char *in = in_all + (size_t)blockIdx.y * R * stride;
    char *out = out_all + (size_t)blockIdx.y * R * stride;
    const int left = nvec - (int)blockIdx.y * R, nrhs = left < R ? left : R;
    const char *ins[R];
#pragma unroll
    for (int r = 0; r < R; ++r) ins[r] = in + (size_t)(r < nrhs ? r : 0) * stride;
    const unsigned mask = (1u << nrhs) - 1u;
    for (int e = blockIdx.x * BLOCK + threadIdx.x; e < g.Vh; e += gridDim.x * BLOCK) {
        T acc[R][6];
        dslash_site_pipe<T, RECON, R, BLOCK, STAGES, VA>(g, W, ins, mask, par, e, acc, ring);
#pragma unroll
        for (int r = 0; r < R; ++r)
            if (r < nrhs) store_vec(out + (size_t)r * stride, g.Vh, e, acc[r]);
    }
}

template <typename T, int RECON, int R, int BLOCK, int STAGES, bool VA>
static int launch_pipe(const stag_ctx *ctx, const void *packed, const void *in, void *out, int par, int nvec,
                       cudaStream_t st) {
    const Geom &g = ctx->g;
    constexpr int smem = STAGES * pipe_stage_bytes<T, RECON, R, BLOCK, VA>();
    if (smem > 227 * 1024 - 1024) return STAG_ERR_UNSUPPORTED;
    auto kern = dslash_pipe_kernel<T, RECON, R, BLOCK, STAGES, VA>;
    STAG_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    const int tiles = (g.Vh + BLOCK - 1) / BLOCK;
    int grid = tiles;
    if (ctx->opt.dslash_ctas_per_sm > 0) {
        const int cap = ctx->num_sms * ctx->opt.dslash_ctas_per_sm;
        if (cap < grid) grid = cap;
    }
    const size_t stride = (size_t)g.Vh * 6 * sizeof(T);
    STAG_LAUNCH_K(ctx, kern, dim3(grid, (nvec + R - 1) / R), BLOCK, smem, st, g, static_cast<const char *>(packed),
                  static_cast<const char *>(in), static_cast<char *>(out), par, stride, nvec);
    STAG_CUDA_OK(cudaGetLastError());
    return STAG_OK;
}

// Tuned at 32^3 x 8 (profiles/README.md, "N1 ring sweep"): the ring pays off where the register-staged
// kernel runs out of registers for loads in flight — fp64 at R = 4, fp32 at R >= 2.  Two stages, not
// more: shared memory per thread bounds the warps per SM, and with fewer than ~8 warps per SM the
// kernel becomes issue-bound (one warp per scheduler issues an instruction every ~4 cycles).
template <typename T, int RECON>
static int pipe_r(const stag_ctx *ctx, const void *packed, const void *in, void *out, int par, int nrhs,
                  cudaStream_t st) {
    // nrhs > 4: groups of four in one launch (blockIdx.y)
    if (sizeof(T) == 8) {
        if (nrhs <= 2) return STAG_ERR_UNSUPPORTED;               // register-staged kernel is as fast
        return launch_pipe<T, RECON, 4, 128, 2, true>(ctx, packed, in, out, par, nrhs, st);
    }
    if (nrhs == 1) return STAG_ERR_UNSUPPORTED;
    if (nrhs == 2) return launch_pipe<T, RECON, 2, 128, 3, true>(ctx, packed, in, out, par, nrhs, st);
    return launch_pipe<T, RECON, 4, 256, 2, true>(ctx, packed, in, out, par, nrhs, st);
}

// STAG_ERR_UNSUPPORTED = "use the register-staged kernel for this case"
int dslash_pipe_dispatch(const stag_ctx *ctx, const void *packed, int prec, int recon, int par, int nrhs,
                         const void *in, void *out, cudaStream_t st) {
    if (prec == STAG_F64)
        return recon == 18 ? pipe_r<double, 18>(ctx, packed, in, out, par, nrhs, st)
                           : pipe_r<double, 12>(ctx, packed, in, out, par, nrhs, st);
    return recon == 18 ? pipe_r<float, 18>(ctx, packed, in, out, par, nrhs, st)
                       : pipe_r<float, 12>(ctx, packed, in, out, par, nrhs, st);
}

}  // namespace stag
