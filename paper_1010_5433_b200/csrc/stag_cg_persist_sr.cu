// stag_cg_persist_sr.cu — instantiations and dispatch of the single-reduction persistent CG kernel
// (stag_cg_persist_sr.cuh): fp64 / fp32 / split-double links, 18- and 12-real, at the default CTA sizes.
#include "stag_cg_persist_sr.cuh"

namespace stag {

int cg_persistent_sr_launch(const stag_ctx *ctx, int prec, int recon, const PersistArgs &a, cudaStream_t st) {
    if (ctx->opt.cg_persistent_threads != 0) return STAG_ERR_UNSUPPORTED;     // other CTA sizes: the two-reduction kernel
    if (prec == STAG_F64)
        return recon == 18 ? launch_persistent_sr<double, 18, 512>(ctx, a, st) : launch_persistent_sr<double, 12, 512>(ctx, a, st);
    if (prec == STAG_F64_SPLIT)
        return recon == 18 ? launch_persistent_sr<double, 18, 512, true>(ctx, a, st)
                           : launch_persistent_sr<double, 12, 512, true>(ctx, a, st);
    return recon == 18 ? launch_persistent_sr<float, 18, 1024>(ctx, a, st) : launch_persistent_sr<float, 12, 1024>(ctx, a, st);
}

}  // namespace stag
