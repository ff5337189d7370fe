// stag_cg_persist_split.cu — the persistent multi-shift CG on split-double links (N3):
// fp64 vectors and scalars, every link rebuilt as (double)b + (double)c in the stencil phases.
// R = 1: stag_mshift_cg(prec = STAG_F64_SPLIT); R = 2, 4: the N2 polish of several shifts per launch.
#include "stag_cg_persist_block.cuh"

namespace stag {

int cg_persistent_launch_split(const stag_ctx *ctx, int recon, int R, const PersistArgs &a, cudaStream_t st) {
    if (R == 1)
        return recon == 12 ? launch_persistent<double, 12, 512, 1, true>(ctx, a, st)
                           : launch_persistent<double, 18, 512, 1, true>(ctx, a, st);
    if (R == 2)
        return recon == 12 ? launch_persistent_block<double, 12, 512, 2, true>(ctx, a, st)
                           : launch_persistent_block<double, 18, 512, 2, true>(ctx, a, st);
    return recon == 12 ? launch_persistent_block<double, 12, 512, 4, true>(ctx, a, st)
                       : launch_persistent_block<double, 18, 512, 4, true>(ctx, a, st);
}

}  // namespace stag
