// stag_cg_persist_split.cu — the persistent multi-shift CG on split-double links (N3):
// fp64 vectors and scalars, every link rebuilt as (double)b + (double)c in the stencil phases.
#include "stag_cg_persist.cuh"

namespace stag {

int cg_persistent_launch_split(const stag_ctx *ctx, int recon, const PersistArgs &a, cudaStream_t st) {
    return recon == 12 ? launch_persistent<double, 12, 512, 1, true>(ctx, a, st)
                       : launch_persistent<double, 18, 512, 1, true>(ctx, a, st);
}

}  // namespace stag
