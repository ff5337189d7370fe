// stag_cg_persist_r2.cu — instantiations of the persistent CG kernel for R = 2 sources per link read.
#include "stag_cg_persist.cuh"
namespace stag {
STAG_DEFINE_PERSIST_R(2)
}
