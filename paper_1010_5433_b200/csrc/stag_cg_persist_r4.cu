// stag_cg_persist_r4.cu — instantiations of the persistent CG kernel for R = 4 sources per link read.
#include "stag_cg_persist.cuh"
namespace stag {
STAG_DEFINE_PERSIST_R(4)
}
