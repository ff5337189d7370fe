// stag_cg_persist_r2.cu — instantiations of the multi-source persistent CG kernel for R = 2 sources per link read.
#include "stag_cg_persist_block.cuh"
namespace stag {
STAG_DEFINE_PERSIST_BLOCK_R(2)
}
