// stag_cg_persist_r4.cu — instantiations of the multi-source persistent CG kernel for R = 4 sources per link read.
#include "stag_cg_persist_block.cuh"
namespace stag {
STAG_DEFINE_PERSIST_BLOCK_R(4)
}
