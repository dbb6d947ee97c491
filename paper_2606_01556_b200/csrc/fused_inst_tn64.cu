// fused_inst_tn64.cu -- explicit instantiations of the fused kernel for the 64-token tile.
#include "fused_kernel.cuh"

namespace twq {
TWQ_DEFINE_INST(64)
}  // namespace twq
