// fused_inst_tn32.cu -- explicit instantiations of the fused kernel for the 32-token tile.
#include "fused_kernel.cuh"

namespace twq {
TWQ_DEFINE_INST(32)
}  // namespace twq
