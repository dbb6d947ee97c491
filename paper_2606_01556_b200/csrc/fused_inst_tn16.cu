// fused_inst_tn16.cu -- explicit instantiations of the fused kernel for the 16-token tile.
#include "fused_kernel.cuh"

namespace twq {
TWQ_DEFINE_INST(16)
}  // namespace twq
