// fused_inst_tn128.cu -- explicit instantiations of the fused kernel for the 128-token tile.
#include "fused_kernel.cuh"

namespace twq {
TWQ_DEFINE_INST(128)
template int max_active_clusters_inst<128, 128, false>(int, int);
}  // namespace twq
