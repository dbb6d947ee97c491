// fused_inst_tn128p.cu -- explicit instantiations of the fused kernel for the 128-token tile in CTA-pair mode
// (cta_group::2: two CTAs of a cluster share one M = 256 MMA, each expanding half of the activation rows).
#include "fused_kernel.cuh"

namespace twq {
template cudaError_t launch_fused_inst<128, 128, false, true>(const FusedMaps&, const FusedParams&, cudaStream_t);
template cudaError_t launch_fused_inst<128, 128, true, true>(const FusedMaps&, const FusedParams&, cudaStream_t);
template cudaError_t launch_fused_inst<128, 64, false, true>(const FusedMaps&, const FusedParams&, cudaStream_t);
template cudaError_t launch_fused_inst<128, 64, true, true>(const FusedMaps&, const FusedParams&, cudaStream_t);
}  // namespace twq
