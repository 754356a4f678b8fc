// tcgen05 / TMA grouped GEMM path (placeholder until the kernels land; the SIMT path serves every shape meanwhile).
#include "common.cuh"

namespace fomoe {
bool umma_supported(const fomoe_config&) { return false; }
int umma_ffn_fwd(const fomoe_config&, int, const void*, const RouteWs&, const ActWs&, const ScratchWs&, const FfnPtrs&, cudaStream_t) {
  return FOMOE_ERR_UNSUPPORTED;
}
int umma_ffn_bwd(const fomoe_config&, int, const void*, const void*, const RouteWs&, const ActWs&, const ScratchWs&, const FfnPtrs&,
                 void*, void*, void*, void*, void*, void*, cudaStream_t) {
  return FOMOE_ERR_UNSUPPORTED;
}
}  // namespace fomoe
