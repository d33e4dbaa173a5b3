// placeholder until the wide kernel lands
#include "spense_internal.cuh"
namespace spense {
int launch_gemm_wide(const GemmParams&, const CUtensorMap&, const CUtensorMap&, const CUtensorMap&, bool, int, int, cudaStream_t) {
  return SPENSE_ERR_CUDA;
}
}  // namespace spense
