// placeholder: replaced by the tcgen05 kernels
#include "internal.h"
namespace pinsage {
bool gemm_tc_supported(const GemmArgs &, const char **why) { if (why) *why = "tcgen05 GEMM not built yet"; return false; }
cudaError_t launch_gemm_tc(const GemmArgs &, int, cudaStream_t, int *) { return cudaErrorNotSupported; }
size_t gemm_tc_scratch_bytes(const GemmArgs &) { return 0; }
}
