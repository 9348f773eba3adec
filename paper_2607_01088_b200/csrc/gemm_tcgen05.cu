#include "rosa_internal.h"
namespace rosa {
bool tc_gemm_supported(int N, int K) { return false; }
cudaError_t launch_gemm_tc(Epi, const bf16*, const bf16*, int, int, int, const EpiArgs&, cudaStream_t) { return cudaErrorNotSupported; }
}
