// placeholder until the tensor-core kernel lands
#include "bf_internal.h"
bool bf_umma_supported(const bf_ctx *, const char **why) { *why = "not built yet"; return false; }
cudaError_t bf_launch_umma(const BfParams &, int, int, cudaStream_t) { return cudaErrorNotSupported; }
