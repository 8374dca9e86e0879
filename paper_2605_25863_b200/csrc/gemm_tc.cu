// gemm_tc.cu -- tensor-core (tcgen05, int8 limb planes) Schur update.  Placeholder until the
// kernel lands: reports "not supported" so callers use the CUDA-core path.
#include "linac_internal.h"

namespace linac {
int gemm_modp_tc(const GemmArgs&, const ModP&, cudaStream_t, Arena*) { return -1; }
size_t gemm_modp_tc_scratch_bytes(int64_t, int64_t, int64_t) { return 0; }
}  // namespace linac
