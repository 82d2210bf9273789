// tcgen05 / TMEM / TMA versions of the two contractions (placeholder until the kernels land).
#include "bip_internal.h"

namespace bip {

bool tc_available() { return false; }

int32_t launch_gemm1_tc(bip_ctx* ctx, const Gemm1Args&) { return fail(ctx, BIP_ERR_UNSUPPORTED, "tensor-core GEMM1 not built"); }
int32_t launch_gemm2_tc(bip_ctx* ctx, const Gemm2Args&) { return fail(ctx, BIP_ERR_UNSUPPORTED, "tensor-core GEMM2 not built"); }

}  // namespace bip
