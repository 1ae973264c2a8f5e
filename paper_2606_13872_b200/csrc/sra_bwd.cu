// SRA backward driver (placeholder until the kernels land in this file).
#include "sra_ctx.h"

namespace sra {
int run_backward(sra_ctx* ctx, const sra_bwd_args*, cudaStream_t) {
  return ctx_fail(ctx, SRA_ERR_UNSUPPORTED, "sra_backward: not implemented yet");
}
}  // namespace sra
