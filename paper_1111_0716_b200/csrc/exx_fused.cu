// exx_fused.cu — fused three-pass pipeline (placeholder until the generic path is parity-green).
#include "exx_internal.h"

namespace exx {
bool fused_supported(const exx_ctx*) { return false; }
int fused_create(exx_ctx*) { return EXX_OK; }
void fused_destroy(exx_ctx*) {}
int fused_apply(exx_ctx*, const double*, const double2*, double2*) { return EXX_ERR_BAD_ARG; }
}  // namespace exx
