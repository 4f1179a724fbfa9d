// cell_tcgen05.cu -- placeholder until the tcgen05 kernel lands: reports "not supported" so that the TF32
// mode runs the SIMT kernel with TF32-rounded operands (same arithmetic contract, slower).
#include "cell_tcgen05.h"

void tc_invalidate(pawfe_ctx*) {}
bool tc_supported(const pawfe_ctx*, int) { return false; }
pawfe_status tc_cell_apply(pawfe_ctx* ctx, const float*, long, float*, long, int, float) {
  ctx->err = "tcgen05 cell kernel not built";
  return PAWFE_EUNSUPPORTED;
}
