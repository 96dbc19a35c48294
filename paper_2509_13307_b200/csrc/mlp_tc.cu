// mlp_tc.cu -- tcgen05/TMEM emulator GEMMs (placeholder: not built yet, SIMT path is used).
#include "internal.cuh"

nsgpu_status mlp_tc_prepare(nsgpu_ctx* ctx, int e, const nsgpu_emulator*) {
  if ((ctx->flags & 3u) == NSGPU_MLP_TC) { ctx->err = "tcgen05 MLP path not built"; return NSGPU_ESHAPE; }
  ctx->emu[e].path = 0;
  return NSGPU_OK;
}
void mlp_tc_release(nsgpu_ctx*, int) {}
nsgpu_status mlp_forward_tc(nsgpu_ctx* ctx, int, const float*, int, const int*, float*, bool, cudaStream_t) {
  ctx->err = "tcgen05 MLP path not built";
  return NSGPU_ESHAPE;
}
