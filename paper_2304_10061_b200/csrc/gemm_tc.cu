// tcgen05 (TF32 / BF16) tensor-core GEMM path — placeholder until the tcgen05 kernel lands.
#include "gemm.h"
#include "internal.h"

int al_gemm_tc(allegro_model* m, const GemmArgs& g) {
  (void)g;
  al_set_error(m, "precision >= 1 (tensor-core GEMMs) not implemented yet");
  return ALLEGRO_ERR_UNIMPLEMENTED;
}

int al_upload_bf16(allegro_model* m, void** dst, const std::vector<float>& h) {
  (void)h;
  *dst = nullptr;
  (void)m;
  return ALLEGRO_OK;
}
