// l_max = 3 forward instantiations: lane-split kernels (tp3_impl.cuh) for the wide layers, the 32-channel
// kernel of tp2_impl.cuh for the scalar-output last layer.
#include "tp3_impl.cuh"

int tp2_l3_fwd(allegro_model* m, const TP2Common& q, int pat) {
  if (pat == P_16_16_31) { TP2<Pat<P_16_16_31>::NNZ> a{}; AL_CHECK(fill2(m, q, a)); return launch_fwd3<P_16_16_31, true, 8, 4>(m, a); }
  if (pat == P_16_31_16) { TP2<Pat<P_16_31_16>::NNZ> a{}; AL_CHECK(fill2(m, q, a)); return launch_fwd3<P_16_31_16, false, 4, 4>(m, a); }
  if (pat == P_16_16_1) { TP2<Pat<P_16_16_1>::NNZ> a{}; AL_CHECK(fill2(m, q, a)); return launch_fwd2<P_16_16_1, 1, false, 3, 4>(m, a); }
  return ALLEGRO_ERR_UNIMPLEMENTED;
}
