// l_max = 3 backward instantiations.  TF32 mode (precision 1): the mma.sync kernels of tp3mb_impl.cuh for the two wide
// layers (NEXT-2; the paper runs the tensor product in TF32); fp32 modes: the blocked
// 32-channel FFMA kernels of tp2_impl.cuh.  The scalar-output last layer always runs the tp2 kernel.
#include "tp3mb_impl.cuh"

int tp2_l3_bwd(allegro_model* m, const TP2Common& q, int pat) {
  const bool mma = tp3m_bwd_active(m);
  if (pat == P_16_16_31) {
    TP2<Pat<P_16_16_31>::NNZ> a{}; AL_CHECK(fill2(m, q, a));
    if (mma) return launch_bwd3m<P_16_16_31, true>(m, a);
    return launch_bwd2<P_16_16_31, 4, true, true, false, 2, 2>(m, a);
  }
  if (pat == P_16_31_16) {
    TP2<Pat<P_16_31_16>::NNZ> a{}; AL_CHECK(fill2(m, q, a));
    if (mma) return launch_bwd3m<P_16_31_16, false>(m, a);
    return launch_bwd2<P_16_31_16, 8, false, true, false, 2, 2>(m, a);
  }
  if (pat == P_16_16_1) { TP2<Pat<P_16_16_1>::NNZ> a{}; AL_CHECK(fill2(m, q, a)); return launch_bwd2<P_16_16_1, 16, false, false, true, 2, 4>(m, a); }
  return ALLEGRO_ERR_UNIMPLEMENTED;
}
