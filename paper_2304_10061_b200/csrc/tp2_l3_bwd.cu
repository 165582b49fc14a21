// l_max = 3 backward instantiations: the blocked 32-channel kernels of tp2_impl.cuh (default), the lane-split
// kernels of tp3_impl.cuh as measured alternatives.
#include "tp3_impl.cuh"

int tp2_l3_bwd(allegro_model* m, const TP2Common& q, int pat) {
  const int lq = t3_bwd_lq();
  if (pat == P_16_16_31) {
    TP2<Pat<P_16_16_31>::NNZ> a{}; AL_CHECK(fill2(m, q, a));
    if (lq == 2) return launch_bwd3<P_16_16_31, true, 2, 4, 4>(m, a);
    if (lq == 3) return launch_bwd3<P_16_16_31, true, 3, 4, 4>(m, a);
    return launch_bwd2<P_16_16_31, 4, true, true, false, 2, 2>(m, a);
  }
  if (pat == P_16_31_16) {
    TP2<Pat<P_16_31_16>::NNZ> a{}; AL_CHECK(fill2(m, q, a));
    if (lq == 2) return launch_bwd3<P_16_31_16, false, 2, 4, 4>(m, a);
    if (lq == 3) return launch_bwd3<P_16_31_16, false, 3, 4, 4>(m, a);
    return launch_bwd2<P_16_31_16, 8, false, true, false, 2, 2>(m, a);
  }
  if (pat == P_16_16_1) { TP2<Pat<P_16_16_1>::NNZ> a{}; AL_CHECK(fill2(m, q, a)); return launch_bwd2<P_16_16_1, 16, false, false, true, 2, 4>(m, a); }
  return ALLEGRO_ERR_UNIMPLEMENTED;
}
