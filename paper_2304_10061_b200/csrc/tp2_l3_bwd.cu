// l_max = 3 backward instantiations of the second-generation tensor-track kernels (tp2_impl.cuh).
#include "tp2_impl.cuh"

int tp2_l3_bwd(allegro_model* m, const TP2& a, int Din, int Dout, bool first, bool hasvb) {
  if (first && hasvb && Din == 16 && Dout == 31) return launch_bwd2<16, 16, 31, 4, true, true, false, 2, 2>(m, a);
  if (!first && hasvb && Din == 31 && Dout == 16) return launch_bwd2<16, 31, 16, 8, false, true, false, 2, 2>(m, a);
  if (!first && !hasvb && Din == 16 && Dout == 1) return launch_bwd2<16, 16, 1, 16, false, false, true, 2, 4>(m, a);
  return ALLEGRO_ERR_UNIMPLEMENTED;
}
