// l_max = 3 forward instantiations of the second-generation tensor-track kernels (tp2_impl.cuh).
#include "tp2_impl.cuh"

int tp2_l3_fwd(allegro_model* m, const TP2& a, int Din, int Dout, bool first) {
  if (first && Din == 16 && Dout == 31) return launch_fwd2<16, 16, 31, 8, true, 3, 4>(m, a);
  if (!first && Din == 31 && Dout == 16) return launch_fwd2<16, 31, 16, 4, false, 3, 4>(m, a);
  if (!first && Din == 16 && Dout == 1) return launch_fwd2<16, 16, 1, 1, false, 3, 4>(m, a);
  return ALLEGRO_ERR_UNIMPLEMENTED;
}
