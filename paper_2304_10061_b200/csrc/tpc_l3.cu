// l_max = 3, three layers (config 4): instantiations of the per-centre-contracted tensor-track kernels (tpc_impl.cuh).
#include "tpc_impl.cuh"

namespace {
template <int L>
int l3_fwd(allegro_model* m, Work& w, int nc, const float* om, int ldo, const float* w0, int ldw, float* xs, int ldx) {
  return tpc_launch_fwd<3, 3, L>(m, w, nc, om, ldo, w0, ldw, xs, ldx);
}
template <int L>
int l3_bwd(allegro_model* m, Work& w, int nc, const float* om, int ldo, const float* w0, int ldw, float* ombar, int ldob, float* w0bar) {
  return tpc_launch_bwd<3, 3, L>(m, w, nc, om, ldo, w0, ldw, ombar, ldob, w0bar);
}
}  // namespace

int tpc_l3_fwd(allegro_model* m, Work& w, int L, int nc, const float* om, int ldo, const float* w0, int ldw, float* xs, int ldx) {
  if (L == 1) return l3_fwd<1>(m, w, nc, om, ldo, w0, ldw, xs, ldx);
  if (L == 2) return l3_fwd<2>(m, w, nc, om, ldo, w0, ldw, xs, ldx);
  return l3_fwd<3>(m, w, nc, om, ldo, w0, ldw, xs, ldx);
}
int tpc_l3_bwd(allegro_model* m, Work& w, int L, int nc, const float* om, int ldo, const float* w0, int ldw, float* ombar,
               int ldob, float* w0bar) {
  if (L == 1) return l3_bwd<1>(m, w, nc, om, ldo, w0, ldw, ombar, ldob, w0bar);
  if (L == 2) return l3_bwd<2>(m, w, nc, om, ldo, w0, ldw, ombar, ldob, w0bar);
  return l3_bwd<3>(m, w, nc, om, ldo, w0, ldw, ombar, ldob, w0bar);
}
