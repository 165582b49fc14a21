// Dispatch of the per-centre-contracted tensor-track kernels (tpc_impl.cuh) for l_max <= 2; the l_max = 3 instantiations
// live in tpc_l3.cu (long straight-line pattern sweeps: separate translation unit for parallel compilation).
#include "tpc_impl.cuh"

int tpc_l3_fwd(allegro_model* m, Work& w, int L, int nc, const float* om, int ldo, const float* w0, int ldw, float* xs, int ldx);
int tpc_l3_bwd(allegro_model* m, Work& w, int L, int nc, const float* om, int ldo, const float* w0, int ldw, float* ombar,
               int ldob, float* w0bar);

// The contracted kernels apply when the per-edge product kernels of tp2_impl.cuh would (tp2_eligible: 32-channel groups, V^0 in
// the environment layout, every layer's pattern a generated one in its expected role), for up to TPC_MAXL layers, unless the
// model was switched to the per-edge product kernels (allegro_set_tensor_track).
bool tpc_eligible(const allegro_model* m) {
  if (m->tt_mode != 0 || m->NL > TPC_MAXL || !tp2_eligible(m)) return false;
  return m->lmax <= 2 || (m->lmax == 3 && m->NL == 3);
}

#define TPC_CASE(LM_, NL_, L_, CALL) if (m->lmax == LM_ && m->NL == NL_ && Lq == L_) return CALL<LM_, NL_, L_>
#define TPC_ALL(LM, CALL, ...)                                                  \
  TPC_CASE(LM, 1, 1, CALL)(__VA_ARGS__); TPC_CASE(LM, 2, 1, CALL)(__VA_ARGS__); \
  TPC_CASE(LM, 2, 2, CALL)(__VA_ARGS__); TPC_CASE(LM, 3, 1, CALL)(__VA_ARGS__); \
  TPC_CASE(LM, 3, 2, CALL)(__VA_ARGS__); TPC_CASE(LM, 3, 3, CALL)(__VA_ARGS__);

int tpc_fwd(allegro_model* m, Work& w, int Lq, int nc, const float* om, int ldo, const float* w0, int ldw, float* xs, int ldx) {
  if (!tpc_eligible(m)) return ALLEGRO_ERR_UNIMPLEMENTED;
  if (m->lmax == 3) return tpc_l3_fwd(m, w, Lq, nc, om, ldo, w0, ldw, xs, ldx);
  TPC_ALL(1, tpc_launch_fwd, m, w, nc, om, ldo, w0, ldw, xs, ldx)
  TPC_ALL(2, tpc_launch_fwd, m, w, nc, om, ldo, w0, ldw, xs, ldx)
  return ALLEGRO_ERR_UNIMPLEMENTED;
}

int tpc_bwd(allegro_model* m, Work& w, int Lq, int nc, const float* om, int ldo, const float* w0, int ldw, float* ombar, int ldob,
            float* w0bar) {
  if (!tpc_eligible(m)) return ALLEGRO_ERR_UNIMPLEMENTED;
  if (m->lmax == 3) return tpc_l3_bwd(m, w, Lq, nc, om, ldo, w0, ldw, ombar, ldob, w0bar);
  TPC_ALL(1, tpc_launch_bwd, m, w, nc, om, ldo, w0, ldw, ombar, ldob, w0bar)
  TPC_ALL(2, tpc_launch_bwd, m, w, nc, om, ldo, w0, ldw, ombar, ldob, w0bar)
  return ALLEGRO_ERR_UNIMPLEMENTED;
}
