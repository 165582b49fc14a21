// Dispatch of the second-generation tensor-track kernels (tp2_impl.cuh) for l_max <= 2, and the
// eligibility test.  The l_max = 3 instantiations live in tp2_l3_fwd.cu / tp2_l3_bwd.cu (separate
// translation units: they dominate the compile time).
#include "tp2_impl.cuh"

int tp2_l3_fwd(allegro_model* m, const TP2& a, int Din, int Dout, bool first);
int tp2_l3_bwd(allegro_model* m, const TP2& a, int Din, int Dout, bool first, bool hasvb);

static bool shape_ok(int de, int di, int dout, bool first, bool last) {
  if (de == 4 || de == 9) return di == de && ((dout == de && !last) || (dout == 1 && last));
  if (de == 16)
    return (first && di == 16 && dout == 31 && !last) || (!first && di == 31 && dout == 16 && !last) ||
           (!first && di == 16 && dout == 1 && last);
  return false;
}

// The kernels apply when every lane of a warp owns a channel, V^0 has the environment layout and every
// layer has one of the instantiated shapes; otherwise tp_kernels.cu / the generic kernels run.
bool tp2_eligible(const allegro_model* m) {
  static const bool off = getenv("B200_ALLEGRO_TP_OLD") != nullptr;
  if (off || m->n % 32 != 0 || (int)m->v0_l.size() != m->Denv) return false;
  for (int k = 0; k < m->Denv; ++k)
    if (m->v0_y[k] != k || m->v0_l[k] != l_of(k)) return false;
  for (int L = 1; L <= m->NL; ++L)
    if (!shape_ok(m->Denv, m->tp[L - 1].Din, m->tp[L - 1].Dout, L == 1, L == m->NL)) return false;
  return true;
}

int tp2_fwd(allegro_model* m, Work& w, int L, int nc, const float* om, int ldo, const float* Vin, const float* w0, int ldw,
            float* Tout, float* xs, int ldx) {
  if (!tp2_eligible(m)) return ALLEGRO_ERR_UNIMPLEMENTED;
  TP2 a{};
  fill2(m, w, L, nc, a, om, ldo, Vin, w0, ldw);
  a.Tout = Tout; a.xs = xs; a.ldx = ldx; a.gamma_out = (float*)w.gamma.p;
  const int DENV = m->Denv, Din = m->tp[L - 1].Din, Dout = m->tp[L - 1].Dout;
  const bool first = (Vin == nullptr);
  if (DENV == 16) return tp2_l3_fwd(m, a, Din, Dout, first);
  if (DENV == 9 && Dout == 9) return first ? launch_fwd2<9, 9, 9, 9, true, 4, 4>(m, a) : launch_fwd2<9, 9, 9, 9, false, 4, 4>(m, a);
  if (DENV == 9 && Dout == 1) return first ? launch_fwd2<9, 9, 1, 1, true, 4, 4>(m, a) : launch_fwd2<9, 9, 1, 1, false, 4, 4>(m, a);
  if (DENV == 4 && Dout == 4) return first ? launch_fwd2<4, 4, 4, 4, true, 4, 4>(m, a) : launch_fwd2<4, 4, 4, 4, false, 4, 4>(m, a);
  if (DENV == 4 && Dout == 1) return first ? launch_fwd2<4, 4, 1, 1, true, 4, 4>(m, a) : launch_fwd2<4, 4, 1, 1, false, 4, 4>(m, a);
  return ALLEGRO_ERR_UNIMPLEMENTED;
}

int tp2_bwd(allegro_model* m, Work& w, int L, int nc, const float* om, int ldo, const float* Vin, const float* w0, int ldw,
            const float* VbarL, const float* sbar, int lds, float* Vbar_prev, float* ombar, int ldob, float* w0bar) {
  if (!tp2_eligible(m)) return ALLEGRO_ERR_UNIMPLEMENTED;
  TP2 a{};
  fill2(m, w, L, nc, a, om, ldo, Vin, w0, ldw);
  a.VbarL = VbarL; a.sbar = sbar; a.lds = lds; a.Vbar_prev = Vbar_prev; a.ombar = ombar; a.ldob = ldob; a.w0bar = w0bar;
  a.Ybar = (float*)w.Ybar.p; a.ybar_gstride = (int64_t)w.cap_edges * m->Denv;
  const int DENV = m->Denv, Din = m->tp[L - 1].Din, Dout = m->tp[L - 1].Dout;
  const bool first = (Vin == nullptr), hasvb = (VbarL != nullptr);
  // Y-bar is initialised by the kernel without a V-bar input, which must be the first of the step (L = NL)
  if (hasvb != (L < m->NL)) { al_set_error(m, "tp2_bwd: unexpected V-bar input"); return ALLEGRO_ERR_BAD_ARG; }
  if (DENV == 16) return tp2_l3_bwd(m, a, Din, Dout, first, hasvb);
  static const bool mreg = getenv("B200_ALLEGRO_TP_MSMEM") == nullptr;
  if (DENV == 9 && Dout == 9) {
    if (mreg) return first ? launch_bwd2<9, 9, 9, 9, true, true, true, 3, 4>(m, a) : launch_bwd2<9, 9, 9, 9, false, true, true, 3, 4>(m, a);
    return first ? launch_bwd2<9, 9, 9, 9, true, true, false, 3, 4>(m, a) : launch_bwd2<9, 9, 9, 9, false, true, false, 3, 4>(m, a);
  }
  if (DENV == 9 && Dout == 1) return first ? launch_bwd2<9, 9, 1, 9, true, false, true, 3, 4>(m, a) : launch_bwd2<9, 9, 1, 9, false, false, true, 3, 4>(m, a);
  if (DENV == 4 && Dout == 4) return first ? launch_bwd2<4, 4, 4, 4, true, true, true, 3, 4>(m, a) : launch_bwd2<4, 4, 4, 4, false, true, true, 3, 4>(m, a);
  if (DENV == 4 && Dout == 1) return first ? launch_bwd2<4, 4, 1, 4, true, false, true, 3, 4>(m, a) : launch_bwd2<4, 4, 1, 4, false, false, true, 3, 4>(m, a);
  return ALLEGRO_ERR_UNIMPLEMENTED;
}
