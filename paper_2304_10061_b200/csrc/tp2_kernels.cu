// Dispatch of the second-generation tensor-track kernels (tp2_impl.cuh) for l_max <= 2, and the
// eligibility test.  The l_max = 3 instantiations live in tp2_l3_fwd.cu / tp2_l3_bwd.cu (separate
// translation units: they dominate the compile time).
#include "tp3_impl.cuh"

int tp2_l3_fwd(allegro_model* m, const TP2Common& q, int pat);
int tp2_l3_bwd(allegro_model* m, const TP2Common& q, int pat);

namespace {

struct Ent { short a, b, c; };
#define XH(k, a, b, c) {a, b, c},
const Ent pat_9_9_9[] = {TP2_PAT_9_9_9(XH)};
const Ent pat_9_9_1[] = {TP2_PAT_9_9_1(XH)};
const Ent pat_4_4_4[] = {TP2_PAT_4_4_4(XH)};
const Ent pat_4_4_1[] = {TP2_PAT_4_4_1(XH)};
const Ent pat_16_16_31[] = {TP2_PAT_16_16_31(XH)};
const Ent pat_16_31_16[] = {TP2_PAT_16_31_16(XH)};
const Ent pat_16_16_1[] = {TP2_PAT_16_16_1(XH)};
#undef XH
struct PatDesc { const Ent* e; int nnz, denv, din, dout; };
const PatDesc pats[P_COUNT] = {
    {pat_9_9_9, TP2_NNZ_9_9_9, 9, 9, 9},        {pat_9_9_1, TP2_NNZ_9_9_1, 9, 9, 1},
    {pat_4_4_4, TP2_NNZ_4_4_4, 4, 4, 4},        {pat_4_4_1, TP2_NNZ_4_4_1, 4, 4, 1},
    {pat_16_16_31, TP2_NNZ_16_16_31, 16, 16, 31}, {pat_16_31_16, TP2_NNZ_16_31_16, 16, 31, 16},
    {pat_16_16_1, TP2_NNZ_16_16_1, 16, 16, 1}};

// index of the generated pattern equal to this layer's dense pair table, or -1
int match_pattern(const TPLayerHost& h) {
  for (int p = 0; p < P_COUNT; ++p) {
    const PatDesc& d = pats[p];
    if (d.denv != h.Denv || d.din != h.Din || d.dout != h.Dout || d.nnz != h.nnz || (int)h.dp_b.size() != d.nnz) continue;
    bool ok = true;
    int k = 0;
    for (int a = 0; a < h.Din && ok; ++a)
      for (int c = 0; c < h.Dout && ok; ++c)
        for (int q = h.dp_ptr[a * h.Dout + c]; q < h.dp_ptr[a * h.Dout + c + 1]; ++q, ++k)
          if (d.e[k].a != a || d.e[k].b != h.dp_b[q] || d.e[k].c != c) { ok = false; break; }
    if (ok && k == d.nnz) return p;
  }
  return -1;
}

}  // namespace

// The kernels apply when every lane of a warp owns a channel, V^0 has the environment layout and every
// layer's sparsity pattern is one of the generated ones with the expected role (first / middle / last
// layer); otherwise tp_kernels.cu / the generic kernels run.
bool tp2_eligible(const allegro_model* m) {
  if (m->n % 32 != 0 || (int)m->v0_l.size() != m->Denv) return false;
  for (int k = 0; k < m->Denv; ++k)
    if (m->v0_y[k] != k || m->v0_l[k] != l_of(k)) return false;
  for (int L = 1; L <= m->NL; ++L) {
    int p = match_pattern(m->tp_host[L - 1]);
    const bool first = (L == 1), last = (L == m->NL);
    bool ok = false;
    switch (p) {
      case P_9_9_9: case P_4_4_4: ok = !last; break;
      case P_9_9_1: case P_4_4_1: ok = last; break;
      case P_16_16_31: ok = first && !last; break;
      case P_16_31_16: ok = !first && !last; break;
      case P_16_16_1: ok = !first && last; break;
      default: ok = false;
    }
    if (!ok) return false;
  }
  return true;
}

// channel groups of the kernel that runs layer L's backward: 8-channel teams for the mma.sync l_max = 3 kernels
// (tp3mb_impl.cuh, TF32 mode), 32-channel warps otherwise
static int bwd_groups(const allegro_model* m, int L) {
  if (tpc_eligible(m)) return m->n / 32;   // contracted kernels: one warp per (centre, 32 channels) in every layer
  int p = match_pattern(m->tp_host[L - 1]);
  return ((p == P_16_16_31 || p == P_16_31_16) && tp3m_bwd_active(m)) ? m->n / 8 : m->n / 32;
}

int al_ybar_layout(const allegro_model* m, int* part0) {
  if (!tp2_eligible(m)) {   // fallback kernels accumulate into one part per 32-channel group
    for (int L = 0; L <= m->NL; ++L) part0[L] = 0;
    return (m->n + 31) / 32;
  }
  int tot = 0;
  part0[0] = tot; tot += bwd_groups(m, 1);
  for (int L = 1; L <= m->NL; ++L) { part0[L] = tot; tot += bwd_groups(m, L); }
  return tot;
}

#define FILL(P)                                \
  TP2<Pat<P>::NNZ> a{};                        \
  { int rc = fill2(m, q, a); if (rc) return rc; }

int tp2_fwd(allegro_model* m, Work& w, int L, int nc, const float* om, int ldo, const float* Vin, const float* w0, int ldw,
            float* Tout, float* xs, int ldx) {
  if (!tp2_eligible(m)) return ALLEGRO_ERR_UNIMPLEMENTED;
  TP2Common q{};
  q.w = &w; q.L = L; q.nc = nc; q.om = om; q.ldo = ldo; q.Vin = Vin; q.w0 = w0; q.ldw = ldw; q.Tout = Tout; q.xs = xs; q.ldx = ldx;
  const int p = match_pattern(m->tp_host[L - 1]);
  const bool first = (Vin == nullptr);
  if (p == P_16_16_31 || p == P_16_31_16 || p == P_16_16_1) return tp2_l3_fwd(m, q, p);
  if (p == P_9_9_9) { FILL(P_9_9_9) return first ? launch_fwd2<P_9_9_9, 9, true, 8, 4>(m, a) : launch_fwd2<P_9_9_9, 9, false, 4, 4>(m, a); }
  if (p == P_9_9_1) { FILL(P_9_9_1) return first ? launch_fwd2<P_9_9_1, 1, true, 8, 4>(m, a) : launch_fwd2<P_9_9_1, 1, false, 4, 4>(m, a); }
  if (p == P_4_4_4) { FILL(P_4_4_4) return first ? launch_fwd2<P_4_4_4, 4, true, 8, 4>(m, a) : launch_fwd2<P_4_4_4, 4, false, 4, 4>(m, a); }
  if (p == P_4_4_1) { FILL(P_4_4_1) return first ? launch_fwd2<P_4_4_1, 1, true, 8, 4>(m, a) : launch_fwd2<P_4_4_1, 1, false, 4, 4>(m, a); }
  return ALLEGRO_ERR_UNIMPLEMENTED;
}

int tp2_bwd(allegro_model* m, Work& w, int L, int nc, const float* om, int ldo, const float* Vin, const float* w0, int ldw,
            const float* VbarL, const float* sbar, int lds, float* Vbar_prev, float* ombar, int ldob, float* w0bar) {
  if (!tp2_eligible(m)) return ALLEGRO_ERR_UNIMPLEMENTED;
  TP2Common q{};
  q.w = &w; q.L = L; q.nc = nc; q.om = om; q.ldo = ldo; q.Vin = Vin; q.w0 = w0; q.ldw = ldw;
  q.VbarL = VbarL; q.sbar = sbar; q.lds = lds; q.Vbar_prev = Vbar_prev; q.ombar = ombar; q.ldob = ldob; q.w0bar = w0bar;
  const int p = match_pattern(m->tp_host[L - 1]);
  const bool first = (Vin == nullptr), hasvb = (VbarL != nullptr);
  if (hasvb != (L < m->NL)) { al_set_error(m, "tp2_bwd: unexpected V-bar input"); return ALLEGRO_ERR_BAD_ARG; }
  if (p == P_16_16_31 || p == P_16_31_16 || p == P_16_16_1) return tp2_l3_bwd(m, q, p);
  // 9 x 9 x 9: M block in the warp's shared slice, 2 ring stages, 12 warps per SM (round-1 measurements: M in registers at
  // 251 registers and deeper rings / smaller blocks were all slower)
  if (p == P_9_9_9) { FILL(P_9_9_9) return first ? launch_bwd2<P_9_9_9, 9, true, true, false, 2, 4>(m, a) : launch_bwd2<P_9_9_9, 9, false, true, false, 2, 4>(m, a); }
  if (p == P_9_9_1) { FILL(P_9_9_1) return first ? launch_bwd2<P_9_9_1, 9, true, false, true, 4, 4>(m, a) : launch_bwd2<P_9_9_1, 9, false, false, true, 4, 4>(m, a); }
  if (p == P_4_4_4) { FILL(P_4_4_4) return first ? launch_bwd2<P_4_4_4, 4, true, true, true, 4, 4>(m, a) : launch_bwd2<P_4_4_4, 4, false, true, true, 4, 4>(m, a); }
  if (p == P_4_4_1) { FILL(P_4_4_1) return first ? launch_bwd2<P_4_4_1, 4, true, false, true, 4, 4>(m, a) : launch_bwd2<P_4_4_1, 4, false, false, true, 4, 4>(m, a); }
  return ALLEGRO_ERR_UNIMPLEMENTED;
}
