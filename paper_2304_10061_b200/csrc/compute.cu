// allegro_compute: center-chunked forward + analytic backward of the Allegro energy (SURVEY.md §3 call
// stack (2), §8(a) steps 2-11).  No host synchronisation inside; the number of active edges of a chunk
// lives on the device (Work::m_act) and every kernel grid is sized for the chunk's candidate count.
#include <algorithm>
#include <cstdlib>
#include <cstring>

#include "gemm.h"
#include <vector>
#include "kernels.h"

static int work_reserve(allegro_model* m, const allegro_nbr* nb, int64_t N) {
  if (!m->work) m->work = new Work();
  m->work_sized = true;
  Work& w = *m->work;
  int64_t M = std::max<int64_t>(nb->max_chunk_edges, 1), Nc = std::max<int64_t>(nb->max_chunk_centers, 1);
  const allegro_hparams& hp = m->hp;
  int d = m->d, n = m->n, nA = m->nA, NL = m->NL;
  const bool tpc = tpc_eligible(m);          // tensor track contracted per centre: no [edges, D, n] tensors at all
  const bool kcat = al_gemm_supports_kcat(m) && (hp.latent_dims[0] % 32 == 0);
  if (m->hfmt >= 0 && (!tpc || !kcat)) {
    al_set_error(m, "16-bit operand modes need the per-centre-contracted tensor track (generated CG patterns, n % 32 == 0, <= 3 layers)");
    return ALLEGRO_ERR_UNIMPLEMENTED;
  }
  if (M > w.cap_edges || w.XS.empty()) {
    auto R = [&](DevBuf& b, size_t floats) { return al_reserve(m, b, floats * 4 + 64); };
    AL_CHECK(R(w.ei, M)); AL_CHECK(R(w.ej, M)); AL_CHECK(R(w.geo, 4 * M)); AL_CHECK(R(w.u, M)); AL_CHECK(R(w.du, M)); AL_CHECK(R(w.sig, M));
    AL_CHECK(R(w.B, M * m->NB)); AL_CHECK(R(w.dB, M * m->NB)); AL_CHECK(R(w.Y, M * m->ldY));
    w.tb_z.resize(hp.n_twobody); w.tb_a.resize(hp.n_twobody);
    int maxw = d + n;
    for (int k = 0; k < hp.n_twobody; ++k) {
      AL_CHECK(R(w.tb_z[k], (size_t)M * hp.twobody_dims[k]));
      if (k < hp.n_twobody - 1) AL_CHECK(R(w.tb_a[k], (size_t)M * hp.twobody_dims[k]));
      maxw = std::max(maxw, hp.twobody_dims[k]);
    }
    w.XS.resize(NL); w.OM.resize(NL + 1); w.T.resize(NL + 1); w.lat_z.resize(NL); w.lat_a.resize(NL);
    int Dmax = 1;
    for (int L = 0; L < NL; ++L) {
      AL_CHECK(R(w.XS[L], (size_t)M * (d + n)));
      if (L >= 1) AL_CHECK(R(w.OM[L + 1], (size_t)M * nA));
      if (L >= 1 && !tpc) AL_CHECK(R(w.T[L], (size_t)M * m->D[L] * n));   // V^L: only the per-edge product kernels store it
      Dmax = std::max(Dmax, m->D[L]);
      w.lat_z[L].resize(hp.n_latent); w.lat_a[L].resize(hp.n_latent);
      for (int k = 0; k < hp.n_latent; ++k) {
        AL_CHECK(R(w.lat_z[L][k], (size_t)M * hp.latent_dims[k]));
        if (k < hp.n_latent - 1) AL_CHECK(R(w.lat_a[L][k], (size_t)M * hp.latent_dims[k]));
        maxw = std::max(maxw, hp.latent_dims[k]);
      }
    }
    AL_CHECK(R(w.XF, (size_t)M * d)); AL_CHECK(R(w.WE, (size_t)M * 2 * nA));
    AL_CHECK(R(w.XB0, (size_t)M * d)); AL_CHECK(R(w.XB1, (size_t)M * d));
    AL_CHECK(R(w.ZB0, (size_t)M * maxw)); AL_CHECK(R(w.ZB1, (size_t)M * maxw));
    AL_CHECK(R(w.G, (size_t)M * (d + n))); AL_CHECK(R(w.OB, (size_t)M * 2 * nA));
    if (!tpc) { AL_CHECK(R(w.VB0, (size_t)M * Dmax * n)); AL_CHECK(R(w.VB1, (size_t)M * Dmax * n)); }
    if (tpc) {
      // s-bar^L of every layer stays alive until layer 1's backward: its own [M][n] rows with the K-concatenated x-bar GEMM,
      // else the whole [x-bar part | s-bar] buffer of each layer
      if (kcat) AL_CHECK(R(w.SB, (size_t)NL * M * n));
      else { w.Gl.resize(NL); for (int L = 0; L < NL; ++L) AL_CHECK(R(w.Gl[L], (size_t)M * (d + n))); }
    }
    w.n_eparts = (d % 32 == 0) ? al_gemm_row_parts(m, d) : 0;   // > 0: last latent layer fused with energy / z-bar (EPI_LATENT_LAST)
    // u-bar partial slots: [0, P) EPI_LATENT_LAST, then P per fused prep stage (NL of them), then one accumulated by k_bwd_prep
    w.n_uparts = (w.n_eparts > 0) ? w.n_eparts * (NL + 1) + 1 : 1;
    AL_CHECK(R(w.ubar, (size_t)M * w.n_uparts)); AL_CHECK(R(w.epart, (size_t)2 * M * std::max(w.n_eparts, 1)));
    { int part0[AL_MAX_LAYERS + 1]; AL_CHECK(R(w.Ybar, (size_t)M * m->Denv * al_ybar_layout(m, part0))); } AL_CHECK(R(w.ge, (size_t)3 * M));
    w.cap_edges = M;
  }
  if (Nc > w.cap_centers) {
    AL_CHECK(al_reserve(m, w.deg, (size_t)Nc * 4 + 64));
    AL_CHECK(al_reserve(m, w.rowa, (size_t)(Nc + 1) * 8 + 64));
    AL_CHECK(al_reserve(m, w.gamma, (size_t)Nc * m->Denv * n * 4 + 64));
    if (tpc) {
      const size_t per = (size_t)NL * Nc * m->Denv * n * 4 + 64;
      AL_CHECK(al_reserve(m, w.tpc_gam, per)); AL_CHECK(al_reserve(m, w.tpc_nvec, per)); AL_CHECK(al_reserve(m, w.tpc_gacc, per));
    }
    w.cap_centers = Nc;
  }
  if (!w.m_act.p) {
    AL_CHECK(al_reserve(m, w.m_act, 64));
    AL_CUDA(m, cudaMemsetAsync(w.m_act.p, 0, 64, m->stream));
  }
  if (N > w.eatom_cap) { AL_CHECK(al_reserve(m, w.eatom, (size_t)N * 8 + 64)); w.eatom_cap = N; }
  return ALLEGRO_OK;
}

void al_work_free(allegro_model* m) {
  if (!m->work) return;
  Work& w = *m->work;
  std::vector<DevBuf*> all = {&w.deg, &w.rowa, &w.scan_tmp, &w.m_act, &w.ei, &w.ej, &w.geo, &w.u, &w.du, &w.sig, &w.B, &w.dB, &w.Y,
                              &w.XF, &w.WE, &w.gamma, &w.XB0, &w.XB1, &w.ZB0, &w.ZB1, &w.G, &w.OB, &w.VB0, &w.VB1,
                              &w.ubar, &w.epart, &w.Ybar, &w.ge, &w.eatom, &w.nh_scal, &w.host_stage, &w.tpc_gam, &w.tpc_nvec, &w.tpc_gacc, &w.SB};
  for (auto* b : all) al_release(m, *b);
  for (auto* v : {&w.tb_z, &w.tb_a, &w.XS, &w.OM, &w.T, &w.Gl}) for (auto& b : *v) al_release(m, b);
  for (auto* vv : {&w.lat_z, &w.lat_a}) for (auto& v : *vv) for (auto& b : v) al_release(m, b);
  delete m->work;
  m->work = nullptr;
}

// io16 (16-bit operand modes only): every epilogue tensor of a 16-bit GEMM (aux rows, second output, prep-stage tensors) is
// 16-bit; its main output C is 16-bit only where a GEMM or an epilogue is the sole reader (IO16_C = gemm_tc.cu's bit) and
// fp32 where the tensor track, k_edge_bwd or a debug tap reads it
enum { IO16_C = 1 };
static GemmArgs mk(const allegro_model* m, const float* A, int lda, const Dense& D, bool transposed_weight, float* C, int ldc, int m_cap,
                   const int* m_ptr, int epi, int io16 = 0) {
  // transposed_weight = false: forward  Y = X W   -> Bt = Wt [fo][fi], N = fo, K = fi
  // transposed_weight = true : backward dX = dY W^T -> Bt = W  [fi][fo], N = fi, K = fo
  GemmArgs g{};
  g.A = A; g.lda = lda;
  if (!transposed_weight) { g.Bt = D.Wt; g.Bt_hi = D.Wt_hi; g.Bt_lo = D.Wt_lo; g.ldb = D.fi; g.N = D.fo; g.K = D.fi; }
  else { g.Bt = D.W; g.Bt_hi = D.W_hi; g.Bt_lo = D.W_lo; g.ldb = D.fo; g.N = D.fi; g.K = D.fo; }
  g.C = C; g.ldc = ldc; g.m_cap = m_cap; g.m_ptr = m_ptr; g.epi = epi;
  if (m->hfmt >= 0) { g.Bt16 = transposed_weight ? D.W16 : D.Wt16; g.hfmt = m->hfmt; g.io16 = io16; }
  return g;
}

static int run_chunk(allegro_model* m, Work& w, const Chunk& ch, const double* pos, const int32_t* species,
                     const double box[3], const allegro_nbr* nb, double* e_atom, double* force, double* e_edge) {
  const allegro_hparams& hp = m->hp;
  const int d = m->d, n = m->n, nA = m->nA, NL = m->NL, ntb = hp.n_twobody, nlat = hp.n_latent;
  const int nc = (int)(ch.c1 - ch.c0);
  const int m_cap = (int)(ch.e1 - ch.e0);
  w.last_nc = nc;
  if (m_cap <= 0) {   // isolated atoms only: E-hat_i = mu_Z
    return k_launch_energy(m, w, species, ch.c0, nc, (float*)w.XF.p, e_atom);   // rowa not valid -> handled below
  }
  const int* mp = (const int*)w.m_act.p;
  cudaStream_t st = m->stream;
  const bool fused_last = w.n_eparts > 0;
  const bool tpc = tpc_eligible(m);
  const bool h16 = m->hfmt >= 0;      // precision 2 / 4: every tensor that only GEMMs and their epilogues touch is 16-bit
  auto el = [&](void* base, size_t elems) { return (float*)((char*)base + elems * (h16 ? 2 : 4)); };   // element offset
  EdgeGeomArgs ga{};
  ga.pos = pos; ga.species = species; memcpy(ga.box, box, 24); ga.rc = hp.r_cut; ga.p = hp.poly_p; ga.NB = m->NB;
  ga.lmax = m->lmax; ga.row_ptr = (const int64_t*)nb->row_ptr.p; ga.j = (const int32_t*)nb->j.p;
  ga.shift = (const int8_t*)nb->shift.p; ga.c0 = ch.c0; ga.nc = nc;
  ga.rc_pair = m->d_rc_pair; ga.S = m->S; ga.bfreq = m->d_bfreq;
  // ---- step 2: compaction + geometry ----------------------------------------------------------------
  AL_CHECK(k_launch_active_count(m, ga, (int*)w.deg.p));
  AL_CHECK(al_exclusive_scan_i64(m, (int*)w.deg.p, (int64_t*)w.rowa.p, nc, w.scan_tmp));
  AL_CHECK(k_launch_set_mact(m, (int64_t*)w.rowa.p, nc, (int*)w.m_act.p));
  AL_CHECK(k_launch_geom_fill(m, ga, (int64_t*)w.rowa.p, w));
  // ---- step 3: two-body latent ------------------------------------------------------------------------
  m->sweep_ctr = 1;   // k_twobody0 walks forward, so the first GEMM after it starts reversed (al_next_rev)
  AL_CHECK(k_launch_twobody0(m, w, species, m->twobody[0], ntb == 1, m_cap));
  for (int k = 1; k < ntb; ++k) {
    bool last = (k == ntb - 1);
    GemmArgs g = mk(m, (float*)w.tb_a[k - 1].p, hp.twobody_dims[k - 1], m->twobody[k], false,
                    last ? (float*)w.XS[0].p : (float*)w.tb_a[k].p, last ? d + n : hp.twobody_dims[k], m_cap, mp,
                    last ? EPI_SILU_U : EPI_SILU_BOTH, IO16_C);
    g.out2 = (float*)w.tb_z[k].p; g.ldo2 = hp.twobody_dims[k]; g.u = (float*)w.u.p;
    AL_CHECK(al_gemm(m, g));
  }
  // ---- step 4: embedding projections  [w^0 | omega^1] = x^0 [A^0 | A^1] ----------------------------------
  AL_CHECK(al_gemm(m, mk(m, (float*)w.XS[0].p, d + n, m->emb01, false, (float*)w.WE.p, 2 * nA, m_cap, mp, EPI_PLAIN)));
  // ---- steps 5-8: layers -----------------------------------------------------------------------------------
  for (int L = 1; L <= NL; ++L) {
    const float* om = (L == 1) ? (float*)w.WE.p + nA : (float*)w.OM[L].p;
    int ldo = (L == 1) ? 2 * nA : nA;
    const float* Vin = (L == 1 || tpc) ? nullptr : (float*)w.T[L - 1].p;
    float* Tout = (L < NL && !tpc) ? (float*)w.T[L].p : nullptr;
    AL_CHECK(k_launch_tp_fwd(m, w, L, nc, om, ldo, Vin, (float*)w.WE.p, 2 * nA, Tout, el(w.XS[L - 1].p, d), d + n));
    for (int k = 0; k < nlat; ++k) {
      bool last = (k == nlat - 1);
      const float* A = (k == 0) ? (float*)w.XS[L - 1].p : (float*)w.lat_a[L - 1][k - 1].p;
      int lda = (k == 0) ? d + n : hp.latent_dims[k - 1];
      float* C; int ldc;
      if (!last) { C = (float*)w.lat_a[L - 1][k].p; ldc = hp.latent_dims[k]; }
      else if (L < NL) { C = (float*)w.XS[L].p; ldc = d + n; }
      else { C = (float*)w.XF.p; ldc = d; }
      GemmArgs g = mk(m, A, lda, m->latent[L - 1][k], false, C, ldc, m_cap, mp, last ? EPI_LATENT : EPI_SILU_BOTH,
                      IO16_C);
      g.out2 = (float*)w.lat_z[L - 1][k].p; g.ldo2 = hp.latent_dims[k];
      g.u = (float*)w.u.p; g.aux1 = (float*)w.XS[L - 1].p; g.ld1 = d + n; g.c0 = m->c_old[L - 1]; g.c1 = m->c_new[L - 1];
      if (last && L == NL && fused_last) {
        // x^{NL} is consumed in the epilogue: edge-energy partials, z-bar^{NL} (in place of z) and u-bar partials
        g.epi = EPI_LATENT_LAST;
        if (!m->debug_keep) g.C = nullptr;
        g.io16 &= ~IO16_C;                         // the debug tap of x^{NL} stays fp32
        g.out2 = (float*)w.ZB0.p; g.ldo2 = d;
        g.sig = (float*)w.sig.p; g.aux3 = m->w_eff_f; g.w_eff_d = m->w_eff_d;
        g.epart = (double*)w.epart.p; g.upart = (float*)w.ubar.p; g.part_stride = w.cap_edges;
      }
      AL_CHECK(al_gemm(m, g));
    }
    if (L < NL)
      AL_CHECK(al_gemm(m, mk(m, (float*)w.XS[L].p, d + n, m->emb[L], false, (float*)w.OM[L + 1].p, nA, m_cap, mp, EPI_PLAIN)));
  }
  // ---- steps 9-10: edge energy, per-atom energy (fp64) -----------------------------------------------------
  AL_CHECK(k_launch_energy(m, w, species, ch.c0, nc, (float*)w.XF.p, e_atom));
  if (m->d_zbl_Z) AL_CHECK(k_launch_zbl(m, ga, m->d_zbl_Z, e_atom, force));           // NEXT-4: ZBL pair repulsion
  if (e_edge) AL_CHECK(k_launch_edge_energy_out(m, ga, w, (float*)w.XF.p, e_edge));   // NEXT-4: per-edge energies
  if (!force) return ALLEGRO_OK;                                                       // NEXT-4: energy only
  // ---- step 11: backward -----------------------------------------------------------------------------------
  // u-bar partials: [0, n_eparts) stored by EPI_LATENT_LAST, the last one accumulated by k_bwd_prep
  AL_CUDA(m, cudaMemsetAsync((float*)w.ubar.p + (size_t)(w.n_uparts - 1) * w.cap_edges, 0, (size_t)m_cap * 4, st));
  // Y-bar partials [part][M][Denv] (al_ybar_layout), summed in fixed order by k_edge_bwd.  The tp2/tp3 kernels
  // store every partial; the fallback kernels accumulate into one part per 32-channel group, zeroed here.
  if (!tp2_eligible(m))
    for (int gq = 0; gq < (n + 31) / 32; ++gq)
      AL_CUDA(m, cudaMemsetAsync((float*)w.Ybar.p + (size_t)gq * w.cap_edges * m->Denv, 0, (size_t)m_cap * m->Denv * 4, st));
  float* xb = (float*)w.XB0.p; float* xb_o = (float*)w.XB1.p;
  float* vb = nullptr; float* vb_a = (float*)w.VB0.p; float* vb_b = (float*)w.VB1.p;
  bool rank1 = true;   // x-bar^{NL} = sigma_e * w_eff is never materialised
  // With fused_last every z-bar that starts an MLP's backward comes out of a GEMM epilogue (EPI_LATENT_LAST for
  // layer NL, the prep stage of EPI_ADD2/ADD2R for the others); otherwise k_bwd_prep computes it.
  bool zb_ready = fused_last;
  const bool fuse_prep = fused_last;
  int prep_slot = 1;
  // K-concatenated x-bar GEMM (tensor-core kernels): x-bar^{L-1} = [z-bar | omega-bar] [W_x | A]^T in one launch, so
  // the x-bar part of dX of the first latent layer never goes through HBM; s-bar comes from its own N = n GEMM.
  const bool kcat = al_gemm_supports_kcat(m) && (hp.latent_dims[0] % 32 == 0);
  float* zstart = (float*)w.ZB0.p;   // where the z-bar entering the next MLP to differentiate lives
  for (int L = NL; L >= 1; --L) {
    float* zb = zstart; float* zb_o = (zstart == (float*)w.ZB0.p) ? (float*)w.ZB1.p : (float*)w.ZB0.p;
    if (!zb_ready)
      AL_CHECK(k_launch_bwd_prep(m, w, rank1 ? nullptr : xb, d, (float*)w.lat_z[L - 1][nlat - 1].p, d, m->c_new[L - 1], zb, d, d, m_cap));
    for (int k = nlat - 1; k >= 1; --k) {
      GemmArgs g = mk(m, zb, hp.latent_dims[k], m->latent[L - 1][k], true, zb_o, hp.latent_dims[k - 1], m_cap, mp, EPI_MUL_DSILU,
                      IO16_C);
      g.aux1 = (float*)w.lat_z[L - 1][k - 1].p; g.ld1 = hp.latent_dims[k - 1];
      AL_CHECK(al_gemm(m, g));
      std::swap(zb, zb_o);
    }
    // [x-bar part | s-bar] of this layer.  Contracted tensor track: s-bar^L of every layer must survive until layer 1's
    // backward (V-bar^0_e = sum_L s-bar^L_e n^L), so each layer has its own rows (SB with the K-concatenated x-bar GEMM,
    // a whole G buffer per layer otherwise); per-edge product kernels: one G buffer re-used by every layer.
    float* Gp = (tpc && !kcat) ? (float*)w.Gl[L - 1].p : (float*)w.G.p;
    float* sbp = (tpc && kcat) ? (float*)w.SB.p + (size_t)(L - 1) * w.cap_edges * n : Gp + d;
    const int sbl = (tpc && kcat) ? n : d + n;
    w.sb_ptr[L - 1] = sbp; w.sb_ld[L - 1] = sbl;
    if (kcat)   // s-bar only: [M, h] x W_lat0[d:, :]^T
      AL_CHECK(al_gemm(m, mk(m, zb, hp.latent_dims[0], m->sbar[L - 1], true, sbp, sbl, m_cap, mp, EPI_PLAIN)));
    else
      AL_CHECK(al_gemm(m, mk(m, zb, hp.latent_dims[0], m->latent[L - 1][0], true, Gp, d + n, m_cap, mp, EPI_PLAIN)));
    const float* om = (L == 1) ? (float*)w.WE.p + nA : (float*)w.OM[L].p;
    int ldo = (L == 1) ? 2 * nA : nA;
    const float* Vin = (L == 1 || tpc) ? nullptr : (float*)w.T[L - 1].p;
    int ldob = (L == 1) ? 2 * nA : nA;
    float* ombar = (L == 1) ? el(w.OB.p, nA) : (float*)w.OB.p;   // (16-bit in the 16-bit modes: the x-bar GEMM's second A operand)
    float* vprev = (vb == vb_a) ? vb_b : vb_a;
    AL_CHECK(k_launch_tp_bwd(m, w, L, nc, om, ldo, Vin, (float*)w.WE.p, 2 * nA, vb, sbp, sbl, vprev, ombar,
                             ldob, (float*)w.OB.p));
    vb = vprev;
    GemmArgs g = mk(m, (float*)w.OB.p, ldob, (L == 1) ? m->emb01 : m->emb[L - 1], true, xb_o, d, m_cap, mp,
                    rank1 ? EPI_ADD2R : EPI_ADD2);
    g.aux1 = xb; g.ld1 = d; g.c0 = m->c_old[L - 1]; g.aux2 = Gp; g.ld2 = d + n;
    g.u = (float*)w.sig.p; g.aux3 = m->w_eff_f;
    if (kcat) {
      const int h = hp.latent_dims[0];
      GemmArgs gc = mk(m, zb, h, m->xcat[L - 1], true, xb_o, d, m_cap, mp, g.epi, IO16_C);
      gc.A2 = (float*)w.OB.p; gc.lda2 = ldob; gc.K1 = h;
      gc.aux1 = g.aux1; gc.ld1 = g.ld1; gc.c0 = g.c0; gc.aux2 = nullptr; gc.ld2 = 0; gc.u = g.u; gc.aux3 = g.aux3;
      g = gc;
    }
    // the prep stage must not overwrite the z-bar this GEMM still reads as its A operand (kcat): use the other buffer
    float* zb_next = (zb == (float*)w.ZB0.p) ? (float*)w.ZB1.p : (float*)w.ZB0.p;
    if (fuse_prep) {
      // prep stage: z-bar of the MLP below (latent MLP of layer L-1, or the two-body MLP when L = 1)
      g.prep = 1;
      g.zp = (L > 1) ? (float*)w.lat_z[L - 2][nlat - 1].p : (float*)w.tb_z[ntb - 1].p; g.ldzp = d;
      g.zbp = zb_next; g.ldzbp = d; g.pu = (float*)w.u.p; g.cp = (L > 1) ? m->c_new[L - 2] : 1.0f;
      g.upart = (float*)w.ubar.p; g.part_stride = w.cap_edges; g.pbase = prep_slot * w.n_eparts;
      ++prep_slot;
      if (L == 1 && !m->debug_keep) g.C = nullptr;   // x-bar^0 itself is not needed afterwards
    }
    AL_CHECK(al_gemm(m, g));
    std::swap(xb, xb_o);
    rank1 = false;
    zb_ready = fuse_prep;
    zstart = fuse_prep ? zb_next : (float*)w.ZB0.p;
  }
  {
    float* zb = zstart; float* zb_o = (zstart == (float*)w.ZB0.p) ? (float*)w.ZB1.p : (float*)w.ZB0.p;
    if (!zb_ready)
      AL_CHECK(k_launch_bwd_prep(m, w, xb, d, (float*)w.tb_z[ntb - 1].p, d, 1.0f, zb, d, d, m_cap));
    for (int k = ntb - 1; k >= 1; --k) {
      GemmArgs g = mk(m, zb, hp.twobody_dims[k], m->twobody[k], true, zb_o, hp.twobody_dims[k - 1], m_cap, mp, EPI_MUL_DSILU,
                      (k > 1 ? IO16_C : 0));   // the last z-bar (read by k_edge_bwd) stays fp32
      g.aux1 = (float*)w.tb_z[k - 1].p; g.ld1 = hp.twobody_dims[k - 1];
      AL_CHECK(al_gemm(m, g));
      std::swap(zb, zb_o);
    }
    AL_CHECK(k_launch_edge_bwd(m, w, zb, hp.twobody_dims[0], m->twobody[0], ntb == 1, force, m_cap));
  }
  return ALLEGRO_OK;
}

int al_compute_impl(allegro_model* m, const double* pos, const int32_t* species, int64_t N, const double box[3],
                    const allegro_nbr* nb, double* e_total, double* e_atom, double* force, double* e_edge) {
  return al_compute_local_impl(m, pos, species, N, N, box, nb, e_total, e_atom, force, e_edge);
}

// n_local < N: only the first n_local atoms are centres (the local atoms of a spatial domain); the others are ghosts that
// appear as neighbours and receive the force -dE_local/dr_ghost.
int al_compute_local_impl(allegro_model* m, const double* pos, const int32_t* species, int64_t N, int64_t n_local,
                          const double box[3], const allegro_nbr* nb, double* e_total, double* e_atom, double* force,
                          double* e_edge) {
  if (!m || !pos || !species || !box || !nb || !e_total) { al_set_error(m, "NULL argument"); return ALLEGRO_ERR_BAD_ARG; }
  if (n_local < 0 || n_local > N) { al_set_error(m, "n_local out of range"); return ALLEGRO_ERR_BAD_ARG; }
  if (nb->n_atoms != N) { al_set_error(m, "neighbor list was built for a different n_atoms"); return ALLEGRO_ERR_BAD_ARG; }
  if (nb->cutoff < m->hp.r_cut) { al_set_error(m, "neighbor list cutoff < r_cut"); return ALLEGRO_ERR_BAD_ARG; }
  AL_CHECK(work_reserve(m, nb, N));
  Work& w = *m->work;
  double* ea = e_atom ? e_atom : (double*)w.eatom.p;
  AL_CHECK(k_launch_begin_compute(m, force, species, N, (int*)w.m_act.p));   // zero the forces, validate the species
  AL_CUDA(m, cudaMemsetAsync((int*)w.m_act.p + 2, 0, 8, m->stream));   // total active edges of this call
  for (Chunk ch : nb->chunks) {
    if (ch.c0 >= n_local) break;
    if (ch.c1 > n_local) {   // the chunk that straddles the local / ghost boundary: keep its local centres only
      ch.c1 = n_local;
      ch.e1 = nb->row_ptr_host[n_local];
    }
    if (ch.e1 == ch.e0) {
      // no candidate edges at all: make rowa all-zero so k_energy yields mu_Z
      AL_CUDA(m, cudaMemsetAsync(w.rowa.p, 0, (size_t)(ch.c1 - ch.c0 + 1) * 8, m->stream));
    }
    AL_CHECK(run_chunk(m, w, ch, pos, species, box, nb, ea, force, e_edge));
  }
  if (n_local < N) AL_CHECK(k_launch_zero_f64(m, ea + n_local, N - n_local));   // ghosts carry no energy here
  AL_CHECK(k_launch_sum_f64(m, ea, n_local, e_total));
  return ALLEGRO_OK;
}

extern "C" int allegro_compute(allegro_model* m, const double* pos, const int32_t* species, int64_t n_atoms,
                               const double box[3], const allegro_nbr* nbr, double* e_total, double* e_atom, double* force) {
  return al_compute_impl(m, pos, species, n_atoms, box, nbr, e_total, e_atom, force, nullptr);
}

extern "C" int allegro_compute_local(allegro_model* m, const double* pos, const int32_t* species, int64_t n_atoms,
                                     int64_t n_local, const double box[3], const allegro_nbr* nbr, double* e_total,
                                     double* e_atom, double* force) {
  return al_compute_local_impl(m, pos, species, n_atoms, n_local, box, nbr, e_total, e_atom, force, nullptr);
}

extern "C" int allegro_edge_energies(allegro_model* m, const double* pos, const int32_t* species, int64_t n_atoms,
                                     const double box[3], const allegro_nbr* nbr, double* e_total, double* e_edge) {
  if (!e_edge) { al_set_error(m, "NULL argument"); return ALLEGRO_ERR_BAD_ARG; }
  return al_compute_impl(m, pos, species, n_atoms, box, nbr, e_total, nullptr, nullptr, e_edge);
}

// Status word written by the kernels (Work::m_act[1]): bit 0 = coincident atoms (r = 0), bit 1 = species out of range.
// Reads it after synchronising the stream, clears it and turns it into an error code.
int al_check_status(allegro_model* m) {
  if (!m->work || !m->work->m_act.p) return ALLEGRO_OK;
  int flags[2] = {0, 0};
  AL_CUDA(m, cudaStreamSynchronize(m->stream));
  AL_CUDA(m, cudaMemcpy(flags, m->work->m_act.p, 8, cudaMemcpyDeviceToHost));
  if (!flags[1]) return ALLEGRO_OK;
  AL_CUDA(m, cudaMemset((int*)m->work->m_act.p + 1, 0, 4));
  if (flags[1] & 2) { al_set_error(m, "species value outside [0, n_species)"); return ALLEGRO_ERR_BAD_ARG; }
  al_set_error(m, "coincident atoms (r = 0)");
  return ALLEGRO_ERR_NONFINITE;
}

extern "C" int allegro_status(allegro_model* m) {
  if (!m) return ALLEGRO_ERR_BAD_ARG;
  return al_check_status(m);
}

extern "C" int allegro_compute_host(allegro_model* m, const double* pos, const int32_t* species, int64_t N,
                                    const double box[3], const allegro_nbr* nbr, double* e_total, double* e_atom,
                                    double* force) {
  if (!m || !pos || !species || !e_total) return ALLEGRO_ERR_BAD_ARG;
  void *dp = nullptr, *ds = nullptr, *de = nullptr, *dea = nullptr, *df = nullptr;
  int rc = ALLEGRO_OK;
  cudaStream_t st = m->stream;
  if ((rc = al_alloc(m, &dp, N * 24 + 16)) || (rc = al_alloc(m, &ds, N * 4 + 16)) || (rc = al_alloc(m, &de, 16)) ||
      (rc = al_alloc(m, &dea, N * 8 + 16)) || (rc = al_alloc(m, &df, N * 24 + 16)))
    goto done;
  {
    cudaError_t e = cudaMemcpyAsync(dp, pos, N * 24, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(ds, species, N * 4, cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) { al_set_error(m, std::string("allegro_compute_host, host->device copy: ") + cudaGetErrorString(e)); rc = ALLEGRO_ERR_CUDA; goto done; }
  }
  rc = al_compute_impl(m, (double*)dp, (int32_t*)ds, N, box, nbr, (double*)de, (double*)dea, force ? (double*)df : nullptr, nullptr);
  if (rc == ALLEGRO_OK) {
    cudaError_t e = cudaMemcpyAsync(e_total, de, 8, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess && e_atom) e = cudaMemcpyAsync(e_atom, dea, N * 8, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess && force) e = cudaMemcpyAsync(force, df, N * 24, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) { al_set_error(m, std::string("allegro_compute_host, device->host copy: ") + cudaGetErrorString(e)); rc = ALLEGRO_ERR_CUDA; }
    else rc = al_check_status(m);
  }
done:
  cudaStreamSynchronize(st);
  al_free(m, dp); al_free(m, ds); al_free(m, de); al_free(m, dea); al_free(m, df);
  return rc;
}

extern "C" int allegro_last_active_edges(allegro_model* m, int64_t* n_active) {
  if (!m || !n_active || !m->work) return ALLEGRO_ERR_BAD_ARG;
  long long v = 0;
  AL_CUDA(m, cudaStreamSynchronize(m->stream));
  AL_CUDA(m, cudaMemcpy(&v, (int*)m->work->m_act.p + 2, 8, cudaMemcpyDeviceToHost));
  *n_active = v;
  return ALLEGRO_OK;
}

// The part of an MD step that follows the (optional) list rebuild.  `with_first_kick`: the half kick + drift that
// precedes the rebuild is included (steps without a rebuild, the ones a CUDA graph can replay).
static int step_tail(allegro_model* m, double* pos, double* vel, double* force, const int32_t* species, const double* mass,
                     int64_t N, const double box[3], double dt_fs, const allegro_nbr* nbr, double* e_pot, double* e_kin,
                     bool with_first_kick) {
  if (with_first_kick) AL_CHECK(k_launch_nve_kick_drift(m, pos, vel, force, species, mass, N, dt_fs, true));
  AL_CHECK(al_compute_impl(m, pos, species, N, box, nbr, e_pot, nullptr, force, nullptr));
  AL_CHECK(k_launch_nve_kick_drift(m, pos, vel, force, species, mass, N, dt_fs, false));
  AL_CHECK(k_launch_kinetic(m, vel, species, mass, N, e_kin, m->work->scan_tmp));
  return ALLEGRO_OK;
}

// Capture one no-rebuild step into a CUDA graph (on a private stream: the caller's may be the legacy default stream,
// which cannot be captured), instantiate or update the executable graph and launch it on the caller's stream.
static int step_capture_and_launch(allegro_model* m, double* pos, double* vel, double* force, const int32_t* species,
                                   const double* mass, int64_t N, const double box[3], double dt_fs, const allegro_nbr* nbr,
                                   double* e_pot, double* e_kin, const std::vector<uint64_t>& key) {
  auto& sg = m->sg;
  auto give_up = [&](const char* why) { cudaGetLastError(); sg.disabled = true; (void)why; return ALLEGRO_ERR_CUDA; };
  if (!sg.cap && cudaStreamCreateWithFlags(&sg.cap, cudaStreamNonBlocking) != cudaSuccess) return give_up("stream");
  cudaStream_t user = m->stream;
  const int64_t l0 = m->launches;
  if (cudaStreamBeginCapture(sg.cap, cudaStreamCaptureModeThreadLocal) != cudaSuccess) return give_up("begin");
  m->stream = sg.cap;
  int rc = step_tail(m, pos, vel, force, species, mass, N, box, dt_fs, nbr, e_pot, e_kin, true);
  m->stream = user;
  cudaGraph_t graph = nullptr;
  cudaError_t e = cudaStreamEndCapture(sg.cap, &graph);
  const int64_t nl = m->launches - l0;
  m->launches = l0;                                    // nothing ran yet
  if (rc != ALLEGRO_OK || e != cudaSuccess || !graph) {
    if (graph) cudaGraphDestroy(graph);
    return give_up("capture");
  }
  if (sg.exec) {
    cudaGraphExecUpdateResultInfo info;
    if (cudaGraphExecUpdate(sg.exec, graph, &info) != cudaSuccess) { cudaGetLastError(); cudaGraphExecDestroy(sg.exec); sg.exec = nullptr; }
  }
  if (!sg.exec && cudaGraphInstantiate(&sg.exec, graph, 0) != cudaSuccess) { cudaGraphDestroy(graph); sg.exec = nullptr; return give_up("instantiate"); }
  cudaGraphDestroy(graph);
  if (cudaGraphLaunch(sg.exec, user) != cudaSuccess) { cudaGraphExecDestroy(sg.exec); sg.exec = nullptr; return give_up("launch"); }
  sg.key = key; sg.nlaunch = nl;
  m->launches += nl;
  return ALLEGRO_OK;
}

extern "C" int allegro_step_nve(allegro_model* m, double* pos, double* vel, double* force, const int32_t* species,
                                const double* mass, int64_t N, const double box[3], double dt_fs, int32_t rebuild_every,
                                double skin, allegro_nbr** nbr, int64_t* step_counter, double* e_pot, double* e_kin) {
  if (!m || !pos || !vel || !force || !species || !mass || !nbr || !step_counter || !e_pot || !e_kin) {
    al_set_error(m, "NULL argument");
    return ALLEGRO_ERR_BAD_ARG;
  }
  if (rebuild_every < 1 || skin < 0) { al_set_error(m, "rebuild_every >= 1 and skin >= 0 required"); return ALLEGRO_ERR_BAD_ARG; }
  const bool rebuild = (*nbr == nullptr || (*step_counter % rebuild_every) == 0);
  static const bool no_graph = getenv("B200_ALLEGRO_NO_GRAPH") != nullptr;
  const bool graphs = !no_graph && !m->prof && !m->sg.disabled;
  auto make_key = [&]() {
    auto bits = [](double x) { uint64_t b; memcpy(&b, &x, 8); return b; };
    return std::vector<uint64_t>{(uint64_t)pos, (uint64_t)vel, (uint64_t)force, (uint64_t)species, (uint64_t)mass, (uint64_t)N,
                                 bits(box[0]), bits(box[1]), bits(box[2]), bits(dt_fs), (uint64_t)*nbr, (*nbr)->version,
                                 (uint64_t)e_pot, (uint64_t)e_kin, (uint64_t)m->stream, m->config_gen, m->alloc_gen};
  };
  if (!rebuild && graphs && m->work) {
    const std::vector<uint64_t> key = make_key();
    if (m->sg.exec && key == m->sg.key) {
      if (cudaGraphLaunch(m->sg.exec, m->stream) == cudaSuccess) {
        m->launches += m->sg.nlaunch;
        m->sg.steps++;
        (*step_counter)++;
        return ALLEGRO_OK;
      }
      cudaGetLastError();
      m->sg.disabled = true;
    } else if (key == m->sg.warm) {
      // a step with exactly this state already ran eagerly (every buffer is sized, every kernel attribute set): capture
      if (step_capture_and_launch(m, pos, vel, force, species, mass, N, box, dt_fs, *nbr, e_pot, e_kin, key) == ALLEGRO_OK) {
        m->sg.steps++;
        (*step_counter)++;
        return ALLEGRO_OK;
      }
    }
  }
  AL_CHECK(k_launch_nve_kick_drift(m, pos, vel, force, species, mass, N, dt_fs, true));
  if (rebuild) {
    AL_CHECK(al_neighbors_impl(m, pos, N, box, m->hp.r_cut + skin, nbr));
    AL_CHECK(al_check_status(m));   // the list build synchronised: surface what the steps since the last rebuild flagged
  }
  AL_CHECK(step_tail(m, pos, vel, force, species, mass, N, box, dt_fs, *nbr, e_pot, e_kin, false));
  if (graphs && !m->sg.disabled) m->sg.warm = make_key();   // the state the next step will see if nothing changes
  (*step_counter)++;
  return ALLEGRO_OK;
}

extern "C" int allegro_nve_kick(allegro_model* m, double* pos, double* vel, const double* force, const int32_t* species,
                                const double* mass, int64_t N, double dt_fs, int32_t drift) {
  if (!m || !vel || !force || !species || !mass || (drift && !pos)) { al_set_error(m, "NULL argument"); return ALLEGRO_ERR_BAD_ARG; }
  return k_launch_nve_kick_drift(m, pos, vel, force, species, mass, N, dt_fs, drift != 0);
}

extern "C" int allegro_kinetic_energy(allegro_model* m, const double* vel, const int32_t* species, const double* mass,
                                      int64_t N, double* e_kin) {
  if (!m || !vel || !species || !mass || !e_kin) { al_set_error(m, "NULL argument"); return ALLEGRO_ERR_BAD_ARG; }
  if (!m->work) m->work = new Work();
  return k_launch_kinetic(m, vel, species, mass, N, e_kin, m->work->scan_tmp);
}

extern "C" int allegro_graph_steps(const allegro_model* m, int64_t* n) {
  if (!m || !n) return ALLEGRO_ERR_BAD_ARG;
  *n = m->sg.disabled ? -1 : m->sg.steps;
  return ALLEGRO_OK;
}

extern "C" int allegro_step_nvt(allegro_model* m, double* pos, double* vel, double* force, const int32_t* species,
                                const double* mass, int64_t N, const double box[3], double dt_fs, int32_t rebuild_every,
                                double skin, allegro_nbr** nbr, int64_t* step_counter, double* e_pot, double* e_kin,
                                double* nh_state, double t0_K, double tau_fs) {
  if (!m || !vel || !species || !mass || !e_kin || !nh_state) { al_set_error(m, "NULL argument"); return ALLEGRO_ERR_BAD_ARG; }
  if (!(t0_K > 0) || !(tau_fs > 0) || N < 1) { al_set_error(m, "t0_K > 0, tau_fs > 0, n_atoms >= 1 required"); return ALLEGRO_ERR_BAD_ARG; }
  if (!m->work) { al_set_error(m, "call allegro_compute once before the first step (force must hold F(r))"); return ALLEGRO_ERR_BAD_ARG; }
  Work& w = *m->work;
  AL_CHECK(al_reserve(m, w.nh_scal, 64));
  const double g = 3.0 * (double)N;
  // [thermostat dt/2] [velocity-Verlet NVE step] [thermostat dt/2]
  AL_CHECK(k_launch_kinetic(m, vel, species, mass, N, e_kin, w.scan_tmp));
  AL_CHECK(k_launch_nh_half(m, vel, N, nh_state, e_kin, g, t0_K, tau_fs, dt_fs, (double*)w.nh_scal.p));
  AL_CHECK(allegro_step_nve(m, pos, vel, force, species, mass, N, box, dt_fs, rebuild_every, skin, nbr, step_counter, e_pot, e_kin));
  AL_CHECK(k_launch_nh_half(m, vel, N, nh_state, e_kin, g, t0_K, tau_fs, dt_fs, (double*)m->work->nh_scal.p));
  return ALLEGRO_OK;
}

extern "C" int allegro_step_nve_host(allegro_model* m, double* pos, double* vel, double* force, const int32_t* species,
                                     const double* mass, int64_t N, const double box[3], double dt_fs,
                                     int32_t rebuild_every, double skin, allegro_nbr** nbr, int64_t* step_counter,
                                     double* e_pot, double* e_kin) {
  if (!m || !pos || !vel || !force || !species || !mass || !e_pot || !e_kin) return ALLEGRO_ERR_BAD_ARG;
  if (!m->work) m->work = new Work();
  DevBuf& stage = m->work->host_stage;   // [pos | vel | force | e_pot, e_kin | mass | species], owned by the model
  size_t b3 = (size_t)N * 24, off_e = 3 * b3, off_m = off_e + 16, off_s = off_m + (size_t)m->S * 8;
  AL_CHECK(al_reserve(m, stage, off_s + (size_t)N * 4 + 64));
  char* d = (char*)stage.p;
  cudaStream_t st = m->stream;
  AL_CUDA(m, cudaMemcpyAsync(d, pos, b3, cudaMemcpyHostToDevice, st));
  AL_CUDA(m, cudaMemcpyAsync(d + b3, vel, b3, cudaMemcpyHostToDevice, st));
  AL_CUDA(m, cudaMemcpyAsync(d + 2 * b3, force, b3, cudaMemcpyHostToDevice, st));
  AL_CUDA(m, cudaMemcpyAsync(d + off_m, mass, (size_t)m->S * 8, cudaMemcpyHostToDevice, st));
  AL_CUDA(m, cudaMemcpyAsync(d + off_s, species, (size_t)N * 4, cudaMemcpyHostToDevice, st));
  AL_CHECK(allegro_step_nve(m, (double*)d, (double*)(d + b3), (double*)(d + 2 * b3), (const int32_t*)(d + off_s),
                            (const double*)(d + off_m), N, box, dt_fs, rebuild_every, skin, nbr, step_counter,
                            (double*)(d + off_e), (double*)(d + off_e + 8)));
  AL_CUDA(m, cudaMemcpyAsync(pos, d, b3, cudaMemcpyDeviceToHost, st));
  AL_CUDA(m, cudaMemcpyAsync(vel, d + b3, b3, cudaMemcpyDeviceToHost, st));
  AL_CUDA(m, cudaMemcpyAsync(force, d + 2 * b3, b3, cudaMemcpyDeviceToHost, st));
  AL_CUDA(m, cudaMemcpyAsync(e_pot, d + off_e, 8, cudaMemcpyDeviceToHost, st));
  AL_CUDA(m, cudaMemcpyAsync(e_kin, d + off_e + 8, 8, cudaMemcpyDeviceToHost, st));
  AL_CUDA(m, cudaStreamSynchronize(st));
  return al_check_status(m);
}

extern "C" int allegro_debug_tensor(allegro_model* m, const char* name, float* out, int64_t* n_floats) {
  if (!m || !name || !out || !n_floats || !m->work) return ALLEGRO_ERR_BAD_ARG;
  Work& w = *m->work;
  if (m->hfmt >= 0 && name[0] != 'Y' && name[0] != 'u' && name[0] != 'B' && name[0] != 'g' && name[0] != 'e') {
    al_set_error(m, "debug taps of latent tensors are fp32-only (16-bit operand mode)");
    return ALLEGRO_ERR_UNIMPLEMENTED;
  }
  int M = 0;
  AL_CUDA(m, cudaStreamSynchronize(m->stream));
  AL_CUDA(m, cudaMemcpy(&M, w.m_act.p, 4, cudaMemcpyDeviceToHost));
  std::string s(name);
  const float* src = nullptr; int width = 0, ld = 0; int64_t rows = M;
  int d = m->d, n = m->n;
  if (s == "Y") { src = (float*)w.Y.p; width = m->Denv; ld = m->ldY; }
  else if (s == "u") { src = (float*)w.u.p; width = ld = 1; }
  else if (s == "B") { src = (float*)w.B.p; width = ld = m->NB; }
  else if (s == "geo") { src = (float*)w.geo.p; width = ld = 4; }
  else if (s == "ge") { src = (float*)w.ge.p; width = ld = 3; }
  else if (s == "ybar") { src = (float*)w.Ybar.p; width = ld = m->Denv; }
  else if (s == "ubar") { src = (float*)w.ubar.p; width = ld = 1; }
  else if (s == "ei") { src = (float*)w.ei.p; width = ld = 1; }
  else if (s == "ej") { src = (float*)w.ej.p; width = ld = 1; }
  else if (s == "we") { src = (float*)w.WE.p; width = ld = 2 * m->nA; }
  else if (s[0] == 'x' && s.size() == 2) {
    int L = s[1] - '0';
    if (L < 0 || L > m->NL) return ALLEGRO_ERR_BAD_ARG;
    if (L == m->NL) { src = (float*)w.XF.p; width = ld = d; } else { src = (float*)w.XS[L].p; width = d; ld = d + n; }
  } else if (s[0] == 's' && s.size() == 2) {
    int L = s[1] - '0';
    if (L < 1 || L > m->NL) return ALLEGRO_ERR_BAD_ARG;
    src = (float*)w.XS[L - 1].p + d; width = n; ld = d + n;
  } else if (s[0] == 'V' && s.size() == 2) {
    int L = s[1] - '0';
    if (L < 1 || L >= m->NL) return ALLEGRO_ERR_BAD_ARG;
    if (!w.T[L].p) { al_set_error(m, "V^L is never formed by the per-centre-contracted tensor track (allegro_set_tensor_track 1 keeps it)"); return ALLEGRO_ERR_BAD_ARG; }
    src = (float*)w.T[L].p; width = ld = m->D[L] * n;
  } else if (s == "gamma") { src = (float*)w.gamma.p; width = ld = m->Denv * n; rows = w.last_nc; }
  else { al_set_error(m, "unknown debug tensor"); return ALLEGRO_ERR_BAD_ARG; }
  int64_t need = rows * width;
  if (need > *n_floats) { *n_floats = need; al_set_error(m, "debug buffer too small"); return ALLEGRO_ERR_CAPACITY; }
  if (need > 0) AL_CUDA(m, cudaMemcpy2D(out, (size_t)width * 4, src, (size_t)ld * 4, (size_t)width * 4, rows, cudaMemcpyDeviceToHost));
  *n_floats = need;
  return ALLEGRO_OK;
}
