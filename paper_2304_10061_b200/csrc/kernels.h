// Launch wrappers of the non-GEMM kernels (edge geometry, tensor track, energy, backward, NVE).
#pragma once
#include "internal.h"

// Per-chunk workspace.  All edge tensors are edge-major over the chunk's ACTIVE edges (r < r_cut),
// sorted by center.  Tensor-track features are [edge][component][channel] (channel fastest).
struct Work {
  int64_t cap_edges = 0, cap_centers = 0;
  DevBuf deg, rowa, scan_tmp, m_act;        // int32[Nc], int64[Nc+1], scan scratch, int32[4]
  DevBuf ei, ej;                            // int32[M] global atom ids
  DevBuf geo;                               // float4[M]: rhat.xyz, r
  DevBuf u, du;                             // float[M]: envelope u(r/rc), du/dr
  DevBuf sig;                               // float[M]: sigma_{Z_i(e)}
  DevBuf B, dB;                             // float[M][NB]: B_n = b_n u, dB_n/dr
  DevBuf Y;                                 // float[M][Denv]
  std::vector<DevBuf> tb_z, tb_a;           // two-body pre-activations / activations, [M][h_k]
  std::vector<DevBuf> XS;                   // [NL] : [M][d+n] = [x^{L-1} | s^L]
  DevBuf XF;                                // [M][d] final latent x^{NL}
  DevBuf WE;                                // [M][2 nA] = [w^0 | omega^1]  (component-major (l,n))
  std::vector<DevBuf> OM;                   // [NL+1]: omega^L for L >= 2, [M][nA]
  std::vector<DevBuf> T;                    // [NL]: T^L = V^L for L < NL, [M][D_L][n]
  std::vector<std::vector<DevBuf>> lat_z, lat_a;   // [NL][n_latent]
  DevBuf gamma;                             // [Nc][Denv][n] of the layer being processed (debug tap)
  // per-centre-contracted tensor track (tpc_impl.cuh): Gamma^L, n^L, Gamma-bar accumulators, each [NL][Nc][Denv][n];
  // s-bar^L of every layer [NL][M][n] (layer 1's backward needs them all); sb_ptr / sb_ld: where each layer's s-bar lives
  DevBuf tpc_gam, tpc_nvec, tpc_gacc, SB;
  std::vector<DevBuf> Gl;                   // [NL] per-layer [x-bar part | s-bar] buffers when the x-bar GEMM is not K-concatenated
  const float* sb_ptr[AL_MAX_LAYERS] = {}; int sb_ld[AL_MAX_LAYERS] = {};
  // backward
  DevBuf XB0, XB1;                          // x-bar ping-pong [M][d]
  DevBuf ZB0, ZB1;                          // z-bar ping-pong [M][max width]
  DevBuf G;                                 // [M][d+n] = [x-bar part | s-bar]
  DevBuf OB;                                // [M][2 nA] omega-bar (and w0-bar)
  DevBuf VB0, VB1;                          // V-bar ping-pong [M][Dmax][n]
  DevBuf ubar, Ybar;                        // u-bar partials [n_uparts][M]; Y-bar partials [groups*(NL+1)][M][Denv]
  int n_uparts = 1;
  DevBuf epart; int n_eparts = 0;           // f64 edge-energy partials [n_eparts][M] (EPI_LATENT_LAST)
  DevBuf ge;                                // float[M][3] dE/dr_e (debug tap)
  DevBuf eatom;                             // f64[N] when the caller passes e_atom = NULL
  DevBuf nh_scal;                           // f64[1]: velocity scale of the Nose-Hoover half step
  DevBuf host_stage;                        // device staging of allegro_step_nve_host
  int64_t eatom_cap = 0;
  int last_nc = 0;
};

struct EdgeGeomArgs {
  const double* pos; const int32_t* species; double box[3]; double rc; int p; int NB; int lmax;
  const double* rc_pair; int S;                                     // ordered species-pair cutoffs [S][S] or null
  const double* bfreq;                                              // Bessel angular frequencies [S][S][NB] or null
  const int64_t* row_ptr; const int32_t* j; const int8_t* shift;   // candidate list (global)
  int64_t c0; int nc;                                               // centers [c0, c0+nc)
};

bool tp2_eligible(const allegro_model* m);   // tp2_kernels.cu
bool tpc_eligible(const allegro_model* m);   // tpc_kernels.cu: the per-centre-contracted kernels run (default when possible)
// Y-bar partial buffers: part0[0] = first part of the V^0 contribution, part0[L] = first part of layer L's
// environment contribution (one part per channel group of the kernel that writes it); returns the total count.
int al_ybar_layout(const allegro_model* m, int* part0);
int k_launch_active_count(allegro_model* m, const EdgeGeomArgs& a, int* deg);
int k_launch_set_mact(allegro_model* m, const int64_t* rowa, int nc, int* m_act);
int k_launch_geom_fill(allegro_model* m, const EdgeGeomArgs& a, const int64_t* rowa, Work& w);
int k_launch_twobody0(allegro_model* m, Work& w, const int32_t* species, const Dense& L0, bool single, int m_cap);
int k_launch_tp_fwd(allegro_model* m, Work& w, int L, int nc, const float* om, int ldo, const float* Vin,
                    const float* w0, int ldw, float* Tout, float* xs, int ldx);
int k_launch_tp_bwd(allegro_model* m, Work& w, int L, int nc, const float* om, int ldo, const float* Vin,
                    const float* w0, int ldw, const float* Vbar_out_in /*V-bar^L or null*/, const float* sbar, int lds,
                    float* Vbar_prev, float* ombar, int ldob, float* w0bar);
int k_launch_energy(allegro_model* m, Work& w, const int32_t* species, int64_t c0, int nc, const float* xf,
                    double* e_atom);
int k_launch_sum_f64(allegro_model* m, const double* x, int64_t n, double* out);
int k_launch_bwd_prep(allegro_model* m, Work& w, const float* xbar, int ldx, const float* z, int ldz, float c,
                      float* zb, int ldzb, int width, int m_cap);
int k_launch_edge_bwd(allegro_model* m, Work& w, const float* zb1, int ldz, const Dense& L0, bool single,
                      double* force, int m_cap);
int k_launch_zero_f64(allegro_model* m, double* p, int64_t n);
int k_launch_begin_compute(allegro_model* m, double* force /*null: energy only*/, const int32_t* species, int64_t n, int* flags);
// ZBL pair repulsion over the candidate rows of the chunk's centres: e_atom[i] += 1/2 sum phi, force[i] += sum phi' rhat
int k_launch_zbl(allegro_model* m, const EdgeGeomArgs& a, const double* zbl_Z, double* e_atom, double* force);
// per-edge energies E_ij in candidate-list order (0 for dropped candidates)
int k_launch_edge_energy_out(allegro_model* m, const EdgeGeomArgs& a, Work& w, const float* xf, double* e_edge);
// Nose-Hoover thermostat half step on device scalars, then v *= s
int k_launch_nh_half(allegro_model* m, double* vel, int64_t n, double* nh_state, double* e_kin, double n_dof, double t0_K,
                     double tau_fs, double dt_fs, double* scratch);
int k_launch_nve_kick_drift(allegro_model* m, double* pos, double* vel, const double* force, const int32_t* species,
                            const double* mass, int64_t n, double dt, bool drift);
int k_launch_kinetic(allegro_model* m, const double* vel, const int32_t* species, const double* mass, int64_t n,
                     double* e_kin, DevBuf& tmp);
