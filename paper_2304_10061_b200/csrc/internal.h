// Internal structures of libb200allegro (not part of the C ABI).
#pragma once
#include <atomic>
#include <cstdlib>
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "b200_allegro.h"

#define AL_MAX_LAYERS 8

// ---- error plumbing ------------------------------------------------------------------------------
void al_set_error(const allegro_model* m, const std::string& msg);
#define AL_CUDA(m, expr)                                                                          \
  do {                                                                                            \
    cudaError_t _e = (expr);                                                                      \
    if (_e != cudaSuccess) {                                                                      \
      al_set_error(m, std::string(#expr) + ": " + cudaGetErrorString(_e));                        \
      return ALLEGRO_ERR_CUDA;                                                                    \
    }                                                                                             \
  } while (0)
#define AL_CHECK(expr)             \
  do {                             \
    int _r = (expr);               \
    if (_r != ALLEGRO_OK) return _r; \
  } while (0)

// cudaFuncSetAttribute is per (kernel, device): one static AttrOnce per launch site remembers which device ordinals
// already carry the attribute, so a second model on another device of the same process sets it again (thread-safe).
struct AttrOnce {
  std::atomic<uint64_t> mask{0};
  bool need(int dev) const { return !(mask.load(std::memory_order_acquire) & (1ull << (dev & 63))); }
  void done(int dev) { mask.fetch_or(1ull << (dev & 63), std::memory_order_release); }
};

// ---- host-side description of the tensor track ---------------------------------------------------
struct Irrep { int l, p; };

struct TPLayerHost {
  std::vector<Irrep> in, out;      // S_{L-1}, S_L
  int Din, Dout, Denv;
  struct Path { int i1, l2, io; };
  std::vector<Path> paths;
  std::vector<int> fan;
  // fused tensor K[a,b,c] as a sparse list, grouped into (a,c) "pairs"
  int npairs;
  std::vector<int> pair_a, pair_c;            // [npairs]
  std::vector<int> pair_ptr;                  // [npairs+1] -> entries (b,val) of K
  std::vector<int> ent_b; std::vector<float> ent_val;
  std::vector<int> ent_idx;                   // [nnz] a*Dout + c of the entry's pair
  // packed entry lists (a | c<<8 | b<<16, val): sorted by c (ce_*, cent_ptr[Dout+1]) and by a (ae_*, aent_ptr[Din+1])
  std::vector<int> ce_pack, cent_ptr, ae_pack, aent_ptr; std::vector<float> ce_val, ae_val;
  // dense pair table: entries (b, val) of pair (a, c) are dp_b/dp_val[dp_ptr[a*Dout+c] .. dp_ptr[a*Dout+c+1])
  std::vector<int> dp_ptr, dp_b; std::vector<float> dp_val;
  // CSR over output component c -> (a, pair)
  std::vector<int> c_ptr, c_a, c_p;
  // CSR over input component a -> (c, pair)
  std::vector<int> a_ptr, a_c, a_p;
  // CSR over env component b -> (pair, val)
  std::vector<int> b_ptr, b_p; std::vector<float> b_val;
  int nnz;
};

// device copy of the tables of one layer
struct TPLayerDev {
  int Din, Dout, Denv, npairs, nnz;
  int *pair_a, *pair_c, *pair_ptr, *ent_b; float* ent_val; int* ent_idx;
  int *c_ptr, *c_a, *c_p;
  int *a_ptr, *a_c, *a_p;
  int *b_ptr, *b_p; float* b_val;
  int *ce_pack, *cent_ptr, *ae_pack, *aent_ptr; float *ce_val, *ae_val;
  int *dp_ptr, *dp_b; float* dp_val;
};

struct Dense {
  int fi = 0, fo = 0;
  float* W = nullptr;    // [fi][fo] row-major  (B operand of dX = dY * W^T, K-major over fo)
  float* Wt = nullptr;   // [fo][fi] row-major  (B operand of Y = X * W, K-major over fi)
  // precision 0 on tensor cores (3xTF32): W_hi = rn_tf32(W), W_lo = rn_tf32(W - W_hi); same two layouts
  float *W_hi = nullptr, *W_lo = nullptr, *Wt_hi = nullptr, *Wt_lo = nullptr;
  // 16-bit operand modes (precision 2 bf16 / 4 fp16): the same two layouts as 16-bit elements
  void *W16 = nullptr, *Wt16 = nullptr;
};

struct DevBuf {
  void* p = nullptr; size_t bytes = 0;
};

struct Chunk { int64_t c0, c1; int64_t e0, e1; };   // centers [c0,c1), candidate edges [e0,e1)

struct allegro_nbr {
  uint64_t version = 0;                // incremented by every build (keys the CUDA-graph replay of the MD step)
  int64_t n_atoms = 0, n_edges = 0;
  double cutoff = 0; double box[3] = {0, 0, 0};
  DevBuf row_ptr, j, shift, keys;      // int64[N+1], int32[E], int8[3E], uint64[E] scratch
  DevBuf wpos, q, cell_of, cell_cnt, cell_start, cell_atoms, deg, scan_tmp;
  std::vector<int64_t> row_ptr_host;
  std::vector<Chunk> chunks; int64_t chunk_cap = 0;
  int64_t max_chunk_edges = 0, max_chunk_centers = 0;
};

struct allegro_model {
  allegro_hparams hp;
  int S, NB, d, n, lmax, NL, Denv, nA, ldY;   // ldY = Denv rounded up to a multiple of 4 (float4 rows of Y)
  std::vector<TPLayerHost> tp_host;       // [NL]
  std::vector<TPLayerDev> tp;             // [NL]
  std::vector<int> D;                     // D_0..D_NL
  // V^0 layout: position -> l, -> index in Y
  std::vector<int> v0_l, v0_y; int *d_v0_l = nullptr, *d_v0_y = nullptr, *d_env_l = nullptr;
  // weights
  std::vector<Dense> twobody;             // twobody[0] is the (2S+NB)-input layer
  Dense emb01;                            // [A0 | A1] : d -> 2 nA, columns permuted to (l, n)
  std::vector<Dense> emb;                 // emb[L] = A^{L+1} for L >= 1 (index 0 unused)
  std::vector<std::vector<Dense>> latent; // [NL][n_latent]
  // backward of layer L: x-bar^{L-1} = z-bar W_x^T + omega-bar A^T as ONE GEMM over the concatenated K axis,
  // xcat[L-1].W = [W_lat0[:d, :] | A] ([d][h + Kx]); sbar[L-1].W = W_lat0[d:, :] ([n][h]) gives s-bar alone
  std::vector<Dense> xcat, sbar;
  float* w_eff_f = nullptr; double* w_eff_d = nullptr;   // product of the edge-MLP layers, [d]
  double *sigma = nullptr, *mu = nullptr; // device [S]
  double* d_rc_pair = nullptr;            // device [S][S] ordered species-pair cutoffs, or null (flat r_cut)
  double* d_bfreq = nullptr;              // device [S][S][NB] trained Bessel angular frequencies, or null (n pi / r_c)
  double* d_zbl_Z = nullptr;              // device [S] atomic numbers: ZBL pair repulsion on, or null
  std::vector<double> sigma_h, mu_h;
  float c_env; float c_old[AL_MAX_LAYERS], c_new[AL_MAX_LAYERS];
  // runtime
  cudaStream_t stream = 0;
  allegro_alloc_fn alloc_fn = nullptr; allegro_free_fn free_fn = nullptr; void* alloc_user = nullptr;
  int64_t chunk_edges = 1 << 20;
  int hfmt = -1;                          // 16-bit operand modes: 0 fp16 (precision 4), 1 bf16 (precision 2); -1: fp32 activations
  int tt_mode = 0;                        // tensor track: 0 contracted per centre (tpc_impl.cuh), 1 per-edge products (allegro_set_tensor_track)
  bool debug_keep = false;                // allegro_set_debug: also store tensors that are otherwise consumed on chip
  int64_t launches = 0;
  // Alternating sweep direction of the edge-ordered kernels (GEMM row tiles, tensor-track centres): every such launch
  // walks the edge range opposite to the one before it, so it starts on the rows its producer wrote last (still in the
  // 126 MB L2) instead of on rows evicted long ago.  Results do not depend on the order.
  unsigned sweep_ctr = 0;
  std::string err;
  int sm_count = 148;
  int device = 0;                         // CUDA device ordinal the model was created on
  void* tmaps = nullptr;                  // tensor-map cache of the tcgen05 GEMMs (gemm_tc.cu), freed by al_gemm_tc_free
  // workspace (per chunk), grown on demand
  struct Work* work = nullptr;
  bool work_sized = false;                // the per-chunk buffers have been laid out (fixes the tensor-track mode)
  // per-kernel-group event timing (allegro_profile_*)
  bool prof = false;
  struct ProfRec { int cat; cudaEvent_t a, b; };
  bool gemm_cta_pairs = true;            // MLP GEMMs on CTA pairs (cta_group::2, 256-row tiles) when the problem is large enough
  bool nvtx = false;                      // allegro_profile_enable bit 1: NVTX range per kernel group (host side)
  std::vector<ProfRec> prof_recs;
  std::vector<cudaEvent_t> prof_pool;
  std::vector<void*> owned;               // device allocations made through al_alloc (weights/tables)
  // CUDA-graph replay of the steps of allegro_step_nve that do not rebuild the list (launch-bound small systems):
  // a step whose key (all arguments, list version, configuration and allocation generations) was seen once eagerly
  // is captured the next time and replayed from then on.
  struct StepGraph {
    cudaGraphExec_t exec = nullptr; cudaStream_t cap = nullptr;
    std::vector<uint64_t> key, warm; int64_t nlaunch = 0, steps = 0; bool disabled = false;
  } sg;
  uint64_t config_gen = 0, alloc_gen = 0; // bumped by every setter / every (re)allocation of a work buffer
};

// direction of the next edge-ordered launch (0 forward, 1 reversed), see allegro_model::sweep_mode
inline int al_next_rev(allegro_model* m) { return (int)(m->sweep_ctr++ & 1u); }

// ---- profiling ------------------------------------------------------------------------------------
enum ProfCat { PC_GEMM = 0, PC_TP_FWD, PC_TP_BWD, PC_GEOM, PC_TWOBODY0, PC_ENERGY, PC_BWD_ELEM, PC_EDGE_BWD, PC_NEIGHBORS,
               PC_NVE, PC_COUNT };
struct ProfScope {
  allegro_model* m; int cat; cudaEvent_t a = nullptr; bool range = false;
  ProfScope(allegro_model* m_, int cat_);
  ~ProfScope();
};

// ---- allocation helpers ---------------------------------------------------------------------------
int al_alloc(allegro_model* m, void** p, size_t bytes);
void al_free(allegro_model* m, void* p);
int al_reserve(allegro_model* m, DevBuf& b, size_t bytes);   // grow-only with +5 % head-room
void al_release(allegro_model* m, DevBuf& b);

// ---- sub-systems ----------------------------------------------------------------------------------
int al_build_tp_tables(allegro_model* m, const std::vector<std::vector<float>>& alphas);   // cg_tables.cpp
void al_enumerate(int lmax, int NL, std::vector<std::vector<Irrep>>& S,
                  std::vector<std::vector<TPLayerHost::Path>>& paths);
int al_neighbors_impl(allegro_model* m, const double* pos, int64_t n_atoms, const double box[3], double cutoff,
                      allegro_nbr** inout);
int al_compute_impl(allegro_model* m, const double* pos, const int32_t* species, int64_t n_atoms,
                    const double box[3], const allegro_nbr* nbr, double* e_total, double* e_atom, double* force /*null: energy only*/,
                    double* e_edge /*null or f64[nbr->n_edges]*/);
int al_compute_local_impl(allegro_model* m, const double* pos, const int32_t* species, int64_t n_atoms, int64_t n_local,
                          const double box[3], const allegro_nbr* nbr, double* e_total, double* e_atom, double* force,
                          double* e_edge);
int al_exclusive_scan_i64(allegro_model* m, const int32_t* in, int64_t* out, int64_t n, DevBuf& tmp);  // out[n] = total
void al_work_free(allegro_model* m);
int al_check_status(allegro_model* m);   // compute.cu: synchronise, read + clear the device status word -> error code
