/* b200_allegro.h — C ABI of the B200-native Allegro energy+force path (arXiv 2304.10061).
 *
 * One library, libb200allegro.so, hand-written CUDA for sm_100a.  Every entry point below is one of
 * the calls of SURVEY.md §8(b); each cites the passage of /root/reference/PAPER.md (or the SURVEY §8(c)
 * reading, where the paper is silent) that defines the operation.
 *
 * Conventions
 *   - C linkage, no C++ type crosses the boundary.  Every function returns int: 0 = ALLEGRO_OK,
 *     negative = error (table below).  allegro_last_error() gives a human-readable message for the
 *     last failing call on that model (or the last failing call without a model).
 *   - Pointer arguments are DEVICE pointers on the current CUDA device unless the parameter comment
 *     says "host".  The `_host` variants take HOST pointers for every array and do the copies inside.
 *   - The caller owns every array it passes in or receives results into.  Opaque handles
 *     (allegro_model, allegro_nbr) are created and destroyed by the library.
 *   - Work is enqueued on the stream set by allegro_set_stream (default: the legacy default stream).
 *     Device-pointer calls return after enqueueing, except allegro_neighbors, which synchronises the
 *     stream once (the edge count is needed on the host to size the list).
 *   - Units: Angstrom, eV, fs, amu.  Species are int32 in [0, n_species).
 *   - Box: orthorhombic, fully periodic, box[3] = edge lengths > 0 (host pointer).
 *   - There is NO CPU fallback: without a CUDA device every compute call returns ALLEGRO_ERR_CUDA.
 */
#ifndef B200_ALLEGRO_H
#define B200_ALLEGRO_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
  ALLEGRO_OK = 0,
  ALLEGRO_ERR_BAD_HPARAMS = -1,   /* inconsistent hyper-parameters (incl. latent width != d, l_max > 3) */
  ALLEGRO_ERR_BLOB_SIZE = -2,     /* blob_bytes != allegro_blob_size()                                */
  ALLEGRO_ERR_BOX_TOO_SMALL = -3, /* an image shift does not fit int8                                 */
  ALLEGRO_ERR_CAPACITY = -4,      /* an internal capacity was exceeded                                */
  ALLEGRO_ERR_NONFINITE = -5,     /* coincident atoms (r = 0) or non-finite input                     */
  ALLEGRO_ERR_CUDA = -6,          /* CUDA runtime error / no device                                   */
  ALLEGRO_ERR_UNIMPLEMENTED = -7,
  ALLEGRO_ERR_BAD_ARG = -8
};

typedef struct allegro_model allegro_model; /* weights, CG tables, workspaces */
typedef struct allegro_nbr allegro_nbr;     /* CSR neighbor list on device     */

/* Hyper-parameters (PAPER.md:222 lists the paper's values; SURVEY §8 table the five configs). */
typedef struct {
  int32_t n_species, l_max, n_layers, n_tensor, n_bessel, poly_p;
  double r_cut;
  int32_t n_twobody;
  int32_t twobody_dims[8]; /* hidden widths; last = latent width d */
  int32_t n_latent;
  int32_t latent_dims[8];  /* same shape for every layer; last must equal d */
  int32_t n_edge;
  int32_t edge_dims[8];    /* hidden widths; the final ->1 layer is implicit */
  double avg_num_neighbors; /* c_env = 1/sqrt(this)                  (S7) */
  double resid_alpha[8];    /* per layer residual mixing coefficient (S7) */
  int32_t precision;        /* MLP GEMM arithmetic (accumulation is fp32 in all modes):
                               0 fp32 on the tensor cores (3xTF32 split operands, meets the fp32 tolerances),
                               1 TF32 tensor cores (the paper's scheme), 3 fp32 on the FFMA pipes (slowest, most accurate),
                               2 / 4 16-bit operand MLPs: every tensor that only the MLP GEMMs and their epilogues touch
                               (activations, pre-activations, latents x^L, their gradients) and the weights are stored as
                               bfloat16 (2) or IEEE fp16 (4), tcgen05 kind::f16, fp32 accumulation, fp32 tensor track and fp64
                               final stage as in the other modes; needs >= 2 two-body layers, d and n_tensor multiples of 32, a
                               first latent width that is a multiple of 64 and a model the contracted tensor track covers
                               (else ALLEGRO_ERR_BAD_HPARAMS at create / ALLEGRO_ERR_UNIMPLEMENTED at the first compute) */
  int64_t max_atoms, max_edges; /* capacity hints, 0 = grow on demand (+5 %) */
} allegro_hparams;

/* Number of bytes of the flat weight blob for these hyper-parameters (layout: SURVEY §8(b),
 * restated in DESIGN.md).  host pointers. */
int allegro_blob_size(const allegro_hparams* hp, size_t* bytes);

/* Tensor-product path table (enumeration SURVEY §8(c) S6).  For layer L (1-based)
 * returns the number of paths; if fan != NULL (host int32[n_paths]) fills, per path in canonical
 * order, how many paths of that layer share the path's output irrep.  dims (host int32[2], may be
 * NULL) receives {D_{L-1}, D_L}, the feature widths sum(2l+1) before / after the layer. */
int allegro_path_info(const allegro_hparams* hp, int32_t layer, int32_t* n_paths, int32_t* fan, int32_t* dims);

/* Create a model from hyper-parameters and the flat blob (host pointers).  Builds irreps, paths, the
 * path-weight-fused real Clebsch-Gordan tensors K^L (Fig. 3) and uploads weights. */
int allegro_create(const allegro_hparams* hp, const void* blob, size_t blob_bytes, allegro_model** out);
int allegro_destroy(allegro_model* m);

/* cudaStream_t to enqueue on, passed as void* (e.g. torch.cuda.current_stream().cuda_stream). */
int allegro_set_stream(allegro_model* m, void* cuda_stream);

/* Optional device allocator hooks (e.g. PyTorch's caching allocator); default cudaMalloc/cudaFree.
 * Must be set before the first neighbors/compute call. */
typedef void* (*allegro_alloc_fn)(size_t bytes, void* user);
typedef void (*allegro_free_fn)(void* ptr, void* user);
int allegro_set_allocator(allegro_model* m, allegro_alloc_fn a, allegro_free_fn f, void* user);

/* Maximum number of active edges processed per center-contiguous chunk (strict locality,
 * PAPER.md:138, makes chunks independent).  Default 1<<20. */
int allegro_set_chunk_edges(allegro_model* m, int64_t max_edges_per_chunk);

/* Periodic cell-list neighbor build (PAPER.md:128 ordered pairs).  Edge set =
 * {(i,j,s): (i!=j or s!=0), d2 < cutoff^2}, dx = (x_j - x_i) + s_x*L_x, d2 = (dx*dx+dy*dy)+dz*dz in
 * fp64 without FMA contraction; CSR by i, each row sorted by (j, sx, sy, sz); positions need not be
 * wrapped (shifts are relative to the positions as given).
 * pos: device f64[n_atoms*3]; box: host f64[3]; *inout: reused (buffers kept) if non-NULL. */
int allegro_neighbors(allegro_model* m, const double* pos, int64_t n_atoms, const double box[3], double cutoff,
                      allegro_nbr** inout);
int allegro_neighbors_host(allegro_model* m, const double* pos_host, int64_t n_atoms, const double box[3],
                           double cutoff, allegro_nbr** inout);
/* Read-only DEVICE views of the list: row_ptr int64[n_atoms+1], j int32[n_edges], shift int8[n_edges*3]. */
int allegro_nbr_info(const allegro_nbr* n, int64_t* n_atoms, int64_t* n_edges, const int64_t** row_ptr,
                     const int32_t** j, const int8_t** shift);
/* Copy the list to host arrays (row_ptr int64[n_atoms+1], j int32[n_edges], shift int8[n_edges*3]). */
int allegro_nbr_copy_host(allegro_model* m, const allegro_nbr* n, int64_t* row_ptr, int32_t* j, int8_t* shift);
int allegro_nbr_free(allegro_model* m, allegro_nbr* n);

/* Energy and forces (PAPER.md:128 energy decomposition; Eq. (2) PAPER.md:132-138 layers
 * fp64 final stage; forces F_i = -dE/dr_i by the hand-written analytic backward).
 * The list may have been built at cutoff >= r_cut (Verlet skin); edges with r >= r_cut are dropped.
 * pos f64[N*3], species i32[N], e_total f64[1], e_atom f64[N] or NULL, force f64[N*3] (device), or NULL for an
 * energy-only evaluation (the backward pass is skipped). */
int allegro_compute(allegro_model* m, const double* pos, const int32_t* species, int64_t n_atoms,
                    const double box[3], const allegro_nbr* nbr, double* e_total, double* e_atom, double* force);
int allegro_compute_host(allegro_model* m, const double* pos, const int32_t* species, int64_t n_atoms,
                         const double box[3], const allegro_nbr* nbr, double* e_total, double* e_atom,
                         double* force);

/* Energy and forces of a spatial domain (the paper runs one rank per GPU over LAMMPS's
 * spatial decomposition).  The first n_local atoms are the domain's own atoms and the only
 * centres; atoms n_local .. n_atoms-1 are ghosts (copies, with their image shift applied, of atoms owned by other
 * domains or by this one across a periodic face) and appear as neighbours only.  e_total = sum of E-hat_i over the local
 * atoms, e_atom[i] = 0 for ghosts, force f64[n_atoms*3] = -d(e_total)/dr for local AND ghost atoms: the ghost part is what
 * the reverse exchange returns to the owners, after which every owner holds its complete force (strict locality,
 * PAPER.md:138).  With ZBL on, local atoms receive their complete pair force and ghosts none.  box is the periodic cell
 * of the coordinates passed in: for a domain it must exceed the extent of local + ghost atoms by more than the cutoff
 * in every direction, so that no pair is found through the boundary.  The list must have been built from the same
 * n_atoms positions.  Arguments otherwise as allegro_compute. */
int allegro_compute_local(allegro_model* m, const double* pos, const int32_t* species, int64_t n_atoms, int64_t n_local,
                          const double box[3], const allegro_nbr* nbr, double* e_total, double* e_atom, double* force);

/* Deferred errors of the device-pointer calls.  allegro_compute / allegro_compute_local / allegro_edge_energies /
 * allegro_step_nve return after enqueueing, so what only the kernels can see -- coincident atoms (r = 0; the survey's
 * ALLEGRO_ERR_NONFINITE) and species values outside [0, n_species) (ALLEGRO_ERR_BAD_ARG; table
 * look-ups clamp, nothing is read out of bounds) -- is recorded in a device status word.  allegro_status synchronises the
 * model's stream, returns the recorded error (ALLEGRO_OK if none) and clears it.  The same check runs inside every call
 * that synchronises anyway: the _host variants, and allegro_step_nve on the steps that rebuild the list. */
int allegro_status(allegro_model* m);

/* Halo kernels of the spatial decomposition (NEXT-3; the paper's ghost-atom forward / reverse communication, PAPER.md:188,
 * 214-216).  The messages themselves travel through torch.distributed (paper_2304_10061_b200/domain.py); these calls do
 * the per-atom work on the device (all pointers DEVICE pointers, enqueued on the model's stream):
 *   allegro_halo_pack: for the n_send ghosts this rank provides, out_rows[k] = {pos[idx[k]] + shift[k], (double)species[idx[k]]}
 *     (f64[n_send*4]); idx int64[n_send] indexes the rank's own atoms, shift f64[n_send*3] is the periodic image shift.
 *   allegro_halo_assemble: pos_all f64[(n_local+n_ghost)*3] = {own positions, received ghost rows} - origin (host f64[3]),
 *     species_all int32[n_local+n_ghost] likewise: the arrays allegro_compute_local takes.
 *   allegro_halo_accumulate: force_out f64[n_local*3] = force_all[0 : n_local] + sum over k of returned[k] at atom idx[k]
 *     (returned f64[n_send*3]: what the other domains accumulated on the ghosts this rank provided; an atom may appear
 *     several times, fp64 atomics). */
int allegro_halo_pack(allegro_model* m, const double* pos, const int32_t* species, const int64_t* idx, const double* shift,
                      int64_t n_send, double* out_rows);
int allegro_halo_assemble(allegro_model* m, const double* pos, const int32_t* species, int64_t n_local,
                          const double* ghost_rows, int64_t n_ghost, const double origin[3], double* pos_all,
                          int32_t* species_all);
int allegro_halo_accumulate(allegro_model* m, const double* force_all, int64_t n_local, const int64_t* idx,
                            const double* returned, int64_t n_send, double* force_out);

/* One velocity-Verlet NVE step: v += dt/2 F/m; r += dt v; [rebuild list at cutoff
 * r_cut+skin if *step_counter % rebuild_every == 0]; F; v += dt/2 F/m.  `force` f64[N*3] (device) must
 * hold F(r) of the current positions on entry (call allegro_compute once before the first step) and
 * holds F of the new positions on exit.  mass: device f64[n_species].  e_pot, e_kin: device f64[1].
 * step_counter: host int64, incremented. */
int allegro_step_nve(allegro_model* m, double* pos, double* vel, double* force, const int32_t* species,
                     const double* mass, int64_t n_atoms, const double box[3], double dt_fs,
                     int32_t rebuild_every, double skin, allegro_nbr** nbr, int64_t* step_counter,
                     double* e_pot, double* e_kin);

/* The two halves of the velocity-Verlet step on their own, for drivers that put something between them (the domain-
 * decomposed step exchanges halos there): v += dt/2 F/m * 9.648533212e-3 and, if drift != 0, r += dt v.
 * allegro_kinetic_energy: e_kin = sum_i m_i v_i^2 / 2 in eV (device f64[1]), fixed-order reduction.  Device pointers. */
int allegro_nve_kick(allegro_model* m, double* pos, double* vel, const double* force, const int32_t* species,
                     const double* mass, int64_t n_atoms, double dt_fs, int32_t drift);
int allegro_kinetic_energy(allegro_model* m, const double* vel, const int32_t* species, const double* mass,
                           int64_t n_atoms, double* e_kin);

/* allegro_kinetic_energy without any allocation, for callers that may not call cudaMalloc (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid it).  Same arguments (device pointers), same fixed-order reduction and the same
 * value as allegro_kinetic_energy; the per-atom scratch that call reserves with cudaMalloc lives here in a fixed __device__
 * array of ALLEGRO_KINETIC_NOALLOC_MAX_ATOMS doubles (8 MiB, held by every GPU that loads the library until the process
 * exits).  n_atoms beyond that limit: ALLEGRO_ERR_CAPACITY, nothing launched.  The model's device must be current
 * (ALLEGRO_ERR_BAD_ARG otherwise).  The call never calls cudaMalloc / cudaFree or an allocating library routine; the kernels
 * run on the model's stream.  Every call on a device shares the one array and nothing in it needs to start at zero (a call
 * reads only what it wrote), so calls ordered on one stream are safe, while calls that OVERLAP on the GPU (other streams, other
 * models on the same device) race on it and must be serialised by the caller.  (csrc/noalloc.cu) */
#define ALLEGRO_KINETIC_NOALLOC_MAX_ATOMS 1048576
int allegro_kinetic_energy_noalloc(allegro_model* m, const double* vel, const int32_t* species, const double* mass,
                                   int64_t n_atoms, double* e_kin);

/* allegro_step_nve replays the steps that do not rebuild the list from a CUDA graph: a step whose arguments, list and
 * configuration are those of the previous (eagerly run) step is captured once and relaunched as one graph from then on
 * (the small configs are launch-bound: ~36 kernels of a few microseconds each); any change of an argument, a rebuild, a
 * setter call or a buffer growth falls back to eager launches and re-captures.  The environment variable
 * B200_ALLEGRO_NO_GRAPH disables it.  n receives the number of steps served by a graph launch so far, -1 if graph
 * capture failed and was switched off (host). */
int allegro_graph_steps(const allegro_model* m, int64_t* n);

/* Same step with HOST arrays (pos, vel, force f64[N*3], species i32[N], mass f64[n_species], e_pot,
 * e_kin f64[1]): copies state host->device, runs allegro_step_nve, copies state and energies back,
 * and synchronises.  Pinned host memory makes the copies asynchronous. */
int allegro_step_nve_host(allegro_model* m, double* pos, double* vel, double* force, const int32_t* species,
                          const double* mass, int64_t n_atoms, const double box[3], double dt_fs,
                          int32_t rebuild_every, double skin, allegro_nbr** nbr, int64_t* step_counter,
                          double* e_pot, double* e_kin);

/* Tile shape of the tensor-core MLP GEMMs.  pairs != 0 (the default): launches large enough to give every pair of SMs a tile run
 * on CTA pairs (thread-block clusters of 2, tcgen05 cta_group::2): 256-row tiles, each CTA loads its 128 rows of the activations
 * and half of the weight tile, so the weights cross L2 -> SM once per 256 rows.  pairs == 0: 128-row tiles on single CTAs
 * everywhere (what small launches always use).  Same arithmetic either way (the accumulation order over K
 * is identical); meant for tests and A/B timing.  Host call, takes effect at the next launch. */
int allegro_set_gemm_pairs(allegro_model* m, int32_t pairs);

/* Per-kernel-group device timing (bench roofline).  While enabled, every kernel group launched by the
 * library is bracketed by CUDA events on the launching stream.  allegro_profile_read synchronises and
 * returns, for group `name` ("gemm", "tp_fwd", "tp_bwd", "geom", "twobody0", "energy", "bwd_elem",
 * "edge_bwd", "neighbors", "nve"), the summed milliseconds and the launch count since enable, plus for
 * "gemm" the summed algorithmic FLOPs (2*M*N*K with M the chunk's candidate-edge capacity is NOT used:
 * flops are computed by the caller from allegro_last_active_edges).  host pointers.
 * `on` is a bit mask: 1 = the CUDA-event timing above; 2 = an NVTX range named after the group around the launches of every
 * group (host side, header-only nvtx3: costs nothing without a tool attached), so a profiler can select a group, e.g.
 * `ncu --nvtx --nvtx-include "tp_bwd/"`. */
int allegro_profile_enable(allegro_model* m, int32_t on);
int allegro_profile_read(allegro_model* m, const char* name, double* ms, int64_t* launches);

/* Roofline denominators for bench.py (the TF32 tensor-core and fp32 FFMA peaks are not in the
 * driver's MEASURED_PEAKS.json and have to be measured on the box).  allegro_probe_ffma: fp32 FMA rate of the SIMT pipes
 * (16 independent FMA chains per thread, no memory traffic).  allegro_probe_tf32: issue rate of tcgen05.mma kind::tf32
 * (128 x 256 x 8 MMAs back to back on shared-memory-resident operands, one CTA per SM, no loads, no epilogue).  Each
 * returns TFLOP/s (host f64): the best of 10 launches (burst) and the average over `sustain_s` seconds of back-to-back
 * launches (sustained, i.e. under the power cap).  Synchronises the model's stream.  Not part of the hot path. */
int allegro_probe_ffma(allegro_model* m, double sustain_s, double* burst_tflops, double* sustained_tflops);
int allegro_probe_tf32(allegro_model* m, double sustain_s, double* burst_tflops, double* sustained_tflops);

/* Counters for tests/bench: number of kernels launched by the library since creation (host). */
int allegro_launch_count(const allegro_model* m, int64_t* launches);
/* Total number of active (r < r_cut) edges, over all chunks, of the last allegro_compute (synchronises the stream). */
int allegro_last_active_edges(allegro_model* m, int64_t* n_active);

/* Ordered species-pair cutoffs ("independent cutoffs for each *ordered* species pair", values
 * :222): rc_pair is a HOST array [n_species][n_species], row = species of the centre i, column = species of the
 * neighbour j, every entry in (0, r_cut].  The ordered pair (i, j) is an edge iff r_ij < rc_pair[Z_i][Z_j]; the
 * envelope argument and the Bessel functions of that edge use the pair's own cutoff.  NULL restores the flat
 * r_cut.  Neighbor lists are still built at a cutoff >= r_cut (the largest pair cutoff). */
int allegro_set_pair_cutoffs(allegro_model* m, const double* rc_pair);

/* Trained Bessel angular frequencies of the "trainable per-ordered-species-pair radial basis":
 * freq is a HOST array [n_species][n_species][n_bessel] in 1/Angstrom (row = centre species, column = neighbour
 * species); b_n(r) = sqrt(2 / r_c) sin(freq_n r) / r with r_c the pair's cutoff.  NULL restores n pi / r_c. */
int allegro_set_bessel_frequencies(allegro_model* m, const double* freq);

/* ZBL pair repulsion ("We also add a repulsive Ziegler-Biersack-Littmark (ZBL) term"; formula: DESIGN.md
 * section 2): atomic_numbers is a HOST array [n_species]; adds 1/2 sum_j phi_ij(r_ij) to every E-hat_i (not scaled by
 * sigma) and the matching forces, phi_ij = k_e Z_i Z_j / r Phi(r / a_ij) u(r / r_cut), over all ordered pairs with
 * r < r_cut (the flat cutoff, also when ordered pair cutoffs are set).  NULL switches the term off. */
int allegro_set_zbl(allegro_model* m, const double* atomic_numbers);

/* Per-edge energies E_ij ("E_i = sum_j E_ij", before the sigma/mu scaling and without ZBL), forward pass
 * only: e_edge is a DEVICE array f64[n_edges of nbr], in the order of the list; candidates that are not edges
 * (r >= the pair's cutoff) receive 0.  e_total f64[1] (device) receives the total energy as allegro_compute does. */
int allegro_edge_energies(allegro_model* m, const double* pos, const int32_t* species, int64_t n_atoms,
                          const double box[3], const allegro_nbr* nbr, double* e_total, double* e_edge);

/* One thermostatted (NVT) step ("thermostat setting of 300K"; reading: DESIGN.md section 2): a single
 * Nose-Hoover variable, Q = g k_B T0 tau^2 with g = 3 n_atoms, split as [thermostat dt/2][allegro_step_nve][thermostat
 * dt/2]; thermostat half step: xi += dt/4 (2K - g k_B T0)/Q; v *= exp(-xi dt/2); xi += dt/4 (2K' - g k_B T0)/Q.
 * nh_state: DEVICE f64[2] = {xi (1/fs), eta = integral of xi dt}, zero-initialised by the caller; the conserved
 * quantity is e_kin + e_pot + Q xi^2/2 + g k_B T0 eta.  All other arguments as allegro_step_nve; e_kin receives the
 * kinetic energy after the final thermostat half step. */
int allegro_step_nvt(allegro_model* m, double* pos, double* vel, double* force, const int32_t* species,
                     const double* mass, int64_t n_atoms, const double box[3], double dt_fs, int32_t rebuild_every,
                     double skin, allegro_nbr** nbr, int64_t* step_counter, double* e_pot, double* e_kin,
                     double* nh_state, double t0_K, double tau_fs);

/* Which kernels run the tensor track (Eq. (2) :132-138; SURVEY.md section 8(a) steps 5-7 and their backward).
 *   0 (default)  contracted per centre: because tensor features only ever leave the track through their scalar block,
 *                s^L_e = V^0_e . (M^1_i ... M^{L-1}_i M^L_i e_0) with the per-centre operators contracted first; no
 *                [edges, D, n] tensor is formed.  Used whenever the model's irreps match the generated
 *                patterns (all five configs), up to 3 layers; other models fall back to mode 1 by themselves.
 *   1            one D_{L-1} x D_L product per edge, channel and layer, V^L_e stored: FFMA kernels (fp32 modes) or warp-level
 *                mma.sync TF32 (precision 1, l_max = 3: SURVEY NEXT-2, the paper's own TF32 tensor product).
 * Same function either way (fp32 summation order differs).  Must be called before the first compute call. */
int allegro_set_tensor_track(allegro_model* m, int32_t mode);

/* Debug mode (tests only; default off): keep every intermediate tensor that allegro_debug_tensor can name.
 * Without it the final latent x^{NL} is consumed inside the epilogue of the last latent GEMM and never stored. */
int allegro_set_debug(allegro_model* m, int on);

/* Debug/parity taps (tests only): copy an intermediate tensor of the LAST chunk of the last
 * allegro_compute to host as fp32.  name: "Y", "u", "x0", "x1".., "V1".., "gamma1".., "ebar".
 * n_floats: in = capacity of out, out = floats written. */
int allegro_debug_tensor(allegro_model* m, const char* name, float* out, int64_t* n_floats);

const char* allegro_last_error(const allegro_model* m);

#ifdef __cplusplus
}
#endif
#endif /* B200_ALLEGRO_H */
