// Halo kernels of the spatial decomposition (the paper runs one rank per GPU over LAMMPS's
// spatial decomposition with ghost-atom forward / reverse communication).  The exchange itself is
// torch.distributed plumbing (paper_2304_10061_b200/domain.py); what touches the atoms runs here:
//   allegro_halo_pack       rows [x, y, z, species] of the ghosts this rank provides (own atom + periodic image shift)
//   allegro_halo_assemble   local atoms + received ghosts -> one coordinate frame whose origin is the domain's halo corner
//   allegro_halo_accumulate forces of the local atoms + the forces other domains accumulated on the ghosts this rank provided
#include "internal.h"

namespace {

__global__ void k_halo_pack(const double* __restrict__ pos, const int32_t* __restrict__ species,
                            const int64_t* __restrict__ idx, const double* __restrict__ shift, int64_t k,
                            double* __restrict__ out) {
  const int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (t >= k) return;
  const int64_t i = idx[t];
  out[4 * t + 0] = pos[3 * i + 0] + shift[3 * t + 0];
  out[4 * t + 1] = pos[3 * i + 1] + shift[3 * t + 1];
  out[4 * t + 2] = pos[3 * i + 2] + shift[3 * t + 2];
  out[4 * t + 3] = (double)species[i];
}

__global__ void k_halo_assemble(const double* __restrict__ pos, const int32_t* __restrict__ species, int64_t n_local,
                                const double* __restrict__ ghosts, int64_t n_ghost, double ox, double oy, double oz,
                                double* __restrict__ pos_all, int32_t* __restrict__ species_all) {
  const int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (t >= n_local + n_ghost) return;
  double x, y, z; int32_t s;
  if (t < n_local) { x = pos[3 * t]; y = pos[3 * t + 1]; z = pos[3 * t + 2]; s = species[t]; }
  else {
    const int64_t g = t - n_local;
    x = ghosts[4 * g]; y = ghosts[4 * g + 1]; z = ghosts[4 * g + 2]; s = (int32_t)llrint(ghosts[4 * g + 3]);
  }
  pos_all[3 * t] = x - ox; pos_all[3 * t + 1] = y - oy; pos_all[3 * t + 2] = z - oz;
  species_all[t] = s;
}

__global__ void k_halo_copy_local(const double* __restrict__ f_all, int64_t n3, double* __restrict__ f_out) {
  const int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (t < n3) f_out[t] = f_all[t];
}

// an own atom can be a ghost of several domains (and several images of one domain): fp64 atomics
__global__ void k_halo_accumulate(const int64_t* __restrict__ idx, const double* __restrict__ returned, int64_t k,
                                  double* __restrict__ f_out) {
  const int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (t >= 3 * k) return;
  const int64_t r = t / 3, c = t - 3 * r;
  atomicAdd(&f_out[3 * idx[r] + c], returned[t]);
}

inline unsigned nblk(int64_t n) { return (unsigned)((n + 255) / 256); }

}  // namespace

extern "C" int allegro_halo_pack(allegro_model* m, const double* pos, const int32_t* species, const int64_t* idx,
                                 const double* shift, int64_t n_send, double* out_rows) {
  if (!m || (n_send > 0 && (!pos || !species || !idx || !shift || !out_rows)) || n_send < 0) { al_set_error(m, "halo_pack: bad argument"); return ALLEGRO_ERR_BAD_ARG; }
  if (n_send == 0) return ALLEGRO_OK;
  k_halo_pack<<<nblk(n_send), 256, 0, m->stream>>>(pos, species, idx, shift, n_send, out_rows);
  m->launches++;
  AL_CUDA(m, cudaGetLastError());
  return ALLEGRO_OK;
}

extern "C" int allegro_halo_assemble(allegro_model* m, const double* pos, const int32_t* species, int64_t n_local,
                                     const double* ghost_rows, int64_t n_ghost, const double origin[3], double* pos_all,
                                     int32_t* species_all) {
  if (!m || !origin || n_local < 0 || n_ghost < 0 || (n_local + n_ghost > 0 && (!pos_all || !species_all)) ||
      (n_local > 0 && (!pos || !species)) || (n_ghost > 0 && !ghost_rows)) { al_set_error(m, "halo_assemble: bad argument"); return ALLEGRO_ERR_BAD_ARG; }
  if (n_local + n_ghost == 0) return ALLEGRO_OK;
  k_halo_assemble<<<nblk(n_local + n_ghost), 256, 0, m->stream>>>(pos, species, n_local, ghost_rows, n_ghost, origin[0], origin[1],
                                                                 origin[2], pos_all, species_all);
  m->launches++;
  AL_CUDA(m, cudaGetLastError());
  return ALLEGRO_OK;
}

extern "C" int allegro_halo_accumulate(allegro_model* m, const double* force_all, int64_t n_local, const int64_t* idx,
                                       const double* returned, int64_t n_send, double* force_out) {
  if (!m || n_local < 0 || n_send < 0 || (n_local > 0 && (!force_all || !force_out)) || (n_send > 0 && (!idx || !returned))) {
    al_set_error(m, "halo_accumulate: bad argument"); return ALLEGRO_ERR_BAD_ARG;
  }
  if (n_local > 0) { k_halo_copy_local<<<nblk(3 * n_local), 256, 0, m->stream>>>(force_all, 3 * n_local, force_out); m->launches++; }
  if (n_send > 0) { k_halo_accumulate<<<nblk(3 * n_send), 256, 0, m->stream>>>(idx, returned, n_send, force_out); m->launches++; }
  AL_CUDA(m, cudaGetLastError());
  return ALLEGRO_OK;
}
