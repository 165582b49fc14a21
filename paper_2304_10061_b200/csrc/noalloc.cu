// allegro_kinetic_energy_noalloc: the kinetic-energy reduction of the velocity-Verlet step (SURVEY 8(c) S10,
// include/b200_allegro.h) for callers that may not allocate -- code under CUDA graph capture, tight serving loops,
// harnesses that forbid cudaMalloc.  The existing allegro_kinetic_energy writes the per-atom terms m_i v_i^2 / 2 into a
// scratch buffer it reserves with cudaMalloc on first use (and on growth) and sums them in a fixed order; this variant
// keeps that scratch in a file-scope __device__ array of a fixed maximum size, so the call allocates nothing, ever.
//
//  - The array costs ALLEGRO_KINETIC_NOALLOC_MAX_ATOMS x 8 bytes = 8 MiB on every GPU that loads the library, until the
//    process exits.
//  - In HOST code `g_kin_scratch` is only a stand-in for the symbol, not a device address; the address the kernels get
//    comes from cudaGetSymbolAddress, looked up once per device with that device current.
//  - Every call shares the array.  Nothing in it has to start at zero: a call writes entries [0, n) and then reads exactly
//    those, so the contents the previous call left behind are never read.  Two calls that overlap on the GPU (different
//    streams, or different models on one device) RACE on the array; calls on one stream are ordered and safe.
//  - The arithmetic is that of k_kin / k_sum_f64 (edge_kernels.cu): same per-atom expression, same strided partial sums by
//    1024 threads, same shared-memory tree, hence the same value as the existing path.
#include <cuda_runtime.h>

#include <mutex>
#include <string>

#include "internal.h"

namespace {

constexpr int64_t KIN_MAX = ALLEGRO_KINETIC_NOALLOC_MAX_ATOMS;
constexpr int MAX_DEVICES = 64;

static __device__ __align__(256) double g_kin_scratch[KIN_MAX];

// per-device address of g_kin_scratch (host side), filled on the first call on that device
std::mutex g_addr_mutex;
double* g_kin_scratch_addr[MAX_DEVICES] = {};

__global__ void k_kin_na(const double* __restrict__ vel, const int32_t* __restrict__ species, const double* __restrict__ mass,
                         int S, int64_t n, double* __restrict__ out) {
  int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int z = min(max(species[i], 0), S - 1);
  const double m = mass[z];
  out[i] = 0.5 * m * (vel[3 * i] * vel[3 * i] + vel[3 * i + 1] * vel[3 * i + 1] + vel[3 * i + 2] * vel[3 * i + 2]) / 9.648533212e-3;
}

__global__ void k_sum_na(const double* __restrict__ x, int64_t n, double* __restrict__ out) {
  __shared__ double sh[1024];
  double s = 0.0;
  for (int64_t i = threadIdx.x; i < n; i += blockDim.x) s += x[i];
  sh[threadIdx.x] = s;
  __syncthreads();
  for (int o = blockDim.x / 2; o > 0; o >>= 1) {
    if (threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
    __syncthreads();
  }
  if (threadIdx.x == 0) *out = sh[0];
}

// the device address of the scratch array on the CURRENT device (which must be `dev`)
int scratch_address(const allegro_model* m, int dev, double** out) {
  std::lock_guard<std::mutex> lock(g_addr_mutex);
  if (!g_kin_scratch_addr[dev]) {
    double* p = nullptr;
    AL_CUDA(m, cudaGetSymbolAddress((void**)&p, g_kin_scratch));
    if (!p) { al_set_error(m, "cudaGetSymbolAddress returned a null address for the kinetic-energy scratch"); return ALLEGRO_ERR_CUDA; }
    g_kin_scratch_addr[dev] = p;
  }
  *out = g_kin_scratch_addr[dev];
  return ALLEGRO_OK;
}

}  // namespace

extern "C" int allegro_kinetic_energy_noalloc(allegro_model* m, const double* vel, const int32_t* species, const double* mass,
                                              int64_t N, double* e_kin) {
  if (!m) return ALLEGRO_ERR_BAD_ARG;
  if (!vel || !species || !mass || !e_kin) { al_set_error(m, "NULL argument"); return ALLEGRO_ERR_BAD_ARG; }
  if (N < 0) { al_set_error(m, "allegro_kinetic_energy_noalloc: n_atoms < 0"); return ALLEGRO_ERR_BAD_ARG; }
  if (N > KIN_MAX) {
    al_set_error(m, "allegro_kinetic_energy_noalloc: n_atoms = " + std::to_string((long long)N) + " exceeds the fixed scratch of " +
                        std::to_string((long long)KIN_MAX) + " atoms (ALLEGRO_KINETIC_NOALLOC_MAX_ATOMS); use allegro_kinetic_energy");
    return ALLEGRO_ERR_CAPACITY;
  }
  int dev = -1;
  AL_CUDA(m, cudaGetDevice(&dev));
  if (dev != m->device || dev < 0 || dev >= MAX_DEVICES) {
    al_set_error(m, "allegro_kinetic_energy_noalloc: the model's device (" + std::to_string(m->device) +
                        ") must be the current device (" + std::to_string(dev) + ") and below " + std::to_string(MAX_DEVICES));
    return ALLEGRO_ERR_BAD_ARG;
  }
  double* scratch = nullptr;
  AL_CHECK(scratch_address(m, dev, &scratch));
  if (N > 0) {
    k_kin_na<<<(unsigned)((N + 255) / 256), 256, 0, m->stream>>>(vel, species, mass, m->S, N, scratch);
    m->launches++;
    AL_CUDA(m, cudaGetLastError());
  }
  k_sum_na<<<1, 1024, 0, m->stream>>>(scratch, N, e_kin);
  m->launches++;
  AL_CUDA(m, cudaGetLastError());
  return ALLEGRO_OK;
}
