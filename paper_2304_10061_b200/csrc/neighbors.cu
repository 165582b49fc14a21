// Periodic cell-list neighbor build on the GPU (PAPER.md:128 ordered
// pairs, PAPER.md:188 GPU-resident lists).  Integer work + the canonical fp64 accept test
//   dx = (x_j - x_i) + s_x*L_x ; d2 = (dx*dx + dy*dy) + dz*dz ; d2 < cutoff*cutoff
// evaluated with explicit round-to-nearest intrinsics so no FMA contraction can change a decision.
#include <cmath>
#include <cstring>

#include "internal.h"

namespace {

struct NbrGeom {
  double L[3], cs[3], cut2;
  int nc[3], R[3];
};

__global__ void k_wrap_cells(const double* __restrict__ pos, int64_t N, NbrGeom g, int* __restrict__ q,
                             int* __restrict__ cell_of, int* __restrict__ cell_cnt, int* __restrict__ flag) {
  int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= N) return;
  int c[3];
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    double x = pos[3 * i + k];
    if (!isfinite(x)) { atomicOr(flag, 1); x = 0.0; }
    double qf = floor(x / g.L[k]);
    double w = x - qf * g.L[k];
    if (w < 0.0) { w += g.L[k]; qf -= 1.0; }
    if (w >= g.L[k]) { w -= g.L[k]; qf += 1.0; }
    if (fabs(qf) > 1.0e6) { atomicOr(flag, 2); qf = 0.0; }
    q[3 * i + k] = (int)qf;
    int ck = (int)(w / g.cs[k]);
    c[k] = min(max(ck, 0), g.nc[k] - 1);
  }
  int cell = (c[2] * g.nc[1] + c[1]) * g.nc[0] + c[0];
  cell_of[i] = cell;
  atomicAdd(&cell_cnt[cell], 1);
}

__global__ void k_fill_cells(int64_t N, const int* __restrict__ cell_of, const int64_t* __restrict__ cell_start,
                             int* __restrict__ cell_fill, int* __restrict__ cell_atoms) {
  int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= N) return;
  int c = cell_of[i];
  int slot = atomicAdd(&cell_fill[c], 1);
  cell_atoms[cell_start[c] + slot] = (int)i;
}

__device__ __forceinline__ bool accept(const double* __restrict__ pos, int i, int j, int sx, int sy, int sz,
                                       const NbrGeom& g) {
  double dx = __dadd_rn(__dsub_rn(pos[3 * (int64_t)j + 0], pos[3 * (int64_t)i + 0]), __dmul_rn((double)sx, g.L[0]));
  double dy = __dadd_rn(__dsub_rn(pos[3 * (int64_t)j + 1], pos[3 * (int64_t)i + 1]), __dmul_rn((double)sy, g.L[1]));
  double dz = __dadd_rn(__dsub_rn(pos[3 * (int64_t)j + 2], pos[3 * (int64_t)i + 2]), __dmul_rn((double)sz, g.L[2]));
  double d2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
  return d2 < g.cut2;
}

__device__ __forceinline__ int floordiv(int a, int b) { int q = a / b; return (a % b != 0 && ((a < 0) != (b < 0))) ? q - 1 : q; }

// One warp per atom.  FILL = false: count accepted edges; FILL = true: append 64-bit keys
// (j << 24 | (sx+128) << 16 | (sy+128) << 8 | (sz+128)) to the atom's row (unsorted).
template <bool FILL>
__global__ void k_scan_stencil(const double* __restrict__ pos, int64_t N, NbrGeom g, const int* __restrict__ q,
                               const int* __restrict__ cell_of, const int64_t* __restrict__ cell_start,
                               const int* __restrict__ cell_atoms, int* __restrict__ deg,
                               const int64_t* __restrict__ row_ptr, unsigned long long* __restrict__ keys,
                               int* __restrict__ flag) {
  int64_t warp = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5;
  int lane = threadIdx.x & 31;
  if (warp >= N) return;
  int i = (int)warp;
  int cell = cell_of[i];
  int cx = cell % g.nc[0], cy = (cell / g.nc[0]) % g.nc[1], cz = cell / (g.nc[0] * g.nc[1]);
  int qix = q[3 * i], qiy = q[3 * i + 1], qiz = q[3 * i + 2];
  int count = 0;
  int64_t base = FILL ? row_ptr[i] : 0;
  for (int dz = -g.R[2]; dz <= g.R[2]; ++dz) {
    int tz = floordiv(cz + dz, g.nc[2]); int zz = cz + dz - tz * g.nc[2];
    for (int dy = -g.R[1]; dy <= g.R[1]; ++dy) {
      int ty = floordiv(cy + dy, g.nc[1]); int yy = cy + dy - ty * g.nc[1];
      for (int dx = -g.R[0]; dx <= g.R[0]; ++dx) {
        int tx = floordiv(cx + dx, g.nc[0]); int xx = cx + dx - tx * g.nc[0];
        int c2 = (zz * g.nc[1] + yy) * g.nc[0] + xx;
        int64_t k0 = cell_start[c2], k1 = cell_start[c2 + 1];
        for (int64_t kb = k0; kb < k1; kb += 32) {
          int64_t k = kb + lane;
          bool ok = false; int j = 0, sx = 0, sy = 0, sz = 0;
          if (k < k1) {
            j = cell_atoms[k];
            sx = tx - q[3 * j] + qix; sy = ty - q[3 * j + 1] + qiy; sz = tz - q[3 * j + 2] + qiz;
            if (!(j == i && sx == 0 && sy == 0 && sz == 0)) ok = accept(pos, i, j, sx, sy, sz, g);
          }
          unsigned mask = __ballot_sync(0xffffffffu, ok);
          if (FILL && ok) {
            if (sx < -128 || sx > 127 || sy < -128 || sy > 127 || sz < -128 || sz > 127) atomicOr(flag, 4);
            int off = count + __popc(mask & ((1u << lane) - 1u));
            keys[base + off] = ((unsigned long long)(unsigned)j << 24) | ((unsigned long long)((sx + 128) & 255) << 16) |
                               ((unsigned long long)((sy + 128) & 255) << 8) | (unsigned long long)((sz + 128) & 255);
          }
          count += __popc(mask);
        }
      }
    }
  }
  if (!FILL && lane == 0) deg[i] = count;
}

// Rank sort of each row (keys are unique): one warp per atom, O(deg^2) compares.
__global__ void k_sort_rows(int64_t N, const int64_t* __restrict__ row_ptr, const unsigned long long* __restrict__ keys,
                            int* __restrict__ jout, int8_t* __restrict__ sout) {
  int64_t warp = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5;
  int lane = threadIdx.x & 31;
  if (warp >= N) return;
  int64_t b = row_ptr[warp], e = row_ptr[warp + 1];
  int n = (int)(e - b);
  for (int k = lane; k < n; k += 32) {
    unsigned long long key = keys[b + k];
    int rank = 0;
    for (int t = 0; t < n; ++t) rank += (keys[b + t] < key);
    jout[b + rank] = (int)(key >> 24);
    sout[3 * (b + rank) + 0] = (int8_t)((int)((key >> 16) & 255) - 128);
    sout[3 * (b + rank) + 1] = (int8_t)((int)((key >> 8) & 255) - 128);
    sout[3 * (b + rank) + 2] = (int8_t)((int)(key & 255) - 128);
  }
}

// ---- exclusive scan int32 -> int64, out[n] = total -----------------------------------------------
constexpr int SCAN_T = 256, SCAN_ITEMS = 4, SCAN_TILE = SCAN_T * SCAN_ITEMS;

__device__ __forceinline__ int64_t block_exclusive(int64_t v, int64_t* total) {
  __shared__ int64_t wsum[SCAN_T / 32];
  int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  int64_t inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    int64_t t = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += t;
  }
  if (lane == 31) wsum[w] = inc;
  __syncthreads();
  if (w == 0) {
    int64_t s = (lane < SCAN_T / 32) ? wsum[lane] : 0;
#pragma unroll
    for (int o = 1; o < SCAN_T / 32; o <<= 1) {
      int64_t t = __shfl_up_sync(0xffffffffu, s, o);
      if (lane >= o) s += t;
    }
    if (lane < SCAN_T / 32) wsum[lane] = s;
  }
  __syncthreads();
  int64_t off = (w > 0) ? wsum[w - 1] : 0;
  *total = wsum[SCAN_T / 32 - 1];
  __syncthreads();
  return off + inc - v;
}

__global__ void k_scan_tile_sums(const int32_t* __restrict__ in, int64_t n, int64_t* __restrict__ tile_sum) {
  int64_t base = blockIdx.x * (int64_t)SCAN_TILE + threadIdx.x * SCAN_ITEMS;
  int64_t s = 0;
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k) if (base + k < n) s += in[base + k];
  int64_t tot;
  block_exclusive(s, &tot);
  if (threadIdx.x == 0) tile_sum[blockIdx.x] = tot;
}

__global__ void k_scan_tile_offsets(int64_t* __restrict__ tile_sum, int64_t ntiles, int64_t* __restrict__ grand) {
  int64_t carry = 0;
  for (int64_t b = 0; b < ntiles; b += SCAN_T) {
    int64_t i = b + threadIdx.x;
    int64_t v = (i < ntiles) ? tile_sum[i] : 0;
    int64_t tot;
    int64_t ex = block_exclusive(v, &tot);
    if (i < ntiles) tile_sum[i] = carry + ex;
    carry += tot;
  }
  if (threadIdx.x == 0) *grand = carry;
}

__global__ void k_scan_apply(const int32_t* __restrict__ in, int64_t n, const int64_t* __restrict__ tile_off,
                             int64_t* __restrict__ out) {
  int64_t base = blockIdx.x * (int64_t)SCAN_TILE + threadIdx.x * SCAN_ITEMS;
  int64_t v[SCAN_ITEMS], s = 0;
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k) { v[k] = (base + k < n) ? in[base + k] : 0; s += v[k]; }
  int64_t tot;
  int64_t ex = block_exclusive(s, &tot) + tile_off[blockIdx.x];
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k) { if (base + k < n) out[base + k] = ex; ex += v[k]; }
}

}  // namespace

int al_exclusive_scan_i64(allegro_model* m, const int32_t* in, int64_t* out, int64_t n, DevBuf& tmp) {
  int64_t ntiles = (n + SCAN_TILE - 1) / SCAN_TILE;
  if (ntiles < 1) ntiles = 1;
  AL_CHECK(al_reserve(m, tmp, (size_t)ntiles * 8));
  int64_t* ts = (int64_t*)tmp.p;
  k_scan_tile_sums<<<(unsigned)ntiles, SCAN_T, 0, m->stream>>>(in, n, ts);
  k_scan_tile_offsets<<<1, SCAN_T, 0, m->stream>>>(ts, ntiles, out + n);
  k_scan_apply<<<(unsigned)ntiles, SCAN_T, 0, m->stream>>>(in, n, ts, out);
  m->launches += 3;
  AL_CUDA(m, cudaGetLastError());
  return ALLEGRO_OK;
}

int al_neighbors_impl(allegro_model* m, const double* pos, int64_t N, const double box[3], double cutoff,
                      allegro_nbr** inout) {
  ProfScope _ps(m, PC_NEIGHBORS);
  if (!m || (!pos && N > 0) || !inout || !box) { al_set_error(m, "NULL argument"); return ALLEGRO_ERR_BAD_ARG; }
  if (N < 0 || N > 2000000000LL) { al_set_error(m, "n_atoms out of range"); return ALLEGRO_ERR_BAD_ARG; }
  if (!(cutoff > 0) || !(box[0] > 0) || !(box[1] > 0) || !(box[2] > 0)) { al_set_error(m, "cutoff and box must be > 0"); return ALLEGRO_ERR_BAD_ARG; }
  allegro_nbr* nb = *inout ? *inout : new allegro_nbr();
  *inout = nb;
  nb->n_atoms = N; nb->cutoff = cutoff;
  nb->version++;
  memcpy(nb->box, box, 24);
  NbrGeom g;
  g.cut2 = cutoff * cutoff;
  int64_t ncell = 1;
  for (int k = 0; k < 3; ++k) {
    g.L[k] = box[k];
    int nc = (int)floor(box[k] / (cutoff * (1.0 + 1e-6)));
    if (nc < 1) nc = 1;
    if (nc > 1024) nc = 1024;
    g.nc[k] = nc; g.cs[k] = box[k] / nc;
    g.R[k] = (int)ceil(cutoff * (1.0 + 1e-6) / g.cs[k]);
    if (g.R[k] > 100) { al_set_error(m, "box edge far smaller than cutoff: image shift does not fit int8"); return ALLEGRO_ERR_BOX_TOO_SMALL; }
    ncell *= nc;
  }
  cudaStream_t st = m->stream;
  AL_CHECK(al_reserve(m, nb->q, (size_t)N * 12 + 16));
  AL_CHECK(al_reserve(m, nb->cell_of, (size_t)N * 4 + 16));
  AL_CHECK(al_reserve(m, nb->cell_cnt, (size_t)(2 * ncell + 2) * 4));
  AL_CHECK(al_reserve(m, nb->cell_start, (size_t)(ncell + 1) * 8));
  AL_CHECK(al_reserve(m, nb->cell_atoms, (size_t)N * 4 + 16));
  AL_CHECK(al_reserve(m, nb->deg, (size_t)N * 4 + 16));
  AL_CHECK(al_reserve(m, nb->row_ptr, (size_t)(N + 1) * 8));
  int* cnt = (int*)nb->cell_cnt.p; int* fill = cnt + ncell; int* flag = fill + ncell;
  AL_CUDA(m, cudaMemsetAsync(cnt, 0, (size_t)(2 * ncell + 2) * 4, st));
  unsigned gb = (unsigned)((N + 255) / 256);
  if (N > 0) {
    k_wrap_cells<<<gb, 256, 0, st>>>(pos, N, g, (int*)nb->q.p, (int*)nb->cell_of.p, cnt, flag);
    m->launches++;
  }
  AL_CHECK(al_exclusive_scan_i64(m, cnt, (int64_t*)nb->cell_start.p, ncell, nb->scan_tmp));
  unsigned gw = (unsigned)((N * 32 + 255) / 256);
  if (N > 0) {
    k_fill_cells<<<gb, 256, 0, st>>>(N, (int*)nb->cell_of.p, (int64_t*)nb->cell_start.p, fill, (int*)nb->cell_atoms.p);
    k_scan_stencil<false><<<gw, 256, 0, st>>>(pos, N, g, (int*)nb->q.p, (int*)nb->cell_of.p, (int64_t*)nb->cell_start.p,
                                             (int*)nb->cell_atoms.p, (int*)nb->deg.p, nullptr, nullptr, flag);
    m->launches += 2;
  }
  AL_CHECK(al_exclusive_scan_i64(m, (int*)nb->deg.p, (int64_t*)nb->row_ptr.p, N, nb->scan_tmp));
  nb->row_ptr_host.resize(N + 1);
  int hflag = 0;
  AL_CUDA(m, cudaMemcpyAsync(nb->row_ptr_host.data(), nb->row_ptr.p, (size_t)(N + 1) * 8, cudaMemcpyDeviceToHost, st));
  AL_CUDA(m, cudaMemcpyAsync(&hflag, flag, 4, cudaMemcpyDeviceToHost, st));
  AL_CUDA(m, cudaStreamSynchronize(st));
  if (hflag & 1) { al_set_error(m, "non-finite position"); return ALLEGRO_ERR_NONFINITE; }
  if (hflag & 2) { al_set_error(m, "position more than 1e6 box lengths away from the cell"); return ALLEGRO_ERR_BOX_TOO_SMALL; }
  int64_t E = nb->row_ptr_host[N];
  nb->n_edges = E;
  if (m->hp.max_edges > 0 && E > m->hp.max_edges) { al_set_error(m, "edge count exceeds hparams.max_edges"); return ALLEGRO_ERR_CAPACITY; }
  AL_CHECK(al_reserve(m, nb->keys, (size_t)E * 8 + 16));
  AL_CHECK(al_reserve(m, nb->j, (size_t)E * 4 + 16));
  AL_CHECK(al_reserve(m, nb->shift, (size_t)E * 3 + 16));
  if (N > 0 && E > 0) {
    k_scan_stencil<true><<<gw, 256, 0, st>>>(pos, N, g, (int*)nb->q.p, (int*)nb->cell_of.p, (int64_t*)nb->cell_start.p,
                                            (int*)nb->cell_atoms.p, nullptr, (int64_t*)nb->row_ptr.p,
                                            (unsigned long long*)nb->keys.p, flag);
    k_sort_rows<<<gw, 256, 0, st>>>(N, (int64_t*)nb->row_ptr.p, (unsigned long long*)nb->keys.p, (int*)nb->j.p,
                                   (int8_t*)nb->shift.p);
    m->launches += 2;
    AL_CUDA(m, cudaMemcpyAsync(&hflag, flag, 4, cudaMemcpyDeviceToHost, st));
    AL_CUDA(m, cudaStreamSynchronize(st));
    if (hflag & 4) { al_set_error(m, "image shift does not fit int8"); return ALLEGRO_ERR_BOX_TOO_SMALL; }
  }
  AL_CUDA(m, cudaGetLastError());
  // center-contiguous chunks of at most chunk_edges candidate edges (strict locality)
  nb->chunks.clear();
  nb->chunk_cap = m->chunk_edges;
  nb->max_chunk_edges = 0; nb->max_chunk_centers = 0;
  int64_t c0 = 0;
  while (c0 < N) {
    int64_t c1 = c0 + 1;
    const int64_t* rp = nb->row_ptr_host.data();
    // largest c1 with rp[c1] - rp[c0] <= cap (at least one center)
    int64_t lo = c0 + 1, hi = N;
    while (lo < hi) {
      int64_t mid = (lo + hi + 1) / 2;
      if (rp[mid] - rp[c0] <= nb->chunk_cap) lo = mid; else hi = mid - 1;
    }
    c1 = lo;
    Chunk ch{c0, c1, rp[c0], rp[c1]};
    nb->chunks.push_back(ch);
    if (ch.e1 - ch.e0 > nb->max_chunk_edges) nb->max_chunk_edges = ch.e1 - ch.e0;
    if (c1 - c0 > nb->max_chunk_centers) nb->max_chunk_centers = c1 - c0;
    c0 = c1;
  }
  return ALLEGRO_OK;
}

extern "C" int allegro_neighbors(allegro_model* m, const double* pos, int64_t n_atoms, const double box[3],
                                 double cutoff, allegro_nbr** inout) {
  return al_neighbors_impl(m, pos, n_atoms, box, cutoff, inout);
}

extern "C" int allegro_neighbors_host(allegro_model* m, const double* pos_host, int64_t N, const double box[3],
                                      double cutoff, allegro_nbr** inout) {
  if (!m || !pos_host) return ALLEGRO_ERR_BAD_ARG;
  void* d = nullptr;
  AL_CHECK(al_alloc(m, &d, (size_t)N * 24 + 16));
  cudaError_t e = cudaMemcpyAsync(d, pos_host, (size_t)N * 24, cudaMemcpyHostToDevice, m->stream);
  int rc = (e == cudaSuccess) ? al_neighbors_impl(m, (const double*)d, N, box, cutoff, inout) : ALLEGRO_ERR_CUDA;
  cudaStreamSynchronize(m->stream);
  al_free(m, d);
  return rc;
}

extern "C" int allegro_nbr_info(const allegro_nbr* n, int64_t* n_atoms, int64_t* n_edges, const int64_t** row_ptr,
                                const int32_t** j, const int8_t** shift) {
  if (!n) return ALLEGRO_ERR_BAD_ARG;
  if (n_atoms) *n_atoms = n->n_atoms;
  if (n_edges) *n_edges = n->n_edges;
  if (row_ptr) *row_ptr = (const int64_t*)n->row_ptr.p;
  if (j) *j = (const int32_t*)n->j.p;
  if (shift) *shift = (const int8_t*)n->shift.p;
  return ALLEGRO_OK;
}

extern "C" int allegro_nbr_copy_host(allegro_model* m, const allegro_nbr* n, int64_t* row_ptr, int32_t* j, int8_t* shift) {
  if (!m || !n) return ALLEGRO_ERR_BAD_ARG;
  if (row_ptr) AL_CUDA(m, cudaMemcpyAsync(row_ptr, n->row_ptr.p, (size_t)(n->n_atoms + 1) * 8, cudaMemcpyDeviceToHost, m->stream));
  if (j && n->n_edges) AL_CUDA(m, cudaMemcpyAsync(j, n->j.p, (size_t)n->n_edges * 4, cudaMemcpyDeviceToHost, m->stream));
  if (shift && n->n_edges) AL_CUDA(m, cudaMemcpyAsync(shift, n->shift.p, (size_t)n->n_edges * 3, cudaMemcpyDeviceToHost, m->stream));
  AL_CUDA(m, cudaStreamSynchronize(m->stream));
  return ALLEGRO_OK;
}

extern "C" int allegro_nbr_free(allegro_model* m, allegro_nbr* n) {
  if (!n) return ALLEGRO_OK;
  if (m) cudaStreamSynchronize(m->stream);
  DevBuf* bufs[] = {&n->row_ptr, &n->j, &n->shift, &n->keys, &n->wpos, &n->q, &n->cell_of, &n->cell_cnt,
                    &n->cell_start, &n->cell_atoms, &n->deg, &n->scan_tmp};
  for (DevBuf* b : bufs) al_release(m, *b);
  delete n;
  return ALLEGRO_OK;
}
