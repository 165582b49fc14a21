// Tensor-track kernels, warp-per-(center, 32-channel group) version (SURVEY.md §8(a) steps 5-7 and their
// backward in step 11; Eq. (2) :132-138, fused path-weighted CG tensor Fig. 3 :180).
//
// The tensor product never mixes channels, so lane = channel.  One warp owns one center
// and 32 channels: it sums the environment Gamma_i over the center's edges (Eq. (2) line 2: sum first,
// product once), contracts it with the sparse fused tensor K into the dense per-center matrix
// M_i[a][c] = sum_b K[a,b,c] Gamma_i[b] held in the warp's private shared-memory slice, then streams
// the center's edges: T_e[c] = sum_a V_e[a] M_i[a][c] with V_e, T_e in registers and fully unrolled
// compile-time loops.  All global accesses are 128-byte coalesced ([edge][component][channel] layout).
// No block-level synchronisation: warps are independent.
#include "kernels.h"

namespace {

#define FULLMASK 0xffffffffu
constexpr int WARPS_PER_BLOCK = 4;

__device__ __forceinline__ float wsum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(FULLMASK, v, o);
  return v;
}

// Sum each of 8 per-lane values over the 32 lanes with 9 shuffles (halving butterfly): on return the
// lane holds the total of value index ((lane>>4)&1)*4 + ((lane>>3)&1)*2 + ((lane>>2)&1).
__device__ __forceinline__ float reduce8(const float* v, int lane) {
  float a[4], b[2], c;
  const bool h16 = lane & 16, h8 = lane & 8, h4 = lane & 4;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    float send = h16 ? v[i] : v[i + 4], keep = h16 ? v[i + 4] : v[i];
    a[i] = keep + __shfl_xor_sync(FULLMASK, send, 16);
  }
#pragma unroll
  for (int i = 0; i < 2; ++i) {
    float send = h8 ? a[i] : a[i + 2], keep = h8 ? a[i + 2] : a[i];
    b[i] = keep + __shfl_xor_sync(FULLMASK, send, 8);
  }
  {
    float send = h4 ? b[0] : b[1], keep = h4 ? b[1] : b[0];
    c = keep + __shfl_xor_sync(FULLMASK, send, 4);
  }
  c += __shfl_xor_sync(FULLMASK, c, 2);
  c += __shfl_xor_sync(FULLMASK, c, 1);
  return c;
}

// Y-bar_e[idx[k]] += sum over lanes of p[k], k < D (D <= 16), deterministic; partial sums live in registers.
template <int D>
__device__ __forceinline__ void ybar_accumulate(float* yrow, const float* p, const int* idx, int lane) {
  const int sel = ((lane >> 4) & 1) * 4 + ((lane >> 3) & 1) * 2 + ((lane >> 2) & 1);
#pragma unroll
  for (int k0 = 0; k0 + 8 <= D; k0 += 8) {
    float r = reduce8(p + k0, lane);
    int t = idx[k0];
#pragma unroll
    for (int q = 1; q < 8; ++q) t = (sel == q) ? idx[k0 + q] : t;
    if ((lane & 3) == 0) yrow[t] += r;
  }
#pragma unroll
  for (int k = (D / 8) * 8; k < D; ++k) {
    float s = wsum(p[k]);
    if (lane == 0) yrow[idx[k]] += s;
  }
}

struct TPW {
  const int64_t* rowa; int nc;
  const float* om; int ldo;
  const float* Y; int ldy;
  const float* Vin;
  const float* w0; int ldw;
  const int *v0_l, *v0_y, *env_l;
  TPLayerDev t;
  int n, ngroups; float c_env;
  float* Tout; float* xs; int ldx; float* gamma_out;
  const float* VbarL; const float* sbar; int lds;
  float* Vbar_prev; float* ombar; int ldob; float* w0bar; float* Ybar; int64_t ybar_gstride;
};

// Gamma_i -> Gs[b][lane] ; M_i -> Ms[a*DOUT+c][lane]      (warp-private smem slices)
struct SmemTables { const int* idx; const int* b; const float* val; int nnz; };

// block-wide: copy the sparse entry list (idx = a*DOUT+c, b, val) of the fused tensor K to shared memory
__device__ __forceinline__ SmemTables load_tables(const TPW& a, float* smem_tab) {
  int nnz = a.t.nnz;
  int* si = (int*)smem_tab; int* sb = si + nnz; float* sv = (float*)(sb + nnz);
  for (int k = threadIdx.x; k < nnz; k += blockDim.x) { si[k] = a.t.ent_idx[k]; sb[k] = a.t.ent_b[k]; sv[k] = a.t.ent_val[k]; }
  __syncthreads();
  return SmemTables{si, sb, sv, nnz};
}

template <int DENV, int DIN, int DOUT>
__device__ __forceinline__ void gamma_and_M(const TPW& a, const SmemTables& tb, int64_t e0, int64_t e1, int nn, bool act,
                                            int lane, float* Gs, float* Ms) {
  constexpr int NLV = (DENV == 1) ? 1 : (DENV == 4) ? 2 : (DENV == 9) ? 3 : 4;
  float G[DENV];
#pragma unroll
  for (int b = 0; b < DENV; ++b) G[b] = 0.f;
#pragma unroll 2
  for (int64_t e = e0; e < e1; ++e) {
    float om[NLV];
#pragma unroll
    for (int l = 0; l < NLV; ++l) om[l] = act ? a.om[e * a.ldo + l * a.n + nn] : 0.f;
#pragma unroll
    for (int l = 0; l < NLV; ++l)
#pragma unroll
      for (int b = l * l; b < (l + 1) * (l + 1); ++b) G[b] = fmaf(om[l], __ldg(&a.Y[e * a.ldy + b]), G[b]);
  }
#pragma unroll
  for (int b = 0; b < DENV; ++b) Gs[b * 32 + lane] = a.c_env * G[b];
#pragma unroll
  for (int k = 0; k < DIN * DOUT; ++k) Ms[k * 32 + lane] = 0.f;
  __syncwarp();
  for (int k = 0; k < tb.nnz; ++k) Ms[tb.idx[k] * 32 + lane] = fmaf(tb.val[k], Gs[tb.b[k] * 32 + lane], Ms[tb.idx[k] * 32 + lane]);
  __syncwarp();
}

template <int DENV, int DIN, bool FIRST>
__device__ __forceinline__ void load_v(const TPW& a, int64_t e, int nn, bool act, const int* vl, const int* vy, float* v) {
  if (FIRST) {
    constexpr int NLV = (DENV == 1) ? 1 : (DENV == 4) ? 2 : (DENV == 9) ? 3 : 4;
    float w[NLV];
#pragma unroll
    for (int l = 0; l < NLV; ++l) w[l] = act ? a.w0[e * a.ldw + l * a.n + nn] : 0.f;
#pragma unroll
    for (int k = 0; k < DIN; ++k) {
      float wl = w[0];
#pragma unroll
      for (int l = 1; l < NLV; ++l) wl = (vl[k] == l) ? w[l] : wl;
      v[k] = wl * __ldg(&a.Y[e * a.ldy + vy[k]]);
    }
  } else {
#pragma unroll
    for (int k = 0; k < DIN; ++k) v[k] = act ? a.Vin[(e * DIN + k) * a.n + nn] : 0.f;
  }
}

template <int DENV, int DIN, int DOUT, bool FIRST>
__global__ void __launch_bounds__(WARPS_PER_BLOCK * 32) k_tpw_fwd(TPW a) {
  extern __shared__ float smem[];
  const int wib = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const SmemTables tb = load_tables(a, smem + WARPS_PER_BLOCK * (DENV + DIN * DOUT) * 32);
  const int64_t wg = (int64_t)blockIdx.x * WARPS_PER_BLOCK + wib;
  if (wg >= (int64_t)a.nc * a.ngroups) return;
  const int c = (int)(wg / a.ngroups), grp = (int)(wg - (int64_t)c * a.ngroups);
  const int nn = grp * 32 + lane;
  const bool act = nn < a.n;
  float* Gs = smem + wib * (DENV + DIN * DOUT) * 32;
  float* Ms = Gs + DENV * 32;
  const int64_t e0 = a.rowa[c], e1 = a.rowa[c + 1];
  if (e1 <= e0) return;
  gamma_and_M<DENV, DIN, DOUT>(a, tb, e0, e1, nn, act, lane, Gs, Ms);
  if (a.gamma_out && act)
#pragma unroll
    for (int b = 0; b < DENV; ++b) a.gamma_out[((size_t)c * DENV + b) * a.n + nn] = Gs[b * 32 + lane];
  int vl[DIN], vy[DIN];
#pragma unroll
  for (int k = 0; k < DIN; ++k) { vl[k] = FIRST ? a.v0_l[k] : 0; vy[k] = FIRST ? a.v0_y[k] : 0; }
  float v[DIN], vn[DIN];
  load_v<DENV, DIN, FIRST>(a, e0, nn, act, vl, vy, v);
  for (int64_t e = e0; e < e1; ++e) {
    if (e + 1 < e1) load_v<DENV, DIN, FIRST>(a, e + 1, nn, act, vl, vy, vn);   // software prefetch of the next edge
    float acc[DOUT];
#pragma unroll
    for (int cc = 0; cc < DOUT; ++cc) acc[cc] = 0.f;
#pragma unroll
    for (int k = 0; k < DIN; ++k)
#pragma unroll
      for (int cc = 0; cc < DOUT; ++cc) acc[cc] = fmaf(v[k], Ms[(k * DOUT + cc) * 32 + lane], acc[cc]);
    if (act) {
      a.xs[e * a.ldx + nn] = acc[0];
      if (a.Tout)
#pragma unroll
        for (int cc = 0; cc < DOUT; ++cc) a.Tout[(e * DOUT + cc) * a.n + nn] = acc[cc];
    }
#pragma unroll
    for (int k = 0; k < DIN; ++k) v[k] = vn[k];
  }
}

template <int DENV, int DIN, int DOUT, bool FIRST>
__global__ void __launch_bounds__(WARPS_PER_BLOCK * 32) k_tpw_bwd(TPW a) {
  extern __shared__ float smem[];
  constexpr int NLV = (DENV == 1) ? 1 : (DENV == 4) ? 2 : (DENV == 9) ? 3 : 4;
  const int wib = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const SmemTables tb = load_tables(a, smem + WARPS_PER_BLOCK * (DENV + DIN * DOUT) * 32);
  const int64_t wg = (int64_t)blockIdx.x * WARPS_PER_BLOCK + wib;
  if (wg >= (int64_t)a.nc * a.ngroups) return;
  const int c = (int)(wg / a.ngroups), grp = (int)(wg - (int64_t)c * a.ngroups);
  const int nn = grp * 32 + lane;
  const bool act = nn < a.n;
  float* Gs = smem + wib * (DENV + DIN * DOUT) * 32;
  float* Ms = Gs + DENV * 32;
  const int64_t e0 = a.rowa[c], e1 = a.rowa[c + 1];
  if (e1 <= e0) return;
  gamma_and_M<DENV, DIN, DOUT>(a, tb, e0, e1, nn, act, lane, Gs, Ms);
  float* Yb = a.Ybar + (size_t)grp * a.ybar_gstride;
  int vl[DIN], vy[DIN];
#pragma unroll
  for (int k = 0; k < DIN; ++k) { vl[k] = FIRST ? a.v0_l[k] : 0; vy[k] = FIRST ? a.v0_y[k] : 0; }
  float Mb[DIN * DOUT];
#pragma unroll
  for (int k = 0; k < DIN * DOUT; ++k) Mb[k] = 0.f;
  // pass 1 over the center's edges: V-bar^{L-1}, and the per-center M-bar accumulated in registers
  for (int64_t e = e0; e < e1; ++e) {
    float v[DIN], tb[DOUT];
    load_v<DENV, DIN, FIRST>(a, e, nn, act, vl, vy, v);
#pragma unroll
    for (int cc = 0; cc < DOUT; ++cc) tb[cc] = (a.VbarL && act) ? a.VbarL[(e * DOUT + cc) * a.n + nn] : 0.f;
    if (act) tb[0] += a.sbar[e * a.lds + nn];
    float vb[DIN];
#pragma unroll
    for (int k = 0; k < DIN; ++k) {
      float acc = 0.f;
#pragma unroll
      for (int cc = 0; cc < DOUT; ++cc) {
        acc = fmaf(Ms[(k * DOUT + cc) * 32 + lane], tb[cc], acc);
        Mb[k * DOUT + cc] = fmaf(v[k], tb[cc], Mb[k * DOUT + cc]);
      }
      vb[k] = acc;
    }
    if (FIRST) {
      // V^0 = w^0 (x) Y : w0-bar[l] = sum_{a in l} V-bar^0[a] Y[a] ; Y-bar[a] += sum_n w0[l(a),n] V-bar^0[a,n]
      float w[NLV], wb[NLV];
#pragma unroll
      for (int l = 0; l < NLV; ++l) { w[l] = act ? a.w0[e * a.ldw + l * a.n + nn] : 0.f; wb[l] = 0.f; }
      float pp[DIN];
#pragma unroll
      for (int k = 0; k < DIN; ++k) {
        float y = __ldg(&a.Y[e * a.ldy + vy[k]]);
        float wl = w[0];
#pragma unroll
        for (int l = 0; l < NLV; ++l) {
          bool m = (vl[k] == l);
          wb[l] = m ? fmaf(vb[k], y, wb[l]) : wb[l];
          wl = m ? w[l] : wl;
        }
        pp[k] = wl * vb[k];
      }
      ybar_accumulate<DIN>(Yb + e * DENV, pp, vy, lane);
      if (act)
#pragma unroll
        for (int l = 0; l < NLV; ++l) a.w0bar[e * a.ldob + l * a.n + nn] = wb[l];
    } else if (act) {
#pragma unroll
      for (int k = 0; k < DIN; ++k) a.Vbar_prev[(e * DIN + k) * a.n + nn] = vb[k];
    }
  }
  // Gamma-bar[b] = sum_{a,c} K[a,b,c] M-bar[a,c] : spill M-bar to the warp's smem slice, walk the sparse list by b
  __syncwarp();
#pragma unroll
  for (int k = 0; k < DIN * DOUT; ++k) Ms[k * 32 + lane] = Mb[k];
  __syncwarp();
#pragma unroll
  for (int b = 0; b < DENV; ++b) Gs[b * 32 + lane] = 0.f;
  __syncwarp();
  for (int k = 0; k < tb.nnz; ++k) Gs[tb.b[k] * 32 + lane] = fmaf(tb.val[k], Ms[tb.idx[k] * 32 + lane], Gs[tb.b[k] * 32 + lane]);
  __syncwarp();
  float Gb[DENV];
  int ident[DENV];
#pragma unroll
  for (int b = 0; b < DENV; ++b) { Gb[b] = a.c_env * Gs[b * 32 + lane]; ident[b] = b; }     // c_env folded in here
  // pass 2: omega-bar_e[l] = sum_m Gamma-bar[(l,m)] Y_e[(l,m)] ; Y-bar_e[b] += sum_n omega_e[l(b),n] Gamma-bar[b,n]
  for (int64_t e = e0; e < e1; ++e) {
    float om[NLV];
#pragma unroll
    for (int l = 0; l < NLV; ++l) om[l] = act ? a.om[e * a.ldo + l * a.n + nn] : 0.f;
    float pp[DENV];
#pragma unroll
    for (int l = 0; l < NLV; ++l) {
      float ob = 0.f;
#pragma unroll
      for (int b = l * l; b < (l + 1) * (l + 1); ++b) {
        ob = fmaf(Gb[b], __ldg(&a.Y[e * a.ldy + b]), ob);
        pp[b] = om[l] * Gb[b];
      }
      if (act) a.ombar[e * a.ldob + l * a.n + nn] = ob;
    }
    ybar_accumulate<DENV>(Yb + e * DENV, pp, ident, lane);
  }
}

// =====================================================================================================
// Blocked variants for wide features (l_max = 3: D = 16 / 31).  M_i no longer fits next to the other live
// values, so the forward walks C-BLOCKS of the output (M block in registers: D_in x CB <= 128) and the
// backward walks A-BLOCKS of the input (M-bar block in registers: AB x D_out <= 128, M block in the warp's
// shared slice).  Entries of the sparse fused tensor are staged per block, sorted by c resp. by a.
// =====================================================================================================
struct PackedTables { const int* pack; const float* val; const int* ptr; };

__device__ __forceinline__ PackedTables load_packed(const int* gpack, const float* gval, const int* gptr, int nnz, int nptr,
                                                    float* smem_tab) {
  int* sp = (int*)smem_tab; float* sv = (float*)(sp + nnz); int* spt = (int*)(sv + nnz);
  for (int k = threadIdx.x; k < nnz; k += blockDim.x) { sp[k] = gpack[k]; sv[k] = gval[k]; }
  for (int k = threadIdx.x; k < nptr; k += blockDim.x) spt[k] = gptr[k];
  __syncthreads();
  return PackedTables{sp, sv, spt};
}

template <int DENV>
__device__ __forceinline__ void gamma_only(const TPW& a, int64_t e0, int64_t e1, int nn, bool act, int lane, float* Gs) {
  constexpr int NLV = (DENV == 1) ? 1 : (DENV == 4) ? 2 : (DENV == 9) ? 3 : 4;
  float G[DENV];
#pragma unroll
  for (int b = 0; b < DENV; ++b) G[b] = 0.f;
#pragma unroll 2
  for (int64_t e = e0; e < e1; ++e) {
    float om[NLV];
#pragma unroll
    for (int l = 0; l < NLV; ++l) om[l] = act ? a.om[e * a.ldo + l * a.n + nn] : 0.f;
#pragma unroll
    for (int l = 0; l < NLV; ++l)
#pragma unroll
      for (int b = l * l; b < (l + 1) * (l + 1); ++b) G[b] = fmaf(om[l], __ldg(&a.Y[e * a.ldy + b]), G[b]);
  }
#pragma unroll
  for (int b = 0; b < DENV; ++b) Gs[b * 32 + lane] = a.c_env * G[b];
  __syncwarp();
}

template <int DENV, int DIN, int DOUT, int CB, bool FIRST>
__global__ void __launch_bounds__(WARPS_PER_BLOCK * 32) k_tpb_fwd(TPW a) {
  extern __shared__ float smem[];
  constexpr int WSL = (DENV + DIN * CB) * 32;          // floats per warp slice
  const int wib = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const PackedTables tb = load_packed(a.t.ce_pack, a.t.ce_val, a.t.cent_ptr, a.t.nnz, DOUT + 1, smem + WARPS_PER_BLOCK * WSL);
  const int64_t wg = (int64_t)blockIdx.x * WARPS_PER_BLOCK + wib;
  if (wg >= (int64_t)a.nc * a.ngroups) return;
  const int c = (int)(wg / a.ngroups), grp = (int)(wg - (int64_t)c * a.ngroups);
  const int nn = grp * 32 + lane;
  const bool act = nn < a.n;
  float* Gs = smem + wib * WSL;
  float* Ms = Gs + DENV * 32;
  const int64_t e0 = a.rowa[c], e1 = a.rowa[c + 1];
  if (e1 <= e0) return;
  gamma_only<DENV>(a, e0, e1, nn, act, lane, Gs);
  if (a.gamma_out && act)
#pragma unroll
    for (int b = 0; b < DENV; ++b) a.gamma_out[((size_t)c * DENV + b) * a.n + nn] = Gs[b * 32 + lane];
  int vl[DIN], vy[DIN];
#pragma unroll
  for (int k = 0; k < DIN; ++k) { vl[k] = FIRST ? a.v0_l[k] : 0; vy[k] = FIRST ? a.v0_y[k] : 0; }
  for (int cb = 0; cb < DOUT; cb += CB) {
    const int cend = (cb + CB < DOUT) ? cb + CB : DOUT;
#pragma unroll
    for (int k = 0; k < DIN * CB; ++k) Ms[k * 32 + lane] = 0.f;
    __syncwarp();
    for (int k = tb.ptr[cb]; k < tb.ptr[cend]; ++k) {
      int pk = tb.pack[k];
      int idx = (pk & 255) * CB + (((pk >> 8) & 255) - cb);
      Ms[idx * 32 + lane] = fmaf(tb.val[k], Gs[(pk >> 16) * 32 + lane], Ms[idx * 32 + lane]);
    }
    __syncwarp();
    float Mr[DIN * CB];
#pragma unroll
    for (int k = 0; k < DIN * CB; ++k) Mr[k] = Ms[k * 32 + lane];
    for (int64_t e = e0; e < e1; ++e) {
      float v[DIN];
      load_v<DENV, DIN, FIRST>(a, e, nn, act, vl, vy, v);
      float acc[CB];
#pragma unroll
      for (int cc = 0; cc < CB; ++cc) acc[cc] = 0.f;
#pragma unroll
      for (int k = 0; k < DIN; ++k)
#pragma unroll
        for (int cc = 0; cc < CB; ++cc) acc[cc] = fmaf(v[k], Mr[k * CB + cc], acc[cc]);
      if (act) {
        if (cb == 0) a.xs[e * a.ldx + nn] = acc[0];
        if (a.Tout)
#pragma unroll
          for (int cc = 0; cc < CB; ++cc)
            if (cb + cc < DOUT) a.Tout[(e * DOUT + cb + cc) * a.n + nn] = acc[cc];
      }
    }
    __syncwarp();
  }
}

template <int DENV, int DIN, int DOUT, int AB, bool FIRST>
__global__ void __launch_bounds__(WARPS_PER_BLOCK * 32) k_tpb_bwd(TPW a) {
  extern __shared__ float smem[];
  constexpr int NLV = (DENV == 1) ? 1 : (DENV == 4) ? 2 : (DENV == 9) ? 3 : 4;
  constexpr int WSL = (2 * DENV + AB * DOUT) * 32;
  const int wib = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const PackedTables tb = load_packed(a.t.ae_pack, a.t.ae_val, a.t.aent_ptr, a.t.nnz, DIN + 1, smem + WARPS_PER_BLOCK * WSL);
  const int64_t wg = (int64_t)blockIdx.x * WARPS_PER_BLOCK + wib;
  if (wg >= (int64_t)a.nc * a.ngroups) return;
  const int c = (int)(wg / a.ngroups), grp = (int)(wg - (int64_t)c * a.ngroups);
  const int nn = grp * 32 + lane;
  const bool act = nn < a.n;
  float* Gs = smem + wib * WSL;
  float* Gbs = Gs + DENV * 32;
  float* Ms = Gbs + DENV * 32;
  const int64_t e0 = a.rowa[c], e1 = a.rowa[c + 1];
  if (e1 <= e0) return;
  gamma_only<DENV>(a, e0, e1, nn, act, lane, Gs);
#pragma unroll
  for (int b = 0; b < DENV; ++b) Gbs[b * 32 + lane] = 0.f;
  float* Yb = a.Ybar + (size_t)grp * a.ybar_gstride;
  if (FIRST && act)
    for (int64_t e = e0; e < e1; ++e)
#pragma unroll
      for (int l = 0; l < NLV; ++l) a.w0bar[e * a.ldob + l * a.n + nn] = 0.f;
  for (int ab = 0; ab < DIN; ab += AB) {
    const int aend = (ab + AB < DIN) ? ab + AB : DIN;
    int vl[AB], vy[AB];
#pragma unroll
    for (int k = 0; k < AB; ++k) {
      int aa = (ab + k < DIN) ? ab + k : DIN - 1;
      vl[k] = FIRST ? a.v0_l[aa] : 0; vy[k] = FIRST ? a.v0_y[aa] : 0;
    }
    // M block [AB][DOUT] -> smem slice
#pragma unroll
    for (int k = 0; k < AB * DOUT; ++k) Ms[k * 32 + lane] = 0.f;
    __syncwarp();
    for (int k = tb.ptr[ab]; k < tb.ptr[aend]; ++k) {
      int pk = tb.pack[k];
      int idx = ((pk & 255) - ab) * DOUT + ((pk >> 8) & 255);
      Ms[idx * 32 + lane] = fmaf(tb.val[k], Gs[(pk >> 16) * 32 + lane], Ms[idx * 32 + lane]);
    }
    __syncwarp();
    float Mb[AB * DOUT];
#pragma unroll
    for (int k = 0; k < AB * DOUT; ++k) Mb[k] = 0.f;
    for (int64_t e = e0; e < e1; ++e) {
      float tbar[DOUT];
#pragma unroll
      for (int cc = 0; cc < DOUT; ++cc) tbar[cc] = (a.VbarL && act) ? a.VbarL[(e * DOUT + cc) * a.n + nn] : 0.f;
      if (act) tbar[0] += a.sbar[e * a.lds + nn];
      float v[AB], vb[AB];
      float w[NLV];
      if (FIRST) {
#pragma unroll
        for (int l = 0; l < NLV; ++l) w[l] = act ? a.w0[e * a.ldw + l * a.n + nn] : 0.f;
      }
#pragma unroll
      for (int k = 0; k < AB; ++k) {
        if (FIRST) {
          float wl = w[0];
#pragma unroll
          for (int l = 1; l < NLV; ++l) wl = (vl[k] == l) ? w[l] : wl;
          v[k] = (ab + k < DIN) ? wl * __ldg(&a.Y[e * a.ldy + vy[k]]) : 0.f;
        } else {
          v[k] = (act && ab + k < DIN) ? a.Vin[(e * DIN + ab + k) * a.n + nn] : 0.f;
        }
        float acc = 0.f;
#pragma unroll
        for (int cc = 0; cc < DOUT; ++cc) {
          acc = fmaf(Ms[(k * DOUT + cc) * 32 + lane], tbar[cc], acc);
          Mb[k * DOUT + cc] = fmaf(v[k], tbar[cc], Mb[k * DOUT + cc]);
        }
        vb[k] = acc;
      }
      if (FIRST) {
        float wb[NLV], pp[AB];
#pragma unroll
        for (int l = 0; l < NLV; ++l) wb[l] = 0.f;
#pragma unroll
        for (int k = 0; k < AB; ++k) {
          float y = __ldg(&a.Y[e * a.ldy + vy[k]]);
          float wl = w[0];
          bool valid = ab + k < DIN;
#pragma unroll
          for (int l = 0; l < NLV; ++l) {
            bool mm = valid && (vl[k] == l);
            wb[l] = mm ? fmaf(vb[k], y, wb[l]) : wb[l];
            wl = (vl[k] == l) ? w[l] : wl;
          }
          pp[k] = valid ? wl * vb[k] : 0.f;
        }
        // (an invalid tail slot aliases vy of the last component and contributes exactly 0)
        ybar_accumulate<AB>(Yb + e * DENV, pp, vy, lane);
        if (act)
#pragma unroll
          for (int l = 0; l < NLV; ++l) a.w0bar[e * a.ldob + l * a.n + nn] += wb[l];
      } else if (act) {
#pragma unroll
        for (int k = 0; k < AB; ++k)
          if (ab + k < DIN) a.Vbar_prev[(e * DIN + ab + k) * a.n + nn] = vb[k];
      }
    }
    // Gamma-bar += K . M-bar(block)
    __syncwarp();
#pragma unroll
    for (int k = 0; k < AB * DOUT; ++k) Ms[k * 32 + lane] = Mb[k];
    __syncwarp();
    for (int k = tb.ptr[ab]; k < tb.ptr[aend]; ++k) {
      int pk = tb.pack[k];
      int idx = ((pk & 255) - ab) * DOUT + ((pk >> 8) & 255);
      Gbs[(pk >> 16) * 32 + lane] = fmaf(tb.val[k], Ms[idx * 32 + lane], Gbs[(pk >> 16) * 32 + lane]);
    }
    __syncwarp();
  }
  float Gb[DENV];
  int ident[DENV];
#pragma unroll
  for (int b = 0; b < DENV; ++b) { Gb[b] = a.c_env * Gbs[b * 32 + lane]; ident[b] = b; }
  for (int64_t e = e0; e < e1; ++e) {
    float om[NLV];
#pragma unroll
    for (int l = 0; l < NLV; ++l) om[l] = act ? a.om[e * a.ldo + l * a.n + nn] : 0.f;
    float pp[DENV];
#pragma unroll
    for (int l = 0; l < NLV; ++l) {
      float ob = 0.f;
#pragma unroll
      for (int b = l * l; b < (l + 1) * (l + 1); ++b) {
        ob = fmaf(Gb[b], __ldg(&a.Y[e * a.ldy + b]), ob);
        pp[b] = om[l] * Gb[b];
      }
      if (act) a.ombar[e * a.ldob + l * a.n + nn] = ob;
    }
    ybar_accumulate<DENV>(Yb + e * DENV, pp, ident, lane);
  }
}

template <int DENV, int DIN, int DOUT, int CB, bool FIRST>
int launch_bfwd(allegro_model* m, const TPW& a) {
  size_t sm = (size_t)WARPS_PER_BLOCK * (DENV + DIN * CB) * 32 * 4 + (size_t)a.t.nnz * 8 + (DOUT + 1) * 4 + 16;
  static AttrOnce once;
  if (once.need(m->device)) { AL_CUDA(m, cudaFuncSetAttribute(k_tpb_fwd<DENV, DIN, DOUT, CB, FIRST>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm)); once.done(m->device); }
  int64_t warps = (int64_t)a.nc * a.ngroups;
  k_tpb_fwd<DENV, DIN, DOUT, CB, FIRST><<<(unsigned)((warps + WARPS_PER_BLOCK - 1) / WARPS_PER_BLOCK), WARPS_PER_BLOCK * 32, sm, m->stream>>>(a);
  m->launches++;
  AL_CUDA(m, cudaGetLastError());
  return ALLEGRO_OK;
}
template <int DENV, int DIN, int DOUT, int AB, bool FIRST>
int launch_bbwd(allegro_model* m, const TPW& a) {
  size_t sm = (size_t)WARPS_PER_BLOCK * (2 * DENV + AB * DOUT) * 32 * 4 + (size_t)a.t.nnz * 8 + (DIN + 1) * 4 + 16;
  static AttrOnce once;
  if (once.need(m->device)) { AL_CUDA(m, cudaFuncSetAttribute(k_tpb_bwd<DENV, DIN, DOUT, AB, FIRST>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm)); once.done(m->device); }
  int64_t warps = (int64_t)a.nc * a.ngroups;
  k_tpb_bwd<DENV, DIN, DOUT, AB, FIRST><<<(unsigned)((warps + WARPS_PER_BLOCK - 1) / WARPS_PER_BLOCK), WARPS_PER_BLOCK * 32, sm, m->stream>>>(a);
  m->launches++;
  AL_CUDA(m, cudaGetLastError());
  return ALLEGRO_OK;
}

template <int DENV, int DIN, int DOUT, bool FIRST>
int launch_fwd(allegro_model* m, const TPW& a) {
  size_t sm = (size_t)WARPS_PER_BLOCK * (DENV + DIN * DOUT) * 32 * 4 + (size_t)a.t.nnz * 12 + 16;
  static AttrOnce once;
  if (once.need(m->device)) { AL_CUDA(m, cudaFuncSetAttribute(k_tpw_fwd<DENV, DIN, DOUT, FIRST>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm)); once.done(m->device); }
  int64_t warps = (int64_t)a.nc * a.ngroups;
  k_tpw_fwd<DENV, DIN, DOUT, FIRST><<<(unsigned)((warps + WARPS_PER_BLOCK - 1) / WARPS_PER_BLOCK), WARPS_PER_BLOCK * 32, sm, m->stream>>>(a);
  m->launches++;
  AL_CUDA(m, cudaGetLastError());
  return ALLEGRO_OK;
}
template <int DENV, int DIN, int DOUT, bool FIRST>
int launch_bwd(allegro_model* m, const TPW& a) {
  size_t sm = (size_t)WARPS_PER_BLOCK * (DENV + DIN * DOUT) * 32 * 4 + (size_t)a.t.nnz * 12 + 16;
  static AttrOnce once;
  if (once.need(m->device)) { AL_CUDA(m, cudaFuncSetAttribute(k_tpw_bwd<DENV, DIN, DOUT, FIRST>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm)); once.done(m->device); }
  int64_t warps = (int64_t)a.nc * a.ngroups;
  k_tpw_bwd<DENV, DIN, DOUT, FIRST><<<(unsigned)((warps + WARPS_PER_BLOCK - 1) / WARPS_PER_BLOCK), WARPS_PER_BLOCK * 32, sm, m->stream>>>(a);
  m->launches++;
  AL_CUDA(m, cudaGetLastError());
  return ALLEGRO_OK;
}

}  // namespace

// Returns ALLEGRO_ERR_UNIMPLEMENTED if no specialisation exists for this layer shape (the caller then
// uses the generic block-per-center kernels of edge_kernels.cu).
#define TPW_DISPATCH(FN, FIRSTV)                                                                      \
  if (DENV == 9 && Din == 9 && Dout == 9) return FN<9, 9, 9, FIRSTV>(m, a);                           \
  if (DENV == 9 && Din == 9 && Dout == 1) return FN<9, 9, 1, FIRSTV>(m, a);                           \
  if (DENV == 4 && Din == 4 && Dout == 4) return FN<4, 4, 4, FIRSTV>(m, a);                           \
  if (DENV == 4 && Din == 4 && Dout == 1) return FN<4, 4, 1, FIRSTV>(m, a);                           \
  if (DENV == 1 && Din == 1 && Dout == 1) return FN<1, 1, 1, FIRSTV>(m, a);

static void fill(allegro_model* m, Work& w, int L, int nc, TPW& a, const float* om, int ldo, const float* Vin,
                 const float* w0, int ldw) {
  a.rowa = (const int64_t*)w.rowa.p; a.nc = nc; a.om = om; a.ldo = ldo; a.Y = (const float*)w.Y.p; a.ldy = m->ldY; a.Vin = Vin;
  a.w0 = w0; a.ldw = ldw; a.v0_l = m->d_v0_l; a.v0_y = m->d_v0_y; a.env_l = m->d_env_l; a.t = m->tp[L - 1];
  a.n = m->n; a.ngroups = (m->n + 31) / 32; a.c_env = m->c_env;
}

int tpw_fwd(allegro_model* m, Work& w, int L, int nc, const float* om, int ldo, const float* Vin, const float* w0, int ldw,
            float* Tout, float* xs, int ldx) {
  TPW a{};
  fill(m, w, L, nc, a, om, ldo, Vin, w0, ldw);
  a.Tout = Tout; a.xs = xs; a.ldx = ldx; a.gamma_out = (float*)w.gamma.p;
  const int DENV = m->Denv, Din = a.t.Din, Dout = a.t.Dout;
  if (Vin == nullptr) { TPW_DISPATCH(launch_fwd, true) } else { TPW_DISPATCH(launch_fwd, false) }
  if (DENV == 16) {   // l_max = 3: blocked kernels
    if (Vin == nullptr) {
      if (Din == 16 && Dout == 31) return launch_bfwd<16, 16, 31, 8, true>(m, a);
      if (Din == 16 && Dout == 16) return launch_bfwd<16, 16, 16, 8, true>(m, a);
      if (Din == 16 && Dout == 1) return launch_bfwd<16, 16, 1, 1, true>(m, a);
    } else {
      if (Din == 31 && Dout == 16) return launch_bfwd<16, 31, 16, 4, false>(m, a);
      if (Din == 16 && Dout == 16) return launch_bfwd<16, 16, 16, 8, false>(m, a);
      if (Din == 16 && Dout == 1) return launch_bfwd<16, 16, 1, 1, false>(m, a);
    }
  }
  return ALLEGRO_ERR_UNIMPLEMENTED;
}

int tpw_bwd(allegro_model* m, Work& w, int L, int nc, const float* om, int ldo, const float* Vin, const float* w0, int ldw,
            const float* VbarL, const float* sbar, int lds, float* Vbar_prev, float* ombar, int ldob, float* w0bar) {
  TPW a{};
  fill(m, w, L, nc, a, om, ldo, Vin, w0, ldw);
  a.VbarL = VbarL; a.sbar = sbar; a.lds = lds; a.Vbar_prev = Vbar_prev; a.ombar = ombar; a.ldob = ldob; a.w0bar = w0bar;
  a.Ybar = (float*)w.Ybar.p; a.ybar_gstride = (int64_t)w.cap_edges * m->Denv;   // one part per 32-channel group
  const int DENV = m->Denv, Din = a.t.Din, Dout = a.t.Dout;
  if (Vin == nullptr) { TPW_DISPATCH(launch_bwd, true) } else { TPW_DISPATCH(launch_bwd, false) }
  if (DENV == 16) {
    if (Vin == nullptr) {
      if (Din == 16 && Dout == 31) return launch_bbwd<16, 16, 31, 4, true>(m, a);
      if (Din == 16 && Dout == 16) return launch_bbwd<16, 16, 16, 8, true>(m, a);
      if (Din == 16 && Dout == 1) return launch_bbwd<16, 16, 1, 16, true>(m, a);
    } else {
      if (Din == 31 && Dout == 16) return launch_bbwd<16, 31, 16, 8, false>(m, a);
      if (Din == 16 && Dout == 16) return launch_bbwd<16, 16, 16, 8, false>(m, a);
      if (Din == 16 && Dout == 1) return launch_bbwd<16, 16, 1, 16, false>(m, a);
    }
  }
  return ALLEGRO_ERR_UNIMPLEMENTED;
}
