// Tensor-track kernels, second generation (SURVEY.md §8(a) steps 5-7 and their backward in step 11;
// PAPER.md Eq. (2) :132-138, fused path-weighted CG tensor Fig. 3 :180).
//
// Same decomposition as tp_kernels.cu -- one warp owns (center i, 32 channels), lane = channel, the
// environment is summed before the product (Eq. (2) line 2) and folded with the sparse fused tensor K into
// the dense per-center matrix M_i[a][c] = sum_b K[a,b,c] Gamma_i[b] -- but built for memory-level
// parallelism and issue rate:
//   * the per-edge operand rows (V_e / w0_e, Y_e, T-bar_e) stream through a per-warp cp.async ring in
//     shared memory (NST stages of one edge each), so the loads in flight do not cost registers;
//   * M_i (and the backward's M-bar_i) live in registers as float2 pairs over the output component and
//     all inner products are packed FFMA2 (two fp32 FMAs per issue slot on sm_100);
//   * wide features (l_max = 3) walk blocks of output components (forward) / input components (backward);
//   * Y-bar is written, not accumulated, by the first kernel of a step that touches it (no memset).
// Requirements (checked on the host, otherwise the kernels of tp_kernels.cu run): n % 32 == 0 and the
// V^0 layout equal to the environment layout (always true for S_0 = env irreps).
#pragma once
#include <cstdlib>

#include "kernels.h"
#include "tp_common.cuh"

struct TP2 {
  const int64_t* rowa; int nc;
  const float* om; int ldo;
  const float* Y; int ldy;
  const float* Vin;
  const float* w0; int ldw;
  const int* dp_ptr; const int* dp_b; const float* dp_val; int nnz;
  int n, ngroups; float c_env;
  float* Tout; float* xs; int ldx; float* gamma_out;
  const float* VbarL; const float* sbar; int lds;
  float* Vbar_prev; float* ombar; int ldob; float* w0bar; float* Ybar; int64_t ybar_gstride;
};

__host__ __device__ constexpr int l_of(int k) { return k < 1 ? 0 : k < 4 ? 1 : k < 9 ? 2 : 3; }
__host__ __device__ constexpr int nlv_of(int denv) { return denv == 1 ? 1 : denv == 4 ? 2 : denv == 9 ? 3 : 4; }
__host__ __device__ constexpr int tab_ints(int din, int dout) { return (din * dout + 1 + 3) & ~3; }

struct Tables { const int* ptr; const int* b; const float* val; };

// block-wide: stage the dense pair table of the fused tensor K in shared memory
template <int DIN, int DOUT>
__device__ __forceinline__ Tables load_tables(const TP2& a, float* smem_tab) {
  int* sp = (int*)smem_tab;
  int* sb = sp + tab_ints(DIN, DOUT);
  float* sv = (float*)(sb + a.nnz);
  for (int k = threadIdx.x; k < DIN * DOUT + 1; k += blockDim.x) sp[k] = a.dp_ptr[k];
  for (int k = threadIdx.x; k < a.nnz; k += blockDim.x) { sb[k] = a.dp_b[k]; sv[k] = a.dp_val[k]; }
  __syncthreads();
  return Tables{sp, sb, sv};
}

// M_i[a][c] for one (a, c) pair from Gamma_i in the warp's shared slice
__device__ __forceinline__ float pair_val(const Tables& t, int p, const float* Gs, int lane) {
  float acc = 0.f;
  for (int k = t.ptr[p]; k < t.ptr[p + 1]; ++k) acc = fmaf(t.val[k], Gs[t.b[k] * 32 + lane], acc);
  return acc;
}

template <int LDY>
__device__ __forceinline__ float ycomp(const float4* y, int b) { return reinterpret_cast<const float*>(y)[b]; }

// Gamma_i[b] = c_env sum_e omega_e[l(b)] Y_e[b]  ->  Gs[b*32 + lane]   (direct loads, 4 edges in flight)
template <int DENV>
__device__ __forceinline__ void gamma_pass(const TP2& a, int64_t e0, int64_t e1, int nn, int lane, float* Gs) {
  constexpr int NLV = nlv_of(DENV), LDY = (DENV + 3) & ~3;
  float G[DENV];
#pragma unroll
  for (int b = 0; b < DENV; ++b) G[b] = 0.f;
  for (int64_t e = e0; e < e1; e += 4) {
    float om[4][NLV];
    float4 yq[4][LDY / 4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const int64_t ee = (e + i < e1) ? e + i : e1 - 1;
#pragma unroll
      for (int l = 0; l < NLV; ++l) om[i][l] = a.om[ee * a.ldo + l * a.n + nn];
#pragma unroll
      for (int q = 0; q < LDY / 4; ++q) yq[i][q] = __ldg(reinterpret_cast<const float4*>(a.Y + ee * a.ldy) + q);
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const bool ok = e + i < e1;
#pragma unroll
      for (int b = 0; b < DENV; ++b) G[b] = fmaf(ok ? om[i][l_of(b)] : 0.f, ycomp<LDY>(yq[i], b), G[b]);
    }
  }
#pragma unroll
  for (int b = 0; b < DENV; ++b) Gs[b * 32 + lane] = a.c_env * G[b];
  __syncwarp();
}

// ======================================================================================================
// forward:  T_e[c] = sum_a V_e[a] M_i[a][c]   (c-blocks of CB output components; CB == DOUT: one pass)
// ======================================================================================================
template <int DENV, int DIN, int DOUT, int CB, bool FIRST, int NST, int WPB>
static __global__ void __launch_bounds__(WPB * 32) k_tp2_fwd(TP2 a) {
  constexpr int NLV = nlv_of(DENV), LDY = (DENV + 3) & ~3, CBH = (CB + 1) / 2;
  constexpr int SF = FIRST ? NLV * 32 + LDY : DIN * 32;   // floats per ring stage (one edge)
  constexpr int SCR = CBH * 64;                           // one row of M as float2 per lane (lane-private scratch)
  constexpr int WSL = DENV * 32 + SCR + NST * SF;         // floats per warp slice
  extern __shared__ float4 smem4[];
  float* smem = reinterpret_cast<float*>(smem4);
  const int wib = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const Tables tb = load_tables<DIN, DOUT>(a, smem + WPB * WSL);
  const int64_t wg = (int64_t)blockIdx.x * WPB + wib;
  if (wg >= (int64_t)a.nc * a.ngroups) return;
  const int c = (int)(wg / a.ngroups), grp = (int)(wg - (int64_t)c * a.ngroups);
  const int nn = grp * 32 + lane;
  float* Gs = smem + wib * WSL;
  float* scr = Gs + DENV * 32;
  float* ring = scr + SCR;
  const int64_t e0 = a.rowa[c], e1 = a.rowa[c + 1];
  const int deg = (int)(e1 - e0);
  if (deg <= 0) return;

  auto issue = [&](int64_t e, float* st) {
    if (FIRST) {
      tp_cp_rows<NLV>(st, a.w0 + e * a.ldw + grp * 32, a.n, lane);
      if (lane < LDY / 4) tp_cp16(st + NLV * 32 + lane * 4, a.Y + e * a.ldy + lane * 4);
    } else {
      tp_cp_rows<DIN>(st, a.Vin + e * DIN * a.n + grp * 32, a.n, lane);
    }
  };
  // start streaming the first edges while Gamma_i is being summed
#pragma unroll
  for (int s = 0; s < NST - 1; ++s) {
    if (s < deg) issue(e0 + s, ring + s * SF);
    tp_cp_commit();
  }
  gamma_pass<DENV>(a, e0, e1, nn, lane, Gs);
  if (a.gamma_out)
#pragma unroll
    for (int b = 0; b < DENV; ++b) a.gamma_out[((size_t)c * DENV + b) * a.n + nn] = Gs[b * 32 + lane];

  for (int cb = 0; cb < DOUT; cb += CB) {
    // M block -> registers, one row at a time through the lane-private scratch (rolled loops: the fully
    // unrolled build overflowed the instruction cache, ncu "no_instructions" 60 %)
    float2 Mr[DIN * CBH];
#pragma unroll
    for (int k = 0; k < DIN; ++k) {
#pragma unroll 1
      for (int cc = 0; cc < 2 * CBH; ++cc) {
        const int ca = cb + cc;
        scr[((cc >> 1) * 32 + lane) * 2 + (cc & 1)] = (cc < CB && ca < DOUT) ? pair_val(tb, k * DOUT + ca, Gs, lane) : 0.f;
      }
#pragma unroll
      for (int j = 0; j < CBH; ++j) Mr[k * CBH + j] = reinterpret_cast<const float2*>(scr)[j * 32 + lane];
    }
    if (cb > 0) {   // restart the ring for this block of output components
      __syncwarp();
#pragma unroll
      for (int s = 0; s < NST - 1; ++s) {
        if (s < deg) issue(e0 + s, ring + s * SF);
        tp_cp_commit();
      }
    }
    int slot = 0;
    for (int i = 0; i < deg; ++i) {
      tp_cp_wait<NST - 2>();
      __syncwarp();
      {
        const int nx = i + NST - 1;
        int ns = slot + NST - 1; if (ns >= NST) ns -= NST;
        if (nx < deg) issue(e0 + nx, ring + ns * SF);
        tp_cp_commit();
      }
      const float* st = ring + slot * SF;
      const int64_t e = e0 + i;
      float2 acc[CBH];
#pragma unroll
      for (int j = 0; j < CBH; ++j) acc[j] = make_float2(0.f, 0.f);
#pragma unroll
      for (int k = 0; k < DIN; ++k) {
        float v = FIRST ? st[l_of(k) * 32 + lane] * st[NLV * 32 + k] : st[k * 32 + lane];
        const float2 v2 = make_float2(v, v);
#pragma unroll
        for (int j = 0; j < CBH; ++j) acc[j] = tp_fma2(v2, Mr[k * CBH + j], acc[j]);
      }
      if (cb == 0) a.xs[e * a.ldx + nn] = acc[0].x;
      if (a.Tout) {
#pragma unroll
        for (int cc = 0; cc < CB; ++cc)
          if (cb + cc < DOUT) a.Tout[(e * DOUT + cb + cc) * a.n + nn] = (cc & 1) ? acc[cc >> 1].y : acc[cc >> 1].x;
      }
      if (++slot == NST) slot = 0;
    }
  }
}

// ======================================================================================================
// backward:  T-bar_e = V-bar^L_e (+ s-bar at the scalar slot)
//   V-bar^{L-1}_e[a] = sum_c M_i[a][c] T-bar_e[c]          M-bar_i[a][c] = sum_e V_e[a] T-bar_e[c]
//   Gamma-bar_i[b]   = sum_{a,c} K[a,b,c] M-bar_i[a][c]
//   omega-bar_e[l]   = c_env sum_m Gamma-bar_i[(l,m)] Y_e[(l,m)]      Y-bar_e[b] += c_env sum_n omega_e[l(b)] Gamma-bar_i[b]
//   FIRST (V^0 = w^0 (x) Y):  w0-bar_e[l] = sum_{a in l} V-bar^0_e[a] Y_e[a] ;  Y-bar_e[a] += sum_n w0_e[l(a)] V-bar^0_e[a]
// a-blocks of AB input components; M block in registers (MREG) or in the warp's shared slice.
// ======================================================================================================
template <int DENV, int DIN, int DOUT, int AB, bool FIRST, bool HASVB, bool MREG, bool YINIT, int NST, int WPB>
static __global__ void __launch_bounds__(WPB * 32) k_tp2_bwd(TP2 a) {
  constexpr int NLV = nlv_of(DENV), LDY = (DENV + 3) & ~3, CH = (DOUT + 1) / 2;
  constexpr int SV = FIRST ? NLV * 32 + LDY : AB * 32;      // operand part of a stage
  constexpr int SF = SV + (HASVB ? DOUT * 32 : 0) + 32;     // + T-bar rows + s-bar row
  constexpr int MSL = MREG ? 0 : AB * CH * 64;              // M block as float2 per lane
  constexpr int SCR = CH * 64;                              // one row of M / M-bar (lane-private scratch)
  constexpr int WSL = 2 * DENV * 32 + MSL + SCR + NST * SF;
  extern __shared__ float4 smem4[];
  float* smem = reinterpret_cast<float*>(smem4);
  const int wib = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const Tables tb = load_tables<DIN, DOUT>(a, smem + WPB * WSL);
  const int64_t wg = (int64_t)blockIdx.x * WPB + wib;
  if (wg >= (int64_t)a.nc * a.ngroups) return;
  const int c = (int)(wg / a.ngroups), grp = (int)(wg - (int64_t)c * a.ngroups);
  const int nn = grp * 32 + lane;
  float* Gs = smem + wib * WSL;
  float* Gbs = Gs + DENV * 32;
  float2* Ms = reinterpret_cast<float2*>(Gbs + DENV * 32);
  float* scr = Gbs + DENV * 32 + MSL;
  float* ring = scr + SCR;
  const int64_t e0 = a.rowa[c], e1 = a.rowa[c + 1];
  const int deg = (int)(e1 - e0);
  if (deg <= 0) return;
  float* Yb = a.Ybar + (size_t)grp * a.ybar_gstride;

  auto issue = [&](int64_t e, float* st, int ab) {
    if (FIRST) {
      tp_cp_rows<NLV>(st, a.w0 + e * a.ldw + grp * 32, a.n, lane);
      if (lane < LDY / 4) tp_cp16(st + NLV * 32 + lane * 4, a.Y + e * a.ldy + lane * 4);
    } else {
      // rows ab .. ab+AB-1 of V_e (a ragged last block re-reads valid rows of the same edge)
      const int a0 = (ab + AB <= DIN) ? ab : DIN - AB;
      tp_cp_rows<AB>(st, a.Vin + (e * DIN + a0) * a.n + grp * 32, a.n, lane);
    }
    if (HASVB) tp_cp_rows<DOUT>(st + SV, a.VbarL + e * DOUT * a.n + grp * 32, a.n, lane);
    if (lane < 8) tp_cp16(st + SF - 32 + lane * 4, a.sbar + e * a.lds + grp * 32 + lane * 4);
  };
#pragma unroll
  for (int s = 0; s < NST - 1; ++s) {
    if (s < deg) issue(e0 + s, ring + s * SF, 0);
    tp_cp_commit();
  }
  gamma_pass<DENV>(a, e0, e1, nn, lane, Gs);
#pragma unroll
  for (int b = 0; b < DENV; ++b) Gbs[b * 32 + lane] = 0.f;

  for (int ab = 0; ab < DIN; ab += AB) {
    // for a ragged last block the staged rows start at a0 = DIN - AB; slot k of the block reads row k + (ab - a0)
    const int a0 = (FIRST || ab + AB <= DIN) ? ab : DIN - AB;
    const int roff = ab - a0;
    float2 Mr[MREG ? AB * CH : 1];
    float2 Mb[AB * CH];
    if constexpr (MREG) {
#pragma unroll
      for (int k = 0; k < AB; ++k) {
#pragma unroll 1
        for (int cc = 0; cc < 2 * CH; ++cc)
          scr[((cc >> 1) * 32 + lane) * 2 + (cc & 1)] = (cc < DOUT && ab + k < DIN) ? pair_val(tb, (ab + k) * DOUT + cc, Gs, lane) : 0.f;
#pragma unroll
        for (int j = 0; j < CH; ++j) Mr[k * CH + j] = reinterpret_cast<const float2*>(scr)[j * 32 + lane];
      }
    } else {
#pragma unroll 1
      for (int k = 0; k < AB; ++k)
#pragma unroll 1
        for (int cc = 0; cc < 2 * CH; ++cc)
          reinterpret_cast<float*>(Ms)[((k * CH + (cc >> 1)) * 32 + lane) * 2 + (cc & 1)] =
              (cc < DOUT && ab + k < DIN) ? pair_val(tb, (ab + k) * DOUT + cc, Gs, lane) : 0.f;
    }
#pragma unroll
    for (int k = 0; k < AB * CH; ++k) Mb[k] = make_float2(0.f, 0.f);
    if (ab > 0) {
      __syncwarp();
#pragma unroll
      for (int s = 0; s < NST - 1; ++s) {
        if (s < deg) issue(e0 + s, ring + s * SF, ab);
        tp_cp_commit();
      }
    }
    __syncwarp();
    int slot = 0;
    for (int i = 0; i < deg; ++i) {
      tp_cp_wait<NST - 2>();
      __syncwarp();
      {
        const int nx = i + NST - 1;
        int ns = slot + NST - 1; if (ns >= NST) ns -= NST;
        if (nx < deg) issue(e0 + nx, ring + ns * SF, ab);
        tp_cp_commit();
      }
      const float* st = ring + slot * SF;
      const int64_t e = e0 + i;
      float2 t2[CH];
#pragma unroll
      for (int j = 0; j < CH; ++j) {
        t2[j].x = HASVB ? st[SV + (2 * j) * 32 + lane] : 0.f;
        t2[j].y = (HASVB && 2 * j + 1 < DOUT) ? st[SV + (2 * j + 1) * 32 + lane] : 0.f;
      }
      t2[0].x += st[SF - 32 + lane];
      float w[NLV], wb[NLV];
      if (FIRST) {
#pragma unroll
        for (int l = 0; l < NLV; ++l) { w[l] = st[l * 32 + lane]; wb[l] = 0.f; }
      }
      float vb[AB], pp[AB];
#pragma unroll
      for (int k = 0; k < AB; ++k) {
        const bool valid = ab + k < DIN;
        const int ka = valid ? ab + k : DIN - 1;     // absolute input component
        float v, y = 0.f, wl = 0.f;
        if (FIRST) {
          y = st[NLV * 32 + ka];
          wl = w[0];
#pragma unroll
          for (int l = 1; l < NLV; ++l) wl = (l_of(ka) == l) ? w[l] : wl;
          v = valid ? wl * y : 0.f;
        } else {
          v = valid ? st[(k + roff) * 32 + lane] : 0.f;
        }
        const float2 v2 = make_float2(v, v);
        float2 s2 = make_float2(0.f, 0.f);
#pragma unroll
        for (int j = 0; j < CH; ++j) {
          float2 m2;
          if constexpr (MREG) m2 = Mr[k * CH + j]; else m2 = Ms[(k * CH + j) * 32 + lane];
          s2 = tp_fma2(m2, t2[j], s2);
          Mb[k * CH + j] = tp_fma2(v2, t2[j], Mb[k * CH + j]);
        }
        vb[k] = s2.x + s2.y;
        if (FIRST) {
#pragma unroll
          for (int l = 0; l < NLV; ++l) wb[l] = (valid && l_of(ka) == l) ? fmaf(vb[k], y, wb[l]) : wb[l];
          pp[k] = valid ? wl * vb[k] : 0.f;
        }
      }
      if (FIRST) {
        const int nvalid = (DIN - ab < AB) ? DIN - ab : AB;
        tp_ybar_rows<AB, YINIT>(Yb + e * DENV, pp, ab, nvalid, lane);
#pragma unroll
        for (int l = 0; l < NLV; ++l) {
          float* p = a.w0bar + e * a.ldob + l * a.n + nn;
          if (ab == 0) *p = wb[l]; else *p += wb[l];
        }
      } else {
#pragma unroll
        for (int k = 0; k < AB; ++k)
          if (ab + k < DIN) a.Vbar_prev[(e * DIN + ab + k) * a.n + nn] = vb[k];
      }
      if (++slot == NST) slot = 0;
    }
    // Gamma-bar += K . M-bar(block)
#pragma unroll
    for (int k = 0; k < AB; ++k) {
#pragma unroll
      for (int j = 0; j < CH; ++j) reinterpret_cast<float2*>(scr)[j * 32 + lane] = Mb[k * CH + j];
      if (ab + k < DIN) {
#pragma unroll 1
        for (int cc = 0; cc < DOUT; ++cc) {
          const float mb = scr[((cc >> 1) * 32 + lane) * 2 + (cc & 1)];
          const int p0 = (ab + k) * DOUT + cc;
          for (int q = tb.ptr[p0]; q < tb.ptr[p0 + 1]; ++q)
            Gbs[tb.b[q] * 32 + lane] = fmaf(tb.val[q], mb, Gbs[tb.b[q] * 32 + lane]);
        }
      }
    }
  }
  // pass 2 (direct loads, 2 edges in flight): omega-bar_e and the environment part of Y-bar_e
  float Gb[DENV];
#pragma unroll
  for (int b = 0; b < DENV; ++b) Gb[b] = a.c_env * Gbs[b * 32 + lane];
  for (int64_t e = e0; e < e1; e += 2) {
    float om[2][NLV];
    float4 yq[2][LDY / 4];
#pragma unroll
    for (int i = 0; i < 2; ++i) {
      const int64_t ee = (e + i < e1) ? e + i : e1 - 1;
#pragma unroll
      for (int l = 0; l < NLV; ++l) om[i][l] = a.om[ee * a.ldo + l * a.n + nn];
#pragma unroll
      for (int q = 0; q < LDY / 4; ++q) yq[i][q] = __ldg(reinterpret_cast<const float4*>(a.Y + ee * a.ldy) + q);
    }
#pragma unroll
    for (int i = 0; i < 2; ++i) {
      if (e + i < e1) {
        float pp[DENV];
#pragma unroll
        for (int l = 0; l < NLV; ++l) {
          float ob = 0.f;
#pragma unroll
          for (int b = l * l; b < (l + 1) * (l + 1); ++b) {
            ob = fmaf(Gb[b], ycomp<LDY>(yq[i], b), ob);
            pp[b] = om[i][l] * Gb[b];
          }
          a.ombar[(e + i) * a.ldob + l * a.n + nn] = ob;
        }
        tp_ybar_rows<DENV, (YINIT && !FIRST)>(Yb + (e + i) * DENV, pp, 0, DENV, lane);
      }
    }
  }
}

// ---- host side ---------------------------------------------------------------------------------------------
template <int DENV, int DIN, int DOUT, int CB, bool FIRST, int NST, int WPB>
int launch_fwd2(allegro_model* m, const TP2& a) {
  constexpr int NLV = nlv_of(DENV), LDY = (DENV + 3) & ~3;
  constexpr int SF = FIRST ? NLV * 32 + LDY : DIN * 32;
  constexpr int WSL = DENV * 32 + ((CB + 1) / 2) * 64 + NST * SF;
  size_t sm = (size_t)WPB * WSL * 4 + (size_t)tab_ints(DIN, DOUT) * 4 + (size_t)a.nnz * 8 + 16;
  static bool set = false;
  if (!set) { AL_CUDA(m, cudaFuncSetAttribute(k_tp2_fwd<DENV, DIN, DOUT, CB, FIRST, NST, WPB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm)); set = true; }
  int64_t warps = (int64_t)a.nc * a.ngroups;
  k_tp2_fwd<DENV, DIN, DOUT, CB, FIRST, NST, WPB><<<(unsigned)((warps + WPB - 1) / WPB), WPB * 32, sm, m->stream>>>(a);
  m->launches++;
  AL_CUDA(m, cudaGetLastError());
  return ALLEGRO_OK;
}

template <int DENV, int DIN, int DOUT, int AB, bool FIRST, bool HASVB, bool MREG, int NST, int WPB>
int launch_bwd2(allegro_model* m, const TP2& a) {
  constexpr int NLV = nlv_of(DENV), LDY = (DENV + 3) & ~3, CH = (DOUT + 1) / 2;
  constexpr int SV = FIRST ? NLV * 32 + LDY : AB * 32;
  constexpr int SF = SV + (HASVB ? DOUT * 32 : 0) + 32;
  constexpr int MSL = MREG ? 0 : AB * CH * 64;
  constexpr int WSL = 2 * DENV * 32 + MSL + CH * 64 + NST * SF;
  size_t sm = (size_t)WPB * WSL * 4 + (size_t)tab_ints(DIN, DOUT) * 4 + (size_t)a.nnz * 8 + 16;
  // Y-bar is initialised by the first backward kernel of the step, which is the one without a V-bar input
  auto kern = k_tp2_bwd<DENV, DIN, DOUT, AB, FIRST, HASVB, MREG, !HASVB, NST, WPB>;
  static bool set = false;
  if (!set) { AL_CUDA(m, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm)); set = true; }
  int64_t warps = (int64_t)a.nc * a.ngroups;
  kern<<<(unsigned)((warps + WPB - 1) / WPB), WPB * 32, sm, m->stream>>>(a);
  m->launches++;
  AL_CUDA(m, cudaGetLastError());
  return ALLEGRO_OK;
}

inline void fill2(allegro_model* m, Work& w, int L, int nc, TP2& a, const float* om, int ldo, const float* Vin, const float* w0, int ldw) {
  const TPLayerDev& t = m->tp[L - 1];
  a.rowa = (const int64_t*)w.rowa.p; a.nc = nc; a.om = om; a.ldo = ldo; a.Y = (const float*)w.Y.p; a.ldy = m->ldY;
  a.Vin = Vin; a.w0 = w0; a.ldw = ldw; a.dp_ptr = t.dp_ptr; a.dp_b = t.dp_b; a.dp_val = t.dp_val; a.nnz = t.nnz;
  a.n = m->n; a.ngroups = m->n / 32; a.c_env = m->c_env;
}

