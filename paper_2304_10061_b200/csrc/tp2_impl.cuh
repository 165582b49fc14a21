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
//     all inner products are packed FFMA2;
//   * the sparsity pattern of K is a compile-time X-macro list (tp2_patterns.inc, generated at build time
//     from cg_tables.cpp), so M_i = K.Gamma_i and Gamma-bar_i = K.M-bar_i are straight-line FFMAs with
//     literal register indices; the values (which carry the path weights) come from the kernel parameters
//     (constant bank);
//   * wide features (l_max = 3) walk blocks of output components (forward) / input components (backward);
//   * every Y-bar contribution (per channel group: V^0 part, environment part of each layer) is a plain
//     store into its own partial buffer; k_edge_bwd sums the partials in fixed order (no memset, no RMW).
// Requirements (checked on the host, otherwise the kernels of tp_kernels.cu run): n % 32 == 0, V^0 layout
// equal to the environment layout, and every layer's pattern equal to a generated one.
#pragma once
#include <cstdlib>
#include <cstring>

#include "kernels.h"
#include "tp2_patterns.inc"
#include "tp_common.cuh"

enum { P_9_9_9 = 0, P_9_9_1, P_4_4_4, P_4_4_1, P_16_16_31, P_16_31_16, P_16_16_1, P_COUNT };
template <int P> struct Pat;
template <> struct Pat<P_9_9_9> { static constexpr int DENV = 9, DIN = 9, DOUT = 9, NNZ = TP2_NNZ_9_9_9; };
template <> struct Pat<P_9_9_1> { static constexpr int DENV = 9, DIN = 9, DOUT = 1, NNZ = TP2_NNZ_9_9_1; };
template <> struct Pat<P_4_4_4> { static constexpr int DENV = 4, DIN = 4, DOUT = 4, NNZ = TP2_NNZ_4_4_4; };
template <> struct Pat<P_4_4_1> { static constexpr int DENV = 4, DIN = 4, DOUT = 1, NNZ = TP2_NNZ_4_4_1; };
template <> struct Pat<P_16_16_31> { static constexpr int DENV = 16, DIN = 16, DOUT = 31, NNZ = TP2_NNZ_16_16_31; };
template <> struct Pat<P_16_31_16> { static constexpr int DENV = 16, DIN = 31, DOUT = 16, NNZ = TP2_NNZ_16_31_16; };
template <> struct Pat<P_16_16_1> { static constexpr int DENV = 16, DIN = 16, DOUT = 1, NNZ = TP2_NNZ_16_16_1; };

// expands X(k, a, b, c) over the entries of pattern P (P is a template parameter at the point of use)
#define TP2_EXPAND(P, X)                                            \
  if constexpr (P == P_9_9_9) { TP2_PAT_9_9_9(X) }                  \
  else if constexpr (P == P_9_9_1) { TP2_PAT_9_9_1(X) }             \
  else if constexpr (P == P_4_4_4) { TP2_PAT_4_4_4(X) }             \
  else if constexpr (P == P_4_4_1) { TP2_PAT_4_4_1(X) }             \
  else if constexpr (P == P_16_16_31) { TP2_PAT_16_16_31(X) }       \
  else if constexpr (P == P_16_31_16) { TP2_PAT_16_31_16(X) }       \
  else if constexpr (P == P_16_16_1) { TP2_PAT_16_16_1(X) }

template <int NNZ>
struct TP2 {
  const int64_t* rowa; int nc;
  const float* om; int ldo;
  const float* Y; int ldy;
  const float* Vin;
  const float* w0; int ldw;
  int n, ngroups; float c_env;
  float* Tout; float* xs; int ldx; float* gamma_out;
  const float* VbarL; const float* sbar; int lds;
  float* Vbar_prev; float* ombar; int ldob; float* w0bar;
  // Y-bar partials [part][M][DENV], plain stores: part = ybar_part0 + group for the V^0 contribution (FIRST, pass 1),
  // ybar_partL + group for this layer's environment contribution (pass 2); see al_ybar_layout()
  float* Ybar; int64_t ybar_pstride; int ybar_part0, ybar_partL;
  int rev;         // 1: warps take the (centre, group) pairs from the last to the first (allegro_model::sweep_mode)
  float kv[NNZ];   // values of the fused tensor K in pattern order (dense pair table order)
};

__host__ __device__ constexpr int l_of(int k) { return k < 1 ? 0 : k < 4 ? 1 : k < 9 ? 2 : 3; }
__host__ __device__ constexpr int nlv_of(int denv) { return denv == 1 ? 1 : denv == 4 ? 2 : denv == 9 ? 3 : 4; }

template <int LDY>
__device__ __forceinline__ float ycomp(const float4* y, int b) { return reinterpret_cast<const float*>(y)[b]; }

// element (r, cc) of a register matrix stored as float2 pairs over the second index, W pairs per row
#define TP2_REF(M, W, r, cc) (((cc) & 1) ? M[(r) * (W) + ((cc) >> 1)].y : M[(r) * (W) + ((cc) >> 1)].x)

// Gamma_i[b] = c_env sum_e omega_e[l(b)] Y_e[b]   (direct loads, 8 edges in flight).  Y_e is the same for every lane:
// the warp loads the 8 rows as one contiguous block (LDY / 4 coalesced loads, one value per lane) and broadcasts the
// components by shuffle, so a batch costs 8 NLV + LDY / 4 registers instead of 8 (NLV + LDY).  (ncu had 29 % of the
// layer-1 forward's stall samples on this serial prologue with 4 edges in flight; holding two batches of 4 with
// per-lane copies of Y took 164 registers in every kernel.)  nn = 32 * group + lane.
template <int DENV, class A>
__device__ __forceinline__ void gamma_pass(const A& a, int64_t e0, int64_t e1, int nn, float* G) {
  constexpr int NLV = nlv_of(DENV), LDY = (DENV + 3) & ~3, NR = LDY / 4;
  const int lane = nn & 31;
  const int64_t ylast = e1 * LDY - 1;
#pragma unroll
  for (int b = 0; b < DENV; ++b) G[b] = 0.f;
  for (int64_t e = e0; e < e1; e += 8) {
    float om[8][NLV], yr[NR];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const int64_t ee = (e + i < e1) ? e + i : e1 - 1;
#pragma unroll
      for (int l = 0; l < NLV; ++l) om[i][l] = a.om[ee * a.ldo + l * a.n + nn];
    }
#pragma unroll
    for (int k = 0; k < NR; ++k) {
      const int64_t idx = e * LDY + k * 32 + lane;     // rows beyond e1 are clamped into this centre's block (masked below)
      yr[k] = __ldg(a.Y + (idx < ylast ? idx : ylast));
    }
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const bool ok = e + i < e1;
#pragma unroll
      for (int b = 0; b < DENV; ++b) {
        const float y = __shfl_sync(TP_FULLMASK, yr[(i * LDY + b) >> 5], (i * LDY + b) & 31);
        G[b] = fmaf(ok ? om[i][l_of(b)] : 0.f, y, G[b]);
      }
    }
  }
#pragma unroll
  for (int b = 0; b < DENV; ++b) G[b] *= a.c_env;
}

// ======================================================================================================
// forward:  T_e[c] = sum_a V_e[a] M_i[a][c]   (c-blocks of CB output components; CB == DOUT: one pass)
// ======================================================================================================
template <int P, int CB, bool FIRST, int NST, int WPB>
static __global__ void __launch_bounds__(WPB * 32) k_tp2_fwd(const __grid_constant__ TP2<Pat<P>::NNZ> a) {
  constexpr int DENV = Pat<P>::DENV, DIN = Pat<P>::DIN, DOUT = Pat<P>::DOUT;
  constexpr int NLV = nlv_of(DENV), LDY = (DENV + 3) & ~3, CBH = (CB + 1) / 2;
  constexpr int SF = FIRST ? NLV * 32 + LDY : DIN * 32;   // floats per ring stage (one edge)
  constexpr int WSL = DENV * 32 + NST * SF;               // floats per warp slice
  extern __shared__ float4 smem4[];
  float* smem = reinterpret_cast<float*>(smem4);
  const int wib = threadIdx.x >> 5, lane = threadIdx.x & 31;
  int64_t wg = (int64_t)blockIdx.x * WPB + wib;
  if (wg >= (int64_t)a.nc * a.ngroups) return;
  if (a.rev) wg = (int64_t)a.nc * a.ngroups - 1 - wg;
  const int c = (int)(wg / a.ngroups), grp = (int)(wg - (int64_t)c * a.ngroups);
  const int nn = grp * 32 + lane;
  float* Gs = smem + wib * WSL;
  float* ring = Gs + DENV * 32;
  const int64_t e0 = a.rowa[c], e1 = a.rowa[c + 1];
  const int deg = (int)(e1 - e0);
  if (deg <= 0) return;

  // per-center base pointers and hoisted per-lane chunk offsets: the edge loop only adds il * stride
  constexpr int OPROWS = FIRST ? NLV : DIN;
  int off_op[(OPROWS * 8 + 31) / 32];
  tp_row_offsets<OPROWS>(off_op, a.n, lane);
  const float* opc = FIRST ? a.w0 + e0 * a.ldw + grp * 32 : a.Vin + e0 * DIN * a.n + grp * 32;
  const int op_stride = FIRST ? a.ldw : DIN * a.n;
  const float* Yc = a.Y + e0 * a.ldy + lane * 4;
  auto issue = [&](int il, float* st) {
    tp_cp_rows_pre<OPROWS>(st, opc + il * op_stride, off_op, lane);
    if (FIRST && lane < LDY / 4) tp_cp16(st + NLV * 32 + lane * 4, Yc + il * a.ldy);
  };
  // start streaming the first edges while Gamma_i is being summed
#pragma unroll
  for (int s = 0; s < NST - 1; ++s) {
    if (s < deg) issue(s, ring + s * SF);
    tp_cp_commit();
  }
  {
    float G[DENV];
    gamma_pass<DENV>(a, e0, e1, nn, G);
#pragma unroll
    for (int b = 0; b < DENV; ++b) Gs[b * 32 + lane] = G[b];
    if (a.gamma_out)
#pragma unroll
      for (int b = 0; b < DENV; ++b) a.gamma_out[((size_t)c * DENV + b) * a.n + nn] = G[b];
  }

#pragma unroll
  for (int cb = 0; cb < DOUT; cb += CB) {
    float2 Mr[DIN * CBH];
    {
      float G[DENV];
#pragma unroll
      for (int b = 0; b < DENV; ++b) G[b] = Gs[b * 32 + lane];
#pragma unroll
      for (int k = 0; k < DIN * CBH; ++k) Mr[k] = make_float2(0.f, 0.f);
#define X(k, a_, b_, c_) \
  if ((c_) >= cb && (c_) < cb + CB) TP2_REF(Mr, CBH, a_, (c_) - cb) = fmaf(a.kv[k], G[b_], TP2_REF(Mr, CBH, a_, (c_) - cb));
      TP2_EXPAND(P, X)
#undef X
    }
    if (cb > 0) {   // restart the ring for this block of output components
      __syncwarp();
#pragma unroll
      for (int s = 0; s < NST - 1; ++s) {
        if (s < deg) issue(s, ring + s * SF);
        tp_cp_commit();
      }
    }
    int slot = 0;
    float* xsp = a.xs + e0 * a.ldx + nn;
    float* Tp = a.Tout ? a.Tout + (e0 * DOUT + cb) * a.n + nn : nullptr;
    for (int i = 0; i < deg; ++i) {
      tp_cp_wait<NST - 2>();
      __syncwarp();
      {
        const int nx = i + NST - 1;
        int ns = slot + NST - 1; if (ns >= NST) ns -= NST;
        if (nx < deg) issue(nx, ring + ns * SF);
        tp_cp_commit();
      }
      const float* st = ring + slot * SF;
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
      if (cb == 0) { *xsp = acc[0].x; xsp += a.ldx; }
      if (Tp) {
#pragma unroll
        for (int cc = 0; cc < CB; ++cc)
          if (cb + cc < DOUT) Tp[cc * a.n] = (cc & 1) ? acc[cc >> 1].y : acc[cc >> 1].x;
        Tp += DOUT * a.n;
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
template <int P, int AB, bool FIRST, bool HASVB, bool MREG, int NST, int WPB>
static __global__ void __launch_bounds__(WPB * 32) k_tp2_bwd(const __grid_constant__ TP2<Pat<P>::NNZ> a) {
  constexpr int DENV = Pat<P>::DENV, DIN = Pat<P>::DIN, DOUT = Pat<P>::DOUT;
  constexpr int NLV = nlv_of(DENV), LDY = (DENV + 3) & ~3, CH = (DOUT + 1) / 2;
  constexpr int SV = FIRST ? NLV * 32 + LDY : AB * 32;      // operand part of a stage
  constexpr int SF = SV + (HASVB ? DOUT * 32 : 0) + 32;     // + T-bar rows + s-bar row
  constexpr int MSL = MREG ? 0 : AB * CH * 64;              // M block as float2 per lane
  constexpr int WSL = 2 * DENV * 32 + MSL + NST * SF;
  extern __shared__ float4 smem4[];
  float* smem = reinterpret_cast<float*>(smem4);
  const int wib = threadIdx.x >> 5, lane = threadIdx.x & 31;
  int64_t wg = (int64_t)blockIdx.x * WPB + wib;
  if (wg >= (int64_t)a.nc * a.ngroups) return;
  if (a.rev) wg = (int64_t)a.nc * a.ngroups - 1 - wg;
  const int c = (int)(wg / a.ngroups), grp = (int)(wg - (int64_t)c * a.ngroups);
  const int nn = grp * 32 + lane;
  float* Gs = smem + wib * WSL;
  float* Gbs = Gs + DENV * 32;
  float2* Ms = reinterpret_cast<float2*>(Gbs + DENV * 32);
  float* ring = Gbs + DENV * 32 + MSL;
  const int64_t e0 = a.rowa[c], e1 = a.rowa[c + 1];
  const int deg = (int)(e1 - e0);
  if (deg <= 0) return;
  float* Yb0 = a.Ybar + (size_t)(a.ybar_part0 + grp) * a.ybar_pstride;
  float* YbL = a.Ybar + (size_t)(a.ybar_partL + grp) * a.ybar_pstride;

  // per-center base pointers and hoisted per-lane chunk offsets: the edge loop only adds il * stride
  constexpr int OPROWS = FIRST ? NLV : AB;
  int off_op[(OPROWS * 8 + 31) / 32], off_vb[HASVB ? (DOUT * 8 + 31) / 32 : 1];
  tp_row_offsets<OPROWS>(off_op, a.n, lane);
  if (HASVB) tp_row_offsets<DOUT>(off_vb, a.n, lane);
  const float* opc = FIRST ? a.w0 + e0 * a.ldw + grp * 32 : a.Vin + e0 * DIN * a.n + grp * 32;
  const int op_stride = FIRST ? a.ldw : DIN * a.n;
  const float* Yc = a.Y + e0 * a.ldy + lane * 4;
  const float* vbc = HASVB ? a.VbarL + e0 * DOUT * a.n + grp * 32 : nullptr;
  const float* sbc = a.sbar + e0 * a.lds + grp * 32 + (lane & 7) * 4;
  auto issue = [&](int il, float* st, int ab) {
    // FIRST: w0 rows + Y; else rows ab .. ab+AB-1 of V_e (a ragged last block re-reads valid rows of the same edge)
    const int a0 = (FIRST || ab + AB <= DIN) ? ab : DIN - AB;
    tp_cp_rows_pre<OPROWS>(st, opc + il * op_stride + (FIRST ? 0 : a0 * a.n), off_op, lane);
    if (FIRST && lane < LDY / 4) tp_cp16(st + NLV * 32 + lane * 4, Yc + il * a.ldy);
    if (HASVB) tp_cp_rows_pre<DOUT>(st + SV, vbc + il * (DOUT * a.n), off_vb, lane);
    if (lane < 8) tp_cp16(st + SF - 32 + lane * 4, sbc + il * a.lds);
  };
#pragma unroll
  for (int s = 0; s < NST - 1; ++s) {
    if (s < deg) issue(s, ring + s * SF, 0);
    tp_cp_commit();
  }
  {
    float G[DENV];
    gamma_pass<DENV>(a, e0, e1, nn, G);
#pragma unroll
    for (int b = 0; b < DENV; ++b) { Gs[b * 32 + lane] = G[b]; Gbs[b * 32 + lane] = 0.f; }
  }

#pragma unroll
  for (int ab = 0; ab < DIN; ab += AB) {
    // for a ragged last block the staged rows start at a0 = DIN - AB; slot k of the block reads row k + (ab - a0)
    const int a0 = (FIRST || ab + AB <= DIN) ? ab : DIN - AB;
    const int roff = ab - a0;
    float2 Mr[MREG ? AB * CH : 1];
    float2 Mb[AB * CH];
    {
      float G[DENV];
#pragma unroll
      for (int b = 0; b < DENV; ++b) G[b] = Gs[b * 32 + lane];
      if constexpr (MREG) {
#pragma unroll
        for (int k = 0; k < AB * CH; ++k) Mr[k] = make_float2(0.f, 0.f);
#define X(k, a_, b_, c_) \
  if ((a_) >= ab && (a_) < ab + AB) TP2_REF(Mr, CH, (a_) - ab, c_) = fmaf(a.kv[k], G[b_], TP2_REF(Mr, CH, (a_) - ab, c_));
        TP2_EXPAND(P, X)
#undef X
      } else {
        // one row of the block at a time: accumulate in registers, park in the warp's shared slice
#pragma unroll
        for (int r = 0; r < AB; ++r) {
          float2 row[CH];
#pragma unroll
          for (int j = 0; j < CH; ++j) row[j] = make_float2(0.f, 0.f);
#define X(k, a_, b_, c_) \
  if ((a_) == ab + r) TP2_REF(row, CH, 0, c_) = fmaf(a.kv[k], G[b_], TP2_REF(row, CH, 0, c_));
          TP2_EXPAND(P, X)
#undef X
#pragma unroll
          for (int j = 0; j < CH; ++j) Ms[(r * CH + j) * 32 + lane] = row[j];
        }
      }
    }
#pragma unroll
    for (int k = 0; k < AB * CH; ++k) Mb[k] = make_float2(0.f, 0.f);
    if (ab > 0) {
      __syncwarp();
#pragma unroll
      for (int s = 0; s < NST - 1; ++s) {
        if (s < deg) issue(s, ring + s * SF, ab);
        tp_cp_commit();
      }
    }
    int slot = 0;
    float* yb0p = Yb0 + e0 * DENV;
    float* outp = FIRST ? a.w0bar + e0 * a.ldob + nn : a.Vbar_prev + (e0 * DIN + ab) * a.n + nn;
    for (int i = 0; i < deg; ++i) {
      tp_cp_wait<NST - 2>();
      __syncwarp();
      {
        const int nx = i + NST - 1;
        int ns = slot + NST - 1; if (ns >= NST) ns -= NST;
        if (nx < deg) issue(nx, ring + ns * SF, ab);
        tp_cp_commit();
      }
      const float* st = ring + slot * SF;
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
          wl = w[l_of(ka)];
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
          if (valid) wb[l_of(ka)] = fmaf(vb[k], y, wb[l_of(ka)]);
          pp[k] = valid ? wl * vb[k] : 0.f;
        }
      }
      if (FIRST) {
        const int nvalid = (DIN - ab < AB) ? DIN - ab : AB;
        tp_ybar_rows<AB, true>(yb0p, pp, ab, nvalid, lane);
        yb0p += DENV;
#pragma unroll
        for (int l = 0; l < NLV; ++l) {
          // (a block only touches the l values of its own components; the first toucher stores)
          const bool touched = l_of(ab) <= l && l <= l_of((ab + AB - 1 < DIN) ? ab + AB - 1 : DIN - 1);
          const bool first_touch = (ab == 0) || l_of(ab - 1) < l;
          if (touched) {
            float* p = outp + l * a.n;
            if (first_touch) *p = wb[l]; else *p += wb[l];
          }
        }
        outp += a.ldob;
      } else {
#pragma unroll
        for (int k = 0; k < AB; ++k)
          if (ab + k < DIN) outp[k * a.n] = vb[k];
        outp += DIN * a.n;
      }
      if (++slot == NST) slot = 0;
    }
    // Gamma-bar += K . M-bar(block)
    {
      float Gb[DENV];
#pragma unroll
      for (int b = 0; b < DENV; ++b) Gb[b] = Gbs[b * 32 + lane];
#define X(k, a_, b_, c_) \
  if ((a_) >= ab && (a_) < ab + AB) Gb[b_] = fmaf(a.kv[k], TP2_REF(Mb, CH, (a_) - ab, c_), Gb[b_]);
      TP2_EXPAND(P, X)
#undef X
#pragma unroll
      for (int b = 0; b < DENV; ++b) Gbs[b * 32 + lane] = Gb[b];
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
        tp_ybar_rows<DENV, true>(YbL + (e + i) * DENV, pp, 0, DENV, lane);
      }
    }
  }
}

// ---- host side ---------------------------------------------------------------------------------------------
template <int P, int CB, bool FIRST, int NST, int WPB>
int launch_fwd2(allegro_model* m, const TP2<Pat<P>::NNZ>& a) {
  constexpr int DENV = Pat<P>::DENV, DIN = Pat<P>::DIN;
  constexpr int NLV = nlv_of(DENV), LDY = (DENV + 3) & ~3;
  constexpr int SF = FIRST ? NLV * 32 + LDY : DIN * 32;
  constexpr int WSL = DENV * 32 + NST * SF;
  size_t sm = (size_t)WPB * WSL * 4 + 16;
  static AttrOnce once;
  if (once.need(m->device)) { AL_CUDA(m, cudaFuncSetAttribute(k_tp2_fwd<P, CB, FIRST, NST, WPB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm)); once.done(m->device); }
  int64_t warps = (int64_t)a.nc * a.ngroups;
  k_tp2_fwd<P, CB, FIRST, NST, WPB><<<(unsigned)((warps + WPB - 1) / WPB), WPB * 32, sm, m->stream>>>(a);
  m->launches++;
  AL_CUDA(m, cudaGetLastError());
  return ALLEGRO_OK;
}

template <int P, int AB, bool FIRST, bool HASVB, bool MREG, int NST, int WPB>
int launch_bwd2(allegro_model* m, const TP2<Pat<P>::NNZ>& a) {
  constexpr int DENV = Pat<P>::DENV, DOUT = Pat<P>::DOUT;
  constexpr int NLV = nlv_of(DENV), LDY = (DENV + 3) & ~3, CH = (DOUT + 1) / 2;
  constexpr int SV = FIRST ? NLV * 32 + LDY : AB * 32;
  constexpr int SF = SV + (HASVB ? DOUT * 32 : 0) + 32;
  constexpr int MSL = MREG ? 0 : AB * CH * 64;
  constexpr int WSL = 2 * DENV * 32 + MSL + NST * SF;
  size_t sm = (size_t)WPB * WSL * 4 + 16;
  auto kern = k_tp2_bwd<P, AB, FIRST, HASVB, MREG, NST, WPB>;
  static AttrOnce once;
  if (once.need(m->device)) { AL_CUDA(m, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm)); once.done(m->device); }
  int64_t warps = (int64_t)a.nc * a.ngroups;
  kern<<<(unsigned)((warps + WPB - 1) / WPB), WPB * 32, sm, m->stream>>>(a);
  m->launches++;
  AL_CUDA(m, cudaGetLastError());
  return ALLEGRO_OK;
}

// common arguments of one layer; the values of K are copied into the parameter block
struct TP2Common {
  Work* w; int L, nc; const float* om; int ldo; const float* Vin; const float* w0; int ldw;
  float* Tout; float* xs; int ldx;
  const float* VbarL; const float* sbar; int lds; float* Vbar_prev; float* ombar; int ldob; float* w0bar;
};

template <int NNZ>
int fill2(allegro_model* m, const TP2Common& q, TP2<NNZ>& a) {
  const TPLayerHost& h = m->tp_host[q.L - 1];
  if ((int)h.dp_val.size() != NNZ) { al_set_error(m, "tp2: pattern size mismatch"); return ALLEGRO_ERR_BAD_ARG; }
  Work& w = *q.w;
  a.rowa = (const int64_t*)w.rowa.p; a.nc = q.nc; a.om = q.om; a.ldo = q.ldo; a.Y = (const float*)w.Y.p; a.ldy = m->ldY;
  a.Vin = q.Vin; a.w0 = q.w0; a.ldw = q.ldw; a.n = m->n; a.ngroups = m->n / 32; a.c_env = m->c_env;
  a.Tout = q.Tout; a.xs = q.xs; a.ldx = q.ldx; a.gamma_out = (float*)w.gamma.p;
  a.VbarL = q.VbarL; a.sbar = q.sbar; a.lds = q.lds; a.Vbar_prev = q.Vbar_prev; a.ombar = q.ombar; a.ldob = q.ldob;
  a.w0bar = q.w0bar; a.Ybar = (float*)w.Ybar.p; a.ybar_pstride = (int64_t)w.cap_edges * m->Denv;
  { int part[AL_MAX_LAYERS + 1]; al_ybar_layout(m, part); a.ybar_part0 = part[0]; a.ybar_partL = part[q.L]; }
  memcpy(a.kv, h.dp_val.data(), sizeof(float) * NNZ);
  a.rev = al_next_rev(m);
  return ALLEGRO_OK;
}
