// Tensor-track kernels for wide features (l_max = 3: D = 16 / 31), lane-split version of tp2_impl.cuh.
//
// With 16 x 31 components the per-(center, channel) matrix M_i no longer fits a lane's registers, and walking
// blocks of it one after another (tp2_impl.cuh) re-reads every operand row once per block: ncu showed the
// blocked kernels at 47-81 % DRAM utilisation on those re-reads.  Here a warp owns (center, 8 channels) and its
// lanes are (channel ch = lane & 7, block q = lane >> 3): lane (ch, q) holds block q of M_i for channel ch --
// output components [q CB, (q+1) CB) in the forward, input components [q AB, (q+1) AB) in the backward -- so
// every operand row is staged once (cp.async ring, 32 B per row and warp) and read by the four lanes that
// share the channel.  The sparsity pattern of K stays compile-time (tp2_patterns.inc): an entry that belongs
// to block blk becomes one FFMA predicated on q == blk.  Row reductions: over the 8 channels with xor-shuffles
// 1, 2, 4; over the 4 blocks with xor-shuffles 8, 16.  Y-bar / w0-bar / omega-bar are split by groups of four
// environment components (group q: b in [4q, 4q+4)), whose l values are {l(4q)} for the first and {l(4q+1)}
// for the other three components.
#pragma once
#include "tp2_impl.cuh"

constexpr int T3_CPW = 8;   // channels per warp

// ROWS rows of 8 floats (32 B): smem dst row r at dst + 8 r, global row r at src + r * rstride
template <int ROWS>
__device__ __forceinline__ void t3_cp_rows(float* dst, const float* src, int rstride, int lane) {
#pragma unroll
  for (int i0 = 0; i0 < ROWS * 2; i0 += 32) {
    int i = i0 + lane;
    if (i < ROWS * 2) tp_cp16(dst + i * 4, src + (i >> 1) * rstride + (i & 1) * 4);
  }
}

// Gamma_i for the warp's 8 channels: lane (ch, q) sums components [4q, 4q+4) -> Gs[b * 8 + ch]
template <class A>
__device__ __forceinline__ void t3_gamma(const A& a, int64_t e0, int64_t e1, int nn, int q, int ch, float* Gs) {
  const int lA = l_of(4 * q), lB = l_of(4 * q + 1);
  float g0 = 0.f, g1 = 0.f, g2 = 0.f, g3 = 0.f;
  for (int64_t e = e0; e < e1; e += 4) {
    float oa[4], ob[4];
    float4 y[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const int64_t ee = (e + i < e1) ? e + i : e1 - 1;
      oa[i] = a.om[ee * a.ldo + lA * a.n + nn];
      ob[i] = a.om[ee * a.ldo + lB * a.n + nn];
      y[i] = __ldg(reinterpret_cast<const float4*>(a.Y + ee * a.ldy + 4 * q));
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      if (e + i < e1) {
        g0 = fmaf(oa[i], y[i].x, g0); g1 = fmaf(ob[i], y[i].y, g1);
        g2 = fmaf(ob[i], y[i].z, g2); g3 = fmaf(ob[i], y[i].w, g3);
      }
    }
  }
  Gs[(4 * q + 0) * 8 + ch] = a.c_env * g0; Gs[(4 * q + 1) * 8 + ch] = a.c_env * g1;
  Gs[(4 * q + 2) * 8 + ch] = a.c_env * g2; Gs[(4 * q + 3) * 8 + ch] = a.c_env * g3;
  __syncwarp();
}

// ======================================================================================================
// forward:  lane (ch, q) computes T_e[c] for c in [q CB, (q+1) CB)
// ======================================================================================================
template <int P, bool FIRST, int NST, int WPB>
static __global__ void __launch_bounds__(WPB * 32) k_tp3_fwd(const __grid_constant__ TP2<Pat<P>::NNZ> a) {
  constexpr int DENV = Pat<P>::DENV, DIN = Pat<P>::DIN, DOUT = Pat<P>::DOUT;
  static_assert(DENV == 16, "lane-split kernels are written for l_max = 3");
  constexpr int CB = (((DOUT + 3) / 4) + 1) & ~1, CBH = CB / 2;   // output components per lane, even
  constexpr int SF = FIRST ? 4 * 8 + 16 : DIN * 8;                 // floats per ring stage (one edge)
  constexpr int WSL = DENV * 8 + NST * SF;
  extern __shared__ float4 smem4[];
  float* smem = reinterpret_cast<float*>(smem4);
  const int wib = threadIdx.x >> 5, lane = threadIdx.x & 31, ch = lane & 7, q = lane >> 3;
  const int ngroups = a.n / T3_CPW;
  const int64_t wg = (int64_t)blockIdx.x * WPB + wib;
  if (wg >= (int64_t)a.nc * ngroups) return;
  const int c = (int)(wg / ngroups), grp = (int)(wg - (int64_t)c * ngroups);
  const int nn = grp * T3_CPW + ch;
  float* Gs = smem + wib * WSL;
  float* ring = Gs + DENV * 8;
  const int64_t e0 = a.rowa[c], e1 = a.rowa[c + 1];
  const int deg = (int)(e1 - e0);
  if (deg <= 0) return;

  const float* opc = FIRST ? a.w0 + e0 * a.ldw + grp * T3_CPW : a.Vin + e0 * DIN * a.n + grp * T3_CPW;
  const int op_stride = FIRST ? a.ldw : DIN * a.n;
  const float* Yc = a.Y + e0 * a.ldy + lane * 4;
  auto issue = [&](int il, float* st) {
    if (FIRST) {
      t3_cp_rows<4>(st, opc + il * op_stride, a.n, lane);
      if (lane < 4) tp_cp16(st + 32 + lane * 4, Yc + il * a.ldy);
    } else {
      t3_cp_rows<DIN>(st, opc + il * op_stride, a.n, lane);
    }
  };
#pragma unroll
  for (int s = 0; s < NST - 1; ++s) {
    if (s < deg) issue(s, ring + s * SF);
    tp_cp_commit();
  }
  t3_gamma(a, e0, e1, nn, q, ch, Gs);
  if (a.gamma_out)
#pragma unroll
    for (int j = 0; j < 4; ++j) a.gamma_out[((size_t)c * DENV + 4 * q + j) * a.n + nn] = Gs[(4 * q + j) * 8 + ch];

  // block q of M_i: entries of block blk are FFMAs predicated on q == blk
  float2 Mr[DIN * CBH];
  {
    float G[DENV];
#pragma unroll
    for (int b = 0; b < DENV; ++b) G[b] = Gs[b * 8 + ch];
#pragma unroll
    for (int k = 0; k < DIN * CBH; ++k) Mr[k] = make_float2(0.f, 0.f);
#define X(k, a_, b_, c_) \
  if (q == (c_) / CB) TP2_REF(Mr, CBH, a_, (c_) % CB) = fmaf(a.kv[k], G[b_], TP2_REF(Mr, CBH, a_, (c_) % CB));
    TP2_EXPAND(P, X)
#undef X
  }
  const int cb = q * CB;
  float* xsp = a.xs + e0 * a.ldx + nn;
  float* Tp = a.Tout ? a.Tout + (e0 * DOUT + cb) * a.n + nn : nullptr;
  int slot = 0;
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
      float v = FIRST ? st[l_of(k) * 8 + ch] * st[32 + k] : st[k * 8 + ch];
      const float2 v2 = make_float2(v, v);
#pragma unroll
      for (int j = 0; j < CBH; ++j) acc[j] = tp_fma2(v2, Mr[k * CBH + j], acc[j]);
    }
    if (q == 0) *xsp = acc[0].x;
    xsp += a.ldx;
    if (Tp) {
#pragma unroll
      for (int cc = 0; cc < CB; ++cc)
        if (cb + cc < DOUT) Tp[cc * a.n] = (cc & 1) ? acc[cc >> 1].y : acc[cc >> 1].x;
      Tp += DOUT * a.n;
    }
    if (++slot == NST) slot = 0;
  }
}

// sum over the 8 channel lanes (xor 1, 2, 4): every lane of the q-group ends with the total
__device__ __forceinline__ float t3_sum_ch(float v) {
  v += __shfl_xor_sync(TP_FULLMASK, v, 1);
  v += __shfl_xor_sync(TP_FULLMASK, v, 2);
  v += __shfl_xor_sync(TP_FULLMASK, v, 4);
  return v;
}

// Per-l sums from the (first, rest) split of the four component groups: group q contributes xa to l(4q) and xb
// to l(4q+1), i.e. l=0: a(0); l=1: b(0); l=2: a(1)+b(1)+a(2); l=3: b(2)+a(3)+b(3).  Lane (ch, q) returns l = q.
__device__ __forceinline__ float t3_gather_l(float xa, float xb, int ch, int q) {
  float a0 = __shfl_sync(TP_FULLMASK, xa, ch), b0 = __shfl_sync(TP_FULLMASK, xb, ch);
  float a1 = __shfl_sync(TP_FULLMASK, xa, ch + 8), b1 = __shfl_sync(TP_FULLMASK, xb, ch + 8);
  float a2 = __shfl_sync(TP_FULLMASK, xa, ch + 16), b2 = __shfl_sync(TP_FULLMASK, xb, ch + 16);
  float a3 = __shfl_sync(TP_FULLMASK, xa, ch + 24), b3 = __shfl_sync(TP_FULLMASK, xb, ch + 24);
  return q == 0 ? a0 : q == 1 ? b0 : q == 2 ? (a1 + b1) + a2 : (b2 + a3) + b3;
}

// ======================================================================================================
// backward:  lane (ch, q) owns input components [q AB, (q+1) AB): V-bar rows, M / M-bar blocks
// ======================================================================================================
template <int P, bool FIRST, int NST, int WPB>
static __global__ void __launch_bounds__(WPB * 32) k_tp3_bwd(const __grid_constant__ TP2<Pat<P>::NNZ> a) {
  constexpr int DENV = Pat<P>::DENV, DIN = Pat<P>::DIN, DOUT = Pat<P>::DOUT;
  static_assert(DENV == 16, "lane-split kernels are written for l_max = 3");
  static_assert(!FIRST || DIN == 16, "FIRST: V^0 has the environment layout");
  constexpr int AB = (DIN + 3) / 4, CH = (DOUT + 1) / 2;
  constexpr int SV = FIRST ? 4 * 8 + 16 : DIN * 8;          // operand part of a stage
  constexpr int SF = SV + DOUT * 8 + 8;                      // + V-bar^L rows + s-bar row
  constexpr int MSL = AB * CH * 64;                          // M block, float2 per lane
  constexpr int WSL = DENV * 8 + MSL + NST * SF;
  extern __shared__ float4 smem4[];
  float* smem = reinterpret_cast<float*>(smem4);
  const int wib = threadIdx.x >> 5, lane = threadIdx.x & 31, ch = lane & 7, q = lane >> 3;
  const int ngroups = a.n / T3_CPW;
  const int64_t wg = (int64_t)blockIdx.x * WPB + wib;
  if (wg >= (int64_t)a.nc * ngroups) return;
  const int c = (int)(wg / ngroups), grp = (int)(wg - (int64_t)c * ngroups);
  const int nn = grp * T3_CPW + ch;
  float* Gs = smem + wib * WSL;
  float2* Ms = reinterpret_cast<float2*>(Gs + DENV * 8);
  float* ring = Gs + DENV * 8 + MSL;
  const int64_t e0 = a.rowa[c], e1 = a.rowa[c + 1];
  const int deg = (int)(e1 - e0);
  if (deg <= 0) return;
  float* Yb0 = a.Ybar + (size_t)(a.ybar_part0 + grp) * a.ybar_pstride;
  float* YbL = a.Ybar + (size_t)(a.ybar_partL + grp) * a.ybar_pstride;

  const float* opc = FIRST ? a.w0 + e0 * a.ldw + grp * T3_CPW : a.Vin + e0 * DIN * a.n + grp * T3_CPW;
  const int op_stride = FIRST ? a.ldw : DIN * a.n;
  const float* Yc = a.Y + e0 * a.ldy + lane * 4;
  const float* vbc = a.VbarL + e0 * DOUT * a.n + grp * T3_CPW;
  const float* sbc = a.sbar + e0 * a.lds + grp * T3_CPW + (lane & 1) * 4;
  auto issue = [&](int il, float* st) {
    if (FIRST) {
      t3_cp_rows<4>(st, opc + il * op_stride, a.n, lane);
      if (lane < 4) tp_cp16(st + 32 + lane * 4, Yc + il * a.ldy);
    } else {
      t3_cp_rows<DIN>(st, opc + il * op_stride, a.n, lane);
    }
    t3_cp_rows<DOUT>(st + SV, vbc + il * (DOUT * a.n), a.n, lane);
    if (lane < 2) tp_cp16(st + SF - 8 + lane * 4, sbc + il * a.lds);
  };
#pragma unroll
  for (int s = 0; s < NST - 1; ++s) {
    if (s < deg) issue(s, ring + s * SF);
    tp_cp_commit();
  }
  t3_gamma(a, e0, e1, nn, q, ch, Gs);

  // M block of this lane (rows q AB + r) -> the lane's shared slice, one row at a time
  {
    float G[DENV];
#pragma unroll
    for (int b = 0; b < DENV; ++b) G[b] = Gs[b * 8 + ch];
#pragma unroll
    for (int r = 0; r < AB; ++r) {
      float2 row[CH];
#pragma unroll
      for (int j = 0; j < CH; ++j) row[j] = make_float2(0.f, 0.f);
#define X(k, a_, b_, c_) \
  if ((a_) % AB == r) { if (q == (a_) / AB) TP2_REF(row, CH, 0, c_) = fmaf(a.kv[k], G[b_], TP2_REF(row, CH, 0, c_)); }
      TP2_EXPAND(P, X)
#undef X
#pragma unroll
      for (int j = 0; j < CH; ++j) Ms[(r * CH + j) * 32 + lane] = row[j];
    }
  }
  float2 Mb[AB * CH];
#pragma unroll
  for (int k = 0; k < AB * CH; ++k) Mb[k] = make_float2(0.f, 0.f);
  const int ab = q * AB;
  // FIRST: shared-memory offsets of w0[l(ab + k)] for this lane's components
  int wrow[AB];
#pragma unroll
  for (int k = 0; k < AB; ++k) wrow[k] = l_of((ab + k < DIN) ? ab + k : DIN - 1) * 8 + ch;
  float* yb0p = Yb0 + e0 * DENV + 4 * q;
  float* outp = FIRST ? a.w0bar + e0 * a.ldob + q * a.n + nn : a.Vbar_prev + (e0 * DIN + ab) * a.n + nn;
  int slot = 0;
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
    float2 t2[CH];
#pragma unroll
    for (int j = 0; j < CH; ++j) {
      t2[j].x = st[SV + (2 * j) * 8 + ch];
      t2[j].y = (2 * j + 1 < DOUT) ? st[SV + (2 * j + 1) * 8 + ch] : 0.f;
    }
    t2[0].x += st[SF - 8 + ch];
    float vb[AB], y[AB], wl[AB];
#pragma unroll
    for (int k = 0; k < AB; ++k) {
      const bool valid = ab + k < DIN;
      float v;
      if (FIRST) {
        y[k] = st[32 + ab + k];
        wl[k] = st[wrow[k]];
        v = wl[k] * y[k];
      } else {
        v = valid ? st[(ab + k) * 8 + ch] : 0.f;
      }
      const float2 v2 = make_float2(v, v);
      float2 s2 = make_float2(0.f, 0.f);
#pragma unroll
      for (int j = 0; j < CH; ++j) {
        const float2 m2 = Ms[(k * CH + j) * 32 + lane];
        s2 = tp_fma2(m2, t2[j], s2);
        Mb[k * CH + j] = tp_fma2(v2, t2[j], Mb[k * CH + j]);
      }
      vb[k] = s2.x + s2.y;
    }
    if (FIRST) {
      // w0-bar[l] = sum_{a in l} V-bar^0[a] Y[a];  Y-bar[a] (V^0 part) = sum_n w0[l(a)] V-bar^0[a]   (AB == 4)
      const float xa = vb[0] * y[0], xb = fmaf(vb[1], y[1], fmaf(vb[2], y[2], vb[3] * y[3]));
      *outp = t3_gather_l(xa, xb, ch, q);
      outp += a.ldob;
      float4 p4 = make_float4(t3_sum_ch(wl[0] * vb[0]), t3_sum_ch(wl[1] * vb[1]), t3_sum_ch(wl[2] * vb[2]), t3_sum_ch(wl[3] * vb[3]));
      if (ch == 0) *reinterpret_cast<float4*>(yb0p) = p4;
      yb0p += DENV;
    } else {
#pragma unroll
      for (int k = 0; k < AB; ++k)
        if (ab + k < DIN) outp[k * a.n] = vb[k];
      outp += DIN * a.n;
    }
    if (++slot == NST) slot = 0;
  }
  // Gamma-bar = K . M-bar: this lane's block, then the sum over the four blocks of the channel
  float Gb[DENV];
#pragma unroll
  for (int b = 0; b < DENV; ++b) Gb[b] = 0.f;
#define X(k, a_, b_, c_) \
  if (q == (a_) / AB) Gb[b_] = fmaf(a.kv[k], TP2_REF(Mb, CH, (a_) % AB, c_), Gb[b_]);
  TP2_EXPAND(P, X)
#undef X
#pragma unroll
  for (int b = 0; b < DENV; ++b) {
    Gb[b] += __shfl_xor_sync(TP_FULLMASK, Gb[b], 8);
    Gb[b] += __shfl_xor_sync(TP_FULLMASK, Gb[b], 16);
  }
  // pass 2: lane (ch, q) takes environment components [4q, 4q+4): omega-bar_e[l], Y-bar_e[b] (environment part)
  float gq[4];
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    float v = Gb[j];
#pragma unroll
    for (int qq = 1; qq < 4; ++qq) v = (q == qq) ? Gb[4 * qq + j] : v;
    gq[j] = a.c_env * v;
  }
  const int lA = l_of(4 * q), lB = l_of(4 * q + 1);
  for (int64_t e = e0; e < e1; e += 2) {
    float oa[2], ob[2];
    float4 y[2];
#pragma unroll
    for (int i = 0; i < 2; ++i) {
      const int64_t ee = (e + i < e1) ? e + i : e1 - 1;
      oa[i] = a.om[ee * a.ldo + lA * a.n + nn];
      ob[i] = a.om[ee * a.ldo + lB * a.n + nn];
      y[i] = __ldg(reinterpret_cast<const float4*>(a.Y + ee * a.ldy + 4 * q));
    }
#pragma unroll
    for (int i = 0; i < 2; ++i) {
      if (e + i < e1) {   // (warp-uniform)
        const float xa = gq[0] * y[i].x, xb = fmaf(gq[1], y[i].y, fmaf(gq[2], y[i].z, gq[3] * y[i].w));
        a.ombar[(e + i) * a.ldob + q * a.n + nn] = t3_gather_l(xa, xb, ch, q);
        float4 p4 = make_float4(t3_sum_ch(oa[i] * gq[0]), t3_sum_ch(ob[i] * gq[1]), t3_sum_ch(ob[i] * gq[2]), t3_sum_ch(ob[i] * gq[3]));
        if (ch == 0) *reinterpret_cast<float4*>(YbL + (e + i) * DENV + 4 * q) = p4;
      }
    }
  }
}

// ---- host side ---------------------------------------------------------------------------------------------
template <int P, bool FIRST, int NST, int WPB>
int launch_fwd3(allegro_model* m, const TP2<Pat<P>::NNZ>& a) {
  constexpr int DIN = Pat<P>::DIN;
  constexpr int SF = FIRST ? 4 * 8 + 16 : DIN * 8;
  constexpr int WSL = 16 * 8 + NST * SF;
  size_t sm = (size_t)WPB * WSL * 4 + 16;
  static bool set = false;
  if (!set) { AL_CUDA(m, cudaFuncSetAttribute(k_tp3_fwd<P, FIRST, NST, WPB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm)); set = true; }
  int64_t warps = (int64_t)a.nc * (a.n / T3_CPW);
  k_tp3_fwd<P, FIRST, NST, WPB><<<(unsigned)((warps + WPB - 1) / WPB), WPB * 32, sm, m->stream>>>(a);
  m->launches++;
  AL_CUDA(m, cudaGetLastError());
  return ALLEGRO_OK;
}

template <int P, bool FIRST, int NST, int WPB>
int launch_bwd3(allegro_model* m, const TP2<Pat<P>::NNZ>& a) {
  constexpr int DIN = Pat<P>::DIN, DOUT = Pat<P>::DOUT;
  constexpr int AB = (DIN + 3) / 4, CH = (DOUT + 1) / 2;
  constexpr int SV = FIRST ? 4 * 8 + 16 : DIN * 8;
  constexpr int SF = SV + DOUT * 8 + 8;
  constexpr int WSL = 16 * 8 + AB * CH * 64 + NST * SF;
  size_t sm = (size_t)WPB * WSL * 4 + 16;
  static bool set = false;
  if (!set) { AL_CUDA(m, cudaFuncSetAttribute(k_tp3_bwd<P, FIRST, NST, WPB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm)); set = true; }
  int64_t warps = (int64_t)a.nc * (a.n / T3_CPW);
  k_tp3_bwd<P, FIRST, NST, WPB><<<(unsigned)((warps + WPB - 1) / WPB), WPB * 32, sm, m->stream>>>(a);
  m->launches++;
  AL_CUDA(m, cudaGetLastError());
  return ALLEGRO_OK;
}
