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

constexpr int T3_CPW = 8;      // channels per warp of the forward kernels (4 blocks)
// The l_max = 3 backward in TF32 mode runs on the tensor cores (tp3mb_impl.cuh: 8-channel teams, so the Y-bar partial
// buffers of those layers are per 8-channel group); the fp32 modes keep the blocked 32-channel kernel of tp2_impl.cuh.
inline bool tp3m_bwd_active(const allegro_model* m) { return m->hp.precision == 1; }

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
  int64_t wg = (int64_t)blockIdx.x * WPB + wib;
  if (wg >= (int64_t)a.nc * ngroups) return;
  if (a.rev) wg = (int64_t)a.nc * ngroups - 1 - wg;
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

// ======================================================================================================
// helpers of the lane-split backward passes (lane = (channel ch, component group q)); used by tp3mb_impl.cuh
// ======================================================================================================
template <int CPW>
__device__ __forceinline__ float t3_sum_ch(float v) {   // sum over the CPW channel lanes of a block
#pragma unroll
  for (int o = 1; o < CPW; o <<= 1) v += __shfl_xor_sync(TP_FULLMASK, v, o);
  return v;
}
// xa belongs to l = lA, xb to l = lB (of this lane's environment components); returns, in the lane with q = l,
// the sum over the blocks of everything that belongs to l (fixed order: xor tree over the block bits)
template <int CPW>
__device__ __forceinline__ float t3_gather_l(float xa, float xb, int lA, int lB, int q) {
  float c[4];
#pragma unroll
  for (int l = 0; l < 4; ++l) c[l] = ((lA == l) ? xa : 0.f) + ((lB == l) ? xb : 0.f);
#pragma unroll
  for (int o = CPW; o < 32; o <<= 1)
#pragma unroll
    for (int l = 0; l < 4; ++l) c[l] += __shfl_xor_sync(TP_FULLMASK, c[l], o);
  return q == 0 ? c[0] : q == 1 ? c[1] : q == 2 ? c[2] : c[3];
}

// rows of CPW floats: smem dst row r at dst + CPW r
template <int ROWS, int CPW>
__device__ __forceinline__ void t3_cp_rows_w(float* dst, const float* src, int rstride, int lane) {
  constexpr int CPR = CPW / 4;   // 16-byte chunks per row
#pragma unroll
  for (int i0 = 0; i0 < ROWS * CPR; i0 += 32) {
    int i = i0 + lane;
    if (i < ROWS * CPR) tp_cp16(dst + i * 4, src + (i / CPR) * rstride + (i % CPR) * 4);
  }
}

// ---- host side ---------------------------------------------------------------------------------------------
template <int P, bool FIRST, int NST, int WPB>
int launch_fwd3(allegro_model* m, const TP2<Pat<P>::NNZ>& a) {
  constexpr int DIN = Pat<P>::DIN;
  constexpr int SF = FIRST ? 4 * 8 + 16 : DIN * 8;
  constexpr int WSL = 16 * 8 + NST * SF;
  size_t sm = (size_t)WPB * WSL * 4 + 16;
  static AttrOnce once;
  if (once.need(m->device)) { AL_CUDA(m, cudaFuncSetAttribute(k_tp3_fwd<P, FIRST, NST, WPB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm)); once.done(m->device); }
  int64_t warps = (int64_t)a.nc * (a.n / T3_CPW);
  k_tp3_fwd<P, FIRST, NST, WPB><<<(unsigned)((warps + WPB - 1) / WPB), WPB * 32, sm, m->stream>>>(a);
  m->launches++;
  AL_CUDA(m, cudaGetLastError());
  return ALLEGRO_OK;
}
