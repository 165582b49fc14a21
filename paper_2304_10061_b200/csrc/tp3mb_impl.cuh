// NEXT-2, backward half: the l_max = 3 tensor product on the tensor cores, TF32 mode.
//
// The paper runs the tensor product as dense TF32 matmuls (Fig. 3 :180).  With the environment folded
// into the per-(centre, channel) matrix M_i[n] = K . Gamma_i[n] (Eq. (2) line 2: sum before product) the backward of one
// layer is, per centre i and channel n, two small dense products over the centre's edges e:
//     V-bar^{L-1}[e, a] = sum_c M[a, c] T-bar[e, c]          (1)   T-bar = V-bar^L, plus s-bar at the scalar slot c = 0
//     M-bar[a, c]       = sum_e V[e, a] T-bar[e, c]          (2)   then Gamma-bar[b] = sum_{a,c} K[a,b,c] M-bar[a, c]
// Both run here as warp-level mma.sync.m16n8k8 (TF32 operands, fp32 accumulate); the B operand of (1) and the A operand
// of (2) differ per channel, which rules out tcgen05 (one B per 128-row tile), as in the forward (tp3m_impl.cuh).
//   (1) as  V-bar^T[a, e] = M[a, c] . T-bar^T[c, e]:  A = M (16 x 8 tiles, parked in shared memory in A-FRAGMENT order, one
//       LDS.128 per MMA), B[k = c][n = e] = T-bar[e][c], N = 8 edges;
//   (2) as  M-bar[a, c] += V^T[a, e] . T-bar[e, c]:   A[row = a][col = e] = V[e][a], B[k = e][n = c] = T-bar[e][c], K = 8 edges,
//       accumulators (16 x 32 or 32 x 16 per channel) live in registers for the whole centre.
// T-bar is the contraction-side operand of (1) and the free-side operand of (2): the two fragment layouts are transposes
// of each other.  So the centre's edges go through shared memory in TILES OF 8 EDGES -- one cp.async pass global ->
// shared (every byte of V, T-bar, s-bar, w0, Y is read from HBM exactly once), double-buffered -- and both fragment
// layouts are read from the tile with conflict-free LDS.128 (16-byte chunk = 4 channels of one (edge, component); chunk
// position XOR-swizzled by the edge row, see t3b_chunk).
// A TEAM of two warps owns (centre, 8 channels): both stage the tile, warp w computes channels [4w, 4w + 4) -- 64
// M-bar accumulator registers per lane instead of 128.  One block = one team (64 threads, __syncthreads as team barrier).
// M_i and Gamma-bar use the same compile-time sparsity pattern of K as every other tensor-track kernel (tp2_patterns.inc).
// FIRST (V^0 = w^0 (x) Y formed on the fly): V-bar^0 goes through a shared tile to the w0-bar / Y-bar reductions.
// Pass 2 (omega-bar, environment part of Y-bar) is the lane-split code of k_tp3_bwd with 8 channels x 4 groups per warp.
#pragma once
#include "tp3m_impl.cuh"

// position (in floats) of the 16-byte chunk (edge row e, component comp) inside a half tile [8 edges][DP components][4 ch];
// the chunk index is XOR-ed with s(e) = 4 (e & 1) + (e & 2): conflict-free for the lane patterns (e = g, comp = t [+4])
// of product (1) and (e = t [+4], comp = g [+8]) of product (2)
template <int DP>
__device__ __forceinline__ int t3b_chunk(int e, int comp) { return (e * DP + (comp ^ (((e & 1) << 2) | (e & 2)))) << 2; }

__device__ __forceinline__ void t3b_st128(float* p, const float4& v) {
  asm volatile("st.global.L1::no_allocate.v4.f32 [%0], {%1,%2,%3,%4};" ::"l"(p), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}

template <int P, bool FIRST>
static __global__ void __launch_bounds__(64) k_tp3m_bwd(const __grid_constant__ TP2<Pat<P>::NNZ> a) {
  constexpr int DENV = Pat<P>::DENV, DIN = Pat<P>::DIN, DOUT = Pat<P>::DOUT;
  static_assert(DENV == 16, "written for l_max = 3");
  static_assert(!FIRST || DIN == 16, "FIRST: V^0 has the environment layout");
  constexpr int DINP = (DIN + 15) & ~15, DOUTP = (DOUT + 7) & ~7;
  constexpr int MT = DINP / 16, KS = DOUTP / 8;            // 16-row tiles over a, 8-wide steps / tiles over c
  static_assert(DINP * DOUTP == 512, "M of one channel: 16 x 32 or 32 x 16");
  constexpr int VDP = FIRST ? 4 : DINP;                    // staged operand rows per edge (FIRST: the four w0 rows)
  constexpr int T_FL = 2 * 8 * DOUTP * 4, V_FL = 2 * 8 * VDP * 4, Y_FL = FIRST ? 8 * 16 : 0, S_FL = 2 * 8 * 4;
  constexpr int ST_FL = T_FL + V_FL + Y_FL + S_FL;         // floats of one stage
  constexpr int MF_FL = 8 * 513;                           // M (A-fragment order, 8 x 512); later M-bar [ch][a][c], channel stride 513
  constexpr int VB_FL = FIRST ? 2 * 8 * 16 * 4 : 0;        // FIRST: V-bar^0 of the tile, [half][edge][a][4]
  constexpr int CB8 = DOUTP / 8;                           // M build: output columns per thread (8 column groups)
  extern __shared__ float4 smem4[];
  float* Gs = reinterpret_cast<float*>(smem4);             // Gamma_i [16][8]
  float* Mf = Gs + 128;
  float* Gbs = Mf + MF_FL;                                 // Gamma-bar partials of the two warps [2][16][8]
  float* stg = Gbs + 256;                                  // two stages
  float* Vb0 = stg + 2 * ST_FL;

  const int tid = threadIdx.x, w = tid >> 5, lane = tid & 31, g = lane >> 2, t = lane & 3;
  const int ch8 = tid & 7, q8 = tid >> 3;
  const int ngroups = a.n / 8;
  int64_t wg = blockIdx.x;
  if (a.rev) wg = (int64_t)a.nc * ngroups - 1 - wg;
  const int c = (int)(wg / ngroups), grp = (int)(wg - (int64_t)c * ngroups);
  const int n0 = grp * 8;
  const int64_t e0 = a.rowa[c], e1 = a.rowa[c + 1];
  const int deg = (int)(e1 - e0);
  if (deg <= 0) return;
  const int ntiles = (deg + 7) >> 3;

  // ---- stage one tile of 8 edges: T-bar [half][e][c][4], V [half][e][a][4] (FIRST: w0 [half][e][l][4] and Y [e][16]), s-bar
  auto issue = [&](int tile, float* st) {
    const int64_t eb = e0 + (int64_t)tile * 8;
    const float4 z4 = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll 4
    for (int i = tid; i < 8 * DOUTP * 2; i += 64) {
      const int half = i & 1, comp = (i >> 1) & (DOUTP - 1), e = (i >> 1) / DOUTP;
      float* dst = st + half * (8 * DOUTP * 4) + t3b_chunk<DOUTP>(e, comp);
      if (eb + e < e1 && comp < DOUT) tp_cp16(dst, a.VbarL + ((eb + e) * DOUT + comp) * a.n + n0 + 4 * half);
      else *reinterpret_cast<float4*>(dst) = z4;
    }
    float* sv = st + T_FL;
    if (FIRST) {
      {
        const int i = tid;                                  // 8 edges x 4 l x 2 halves = 64 chunks
        const int half = i & 1, l = (i >> 1) & 3, e = i >> 3;
        float* dst = sv + half * (8 * 4 * 4) + (e * 4 + l) * 4;
        if (eb + e < e1) tp_cp16(dst, a.w0 + (eb + e) * a.ldw + l * a.n + n0 + 4 * half);
        else *reinterpret_cast<float4*>(dst) = z4;
      }
      if (tid < 32) {
        const int e = tid >> 2, j = tid & 3;
        float* dst = sv + V_FL + e * 16 + j * 4;
        if (eb + e < e1) tp_cp16(dst, a.Y + (eb + e) * a.ldy + j * 4);
        else *reinterpret_cast<float4*>(dst) = z4;
      }
    } else {
#pragma unroll 4
      for (int i = tid; i < 8 * DINP * 2; i += 64) {
        const int half = i & 1, comp = (i >> 1) & (DINP - 1), e = (i >> 1) / DINP;
        float* dst = sv + half * (8 * DINP * 4) + t3b_chunk<DINP>(e, comp);
        if (eb + e < e1 && comp < DIN) tp_cp16(dst, a.Vin + ((eb + e) * DIN + comp) * a.n + n0 + 4 * half);
        else *reinterpret_cast<float4*>(dst) = z4;
      }
    }
    if (tid < 16) {
      const int half = tid & 1, e = tid >> 1;
      float* dst = sv + V_FL + Y_FL + half * 32 + e * 4;
      if (eb + e < e1) tp_cp16(dst, a.sbar + (eb + e) * a.lds + n0 + 4 * half);
      else *reinterpret_cast<float4*>(dst) = z4;
    }
  };
  issue(0, stg);
  tp_cp_commit();

  // ---- Gamma_i (k_tp3m_gamma) and M_i of the team's 8 channels, M parked in A-fragment order --------------------------
  for (int i = tid; i < MF_FL / 4; i += 64) reinterpret_cast<float4*>(Mf)[i] = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
  for (int i = 0; i < 2; ++i) {
    const int b = q8 * 2 + i;
    Gs[b * 8 + ch8] = a.gamma_out[((size_t)c * DENV + b) * a.n + n0 + ch8];
  }
  __syncthreads();
  {
    float Mr[DIN * CB8];
    float G[DENV];
#pragma unroll
    for (int b = 0; b < DENV; ++b) G[b] = Gs[b * 8 + ch8];
#pragma unroll
    for (int k = 0; k < DIN * CB8; ++k) Mr[k] = 0.f;
#define X(k, a_, b_, c_) \
  if (q8 == (c_) / CB8) Mr[(a_) * CB8 + (c_) % CB8] = fmaf(a.kv[k], G[b_], Mr[(a_) * CB8 + (c_) % CB8]);
    TP2_EXPAND(P, X)
#undef X
    // A fragment of (m, k): lane L = (row & 7) * 4 + (col & 3), register (row >> 3) + 2 * (col >> 2), row = a & 15, col = c & 7
#pragma unroll
    for (int aa = 0; aa < DIN; ++aa) {
      const int m = aa >> 4, r = aa & 15;
#pragma unroll
      for (int cc = 0; cc < CB8; ++cc) {
        const int co = q8 * CB8 + cc;
        if (co < DOUT) {
          const int k = co >> 3, cl = co & 7;
          Mf[(((ch8 * MT + m) * KS + k) * 32 + (r & 7) * 4 + (cl & 3)) * 4 + (r >> 3) + 2 * (cl >> 2)] =
              __uint_as_float(t3m_tf32(Mr[aa * CB8 + cc]));
        }
      }
    }
  }

  // ---- the centre's edges, 8 at a time ------------------------------------------------------------------------------------
  float Mb[MT][KS][4][4];                                  // M-bar accumulators of this warp's 4 channels
#pragma unroll
  for (int m = 0; m < MT; ++m)
#pragma unroll
    for (int j = 0; j < KS; ++j)
#pragma unroll
      for (int cq = 0; cq < 4; ++cq) { Mb[m][j][cq][0] = 0.f; Mb[m][j][cq][1] = 0.f; Mb[m][j][cq][2] = 0.f; Mb[m][j][cq][3] = 0.f; }
  float* Yb0 = a.Ybar + (size_t)(a.ybar_part0 + grp) * a.ybar_pstride;
  float* YbL = a.Ybar + (size_t)(a.ybar_partL + grp) * a.ybar_pstride;

  for (int tile = 0; tile < ntiles; ++tile) {
    float* st = stg + (tile & 1) * ST_FL;
    tp_cp_wait<0>();
    __syncthreads();                                       // tile landed (and M_i built, first round); the other stage is free
    if (tile + 1 < ntiles) issue(tile + 1, stg + ((tile + 1) & 1) * ST_FL);
    tp_cp_commit();
    const float* Th = st + w * (8 * DOUTP * 4);
    const float* sv = st + T_FL;
    const float* Sh = sv + V_FL + Y_FL + w * 32;
    const int64_t eb = e0 + (int64_t)tile * 8;

    // (1) V-bar^T[a, e] = sum_c M[a, c] T-bar[e, c]: D1[m][ch] holds (a = 16m + g [+8], e = 2t [+1])
    float D1[MT][4][4];
    {
      uint32_t B0[KS][4], B1[KS][4];
#pragma unroll
      for (int k = 0; k < KS; ++k) {
        float4 x0 = *reinterpret_cast<const float4*>(Th + t3b_chunk<DOUTP>(g, 8 * k + t));
        const float4 x1 = *reinterpret_cast<const float4*>(Th + t3b_chunk<DOUTP>(g, 8 * k + t + 4));
        if (k == 0 && t == 0) {                            // s-bar enters at the scalar slot c = 0
          const float4 s = *reinterpret_cast<const float4*>(Sh + g * 4);
          x0.x += s.x; x0.y += s.y; x0.z += s.z; x0.w += s.w;
        }
        B0[k][0] = t3m_tf32(x0.x); B0[k][1] = t3m_tf32(x0.y); B0[k][2] = t3m_tf32(x0.z); B0[k][3] = t3m_tf32(x0.w);
        B1[k][0] = t3m_tf32(x1.x); B1[k][1] = t3m_tf32(x1.y); B1[k][2] = t3m_tf32(x1.z); B1[k][3] = t3m_tf32(x1.w);
      }
#pragma unroll
      for (int m = 0; m < MT; ++m)
#pragma unroll
        for (int cq = 0; cq < 4; ++cq) {
          D1[m][cq][0] = 0.f; D1[m][cq][1] = 0.f; D1[m][cq][2] = 0.f; D1[m][cq][3] = 0.f;
#pragma unroll
          for (int k = 0; k < KS; ++k) {
            const float4 af = *reinterpret_cast<const float4*>(Mf + ((((4 * w + cq) * MT + m) * KS + k) * 32 + lane) * 4);
            t3m_mma(D1[m][cq], __float_as_uint(af.x), __float_as_uint(af.y), __float_as_uint(af.z), __float_as_uint(af.w),
                    B0[k][cq], B1[k][cq]);
          }
        }
    }
    if (!FIRST) {
#pragma unroll
      for (int m = 0; m < MT; ++m)
#pragma unroll
        for (int rs = 0; rs < 2; ++rs)
#pragma unroll
          for (int cs = 0; cs < 2; ++cs) {
            const int aa = 16 * m + g + 8 * rs;
            const int64_t ee = eb + 2 * t + cs;
            if (aa < DIN && ee < e1)
              t3b_st128(a.Vbar_prev + (ee * DIN + aa) * a.n + n0 + 4 * w,
                        make_float4(D1[m][0][rs * 2 + cs], D1[m][1][rs * 2 + cs], D1[m][2][rs * 2 + cs], D1[m][3][rs * 2 + cs]));
          }
    } else {
      // V-bar^0 of the tile -> shared, then w0-bar[e, l] = sum_{a in l} V-bar^0[e, a] Y[e, a] and the V^0 part of
      // Y-bar[e, a] = sum_n w0[e, l(a), n] V-bar^0[e, a, n], thread = (edge, group of 4 components, channel half)
#pragma unroll
      for (int rs = 0; rs < 2; ++rs)
#pragma unroll
        for (int cs = 0; cs < 2; ++cs)
          *reinterpret_cast<float4*>(Vb0 + ((w * 8 + 2 * t + cs) * 16 + g + 8 * rs) * 4) =
              make_float4(D1[0][0][rs * 2 + cs], D1[0][1][rs * 2 + cs], D1[0][2][rs * 2 + cs], D1[0][3][rs * 2 + cs]);
      __syncthreads();
      {
        const int e = tid >> 3, q = (tid >> 1) & 3, h = tid & 1;
        const int lA = l_of(4 * q), lB = l_of(4 * q + 1);
        const bool valid = eb + e < e1;
        const float* w0h = sv + h * (8 * 4 * 4);
        const float4 wA = *reinterpret_cast<const float4*>(w0h + (e * 4 + lA) * 4);
        const float4 wB = *reinterpret_cast<const float4*>(w0h + (e * 4 + lB) * 4);
        const float4 y4 = *reinterpret_cast<const float4*>(sv + V_FL + e * 16 + 4 * q);
        const float yv[4] = {y4.x, y4.y, y4.z, y4.w};
        float xa[4], xb[4] = {0.f, 0.f, 0.f, 0.f}, pj[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          const float4 v = *reinterpret_cast<const float4*>(Vb0 + ((h * 8 + e) * 16 + 4 * q + k) * 4);
          const float4 wl = (k == 0) ? wA : wB;
          pj[k] = wl.x * v.x + wl.y * v.y + wl.z * v.z + wl.w * v.w;
          if (k == 0) { xa[0] = v.x * yv[0]; xa[1] = v.y * yv[0]; xa[2] = v.z * yv[0]; xa[3] = v.w * yv[0]; }
          else { xb[0] = fmaf(v.x, yv[k], xb[0]); xb[1] = fmaf(v.y, yv[k], xb[1]); xb[2] = fmaf(v.z, yv[k], xb[2]); xb[3] = fmaf(v.w, yv[k], xb[3]); }
        }
#pragma unroll
        for (int k = 0; k < 4; ++k) pj[k] += __shfl_xor_sync(TP_FULLMASK, pj[k], 1);      // the two channel halves
        if (valid && h == 0)
          *reinterpret_cast<float4*>(Yb0 + (eb + e) * DENV + 4 * q) = make_float4(pj[0], pj[1], pj[2], pj[3]);
        float o[4];
#pragma unroll
        for (int cq = 0; cq < 4; ++cq) {
          float cl[4];
#pragma unroll
          for (int l = 0; l < 4; ++l) cl[l] = ((lA == l) ? xa[cq] : 0.f) + ((lB == l) ? xb[cq] : 0.f);
#pragma unroll
          for (int off = 2; off <= 4; off <<= 1)
#pragma unroll
            for (int l = 0; l < 4; ++l) cl[l] += __shfl_xor_sync(TP_FULLMASK, cl[l], off);   // over the 4 component groups
          o[cq] = q == 0 ? cl[0] : q == 1 ? cl[1] : q == 2 ? cl[2] : cl[3];
        }
        if (valid) t3b_st128(a.w0bar + (eb + e) * a.ldob + q * a.n + n0 + 4 * h, make_float4(o[0], o[1], o[2], o[3]));
      }
    }

    // (2) M-bar[a, c] += sum_{e in tile} V[e, a] T-bar[e, c]
    {
      uint32_t A[MT][4][4];                                // [m][a0..a3][channel]
#pragma unroll
      for (int m = 0; m < MT; ++m)
#pragma unroll
        for (int r = 0; r < 4; ++r) {
          const int ee = t + 4 * (r >> 1), aa = 16 * m + g + 8 * (r & 1);
          float4 v;
          if (FIRST) {
            const float y = sv[V_FL + ee * 16 + aa];
            const float4 wv = *reinterpret_cast<const float4*>(sv + w * (8 * 4 * 4) + (ee * 4 + l_of(aa)) * 4);
            v = make_float4(wv.x * y, wv.y * y, wv.z * y, wv.w * y);
          } else {
            v = *reinterpret_cast<const float4*>(sv + w * (8 * DINP * 4) + t3b_chunk<DINP>(ee, aa));
          }
          A[m][r][0] = t3m_tf32(v.x); A[m][r][1] = t3m_tf32(v.y); A[m][r][2] = t3m_tf32(v.z); A[m][r][3] = t3m_tf32(v.w);
        }
#pragma unroll
      for (int j = 0; j < KS; ++j) {
        float4 x0 = *reinterpret_cast<const float4*>(Th + t3b_chunk<DOUTP>(t, 8 * j + g));
        float4 x1 = *reinterpret_cast<const float4*>(Th + t3b_chunk<DOUTP>(t + 4, 8 * j + g));
        if (j == 0 && g == 0) {
          const float4 s0 = *reinterpret_cast<const float4*>(Sh + t * 4), s1 = *reinterpret_cast<const float4*>(Sh + (t + 4) * 4);
          x0.x += s0.x; x0.y += s0.y; x0.z += s0.z; x0.w += s0.w;
          x1.x += s1.x; x1.y += s1.y; x1.z += s1.z; x1.w += s1.w;
        }
        const uint32_t b0[4] = {t3m_tf32(x0.x), t3m_tf32(x0.y), t3m_tf32(x0.z), t3m_tf32(x0.w)};
        const uint32_t b1[4] = {t3m_tf32(x1.x), t3m_tf32(x1.y), t3m_tf32(x1.z), t3m_tf32(x1.w)};
#pragma unroll
        for (int m = 0; m < MT; ++m)
#pragma unroll
          for (int cq = 0; cq < 4; ++cq)
            t3m_mma(Mb[m][j][cq], A[m][0][cq], A[m][1][cq], A[m][2][cq], A[m][3][cq], b0[cq], b1[cq]);
      }
    }
  }

  // ---- Gamma-bar = K . M-bar: accumulators -> shared [ch][a][c] (channel stride 513), pattern entries split by a & 7 ----
  __syncthreads();                                         // every read of M_i is done: the region is re-used for M-bar
#pragma unroll
  for (int m = 0; m < MT; ++m)
#pragma unroll
    for (int j = 0; j < KS; ++j)
#pragma unroll
      for (int cq = 0; cq < 4; ++cq) {
        float* p = Mf + (4 * w + cq) * 513 + (16 * m + g) * DOUTP + 8 * j + 2 * t;
        p[0] = Mb[m][j][cq][0]; p[1] = Mb[m][j][cq][1];
        p[8 * DOUTP] = Mb[m][j][cq][2]; p[8 * DOUTP + 1] = Mb[m][j][cq][3];
      }
  __syncthreads();
  {
    float Gb[DENV];
#pragma unroll
    for (int b = 0; b < DENV; ++b) Gb[b] = 0.f;
    const float* Mc = Mf + ch8 * 513;
#define X(k, a_, b_, c_) \
  if (q8 == ((a_) & 7)) Gb[b_] = fmaf(a.kv[k], Mc[(a_) * DOUTP + (c_)], Gb[b_]);
    TP2_EXPAND(P, X)
#undef X
#pragma unroll
    for (int b = 0; b < DENV; ++b) {
      Gb[b] += __shfl_xor_sync(TP_FULLMASK, Gb[b], 8);
      Gb[b] += __shfl_xor_sync(TP_FULLMASK, Gb[b], 16);
    }
    if (lane < 8)
#pragma unroll
      for (int b = 0; b < DENV; ++b) Gbs[w * 128 + b * 8 + lane] = Gb[b];
  }
  __syncthreads();

  // ---- pass 2: omega-bar_e[l] = c_env sum_{m in l} Gamma-bar[(l,m)] Y_e[(l,m)];  Y-bar_e[b] (environment part) =
  //      c_env sum_n omega_e[l(b)] Gamma-bar[b]; lane (ch, q) takes components [4q, 4q + 4), the warps alternate edge pairs
  {
    const int ch = lane & 7, q = lane >> 3, nn = n0 + ch;
    const int lA = l_of(4 * q), lB = l_of(4 * q + 1);
    float gq[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) gq[j] = a.c_env * (Gbs[(4 * q + j) * 8 + ch] + Gbs[128 + (4 * q + j) * 8 + ch]);
    for (int64_t e = e0 + 2 * w; e < e1; e += 4) {
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
        if (e + i < e1) {                                  // (warp-uniform)
          const float xa = gq[0] * y[i].x, xb = fmaf(gq[1], y[i].y, fmaf(gq[2], y[i].z, gq[3] * y[i].w));
          const float osum = t3_gather_l<8>(xa, xb, lA, lB, q);
          a.ombar[(e + i) * a.ldob + q * a.n + nn] = osum;
          float pj[4];
          pj[0] = t3_sum_ch<8>(oa[i] * gq[0]);
#pragma unroll
          for (int j = 1; j < 4; ++j) pj[j] = t3_sum_ch<8>(ob[i] * gq[j]);
          if (ch == 0) *reinterpret_cast<float4*>(YbL + (e + i) * DENV + 4 * q) = make_float4(pj[0], pj[1], pj[2], pj[3]);
        }
      }
    }
  }
}

template <int P, bool FIRST>
int launch_bwd3m(allegro_model* m, const TP2<Pat<P>::NNZ>& a) {
  constexpr int DIN = Pat<P>::DIN, DOUT = Pat<P>::DOUT;
  constexpr int DINP = (DIN + 15) & ~15, DOUTP = (DOUT + 7) & ~7, VDP = FIRST ? 4 : DINP;
  constexpr int ST_FL = 2 * 8 * DOUTP * 4 + 2 * 8 * VDP * 4 + (FIRST ? 8 * 16 : 0) + 2 * 8 * 4;
  constexpr int TEAM_FL = 128 + 8 * 513 + 256 + 2 * ST_FL + (FIRST ? 2 * 8 * 16 * 4 : 0);
  const size_t sm = (size_t)TEAM_FL * 4;
  static AttrOnce once;
  if (once.need(m->device)) { AL_CUDA(m, cudaFuncSetAttribute(k_tp3m_bwd<P, FIRST>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm)); once.done(m->device); }
  {
    int64_t gw = (int64_t)a.nc * (a.n / 32);
    k_tp3m_gamma<P, 8><<<(unsigned)((gw + 7) / 8), 256, 0, m->stream>>>(a);
    m->launches++;
  }
  const int64_t teams = (int64_t)a.nc * (a.n / 8);
  k_tp3m_bwd<P, FIRST><<<(unsigned)teams, 64, sm, m->stream>>>(a);
  m->launches++;
  AL_CUDA(m, cudaGetLastError());
  return ALLEGRO_OK;
}
