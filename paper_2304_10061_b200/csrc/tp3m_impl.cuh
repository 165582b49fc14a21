// NEXT-2: the l_max = 3 tensor product on the tensor cores, forward pass, TF32 mode.
//
// The paper runs the tensor product as dense TF32 matmuls.  Here the environment is folded into the
// per-(centre, channel) matrix first (M_i[n] = K . Gamma_i[n], sum before product, Eq. (2) line 2), which leaves, per
// centre and channel, the small dense product  T[e, c] = sum_a V[e, a] M_i[n][a, c]  over the centre's edges: M = deg,
// K = D_in (16 / 31), N = D_out (31 / 16).  The B operand changes with the channel, so this is warp-level
// mma.sync.m16n8k8 (TF32, fp32 accumulate), not tcgen05: a warp owns (centre, 8 channels);
//   * M_i of the 8 channels is built once per centre by the lanes (channel = lane & 7, block q = lane >> 3) exactly as in
//     k_tp3_fwd and parked in shared memory in B-FRAGMENT ORDER (one conflict-free LDS.64 per MMA), rounded to TF32;
//   * with the channel-fastest layout [edge][component][channel] the A-fragment element (row = edge, col = component) of
//     the 8 per-channel MMAs is one 32-byte sector V[e][a][n0..n0+7]: every lane loads whole sectors, no staging;
//   * the accumulators of the 8 channels stay in registers for two 8-column tiles at a time, so a lane also STORES whole
//     32-byte sectors T[e][c][n0..n0+7].
// Measured rates on this part: mma.sync TF32 279 TFLOP/s against 68 TFLOP/s for packed FFMA.
// Measured result (config 4, forward of the tensor track): 24.3 ms against 30.3 ms for the FFMA kernels of tp3_impl.cuh.
// The arithmetic is gone from the profile (tensor pipe 8 % busy, 4x fewer instructions); what remains is the L1: with
// channels fastest and 8 channels per warp every 32-byte sector sits in its own 128-byte line (l1tex 82 % busy).
// Marking the sector loads and stores L1::no_allocate took the kernel from 29.5 to 24.3 ms (66 % of the copy bandwidth);
// the same hint on the 4-byte stores of the FFMA kernels changed nothing.  A layout with the 8-channel group fastest
// after the component ([edge][group][component][8]) would make the 4 lanes of a fragment row read one line; that, and
// the backward, are the open part of NEXT-2.
#pragma once
#include "tp3_impl.cuh"

// round to the nearest TF32 value, ties away from zero (two integer instructions; cvt.rna.tf32.f32 expands to six)
__device__ __forceinline__ uint32_t t3m_tf32(float x) { return (__float_as_uint(x) + 0x1000u) & 0xFFFFE000u; }
__device__ __forceinline__ void t3m_mma(float* c, uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3, uint32_t b0, uint32_t b1) {
  asm volatile("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
               : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
               : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}

// one whole 32-byte sector per lane (sm_100: 256-bit global loads / stores); p must be 32-byte aligned
__device__ __forceinline__ void t3m_ld256(const float* p, float4& lo, float4& hi) {
  asm volatile("ld.global.nc.L1::no_allocate.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
               : "=f"(lo.x), "=f"(lo.y), "=f"(lo.z), "=f"(lo.w), "=f"(hi.x), "=f"(hi.y), "=f"(hi.z), "=f"(hi.w) : "l"(p));
}
__device__ __forceinline__ void t3m_st256(float* p, const float4& lo, const float4& hi) {
  asm volatile("st.global.L1::no_allocate.v8.f32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"l"(p), "f"(lo.x), "f"(lo.y), "f"(lo.z), "f"(lo.w),
               "f"(hi.x), "f"(hi.y), "f"(hi.z), "f"(hi.w) : "memory");
}

// Gamma_i for every (centre, channel) of the chunk, one warp per (centre, 32 channels), into a.gamma_out: the pass over
// the centre's edges is latency-bound, so it runs once here at full occupancy instead of in front of the MMA tiles of
// every 8-channel warp (where it was 23 % of the stall samples)
template <int P, int WPB>
static __global__ void __launch_bounds__(WPB * 32) k_tp3m_gamma(const __grid_constant__ TP2<Pat<P>::NNZ> a) {
  const int wib = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int ng = a.n / 32;
  int64_t wg = (int64_t)blockIdx.x * WPB + wib;
  if (wg >= (int64_t)a.nc * ng) return;
  if (a.rev) wg = (int64_t)a.nc * ng - 1 - wg;
  const int c = (int)(wg / ng), nn = (int)(wg - (int64_t)c * ng) * 32 + lane;
  const int64_t e0 = a.rowa[c], e1 = a.rowa[c + 1];
  float G[16];
  gamma_pass<16>(a, e0, e1, nn, G);
#pragma unroll
  for (int b = 0; b < 16; ++b) a.gamma_out[((size_t)c * 16 + b) * a.n + nn] = G[b];
}

template <int P, bool FIRST, int WPB, bool PIPE>
static __global__ void __launch_bounds__(WPB * 32) k_tp3m_fwd(const __grid_constant__ TP2<Pat<P>::NNZ> a) {
  constexpr int DENV = Pat<P>::DENV, DIN = Pat<P>::DIN, DOUT = Pat<P>::DOUT;
  static_assert(DENV == 16, "written for l_max = 3");
  constexpr int KH = (DIN + 7) / 8, NJ = (DOUT + 7) / 8;       // k-steps and 8-column tiles of the per-channel product
  static_assert(KH % 2 == 0 && NJ % 2 == 0, "pairs of k-steps / column tiles");
  constexpr int NKC = KH / 2, NJC = NJ / 2;
  constexpr int CB = (((DOUT + 3) / 4) + 1) & ~1, CBH = CB / 2;  // M build: output components per lane (as k_tp3_fwd)
  // M_i of 8 channels in fragment order: 64 floats per (channel, k-step, column tile) block, padded to 72, channel stride
  // padded by 2, so the build's scattered 4-byte stores spread over 16 banks instead of hitting one
  constexpr int BS = 72, CHS = KH * NJ * BS + 2, MS = 8 * CHS;
  static_assert(MS % 4 == 0, "float4 zero fill");
  constexpr int WSL = DENV * 8 + MS;
  extern __shared__ float4 smem4[];
  float* smem = reinterpret_cast<float*>(smem4);
  const int wib = threadIdx.x >> 5, lane = threadIdx.x & 31, ch = lane & 7, q = lane >> 3;
  const int ngroups = a.n / T3_CPW;
  int64_t wg = (int64_t)blockIdx.x * WPB + wib;
  if (wg >= (int64_t)a.nc * ngroups) return;
  if (a.rev) wg = (int64_t)a.nc * ngroups - 1 - wg;
  const int c = (int)(wg / ngroups), grp = (int)(wg - (int64_t)c * ngroups);
  const int n0 = grp * T3_CPW, nn = n0 + ch;
  float* Gs = smem + wib * WSL;
  float* Ms = Gs + DENV * 8;
  const int64_t e0 = a.rowa[c], e1 = a.rowa[c + 1];
  const int deg = (int)(e1 - e0);
  if (deg <= 0) return;

  // ---- Gamma_i and M_i of the warp's 8 channels ----------------------------------------------------------------------
  {
    float4* z = reinterpret_cast<float4*>(Ms);
#pragma unroll 4
    for (int i = lane; i < MS / 4; i += 32) z[i] = make_float4(0.f, 0.f, 0.f, 0.f);   // padded rows / columns stay 0
  }
#pragma unroll
  for (int j = 0; j < 4; ++j) Gs[(4 * q + j) * 8 + ch] = a.gamma_out[((size_t)c * DENV + 4 * q + j) * a.n + nn];   // k_tp3m_gamma
  __syncwarp();
  {
    float2 Mr[DIN * CBH];
    float G[DENV];
#pragma unroll
    for (int b = 0; b < DENV; ++b) G[b] = Gs[b * 8 + ch];
#pragma unroll
    for (int k = 0; k < DIN * CBH; ++k) Mr[k] = make_float2(0.f, 0.f);
#define X(k, a_, b_, c_) \
  if (q == (c_) / CB) TP2_REF(Mr, CBH, a_, (c_) % CB) = fmaf(a.kv[k], G[b_], TP2_REF(Mr, CBH, a_, (c_) % CB));
    TP2_EXPAND(P, X)
#undef X
    // B fragment of (channel, k-step h, column tile j): lane (g', t') holds b0 = M[8h + t'][8j + g'], b1 = M[8h + t' + 4][8j + g']
    const int cb = q * CB;
#pragma unroll
    for (int k = 0; k < DIN; ++k) {
      const int h = k >> 3, tq = k & 3, hi = (k & 7) >> 2;
#pragma unroll
      for (int cc = 0; cc < CB; ++cc) {
        const int co = cb + cc;
        if (co < DOUT) {
          const float v = (cc & 1) ? Mr[k * CBH + (cc >> 1)].y : Mr[k * CBH + (cc >> 1)].x;
          const int j = co >> 3, gq = co & 7;
          Ms[ch * CHS + (h * NJ + j) * BS + (gq * 4 + tq) * 2 + hi] = __uint_as_float(t3m_tf32(v));
        }
      }
    }
  }
  __syncwarp();

  // ---- the centre's edges in tiles of 16 rows; a CHUNK is one pair of k-steps of one tile ----------------------------
  // Software pipeline over chunks: the 32-byte sectors of chunk s + 1 are in flight (raw registers) while chunk s runs
  // through the tensor cores.  K = 16: one chunk per tile and two column-tile pairs per chunk; K = 32: two chunks per
  // tile accumulate into the same registers.
  const int g = lane >> 2, t = lane & 3;
  const float2* Ms2 = reinterpret_cast<const float2*>(Ms);
  const int nchunks = ((deg + 15) >> 4) * NKC;
  float4 R[2][2][2][2];                        // raw sectors of the next chunk: [k-step][row][column][low / high channels]
  float Yv[2][2][2];                           // FIRST: the Y factor of each raw sector
  uint32_t A[2][2][2][8];                      // current chunk as TF32: [k-step of the pair][row g / g+8][column t / t+4][channel]
  float C[8][2][4];
  auto rows_of = [&](int tile, int64_t* er, bool* ok) {
    int r0 = tile * 16 + g, r1 = r0 + 8;
    ok[0] = r0 < deg; ok[1] = r1 < deg;
    er[0] = e0 + (ok[0] ? r0 : deg - 1); er[1] = e0 + (ok[1] ? r1 : deg - 1);
  };
  auto issue = [&](int sidx) {
    const int tile = sidx / NKC, hp = sidx - tile * NKC;
    int64_t er[2]; bool ok[2];
    rows_of(tile, er, ok);
#pragma unroll
    for (int hh = 0; hh < 2; ++hh)
#pragma unroll
      for (int cs = 0; cs < 2; ++cs) {
        const int acol = 8 * (2 * hp + hh) + t + 4 * cs;
#pragma unroll
        for (int rs = 0; rs < 2; ++rs) {
          R[hh][rs][cs][0] = make_float4(0.f, 0.f, 0.f, 0.f); R[hh][rs][cs][1] = R[hh][rs][cs][0];
          Yv[hh][rs][cs] = 1.f;
          if (acol < DIN) {
            if (FIRST) {
              Yv[hh][rs][cs] = __ldg(a.Y + er[rs] * a.ldy + acol);
              t3m_ld256(a.w0 + er[rs] * a.ldw + l_of(acol) * a.n + n0, R[hh][rs][cs][0], R[hh][rs][cs][1]);
            } else {
              t3m_ld256(a.Vin + (er[rs] * DIN + acol) * a.n + n0, R[hh][rs][cs][0], R[hh][rs][cs][1]);
            }
          }
        }
      }
  };
  auto convert = [&]() {
#pragma unroll
    for (int hh = 0; hh < 2; ++hh)
#pragma unroll
      for (int cs = 0; cs < 2; ++cs)
#pragma unroll
        for (int rs = 0; rs < 2; ++rs) {
          const float y = Yv[hh][rs][cs];
          const float4 v0 = R[hh][rs][cs][0], v1 = R[hh][rs][cs][1];
          A[hh][rs][cs][0] = t3m_tf32(v0.x * y); A[hh][rs][cs][1] = t3m_tf32(v0.y * y);
          A[hh][rs][cs][2] = t3m_tf32(v0.z * y); A[hh][rs][cs][3] = t3m_tf32(v0.w * y);
          A[hh][rs][cs][4] = t3m_tf32(v1.x * y); A[hh][rs][cs][5] = t3m_tf32(v1.y * y);
          A[hh][rs][cs][6] = t3m_tf32(v1.z * y); A[hh][rs][cs][7] = t3m_tf32(v1.w * y);
        }
  };
  auto zero_C = [&]() {
#pragma unroll
    for (int x = 0; x < 8; ++x)
#pragma unroll
      for (int y = 0; y < 2; ++y) { C[x][y][0] = 0.f; C[x][y][1] = 0.f; C[x][y][2] = 0.f; C[x][y][3] = 0.f; }
  };
  auto mmas = [&](int hp, int jp) {
#pragma unroll
    for (int cq = 0; cq < 8; ++cq)
#pragma unroll
      for (int jj = 0; jj < 2; ++jj)
#pragma unroll
        for (int hh = 0; hh < 2; ++hh) {
          const float2 b = Ms2[(cq * CHS + ((2 * hp + hh) * NJ + 2 * jp + jj) * BS) / 2 + lane];
          t3m_mma(C[cq][jj], A[hh][0][0][cq], A[hh][1][0][cq], A[hh][0][1][cq], A[hh][1][1][cq], __float_as_uint(b.x),
                  __float_as_uint(b.y));
        }
  };
  // C fragment: c0 (row g, col 2t), c1 (row g, col 2t+1), c2 (row g+8, col 2t), c3 (row g+8, col 2t+1); the lane holds the
  // same element of all 8 channels = one 32-byte sector of T[e][c][n0..n0+7]
  auto store = [&](int tile, int jp) {
    int64_t er[2]; bool ok[2];
    rows_of(tile, er, ok);
#pragma unroll
    for (int jj = 0; jj < 2; ++jj)
#pragma unroll
      for (int cs = 0; cs < 2; ++cs) {
        const int co = 8 * (2 * jp + jj) + 2 * t + cs;
        if (co < DOUT) {
#pragma unroll
          for (int rs = 0; rs < 2; ++rs) {
            if (ok[rs]) {
              const int el = rs * 2 + cs;
              const float4 lo = make_float4(C[0][jj][el], C[1][jj][el], C[2][jj][el], C[3][jj][el]);
              const float4 hi = make_float4(C[4][jj][el], C[5][jj][el], C[6][jj][el], C[7][jj][el]);
              if (a.Tout) t3m_st256(a.Tout + (er[rs] * DOUT + co) * a.n + n0, lo, hi);
              if (co == 0) t3m_st256(a.xs + er[rs] * a.ldx + n0, lo, hi);
            }
          }
        }
      }
  };
  if (PIPE) issue(0);
  for (int sidx = 0; sidx < nchunks; ++sidx) {
    if (!PIPE) issue(sidx);
    convert();
    if (PIPE && sidx + 1 < nchunks) issue(sidx + 1);
    const int tile = sidx / NKC, hp = sidx - tile * NKC;
    if (NKC == 1) {
#pragma unroll
      for (int jp = 0; jp < NJC; ++jp) {
        zero_C();
        mmas(0, jp);
        store(tile, jp);
      }
    } else {
      static_assert(NKC == 1 || NJC == 1, "K = 32 layers have 16 output columns");
      if (hp == 0) zero_C();
      mmas(hp, 0);
      if (hp == NKC - 1) store(tile, 0);
    }
  }
}

template <int P, bool FIRST, int WPB, bool PIPE>
int launch_fwd3m(allegro_model* m, const TP2<Pat<P>::NNZ>& a) {
  constexpr int KH = (Pat<P>::DIN + 7) / 8, NJ = (Pat<P>::DOUT + 7) / 8;
  constexpr int WSL = 16 * 8 + 8 * (KH * NJ * 72 + 2);
  size_t sm = (size_t)WPB * WSL * 4 + 16;
  static AttrOnce once;
  if (once.need(m->device)) { AL_CUDA(m, cudaFuncSetAttribute(k_tp3m_fwd<P, FIRST, WPB, PIPE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm)); once.done(m->device); }
  {
    int64_t gw = (int64_t)a.nc * (a.n / 32);
    k_tp3m_gamma<P, 8><<<(unsigned)((gw + 7) / 8), 256, 0, m->stream>>>(a);
    m->launches++;
  }
  int64_t warps = (int64_t)a.nc * (a.n / T3_CPW);
  k_tp3m_fwd<P, FIRST, WPB, PIPE><<<(unsigned)((warps + WPB - 1) / WPB), WPB * 32, sm, m->stream>>>(a);
  m->launches++;
  AL_CUDA(m, cudaGetLastError());
  return ALLEGRO_OK;
}
