// Tensor track, contracted per centre ("collapsed"): the default tensor-track kernels (SURVEY.md section 8(a) steps 5-7 and
// their backward in step 11; Eq. (2) :132-138, fused path-weighted CG tensor :160-164, Fig. 3 :180).
//
// The paper sums the environment before the product because the tensor product is bilinear (Eq. (2) line 2).
// The same linearity reaches across layers: tensor features never pass through a nonlinearity -- only the scalar block
// s^L_e = V^L_e[(0,+)] leaves the tensor track -- so with  M^k_i[a,c] = sum_b K^k[a,b,c] Gamma^k_i[b]  (per centre
// i and channel n, the same for all edges of the centre)
//     V^L_e = V^0_e M^1_i M^2_i ... M^L_i        and        s^L_e = V^0_e . n^L_i,     n^L_i = M^1_i ... M^{L-1}_i M^L_i[:, 0].
// Contracting the per-centre operators FIRST leaves one D_0-long dot product per edge, channel and layer, instead of a
// D_{L-1} x D_L product per edge: V^L_e is never formed, nothing of size [edges, D, n] is read or written, and the work that
// involves the sparse tensors K^k happens once per centre.  It is the same function up to the order of the fp32 sums
// (the fp64 reference of the test suite follows the paper's order, layer by layer and edge by edge).  Matrix-free: M^k is never built either;
// the three trilinear forms of K^k(Gamma^k) that are needed run straight off the compile-time sparsity pattern
// (tp2_patterns.inc) with every operand in registers:
//     fwd :  y[a]  = sum K[a,b,c] Gamma[b] x[c]      (y = M x)
//     tr  :  v[c]  = sum K[a,b,c] Gamma[b] u[a]      (v = M^T u)
//     gb  :  g[b]  = sum K[a,b,c] u[a] w[c]          (d(u^T M w) / dGamma)
// Forward, layer L (one warp = centre x 32 channels, lane = channel):
//     Gamma^L_i = c_env sum_e omega^L_e (x) Y_e  ->  n^L_i (needs Gamma^1..Gamma^L)  ->  s^L_e = sum_a w0_e[l(a)] Y_e[a] n^L_i[a].
// Backward, layer L (reverse order), with s-bar^L_e from the latent MLP's backward:
//     n-bar^L_i = sum_e s-bar^L_e V^0_e;   u_0 = n-bar^L, w_L = e_0, w_k = M^{k+1} w_{k+1}, u_k = M^{k T} u_{k-1}:
//     Gamma-bar^k_i += gb_k(u_{k-1}, w_k) for k = 1..L   (contributions to k < L wait in a per-centre accumulator until layer
//     k's own backward, which then has the complete Gamma-bar^k);
//     pass B: omega-bar^L_e[l] = c_env sum_{m} Gamma-bar^L[(l,m)] Y_e[(l,m)],  Y-bar_e[b] += c_env sum_n omega^L_e[l(b)] Gamma-bar^L[b];
//     layer 1 also: V-bar^0_e = sum_L s-bar^L_e n^L_i  ->  w0-bar_e[l] = sum_{a in l} V-bar^0_e[a] Y_e[a],  Y-bar_e[a] += sum_n w0_e[l(a)] V-bar^0_e[a].
// HBM traffic per edge at config 2/3 (n = 64): forward 2 x (omega 768 + w0 768 + s 256 B), backward 6.3 KB, against
// 7.4 + 12.0 KB for the per-edge product kernels (tp2_impl.cuh), and the [edges, D, n] buffers T, V-bar are not allocated.
#pragma once
#include "h16.cuh"
#include "tp2_impl.cuh"

constexpr int TPC_MAXL = 3;   // layers the contracted kernels are instantiated for

// pattern of layer k (1-based) of an (l_max, NL) model: the eligibility test (tp2_eligible) guarantees these roles
template <int LM, int NL, int K> struct TpcPat {
  static constexpr int P = (LM == 1) ? (K < NL ? P_4_4_4 : P_4_4_1) : (LM == 2) ? (K < NL ? P_9_9_9 : P_9_9_1)
                                     : (K == 1 ? P_16_16_31 : K == 2 ? P_16_31_16 : P_16_16_1);
};
template <int LM> struct TpcEnv { static constexpr int DENV = (LM + 1) * (LM + 1); };

template <int LM, int NL>
struct TPC {
  static constexpr int NNZ1 = Pat<TpcPat<LM, NL, 1>::P>::NNZ;
  static constexpr int NNZ2 = NL >= 2 ? Pat<TpcPat<LM, NL, (NL >= 2 ? 2 : 1)>::P>::NNZ : 1;
  static constexpr int NNZ3 = NL >= 3 ? Pat<TpcPat<LM, NL, (NL >= 3 ? 3 : 1)>::P>::NNZ : 1;
  const int64_t* rowa; int nc, n; float c_env; int rev;
  int hfmt;                                   // >= 0 (16-bit operand modes): xs, ombar, w0bar are 16-bit tensors (GEMM A operands)
  const float* Y; int ldy;
  const float* w0; int ldw;                   // w^0_e[l][n]
  const float* om; int ldo;                   // omega^L_e[l][n] of THIS layer
  float* xs; int ldx;                         // forward: s^L_e[n]
  float* gam; float* nvec; float* gacc; int64_t cstride;   // per-centre [layer][centre][DENV][n]; cstride = centres * DENV * n
  const float* sb[TPC_MAXL]; int lds[TPC_MAXL];            // backward: s-bar^k_e[n] of every layer k (layer 1 needs them all)
  float* ombar; int ldob; float* w0bar;
  float* Ybar; int64_t ybar_pstride; int ybar_part0, ybar_partL;
  float kv1[NNZ1], kv2[NNZ2], kv3[NNZ3];      // values of K^1, K^2, K^3 in pattern order
};

// ---- the three trilinear sweeps over the pattern of P ------------------------------------------------------------------------
// E0: the right-hand vector is e_0 (only the entries with c = 0 contribute).  Each sweep multiplies K's value by a DIFFERENT
// operand first -- fwd (k G) x, tr (k u) G, gb (k w) u -- so the compiler finds no common sub-expression between two sweeps over
// the same pattern (it would otherwise keep all nnz = 611 products kv[k] * G[b] of an l_max = 3 layer alive: 3 KB of spills).
template <int P, bool E0, int NNZ>
__device__ __forceinline__ void tpc_fwd(const float (&kv)[NNZ], const float* G, const float* x, float* y) {
#pragma unroll
  for (int a = 0; a < Pat<P>::DIN; ++a) y[a] = 0.f;
#define X(k, a_, b_, c_) \
  if (!E0) y[a_] = fmaf(kv[k] * G[b_], x[c_], y[a_]); else if ((c_) == 0) y[a_] = fmaf(kv[k], G[b_], y[a_]);
  TP2_EXPAND(P, X)
#undef X
}
template <int P, int NNZ>
__device__ __forceinline__ void tpc_tr(const float (&kv)[NNZ], const float* G, const float* u, float* v) {
#pragma unroll
  for (int c = 0; c < Pat<P>::DOUT; ++c) v[c] = 0.f;
#define X(k, a_, b_, c_) v[c_] = fmaf(kv[k] * u[a_], G[b_], v[c_]);
  TP2_EXPAND(P, X)
#undef X
}
// g[b] += ...  (accumulates)
template <int P, bool E0, int NNZ>
__device__ __forceinline__ void tpc_gb(const float (&kv)[NNZ], const float* u, const float* w, float* g) {
#define X(k, a_, b_, c_) \
  if (!E0) g[b_] = fmaf(kv[k] * w[c_], u[a_], g[b_]); else if ((c_) == 0) g[b_] = fmaf(kv[k], u[a_], g[b_]);
  TP2_EXPAND(P, X)
#undef X
}

// tr and gb over the same pattern with the same left vector u in one sweep: v = M^T u and g[b] += sum K[a,b,c] u[a] w[c] share
// the product kv[k] * u[a] (3 instead of 4 instructions per entry; the shared product lives for two instructions only)
template <int P, int NNZ>
__device__ __forceinline__ void tpc_tr_gb(const float (&kv)[NNZ], const float* G, const float* u, const float* w, float* v, float* g) {
#pragma unroll
  for (int c = 0; c < Pat<P>::DOUT; ++c) v[c] = 0.f;
#define X(k, a_, b_, c_) { const float t_ = kv[k] * u[a_]; v[c_] = fmaf(t_, G[b_], v[c_]); g[b_] = fmaf(t_, w[c_], g[b_]); }
  TP2_EXPAND(P, X)
#undef X
}

// Sum each of N per-lane values (N = 4, 16, 32) over the 32 lanes with the halving butterfly: N - 1 shuffles for the halving
// steps, one more per remaining stride.  On return the lane holds the total of value index lane >> (5 - log2 N).
template <int N>
__device__ __forceinline__ float tpc_reduce(float* v, int lane) {
  int cnt = N, stride = 16;
#pragma unroll
  for (int step = 0; step < 5; ++step) {
    if (cnt > 1) {
      const bool hi = lane & stride;
      cnt >>= 1;
#pragma unroll
      for (int i = 0; i < N / 2; ++i) {
        if (i < cnt) {
          const float send = hi ? v[i] : v[i + cnt], keep = hi ? v[i + cnt] : v[i];
          v[i] = keep + __shfl_xor_sync(TP_FULLMASK, send, stride);
        }
      }
    } else {
      v[0] += __shfl_xor_sync(TP_FULLMASK, v[0], stride);
    }
    stride >>= 1;
  }
  return v[0];
}

// Y-bar partial rows of four consecutive edges (rows il0 .. il0 + 3 of yrows, rows >= deg not stored; pp of those must be 0):
// pp[j][b] summed over the lanes, 32 values per butterfly instead of one tree per value (1.0 instead of 1.55 shuffles per
// value).  DENV = 9: the 8 leading components of the 4 edges in one butterfly (lane -> edge lane / 8, component lane % 8),
// the 9th components in a 4-value butterfly; DENV = 16: two edges per butterfly; DENV = 4: one 16-value butterfly.
template <int DENV>
__device__ __forceinline__ void tpc_ybar_store(float* yrows, float (*pp)[DENV], int il0, int deg, int lane) {
  if constexpr (DENV == 9) {
    float v[32];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
      for (int b = 0; b < 8; ++b) v[i * 8 + b] = pp[i][b];
    const float r = tpc_reduce<32>(v, lane);
    if (il0 + (lane >> 3) < deg) yrows[(int64_t)(il0 + (lane >> 3)) * DENV + (lane & 7)] = r;
    float t[4] = {pp[0][8], pp[1][8], pp[2][8], pp[3][8]};
    const float r8 = tpc_reduce<4>(t, lane);
    if ((lane & 7) == 0 && il0 + (lane >> 3) < deg) yrows[(int64_t)(il0 + (lane >> 3)) * DENV + 8] = r8;
  } else if constexpr (DENV == 16) {
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      float v[32];
#pragma unroll
      for (int i = 0; i < 2; ++i)
#pragma unroll
        for (int b = 0; b < 16; ++b) v[i * 16 + b] = pp[2 * h + i][b];
      const float r = tpc_reduce<32>(v, lane);
      if (il0 + 2 * h + (lane >> 4) < deg) yrows[(int64_t)(il0 + 2 * h + (lane >> 4)) * DENV + (lane & 15)] = r;
    }
  } else {
    static_assert(DENV == 4, "l_max <= 3");
    float v[16];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
      for (int b = 0; b < 4; ++b) v[i * 4 + b] = pp[i][b];
    const float r = tpc_reduce<16>(v, lane);                          // lane holds value lane >> 1
    if ((lane & 1) == 0 && il0 + (lane >> 3) < deg) yrows[(int64_t)(il0 + (lane >> 3)) * DENV + ((lane >> 1) & 3)] = r;
  }
}

// ---- streaming the centre's edges: a per-warp cp.async ring in shared memory (the loads in flight cost no registers; the
//      passes are pure streams whose speed is the number of bytes in flight).  One stage = one edge: NR rows of 32 channels
//      (rows 0 .. NLV-1 from `src1`, one per l; then up to two single rows from `xa`, `xb`) + the LDY floats of Y_e. ------------
template <int DENV, int NX>
struct TpcStage {
  static constexpr int NLV = nlv_of(DENV), LDY = (DENV + 3) & ~3, NR = NLV + NX, SF = NR * 32 + LDY, NCH = NR * 8 + LDY / 4;
};
constexpr int TPC_NST = 8;        // ring stages per warp

struct TpcSrc {
  const float* src1; int ld1;     // NLV rows: src1 + e * ld1 + l * n
  const float* xa; int lda;       // optional single rows: xa + e * lda, xb + e * ldb
  const float* xb; int ldb;
  const float* Y; int ldy; int n;
};

// per-lane copy plan of a pass, computed once per centre: chunk it * 32 + lane of a stage comes from p[it] + il * ld[it]
template <int DENV, int NX>
struct TpcPlan {
  using S = TpcStage<DENV, NX>;
  static constexpr int NIT = (S::NCH + 31) / 32;
  const float* p[NIT]; int ld[NIT], dst[NIT];
  __device__ __forceinline__ TpcPlan(const TpcSrc& q, int64_t e0, int ch0, int lane) {
#pragma unroll
    for (int it = 0; it < NIT; ++it) {
      const int i = it * 32 + lane;
      if (i < S::NR * 8) {
        const int row = i >> 3;
        if (row < S::NLV) { p[it] = q.src1 + e0 * q.ld1 + row * q.n; ld[it] = q.ld1; }
        else if (row == S::NLV) { p[it] = q.xa + e0 * q.lda; ld[it] = q.lda; }
        else { p[it] = q.xb + e0 * q.ldb; ld[it] = q.ldb; }
        p[it] += ch0 + (i & 7) * 4; dst[it] = i * 4;
      } else if (i < S::NCH) {
        p[it] = q.Y + e0 * q.ldy + (i - S::NR * 8) * 4; ld[it] = q.ldy; dst[it] = S::NR * 32 + (i - S::NR * 8) * 4;
      } else {
        p[it] = nullptr; ld[it] = 0; dst[it] = 0;
      }
    }
  }
  __device__ __forceinline__ void issue(float* st, int il) const {
#pragma unroll
    for (int it = 0; it < NIT; ++it)
      if (p[it]) tp_cp16(st + dst[it], p[it] + (int64_t)il * ld[it]);
  }
};

// body(il, j, stage pointer) for il = 0 .. deg-1 in groups of four (j = il & 3, compile-time in the unrolled group), then
// post(first il of the group) once per group; the next TPC_NST - 1 edges are in flight
template <int DENV, int NX, class F, class G>
__device__ __forceinline__ void tpc_stream(float* ring, const TpcSrc& q, int64_t e0, int deg, int ch0, int lane, F body, G post) {
  using S = TpcStage<DENV, NX>;
  const TpcPlan<DENV, NX> plan(q, e0, ch0, lane);
#pragma unroll
  for (int s = 0; s < TPC_NST - 1; ++s) {
    if (s < deg) plan.issue(ring + s * S::SF, s);
    tp_cp_commit();
  }
  int slot = 0;
  for (int g0 = 0; g0 < deg; g0 += 4) {
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int il = g0 + j;
      if (il < deg) {                                                // (warp-uniform)
        tp_cp_wait<TPC_NST - 2>();
        __syncwarp();
        const int nx = il + TPC_NST - 1;
        int ns = slot + TPC_NST - 1; if (ns >= TPC_NST) ns -= TPC_NST;
        if (nx < deg) plan.issue(ring + ns * S::SF, nx);
        tp_cp_commit();
        body(il, j, ring + slot * S::SF);
        if (++slot == TPC_NST) slot = 0;
      }
    }
    post(g0);
  }
  tp_cp_wait<0>();
  __syncwarp();                   // the ring may be re-used by the next pass
}

// floats of ring per warp: the widest stage of the kernel's passes
template <int DENV> __host__ __device__ constexpr int tpc_ring_floats(int nx_max) { return TPC_NST * ((nlv_of(DENV) + nx_max) * 32 + ((DENV + 3) & ~3)); }

// ======================================================================================================
// forward of layer L
// ======================================================================================================
template <int LM, int NL, int L, int WPB>
static __global__ void __launch_bounds__(WPB * 32) k_tpc_fwd(const __grid_constant__ TPC<LM, NL> a) {
  constexpr int DENV = TpcEnv<LM>::DENV, NLV = nlv_of(DENV);
  constexpr int P1 = TpcPat<LM, NL, 1>::P, P2 = TpcPat<LM, NL, (NL >= 2 ? 2 : 1)>::P, P3 = TpcPat<LM, NL, (NL >= 3 ? 3 : 1)>::P;
  using S0 = TpcStage<DENV, 0>;
  extern __shared__ float4 smem4[];
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5, ng = a.n / 32;
  float* ring = reinterpret_cast<float*>(smem4) + wib * tpc_ring_floats<DENV>(0);
  int64_t wg = (int64_t)blockIdx.x * WPB + wib;
  if (wg >= (int64_t)a.nc * ng) return;
  if (a.rev) wg = (int64_t)a.nc * ng - 1 - wg;
  const int c = (int)(wg / ng), grp = (int)(wg - (int64_t)c * ng), nn = grp * 32 + lane;
  const int64_t e0 = a.rowa[c], e1 = a.rowa[c + 1];
  const int deg = (int)(e1 - e0);
  if (deg <= 0) return;
  TpcSrc q{a.om, a.ldo, nullptr, 0, nullptr, 0, a.Y, a.ldy, a.n};
  float nv[DENV];
  {
    float G[L][DENV];
    // Gamma^L_i[b] = c_env sum_e omega^L_e[l(b)] Y_e[b]   (Eq. (2) line 2: the environment is summed before the product)
#pragma unroll
    for (int b = 0; b < DENV; ++b) G[L - 1][b] = 0.f;
    tpc_stream<DENV, 0>(ring, q, e0, deg, grp * 32, lane, [&](int, int, const float* st) {
      float om[NLV];
#pragma unroll
      for (int l = 0; l < NLV; ++l) om[l] = st[l * 32 + lane];
#pragma unroll
      for (int b = 0; b < DENV; ++b) G[L - 1][b] = fmaf(om[l_of(b)], st[S0::NR * 32 + b], G[L - 1][b]);
    }, [](int) {});
    float* gp = a.gam + ((size_t)c * DENV) * a.n + nn;
#pragma unroll
    for (int b = 0; b < DENV; ++b) { G[L - 1][b] *= a.c_env; gp[(L - 1) * a.cstride + (size_t)b * a.n] = G[L - 1][b]; }
#pragma unroll
    for (int k = 0; k < L - 1; ++k)
#pragma unroll
      for (int b = 0; b < DENV; ++b) G[k][b] = gp[k * a.cstride + (size_t)b * a.n];
    // n^L = M^1 ... M^{L-1} M^L e_0
    if constexpr (L == 1) {
      tpc_fwd<P1, true>(a.kv1, G[0], nullptr, nv);
    } else if constexpr (L == 2) {
      float x1[Pat<P2>::DIN];
      tpc_fwd<P2, true>(a.kv2, G[1], nullptr, x1);
      tpc_fwd<P1, false>(a.kv1, G[0], x1, nv);
    } else {
      float x2[Pat<P3>::DIN], x1[Pat<P2>::DIN];
      tpc_fwd<P3, true>(a.kv3, G[2], nullptr, x2);
      tpc_fwd<P2, false>(a.kv2, G[1], x2, x1);
      tpc_fwd<P1, false>(a.kv1, G[0], x1, nv);
    }
    float* np = a.nvec + (L - 1) * a.cstride + ((size_t)c * DENV) * a.n + nn;
#pragma unroll
    for (int b = 0; b < DENV; ++b) np[(size_t)b * a.n] = nv[b];
  }
  // s^L_e = sum_a w0_e[l(a)] Y_e[a] n^L[a]
  q.src1 = a.w0; q.ld1 = a.ldw;
  const size_t xs0 = (size_t)e0 * a.ldx + nn;
  tpc_stream<DENV, 0>(ring, q, e0, deg, grp * 32, lane, [&](int il, int, const float* st) {
    float t[NLV];
#pragma unroll
    for (int l = 0; l < NLV; ++l) t[l] = 0.f;
#pragma unroll
    for (int b = 0; b < DENV; ++b) t[l_of(b)] = fmaf(st[S0::NR * 32 + b], nv[b], t[l_of(b)]);
    float sv = 0.f;
#pragma unroll
    for (int l = 0; l < NLV; ++l) sv = fmaf(st[l * 32 + lane], t[l], sv);
    h16_store(a.xs, xs0 + (size_t)il * a.ldx, sv, a.hfmt);
  }, [](int) {});
}

// ======================================================================================================
// forward of layer L, register-batch variant (l_max <= 2): 8 edges in flight per warp by direct loads, Y rows broadcast by
// shuffle.  The per-edge work of the forward passes is so small (9 FMAs) that the ring's per-edge wait / issue bookkeeping costs
// more than it hides: measured 2.58 ms (this) against 2.81 ms (ring) per step at config 2; at l_max = 3 (16 components, 4 rows
// per edge) the ring wins, 5.5 against 7.7 ms at config 4.
// ======================================================================================================
// ---- one batch of up to 8 edges of a centre: NLV rows of 32 channels each + the Y rows (one contiguous block, one value per
//      lane, components broadcast by shuffle as in gamma_pass) ------------------------------------------------------------------
template <int DENV>
struct TpcBatch {
  static constexpr int NLV = nlv_of(DENV), LDY = (DENV + 3) & ~3, NR = LDY / 4;
  float yr[NR];
  __device__ __forceinline__ void load_y(const float* Y, int64_t e, int64_t e1, int lane) {
    const int64_t ylast = e1 * LDY - 1;
#pragma unroll
    for (int k = 0; k < NR; ++k) {
      const int64_t idx = e * LDY + k * 32 + lane;
      yr[k] = __ldg(Y + (idx < ylast ? idx : ylast));
    }
  }
  __device__ __forceinline__ float y(int i, int b) const { return __shfl_sync(TP_FULLMASK, yr[(i * LDY + b) >> 5], (i * LDY + b) & 31); }
};

template <int LM, int NL, int L, int WPB>
static __global__ void __launch_bounds__(WPB * 32) k_tpc_fwd_rb(const __grid_constant__ TPC<LM, NL> a) {
  constexpr int DENV = TpcEnv<LM>::DENV, NLV = nlv_of(DENV);
  constexpr int P1 = TpcPat<LM, NL, 1>::P, P2 = TpcPat<LM, NL, (NL >= 2 ? 2 : 1)>::P, P3 = TpcPat<LM, NL, (NL >= 3 ? 3 : 1)>::P;
  const int lane = threadIdx.x & 31, ng = a.n / 32;
  int64_t wg = (int64_t)blockIdx.x * WPB + (threadIdx.x >> 5);
  if (wg >= (int64_t)a.nc * ng) return;
  if (a.rev) wg = (int64_t)a.nc * ng - 1 - wg;
  const int c = (int)(wg / ng), nn = (int)(wg - (int64_t)c * ng) * 32 + lane;
  const int64_t e0 = a.rowa[c], e1 = a.rowa[c + 1];
  if (e1 <= e0) return;
  float nv[DENV];
  {
    float G[L][DENV];
    gamma_pass<DENV>(a, e0, e1, nn, G[L - 1]);                       // Gamma^L_i (Eq. (2) line 2: sum before product)
    float* gp = a.gam + ((size_t)c * DENV) * a.n + nn;
#pragma unroll
    for (int b = 0; b < DENV; ++b) gp[(L - 1) * a.cstride + (size_t)b * a.n] = G[L - 1][b];
#pragma unroll
    for (int k = 0; k < L - 1; ++k)
#pragma unroll
      for (int b = 0; b < DENV; ++b) G[k][b] = gp[k * a.cstride + (size_t)b * a.n];
    // n^L = M^1 ... M^{L-1} M^L e_0
    if constexpr (L == 1) {
      tpc_fwd<P1, true>(a.kv1, G[0], nullptr, nv);
    } else if constexpr (L == 2) {
      float x1[Pat<P2>::DIN];
      tpc_fwd<P2, true>(a.kv2, G[1], nullptr, x1);
      tpc_fwd<P1, false>(a.kv1, G[0], x1, nv);
    } else {
      float x2[Pat<P3>::DIN], x1[Pat<P2>::DIN];
      tpc_fwd<P3, true>(a.kv3, G[2], nullptr, x2);
      tpc_fwd<P2, false>(a.kv2, G[1], x2, x1);
      tpc_fwd<P1, false>(a.kv1, G[0], x1, nv);
    }
    float* np = a.nvec + (L - 1) * a.cstride + ((size_t)c * DENV) * a.n + nn;
#pragma unroll
    for (int b = 0; b < DENV; ++b) np[(size_t)b * a.n] = nv[b];
  }
  // s^L_e = sum_a w0_e[l(a)] Y_e[a] n^L[a], 8 edges in flight
  for (int64_t e = e0; e < e1; e += 8) {
    float w[8][NLV];
    TpcBatch<DENV> yb;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const int64_t ee = (e + i < e1) ? e + i : e1 - 1;
#pragma unroll
      for (int l = 0; l < NLV; ++l) w[i][l] = a.w0[ee * a.ldw + l * a.n + nn];
    }
    yb.load_y(a.Y, e, e1, lane);
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      float t[NLV];
#pragma unroll
      for (int l = 0; l < NLV; ++l) t[l] = 0.f;
#pragma unroll
      for (int b = 0; b < DENV; ++b) t[l_of(b)] = fmaf(yb.y(i, b), nv[b], t[l_of(b)]);
      float s = 0.f;
#pragma unroll
      for (int l = 0; l < NLV; ++l) s = fmaf(w[i][l], t[l], s);
      if (e + i < e1) h16_store(a.xs, (size_t)(e + i) * a.ldx + nn, s, a.hfmt);
    }
  }
}

// ======================================================================================================
// backward of layer L
// ======================================================================================================
template <int LM, int NL, int L, int WPB>
static __global__ void __launch_bounds__(WPB * 32) k_tpc_bwd(const __grid_constant__ TPC<LM, NL> a) {
  constexpr int DENV = TpcEnv<LM>::DENV, NLV = nlv_of(DENV);
  constexpr int P1 = TpcPat<LM, NL, 1>::P, P2 = TpcPat<LM, NL, (NL >= 2 ? 2 : 1)>::P, P3 = TpcPat<LM, NL, (NL >= 3 ? 3 : 1)>::P;
  constexpr int NXA = (L == 1) ? (NL < 2 ? 1 : 2) : 1;               // single rows of pass A staged in the ring (s-bar rows)
  using SA = TpcStage<DENV, NXA>;
  using SB = TpcStage<DENV, 0>;
  extern __shared__ float4 smem4[];
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5, ng = a.n / 32;
  float* ring = reinterpret_cast<float*>(smem4) + wib * tpc_ring_floats<DENV>(NXA);
  int64_t wg = (int64_t)blockIdx.x * WPB + wib;
  if (wg >= (int64_t)a.nc * ng) return;
  if (a.rev) wg = (int64_t)a.nc * ng - 1 - wg;
  const int c = (int)(wg / ng), grp = (int)(wg - (int64_t)c * ng), nn = grp * 32 + lane;
  const int64_t e0 = a.rowa[c], e1 = a.rowa[c + 1];
  const int deg = (int)(e1 - e0);
  if (deg <= 0) return;
  const size_t cb = ((size_t)c * DENV) * a.n + nn;                   // + layer * cstride + b * n
  float* Yb0 = a.Ybar + (size_t)(a.ybar_part0 + grp) * a.ybar_pstride + e0 * DENV;
  float* YbL = a.Ybar + (size_t)(a.ybar_partL + grp) * a.ybar_pstride + e0 * DENV;

  // ---- pass A: n-bar^L[a] = sum_e s-bar^L_e w0_e[l(a)] Y_e[a]; layer 1 also turns V-bar^0_e = sum_k s-bar^k_e n^k into
  //      w0-bar_e and the V^0 part of Y-bar_e (a third layer's s-bar row is read directly) ------------------------------------------
  float nb[DENV];
#pragma unroll
  for (int b = 0; b < DENV; ++b) nb[b] = 0.f;
  {
    constexpr int NK = (L == 1) ? NL : 1;
    float nk[NK][DENV];                                              // layer 1: n^k of every layer
    if constexpr (L == 1) {
#pragma unroll
      for (int k = 0; k < NL; ++k)
#pragma unroll
        for (int b = 0; b < DENV; ++b) nk[k][b] = a.nvec[k * a.cstride + cb + (size_t)b * a.n];
    }
    TpcSrc q{a.w0, a.ldw, a.sb[L - 1], a.lds[L - 1], (L == 1 && NL >= 2) ? a.sb[1] : nullptr, (L == 1 && NL >= 2) ? a.lds[1] : 0,
             a.Y, a.ldy, a.n};
    size_t wbo = (size_t)e0 * a.ldob + nn;       // element offset into w0bar
    // Y-bar sums over the lanes: batched over four edges (l_max <= 2: 36 values per butterfly pass) or one tree per edge
    // (l_max = 3: the four-edge batch costs 64 registers and measured slower, 20.9 against 17.0 ms per step at config 4)
    constexpr bool BATCHY = DENV <= 9;
    float pp[(L == 1 && BATCHY) ? 4 : 1][DENV];
    tpc_stream<DENV, NXA>(ring, q, e0, deg, grp * 32, lane, [&](int il, int j, const float* st) {
      float w[NLV], sb[NK];
#pragma unroll
      for (int l = 0; l < NLV; ++l) w[l] = st[l * 32 + lane];
      sb[0] = st[NLV * 32 + lane];                                   // s-bar of THIS layer
      if constexpr (L == 1 && NL >= 2) sb[1] = st[(NLV + 1) * 32 + lane];
      if constexpr (L == 1 && NL >= 3) sb[2] = a.sb[2][(e0 + il) * a.lds[2] + nn];
      float ws[NLV];
#pragma unroll
      for (int l = 0; l < NLV; ++l) ws[l] = w[l] * sb[0];
      if constexpr (L == 1) {
        float wbar[NLV];
#pragma unroll
        for (int l = 0; l < NLV; ++l) wbar[l] = 0.f;
#pragma unroll
        for (int b = 0; b < DENV; ++b) {
          const float yb = st[SA::NR * 32 + b];
          nb[b] = fmaf(ws[l_of(b)], yb, nb[b]);
          float vb = 0.f;                                            // V-bar^0_e[b]
#pragma unroll
          for (int k = 0; k < NL; ++k) vb = fmaf(sb[k], nk[k][b], vb);
          wbar[l_of(b)] = fmaf(vb, yb, wbar[l_of(b)]);
          pp[BATCHY ? j : 0][b] = w[l_of(b)] * vb;
        }
#pragma unroll
        for (int l = 0; l < NLV; ++l) h16_store(a.w0bar, wbo + (size_t)l * a.n, wbar[l], a.hfmt);
        wbo += a.ldob;
        if constexpr (!BATCHY) tp_ybar_rows<DENV, true>(Yb0 + (int64_t)il * DENV, pp[0], 0, DENV, lane);
      } else {
#pragma unroll
        for (int b = 0; b < DENV; ++b) nb[b] = fmaf(ws[l_of(b)], st[SA::NR * 32 + b], nb[b]);
      }
    }, [&](int il0) {
      if constexpr (L == 1 && BATCHY) {
#pragma unroll
        for (int j = 1; j < 4; ++j)
          if (il0 + j >= deg)
#pragma unroll
            for (int b = 0; b < DENV; ++b) pp[j][b] = 0.f;
        tpc_ybar_store<DENV>(Yb0, pp, il0, deg, lane);
      }
    });
  }

  // ---- per centre: Gamma-bar^k contributions of this layer's scalars, k = 1..L ------------------------------------------------------
  float Gb[DENV];                                                    // Gamma-bar^L, complete after this block
  {
    float G[L][DENV];
#pragma unroll
    for (int k = 0; k < L; ++k)
#pragma unroll
      for (int b = 0; b < DENV; ++b) G[k][b] = a.gam[k * a.cstride + cb + (size_t)b * a.n];
    // what the later layers (processed before this one) left for Gamma-bar^L
#pragma unroll
    for (int b = 0; b < DENV; ++b) Gb[b] = (L < NL) ? a.gacc[(L - 1) * a.cstride + cb + (size_t)b * a.n] : 0.f;
    auto put = [&](int k, const float* g) {                          // Gamma-bar^k accumulator, k < L: layer NL writes, the others add
      float* p = a.gacc + (k - 1) * a.cstride + cb;
#pragma unroll
      for (int b = 0; b < DENV; ++b) {
        if (L == NL) p[(size_t)b * a.n] = g[b]; else p[(size_t)b * a.n] += g[b];
      }
    };
    if constexpr (L == 1) {
      tpc_gb<P1, true>(a.kv1, nb, nullptr, Gb);
    } else if constexpr (L == 2) {
      float w1[Pat<P2>::DIN], u1[Pat<P1>::DOUT], g1[DENV];
      tpc_fwd<P2, true>(a.kv2, G[1], nullptr, w1);                   // w_1 = M^2 e_0
#pragma unroll
      for (int b = 0; b < DENV; ++b) g1[b] = 0.f;
      tpc_tr_gb<P1>(a.kv1, G[0], nb, w1, u1, g1);                    // u_1 = M^1T n-bar;  Gamma-bar^1 += g_1(n-bar, w_1)
      put(1, g1);
      tpc_gb<P2, true>(a.kv2, u1, nullptr, Gb);
    } else {
      float w2[Pat<P3>::DIN], w1[Pat<P2>::DIN], u1[Pat<P1>::DOUT], u2[Pat<P2>::DOUT], g[DENV];
      tpc_fwd<P3, true>(a.kv3, G[2], nullptr, w2);                   // w_2 = M^3 e_0
      tpc_fwd<P2, false>(a.kv2, G[1], w2, w1);                       // w_1 = M^2 w_2
#pragma unroll
      for (int b = 0; b < DENV; ++b) g[b] = 0.f;
      tpc_tr_gb<P1>(a.kv1, G[0], nb, w1, u1, g);
      put(1, g);
#pragma unroll
      for (int b = 0; b < DENV; ++b) g[b] = 0.f;
      tpc_tr_gb<P2>(a.kv2, G[1], u1, w2, u2, g);
      put(2, g);
      tpc_gb<P3, true>(a.kv3, u2, nullptr, Gb);
    }
  }

  // ---- pass B: omega-bar^L_e and the environment part of Y-bar_e -------------------------------------------------------------------
#pragma unroll
  for (int b = 0; b < DENV; ++b) Gb[b] *= a.c_env;
  {
    TpcSrc q{a.om, a.ldo, nullptr, 0, nullptr, 0, a.Y, a.ldy, a.n};
    size_t obo = (size_t)e0 * a.ldob + nn;       // element offset into ombar
    constexpr bool BATCHY = DENV <= 9;
    float pp[BATCHY ? 4 : 1][DENV];
    tpc_stream<DENV, 0>(ring, q, e0, deg, grp * 32, lane, [&](int il, int j, const float* st) {
      float om[NLV], ob[NLV];
#pragma unroll
      for (int l = 0; l < NLV; ++l) { om[l] = st[l * 32 + lane]; ob[l] = 0.f; }
#pragma unroll
      for (int b = 0; b < DENV; ++b) {
        ob[l_of(b)] = fmaf(Gb[b], st[SB::NR * 32 + b], ob[l_of(b)]);
        pp[BATCHY ? j : 0][b] = om[l_of(b)] * Gb[b];
      }
#pragma unroll
      for (int l = 0; l < NLV; ++l) h16_store(a.ombar, obo + (size_t)l * a.n, ob[l], a.hfmt);
      obo += a.ldob;
      if constexpr (!BATCHY) tp_ybar_rows<DENV, true>(YbL + (int64_t)il * DENV, pp[0], 0, DENV, lane);
    }, [&](int il0) {
      if constexpr (BATCHY) {
#pragma unroll
        for (int j = 1; j < 4; ++j)
          if (il0 + j >= deg)
#pragma unroll
            for (int b = 0; b < DENV; ++b) pp[j][b] = 0.f;
        tpc_ybar_store<DENV>(YbL, pp, il0, deg, lane);
      }
    });
  }
}

// ---- host side ---------------------------------------------------------------------------------------------
template <int LM, int NL>
int tpc_fill(allegro_model* m, Work& w, int L, int nc, const float* om, int ldo, const float* w0, int ldw, TPC<LM, NL>& a) {
  a.rowa = (const int64_t*)w.rowa.p; a.nc = nc; a.n = m->n; a.c_env = m->c_env; a.rev = al_next_rev(m); a.hfmt = m->hfmt;
  a.Y = (const float*)w.Y.p; a.ldy = m->ldY; a.w0 = w0; a.ldw = ldw; a.om = om; a.ldo = ldo;
  a.gam = (float*)w.tpc_gam.p; a.nvec = (float*)w.tpc_nvec.p; a.gacc = (float*)w.tpc_gacc.p;
  a.cstride = (int64_t)w.cap_centers * m->Denv * m->n;
  for (int k = 0; k < TPC_MAXL; ++k) { a.sb[k] = w.sb_ptr[k]; a.lds[k] = w.sb_ld[k]; }
  a.Ybar = (float*)w.Ybar.p; a.ybar_pstride = (int64_t)w.cap_edges * m->Denv;
  { int part[AL_MAX_LAYERS + 1]; al_ybar_layout(m, part); a.ybar_part0 = part[0]; a.ybar_partL = part[L]; }
  const int want[3] = {TPC<LM, NL>::NNZ1, TPC<LM, NL>::NNZ2, TPC<LM, NL>::NNZ3};
  float* dst[3] = {a.kv1, a.kv2, a.kv3};
  for (int k = 0; k < NL; ++k) {
    const TPLayerHost& h = m->tp_host[k];
    if ((int)h.dp_val.size() != want[k]) { al_set_error(m, "tpc: pattern size mismatch"); return ALLEGRO_ERR_BAD_ARG; }
    memcpy(dst[k], h.dp_val.data(), sizeof(float) * want[k]);
  }
  return ALLEGRO_OK;
}

template <int LM, int NL, int L>
int tpc_launch_fwd(allegro_model* m, Work& w, int nc, const float* om, int ldo, const float* w0, int ldw, float* xs, int ldx) {
  TPC<LM, NL> a{};
  AL_CHECK((tpc_fill<LM, NL>(m, w, L, nc, om, ldo, w0, ldw, a)));
  a.xs = xs; a.ldx = ldx;
  constexpr int WPB = 4;
  const int64_t warps = (int64_t)nc * (m->n / 32);
  const size_t sm = (size_t)WPB * tpc_ring_floats<TpcEnv<LM>::DENV>(0) * 4;
  if constexpr (LM <= 2) {
    k_tpc_fwd_rb<LM, NL, L, WPB><<<(unsigned)((warps + WPB - 1) / WPB), WPB * 32, 0, m->stream>>>(a);
  } else {
    static AttrOnce once;
    if (once.need(m->device)) { AL_CUDA(m, cudaFuncSetAttribute(k_tpc_fwd<LM, NL, L, WPB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm)); once.done(m->device); }
    k_tpc_fwd<LM, NL, L, WPB><<<(unsigned)((warps + WPB - 1) / WPB), WPB * 32, sm, m->stream>>>(a);
  }
  m->launches++;
  AL_CUDA(m, cudaGetLastError());
  return ALLEGRO_OK;
}

template <int LM, int NL, int L>
int tpc_launch_bwd(allegro_model* m, Work& w, int nc, const float* om, int ldo, const float* w0, int ldw, float* ombar, int ldob,
                   float* w0bar) {
  TPC<LM, NL> a{};
  AL_CHECK((tpc_fill<LM, NL>(m, w, L, nc, om, ldo, w0, ldw, a)));
  a.ombar = ombar; a.ldob = ldob; a.w0bar = w0bar;
  constexpr int WPB = 4;
  const int64_t warps = (int64_t)nc * (m->n / 32);
  constexpr int NXA = (L == 1) ? (NL < 2 ? 1 : 2) : 1;
  const size_t sm = (size_t)WPB * tpc_ring_floats<TpcEnv<LM>::DENV>(NXA) * 4;
  static AttrOnce once;
  if (once.need(m->device)) { AL_CUDA(m, cudaFuncSetAttribute(k_tpc_bwd<LM, NL, L, WPB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm)); once.done(m->device); }
  k_tpc_bwd<LM, NL, L, WPB><<<(unsigned)((warps + WPB - 1) / WPB), WPB * 32, sm, m->stream>>>(a);
  m->launches++;
  AL_CUDA(m, cudaGetLastError());
  return ALLEGRO_OK;
}

