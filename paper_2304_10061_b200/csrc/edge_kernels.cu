// Non-GEMM kernels of the hot path: active-edge compaction + edge geometry / radial / angular basis
// (SURVEY.md §8(a) step 2), first two-body layer (step 3), environment sum + tensor product (steps 5-7,
// PAPER.md Eq. (2) :132-138 and Fig. 3 :180), energies (steps 9-10), and the
// hand-written backward of all of them (step 11), NVE helpers (step 12).
#include <cmath>

#include "kernels.h"
#include "h16.cuh"

namespace {
// streamed rows (written or read once per step): keep them out of L1
__device__ __forceinline__ void ek_st4(float* p, const float4 v) {
  asm volatile("st.global.L1::no_allocate.v4.f32 [%0], {%1,%2,%3,%4};" ::"l"(p), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}
__device__ __forceinline__ float4 ek_ld4(const float* p) {
  float4 v;
  asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
  return v;
}

#define FULLMASK 0xffffffffu

__device__ __forceinline__ float silu_f(float z) { return z / (1.0f + expf(-z)); }
// tensor-core modes (TF32 / 16-bit operands): the value feeds a TF32 / fp16 MMA operand, ex2.approx + rcp.approx (error ~1e-7)
// is far below its rounding; the fp32 modes keep expf and the IEEE division
__device__ __forceinline__ float silu_fast(float z) {
  float e, r;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(e) : "f"(z * -1.4426950408889634f));
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(1.0f + e));
  return z * r;
}
__device__ __forceinline__ float dsilu_f(float z) {
  float s = 1.0f / (1.0f + expf(-z));
  return s * (1.0f + z * (1.0f - s));
}
__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(FULLMASK, v, o);
  return v;
}
__device__ __forceinline__ double warp_sum_d(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(FULLMASK, v, o);
  return v;
}

// ---- real spherical harmonics, component normalisation, l <= 3 (SURVEY §8(c) S4 closed forms) ------
#define SQ3 1.7320508075688772f
#define SQ5 2.23606797749979f
#define SQ15 3.872983346207417f
#define SQ7 2.6457513110645907f
#define C3A 2.091650066335189f    /* sqrt(35/8) */
#define C3B 10.246950765959598f   /* sqrt(105)  */
#define C3C 1.620185174601965f    /* sqrt(21/8) */

__device__ __forceinline__ void sph_harm(float x, float y, float z, int lmax, float* Y) {
  Y[0] = 1.0f;
  if (lmax >= 1) { Y[1] = SQ3 * y; Y[2] = SQ3 * z; Y[3] = SQ3 * x; }
  if (lmax >= 2) {
    Y[4] = SQ15 * x * y; Y[5] = SQ15 * y * z; Y[6] = 0.5f * SQ5 * (3.0f * z * z - 1.0f);
    Y[7] = SQ15 * x * z; Y[8] = 0.5f * SQ15 * (x * x - y * y);
  }
  if (lmax >= 3) {
    Y[9] = C3A * y * (3.0f * x * x - y * y); Y[10] = C3B * x * y * z; Y[11] = C3C * y * (5.0f * z * z - 1.0f);
    Y[12] = 0.5f * SQ7 * (5.0f * z * z * z - 3.0f * z); Y[13] = C3C * x * (5.0f * z * z - 1.0f);
    Y[14] = 0.5f * C3B * z * (x * x - y * y); Y[15] = C3A * x * (x * x - 3.0f * y * y);
  }
}

// v = sum_b Ybar[b] * grad Y_b (gradient of the polynomial forms above; only its tangential part is used)
__device__ __forceinline__ void sph_harm_vjp(float x, float y, float z, int lmax, const float* g, float& vx, float& vy,
                                             float& vz) {
  vx = vy = vz = 0.f;
  if (lmax >= 1) { vy += SQ3 * g[1]; vz += SQ3 * g[2]; vx += SQ3 * g[3]; }
  if (lmax >= 2) {
    vx += SQ15 * (y * g[4] + z * g[7] + x * g[8]);
    vy += SQ15 * (x * g[4] + z * g[5] - y * g[8]);
    vz += SQ15 * (y * g[5] + x * g[7]) + 3.0f * SQ5 * z * g[6];
  }
  if (lmax >= 3) {
    float xx = x * x, yy = y * y, zz = z * z;
    vx += 6.0f * C3A * x * y * g[9] + C3B * y * z * g[10] + C3C * (5.0f * zz - 1.0f) * g[13] + C3B * x * z * g[14] +
          3.0f * C3A * (xx - yy) * g[15];
    vy += 3.0f * C3A * (xx - yy) * g[9] + C3B * x * z * g[10] + C3C * (5.0f * zz - 1.0f) * g[11] - C3B * y * z * g[14] -
          6.0f * C3A * x * y * g[15];
    vz += C3B * x * y * g[10] + 10.0f * C3C * y * z * g[11] + 0.5f * SQ7 * (15.0f * zz - 3.0f) * g[12] +
          10.0f * C3C * x * z * g[13] + 0.5f * C3B * (xx - yy) * g[14];
  }
}

// x^n for a small non-negative integer n (the envelope exponent), fp64
__device__ __forceinline__ double ipow_d(double x, int n) {
  double r = 1.0, b = x;
  while (n > 0) {
    if (n & 1) r *= b;
    b *= b;
    n >>= 1;
  }
  return r;
}

// species index clamped into [0, S): an out-of-range value (caller error) is reported through the status flag by
// k_zero_check (ALLEGRO_ERR_BAD_ARG at the next host synchronisation) and must never index a table out of bounds
__device__ __forceinline__ int zc(int z, int S) { return min(max(z, 0), S - 1); }

// ---- active-edge count / compaction + geometry ------------------------------------------------------
// rc: the cutoff of this ordered pair, r_cut or r_c[Z_i][Z_j] (allegro_set_pair_cutoffs)
__device__ __forceinline__ bool edge_vec(const EdgeGeomArgs& a, int i, int64_t e, int& j, double& dx, double& dy,
                                         double& dz, double& r2, double& rc) {
  j = a.j[e];
  rc = a.rc_pair ? a.rc_pair[zc(a.species[i], a.S) * a.S + zc(a.species[j], a.S)] : a.rc;
  dx = __dadd_rn(a.pos[3 * (int64_t)j + 0] - a.pos[3 * (int64_t)i + 0], __dmul_rn((double)a.shift[3 * e + 0], a.box[0]));
  dy = __dadd_rn(a.pos[3 * (int64_t)j + 1] - a.pos[3 * (int64_t)i + 1], __dmul_rn((double)a.shift[3 * e + 1], a.box[1]));
  dz = __dadd_rn(a.pos[3 * (int64_t)j + 2] - a.pos[3 * (int64_t)i + 2], __dmul_rn((double)a.shift[3 * e + 2], a.box[2]));
  // the canonical expression of the list build: (dx*dx + dy*dy) + dz*dz, fp64, no FMA contraction, so the
  // active-edge decision r2 < rc^2 is the same one an IEEE host evaluation takes (bit-exact counts with pair cutoffs)
  r2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
  return r2 < __dmul_rn(rc, rc);
}

__global__ void k_active_count(EdgeGeomArgs a, int* __restrict__ deg) {
  int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (warp >= a.nc) return;
  int i = (int)(a.c0 + warp);
  int64_t b = a.row_ptr[i], e = a.row_ptr[i + 1];
  int cnt = 0;
  for (int64_t k = b + lane; k < e; k += 32) {
    int j; double dx, dy, dz, r2, rc;
    cnt += edge_vec(a, i, k, j, dx, dy, dz, r2, rc) ? 1 : 0;
  }
  cnt = (int)warp_sum((float)cnt);
  if (lane == 0) deg[warp] = cnt;
}

// m_act[0] = active edges of this chunk; (int64*)(m_act + 2) accumulates the total over the chunks of one compute call
__global__ void k_set_mact(const int64_t* __restrict__ rowa, int nc, int* __restrict__ m_act) {
  m_act[0] = (int)rowa[nc];
  *reinterpret_cast<long long*>(m_act + 2) += (long long)rowa[nc];
}

__global__ void k_geom_fill(EdgeGeomArgs a, const int64_t* __restrict__ rowa, int* __restrict__ ei, int* __restrict__ ej,
                            float4* __restrict__ geo, float* __restrict__ u, float* __restrict__ du,
                            float* __restrict__ B, float* __restrict__ dB, float* __restrict__ Y, int Denv, int ldy,
                            int* __restrict__ flags, float* __restrict__ sig, const double* __restrict__ sigma) {
  int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (warp >= a.nc) return;
  int i = (int)(a.c0 + warp);
  int64_t b = a.row_ptr[i], e = a.row_ptr[i + 1];
  int64_t out0 = rowa[warp];
  int cnt = 0;
  for (int64_t kb = b; kb < e; kb += 32) {
    int64_t k = kb + lane;
    int j = 0; double dx = 0, dy = 0, dz = 0, r2 = 0, rc = a.rc;
    bool ok = (k < e) && edge_vec(a, i, k, j, dx, dy, dz, r2, rc);
    unsigned mask = __ballot_sync(FULLMASK, ok);
    if (ok) {
      int64_t o = out0 + cnt + __popc(mask & ((1u << lane) - 1u));
      double r = sqrt(r2);
      if (!(r > 0.0)) { atomicOr(&flags[1], 1); r = 1.0; }
      double inv = 1.0 / r;
      float hx = (float)(dx * inv), hy = (float)(dy * inv), hz = (float)(dz * inv);
      ei[o] = i; ej[o] = j;
      sig[o] = (float)sigma[zc(a.species[i], a.S)];
      geo[o] = make_float4(hx, hy, hz, (float)r);
      // envelope (fp64; PAPER.md:222 via SURVEY S2)
      double x = r / rc, p = (double)a.p;
      double xp1 = ipow_d(x, a.p - 1), xp = xp1 * x;   // integer power by repeated squaring instead of pow()
      double uu = 1.0 - 0.5 * (p + 1.0) * (p + 2.0) * xp + p * (p + 2.0) * xp * x - 0.5 * p * (p + 1.0) * xp * x * x;
      double dud = -0.5 * p * (p + 1.0) * (p + 2.0) * xp1 * (1.0 - x) * (1.0 - x) / rc;
      u[o] = (float)uu; du[o] = (float)dud;
      double pref = sqrt(2.0 / rc);
      if (a.bfreq) {
        // trained per-ordered-pair angular frequencies w_n: b_n = sqrt(2/rc) sin(w_n r) / r
        const double* wq = a.bfreq + ((size_t)zc(a.species[i], a.S) * a.S + zc(a.species[j], a.S)) * a.NB;
        for (int nb = 0; nb < a.NB; ++nb) {
          double wn = wq[nb], sn, cn;
          sincos(wn * r, &sn, &cn);
          double bn = pref * sn * inv;
          double dbn = pref * (wn * cn * inv - sn * inv * inv);
          B[o * a.NB + nb] = (float)(bn * uu);
          dB[o * a.NB + nb] = (float)(dbn * uu + bn * dud);
        }
      } else {
        // Bessel basis by the angle-addition recurrence in fp64
        double th = M_PI * x, s1, c1;
        sincos(th, &s1, &c1);
        double sn = s1, cn = c1;
        for (int nb = 1; nb <= a.NB; ++nb) {
          double bn = pref * sn * inv;
          double dbn = pref * ((double)nb * M_PI / rc * cn * inv - sn * inv * inv);
          B[o * a.NB + nb - 1] = (float)(bn * uu);
          dB[o * a.NB + nb - 1] = (float)(dbn * uu + bn * dud);
          double s2 = sn * c1 + cn * s1, c2 = cn * c1 - sn * s1;
          sn = s2; cn = c2;
        }
      }
      float yy[16];
      sph_harm(hx, hy, hz, a.lmax, yy);
      for (int q = 0; q < ldy; ++q) Y[o * ldy + q] = (q < Denv) ? yy[q] : 0.f;
    }
    cnt += __popc(mask);
  }
}

// ---- first two-body layer: one-hot rows + Bessel matvec ----------------------------------
// z_0[e, :] = W[Z_i, :] + W[S + Z_j, :] + sum_q B_q(e) W[2S + q, :]; a thread owns 4 consecutive outputs
// (float4 I/O, the weight rows come from L1) of one edge at a time.
constexpr int TB0_EDGES = 64;
__global__ void __launch_bounds__(256)
k_twobody0(const int* __restrict__ m_ptr, const int* __restrict__ ei, const int* __restrict__ ej,
           const int32_t* __restrict__ species, const float* __restrict__ B, const float* __restrict__ u,
           const float* __restrict__ W, int S, int NB, int H, float* __restrict__ z, float* __restrict__ act, int ldact,
           int scale_u, int hfmt /* -1: fp32 outputs; 0 / 1: z and act stored as fp16 / bf16 (16-bit operand modes) */,
           int fast /* 1: silu_fast (tensor-core precision modes) */) {
  const int M = *m_ptr;
  const int64_t e_base = (int64_t)blockIdx.x * TB0_EDGES;
  if (e_base >= M) return;
  __shared__ float sB[TB0_EDGES][16];
  __shared__ int sZi[TB0_EDGES], sZj[TB0_EDGES];
  __shared__ float sU[TB0_EDGES];
  const int tid = threadIdx.x;
  for (int idx = tid; idx < TB0_EDGES * 16; idx += 256) {
    int r = idx >> 4, q = idx & 15;
    sB[r][q] = (q < NB && e_base + r < M) ? B[(e_base + r) * NB + q] : 0.f;
  }
  if (tid < TB0_EDGES) {
    int64_t e = e_base + tid;
    sZi[tid] = (e < M) ? zc(species[ei[e]], S) : 0;
    sZj[tid] = (e < M) ? zc(species[ej[e]], S) : 0;
    sU[tid] = (e < M) ? u[e] : 0.f;
  }
  __syncthreads();
  const int H4 = H >> 2;
  if (256 % H4 == 0 && NB <= 8) {
    // a thread keeps its 4 output columns for all its edges: the Bessel weight rows stay in registers
    const int k4 = (tid % H4) * 4, rstep = 256 / H4;
    float4 wb[8];
#pragma unroll
    for (int q = 0; q < 8; ++q)
      wb[q] = (q < NB) ? __ldg(reinterpret_cast<const float4*>(W + (size_t)(2 * S + q) * H + k4)) : make_float4(0.f, 0.f, 0.f, 0.f);
    for (int r = tid / H4; r < TB0_EDGES; r += rstep) {
      const int64_t e = e_base + r;
      if (e >= M) break;
      float4 a0 = __ldg(reinterpret_cast<const float4*>(W + (size_t)sZi[r] * H + k4));
      float4 a1 = __ldg(reinterpret_cast<const float4*>(W + (size_t)(S + sZj[r]) * H + k4));
      float4 acc = make_float4(a0.x + a1.x, a0.y + a1.y, a0.z + a1.z, a0.w + a1.w);
#pragma unroll
      for (int q = 0; q < 8; ++q) {
        const float b = sB[r][q];   // (zero beyond NB)
        acc.x = fmaf(b, wb[q].x, acc.x); acc.y = fmaf(b, wb[q].y, acc.y); acc.z = fmaf(b, wb[q].z, acc.z); acc.w = fmaf(b, wb[q].w, acc.w);
      }
      if (hfmt < 0) ek_st4(z + e * H + k4, acc); else h16_store4(z, (size_t)e * H + k4, acc, hfmt);
      const float us = scale_u ? sU[r] : 1.0f;
      { const float4 o4 = fast ? make_float4(us * silu_fast(acc.x), us * silu_fast(acc.y), us * silu_fast(acc.z), us * silu_fast(acc.w))
                               : make_float4(us * silu_f(acc.x), us * silu_f(acc.y), us * silu_f(acc.z), us * silu_f(acc.w));
        if (hfmt < 0) ek_st4(act + e * ldact + k4, o4); else h16_store4(act, (size_t)e * ldact + k4, o4, hfmt); }
    }
    return;
  }
  for (int idx = tid; idx < TB0_EDGES * H4; idx += 256) {
    const int r = idx / H4, k4 = (idx - r * H4) * 4;
    const int64_t e = e_base + r;
    if (e >= M) break;
    float4 a0 = __ldg(reinterpret_cast<const float4*>(W + (size_t)sZi[r] * H + k4));
    float4 a1 = __ldg(reinterpret_cast<const float4*>(W + (size_t)(S + sZj[r]) * H + k4));
    float4 acc = make_float4(a0.x + a1.x, a0.y + a1.y, a0.z + a1.z, a0.w + a1.w);
    for (int q = 0; q < NB; ++q) {
      float4 w4 = __ldg(reinterpret_cast<const float4*>(W + (size_t)(2 * S + q) * H + k4));
      float b = sB[r][q];
      acc.x = fmaf(b, w4.x, acc.x); acc.y = fmaf(b, w4.y, acc.y); acc.z = fmaf(b, w4.z, acc.z); acc.w = fmaf(b, w4.w, acc.w);
    }
    if (hfmt < 0) ek_st4(z + e * H + k4, acc); else h16_store4(z, (size_t)e * H + k4, acc, hfmt);
    const float us = scale_u ? sU[r] : 1.0f;
    { const float4 o4 = make_float4(us * silu_f(acc.x), us * silu_f(acc.y), us * silu_f(acc.z), us * silu_f(acc.w));
        if (hfmt < 0) ek_st4(act + e * ldact + k4, o4); else h16_store4(act, (size_t)e * ldact + k4, o4, hfmt); }
  }
}

// ---- tensor track -------------------------------------------------------------------------------------
struct TPArgs {
  const int64_t* rowa;
  const float* om; int ldo;       // omega^L  [M][(l,n)]
  const float* Y; int Denv, ldy;
  const float* Vin;               // [M][Din][n] or null (FIRST)
  const float* w0; int ldw;       // FIRST: w^0 [M][(l,n)]
  const int *v0_l, *v0_y, *env_l;
  TPLayerDev t;
  int n, lmax; float c_env;
  float* Tout;                    // [M][Dout][n] or null
  float* xs; int ldx;             // scalars s -> xs[e*ldx + nn]
  float* gamma_out;               // [Nc][Denv][n] or null
  // backward
  const float* VbarL;             // [M][Dout][n] or null
  const float* sbar; int lds;
  float* Vbar_prev;               // [M][Din][n]
  float* ombar; int ldob;
  float* w0bar;                   // FIRST: [M][(l,n)] with ld = ldob
  float* Ybar;
};

template <bool FIRST>
__device__ __forceinline__ float v_load(const TPArgs& a, int64_t e, int comp, int nn) {
  if (FIRST) return a.w0[e * a.ldw + a.v0_l[comp] * a.n + nn] * a.Y[e * a.ldy + a.v0_y[comp]];
  return a.Vin[(e * a.t.Din + comp) * a.n + nn];
}

__device__ __forceinline__ void tp_gamma_M(const TPArgs& a, int64_t e0, int64_t e1, float* G, float* Ms) {
  const int n = a.n;
  for (int idx = threadIdx.x; idx < a.Denv * n; idx += blockDim.x) {
    int b = idx / n, nn = idx - b * n, l = a.env_l[b];
    float acc = 0.f;
    for (int64_t e = e0; e < e1; ++e) acc = fmaf(a.om[e * a.ldo + l * n + nn], a.Y[e * a.ldy + b], acc);
    G[idx] = a.c_env * acc;
  }
  __syncthreads();
  for (int idx = threadIdx.x; idx < a.t.npairs * n; idx += blockDim.x) {
    int p = idx / n, nn = idx - p * n;
    float acc = 0.f;
    for (int k = a.t.pair_ptr[p]; k < a.t.pair_ptr[p + 1]; ++k) acc = fmaf(a.t.ent_val[k], G[a.t.ent_b[k] * n + nn], acc);
    Ms[idx] = acc;
  }
  __syncthreads();
}

// One block per center: Gamma_i (Eq. (2) line 2), M_i = K . Gamma_i, then T_e = V_e . M_i for its edges.
template <bool FIRST>
__global__ void __launch_bounds__(256) k_tp_fwd(TPArgs a) {
  extern __shared__ float smem[];
  const int n = a.n;
  float* G = smem;
  float* Ms = smem + a.Denv * n;
  int c = blockIdx.x;
  int64_t e0 = a.rowa[c], e1 = a.rowa[c + 1];
  if (e1 <= e0) return;
  tp_gamma_M(a, e0, e1, G, Ms);
  if (a.gamma_out)
    for (int idx = threadIdx.x; idx < a.Denv * n; idx += blockDim.x) a.gamma_out[(size_t)c * a.Denv * n + idx] = G[idx];
  int deg = (int)(e1 - e0);
  for (int idx = threadIdx.x; idx < deg * n; idx += blockDim.x) {
    int el = idx / n, nn = idx - el * n;
    int64_t e = e0 + el;
    for (int cc = 0; cc < a.t.Dout; ++cc) {
      float acc = 0.f;
      for (int k = a.t.c_ptr[cc]; k < a.t.c_ptr[cc + 1]; ++k)
        acc = fmaf(v_load<FIRST>(a, e, a.t.c_a[k], nn), Ms[a.t.c_p[k] * n + nn], acc);
      if (cc == 0) a.xs[e * a.ldx + nn] = acc;
      if (a.Tout) a.Tout[(e * a.t.Dout + cc) * n + nn] = acc;
    }
  }
}

__device__ __forceinline__ float tbar_load(const TPArgs& a, int64_t e, int cc, int nn) {
  float v = a.VbarL ? a.VbarL[(e * a.t.Dout + cc) * a.n + nn] : 0.f;
  if (cc == 0) v += a.sbar[e * a.lds + nn];
  return v;
}

template <bool FIRST>
__global__ void __launch_bounds__(256) k_tp_bwd(TPArgs a) {
  extern __shared__ float smem[];
  const int n = a.n, nl = a.lmax + 1;
  float* G = smem;
  float* Ms = smem + a.Denv * n;
  int c = blockIdx.x;
  int64_t e0 = a.rowa[c], e1 = a.rowa[c + 1];
  if (e1 <= e0) return;
  int deg = (int)(e1 - e0);
  tp_gamma_M(a, e0, e1, G, Ms);
  // V-bar^{L-1}_e[a] = sum_c M[a,c] T-bar_e[c]
  for (int idx = threadIdx.x; idx < deg * n; idx += blockDim.x) {
    int el = idx / n, nn = idx - el * n;
    int64_t e = e0 + el;
    for (int aa = 0; aa < a.t.Din; ++aa) {
      float acc = 0.f;
      for (int k = a.t.a_ptr[aa]; k < a.t.a_ptr[aa + 1]; ++k)
        acc = fmaf(Ms[a.t.a_p[k] * n + nn], tbar_load(a, e, a.t.a_c[k], nn), acc);
      a.Vbar_prev[(e * a.t.Din + aa) * n + nn] = acc;
    }
  }
  __syncthreads();
  // M-bar[p] = sum_e V_e[a_p] T-bar_e[c_p]   (overwrites M)
  for (int idx = threadIdx.x; idx < a.t.npairs * n; idx += blockDim.x) {
    int p = idx / n, nn = idx - p * n;
    int aa = a.t.pair_a[p], cc = a.t.pair_c[p];
    float acc = 0.f;
    for (int64_t e = e0; e < e1; ++e) acc = fmaf(v_load<FIRST>(a, e, aa, nn), tbar_load(a, e, cc, nn), acc);
    Ms[idx] = acc;
  }
  __syncthreads();
  // Gamma-bar[b] = sum_{(a,c)} K[a,b,c] M-bar[a,c]   (overwrites Gamma)
  for (int idx = threadIdx.x; idx < a.Denv * n; idx += blockDim.x) {
    int b = idx / n, nn = idx - b * n;
    float acc = 0.f;
    for (int k = a.t.b_ptr[b]; k < a.t.b_ptr[b + 1]; ++k) acc = fmaf(a.t.b_val[k], Ms[a.t.b_p[k] * n + nn], acc);
    G[idx] = acc;
  }
  __syncthreads();
  // omega-bar_e[l,n] = c_env sum_m Gamma-bar[(l,m),n] Y_e[(l,m)]
  for (int idx = threadIdx.x; idx < deg * nl * n; idx += blockDim.x) {
    int el = idx / (nl * n), rem = idx - el * nl * n, l = rem / n, nn = rem - l * n;
    int64_t e = e0 + el;
    float acc = 0.f;
    for (int b = l * l; b < (l + 1) * (l + 1); ++b) acc = fmaf(G[b * n + nn], a.Y[e * a.ldy + b], acc);
    a.ombar[e * a.ldob + l * n + nn] = a.c_env * acc;
  }
  // Y-bar_e[b] += c_env sum_n omega_e[l(b),n] Gamma-bar[b,n]
  int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nw = blockDim.x >> 5;
  for (int item = warp; item < deg * a.Denv; item += nw) {
    int el = item / a.Denv, b = item - el * a.Denv, l = a.env_l[b];
    int64_t e = e0 + el;
    float acc = 0.f;
    for (int nn = lane; nn < n; nn += 32) acc = fmaf(a.om[e * a.ldo + l * n + nn], G[b * n + nn], acc);
    acc = warp_sum(acc);
    if (lane == 0) a.Ybar[e * a.Denv + b] += a.c_env * acc;
  }
  if (FIRST) {
    __syncthreads();
    // V^0 = w^0 (x) Y :  w0-bar[l,n] = sum_{a in l} V-bar^0[a,n] Y[a] ; Y-bar[a] += sum_n w0[l(a),n] V-bar^0[a,n]
    for (int idx = threadIdx.x; idx < deg * nl * n; idx += blockDim.x) {
      int el = idx / (nl * n), rem = idx - el * nl * n, l = rem / n, nn = rem - l * n;
      int64_t e = e0 + el;
      float acc = 0.f;
      for (int aa = 0; aa < a.t.Din; ++aa)
        if (a.v0_l[aa] == l) acc = fmaf(a.Vbar_prev[(e * a.t.Din + aa) * n + nn], a.Y[e * a.ldy + a.v0_y[aa]], acc);
      a.w0bar[e * a.ldob + l * n + nn] = acc;
    }
    for (int item = warp; item < deg * a.t.Din; item += nw) {
      int el = item / a.t.Din, aa = item - el * a.t.Din;
      int64_t e = e0 + el;
      float acc = 0.f;
      for (int nn = lane; nn < n; nn += 32)
        acc = fmaf(a.w0[e * a.ldw + a.v0_l[aa] * n + nn], a.Vbar_prev[(e * a.t.Din + aa) * n + nn], acc);
      acc = warp_sum(acc);
      if (lane == 0) a.Ybar[e * a.Denv + a.v0_y[aa]] += acc;
    }
  }
}

// ---- energies (fp64 final stage) -------------------------------------------------------------
__global__ void k_energy(const int64_t* __restrict__ rowa, int nc, int64_t c0, const float* __restrict__ xf, int d,
                         const double* __restrict__ w_eff, const int32_t* __restrict__ species, int S,
                         const double* __restrict__ sigma, const double* __restrict__ mu, double* __restrict__ e_atom) {
  int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (warp >= nc) return;
  int64_t e0 = rowa[warp], e1 = rowa[warp + 1];
  double acc = 0.0;
  for (int64_t e = e0; e < e1; ++e)
    for (int k = lane; k < d; k += 32) acc += (double)xf[e * d + k] * w_eff[k];
  acc = warp_sum_d(acc);
  if (lane == 0) {
    int z = zc(species[c0 + warp], S);
    e_atom[c0 + warp] = sigma[z] * acc + mu[z];
  }
}

// E-hat_i from the edge-energy partials written by the last latent GEMM (EPI_LATENT_LAST): lanes take the
// center's edges, each sums its partials in fixed order, then a fixed-order warp reduction in fp64.
__global__ void k_energy_parts(const int64_t* __restrict__ rowa, int nc, int64_t c0, const double* __restrict__ epart,
                               int nparts, int64_t pstride, const int32_t* __restrict__ species, int S,
                               const double* __restrict__ sigma, const double* __restrict__ mu, double* __restrict__ e_atom) {
  int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (warp >= nc) return;
  int64_t e0 = rowa[warp], e1 = rowa[warp + 1];
  double acc = 0.0;
  for (int64_t e = e0 + lane; e < e1; e += 32) {
    double s = 0.0;
    for (int p = 0; p < nparts; ++p) s += epart[(int64_t)p * pstride + e];
    acc += s;
  }
  acc = warp_sum_d(acc);
  if (lane == 0) {
    int z = zc(species[c0 + warp], S);
    e_atom[c0 + warp] = sigma[z] * acc + mu[z];
  }
}

__global__ void k_sum_f64(const double* __restrict__ x, int64_t n, double* __restrict__ out) {
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

// zb = c * u * xbar * silu'(z) ; ubar += c * <xbar, silu(z)>      (one warp per edge, float4 lanes)
// xbar == nullptr: the incoming gradient is the rank-1 x-bar^{NL}_e = sigma_{Z_i(e)} * w_eff (never materialised).
__global__ void k_bwd_prep(const int* __restrict__ m_ptr, const float* __restrict__ xbar, int ldx, const float* __restrict__ z,
                           int ldz, const float* __restrict__ u, float c, float* __restrict__ zb, int ldzb, int width,
                           float* __restrict__ ubar, const float* __restrict__ sig, const float* __restrict__ w_eff) {
  const int M = *m_ptr;
  int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (warp >= M) return;
  int64_t e = warp;
  float cu = c * u[e], acc = 0.f;
  float sg = xbar ? 0.f : sig[e];
  for (int k = lane * 4; k < width; k += 128) {
    float4 x4 = xbar ? *reinterpret_cast<const float4*>(xbar + e * ldx + k) : *reinterpret_cast<const float4*>(w_eff + k);
    float4 z4 = *reinterpret_cast<const float4*>(z + e * ldz + k);
    float xb[4] = {x4.x, x4.y, x4.z, x4.w}, zz[4] = {z4.x, z4.y, z4.z, z4.w}, o[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      if (!xbar) xb[j] *= sg;
      float s = 1.0f / (1.0f + expf(-zz[j]));
      acc = fmaf(xb[j], zz[j] * s, acc);
      o[j] = cu * xb[j] * (s * (1.0f + zz[j] * (1.0f - s)));
    }
    *reinterpret_cast<float4*>(zb + e * ldzb + k) = make_float4(o[0], o[1], o[2], o[3]);
  }
  acc = warp_sum(acc);
  if (lane == 0) ubar[e] += c * acc;
}

// Last backward stage: B-bar through the first two-body layer, r-bar, angular part, dE/dr_e, force scatter.
// Block = 32 edges x 8 lanes.  The block stages its 32 rows of z-bar_0 [H] and the Bessel rows of the first
// two-body weight matrix in shared memory; lane q of an edge forms B-bar_q = <z-bar_0, W[2S+q,:]> (and q+8 when
// n_bessel > 8), the 8 lanes then share the sums over the u-bar and Y-bar partial buffers (fixed order), one
// lane evaluates the spherical-harmonic vjp and six lanes issue the fp64 force atomics (F_i += g, F_j -= g).
constexpr int EB_EDGES = 32;
__global__ void __launch_bounds__(256)
k_edge_bwd(const int* __restrict__ m_ptr, const float* __restrict__ zb1, int ldz, const float* __restrict__ W, int S, int NB,
           int H, const float4* __restrict__ geo, const float* __restrict__ du, const float* __restrict__ dB,
           const float* __restrict__ ubar, int n_uparts, int64_t ubar_pstride, const float* __restrict__ Ybar, int nparts,
           int64_t ybar_pstride, int Denv, int lmax, const int* __restrict__ ei, const int* __restrict__ ej,
           float* __restrict__ ge, double* __restrict__ force) {
  extern __shared__ float4 eb_smem4[];
  float* Ws = reinterpret_cast<float*>(eb_smem4);     // [NB][H + 4]
  const int HP = H + 4;
  float* zs = Ws + NB * HP;                           // [32][H + 4]
  const int M = *m_ptr;
  const int64_t e_base = (int64_t)blockIdx.x * EB_EDGES;
  if (e_base >= M) return;
  const int tid = threadIdx.x;
  const int el = tid >> 3, q = tid & 7, lane = tid & 31;
  const int64_t e = e_base + el;
  const bool live = e < M;
  const int64_t ee = live ? e : (int64_t)M - 1;
  // Per-edge operands first: the first batch of u-bar partials (lane q takes parts q, q+8, ...), of Y-bar partials
  // (lane q sums components q and q+8 over the parts), du and dB are independent loads issued before the staging
  // loops, so their latency overlaps the staging (ncu had 65 % of this kernel's stall samples on the serial
  // partial-sum loops that used to follow the barrier).  The order of every sum is fixed.
  float ut[4], ya[4], yc[4];
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    const int pu = q + 8 * k;
    ut[k] = (pu < n_uparts) ? ubar[(int64_t)pu * ubar_pstride + ee] : 0.f;
    const float* yp = Ybar + (int64_t)k * ybar_pstride + ee * Denv;
    ya[k] = (k < nparts && q < Denv) ? yp[q] : 0.f;
    yc[k] = (k < nparts && q + 8 < Denv) ? yp[q + 8] : 0.f;
  }
  const float duv = du[ee];
  const float dB0 = (q < NB) ? dB[ee * NB + q] : 0.f, dB1 = (q + 8 < NB) ? dB[ee * NB + q + 8] : 0.f;
  for (int idx = tid; idx < NB * (H / 4); idx += 256) {
    int qw = idx / (H / 4), k4 = (idx - qw * (H / 4)) * 4;
    *reinterpret_cast<float4*>(Ws + qw * HP + k4) = __ldg(reinterpret_cast<const float4*>(W + (size_t)(2 * S + qw) * H + k4));
  }
  for (int idx = tid; idx < EB_EDGES * (H / 4); idx += 256) {
    int r = idx / (H / 4), k4 = (idx - r * (H / 4)) * 4;
    float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
    if (e_base + r < M) v = ek_ld4(zb1 + (e_base + r) * ldz + k4);
    *reinterpret_cast<float4*>(zs + r * HP + k4) = v;
  }
  __syncthreads();
  // B-bar_q . dB_q
  float pr = 0.f;
  for (int qq = q; qq < NB; qq += 8) {
    float acc = 0.f;
    const float* zr = zs + el * HP;
    const float* wr = Ws + qq * HP;
    for (int k4 = 0; k4 < H; k4 += 4) {
      float4 z4 = *reinterpret_cast<const float4*>(zr + k4);
      float4 w4 = *reinterpret_cast<const float4*>(wr + k4);
      acc = fmaf(z4.x, w4.x, acc); acc = fmaf(z4.y, w4.y, acc); acc = fmaf(z4.z, w4.z, acc); acc = fmaf(z4.w, w4.w, acc);
    }
    pr = fmaf(acc, (qq == q) ? dB0 : (qq == q + 8) ? dB1 : dB[ee * NB + qq], pr);
  }
  // remaining u-bar / Y-bar partials (more than 32 / 4 parts), four independent loads at a time
  float ub = (ut[0] + ut[1]) + (ut[2] + ut[3]);
  for (int p0 = q + 32; p0 < n_uparts; p0 += 32) {
    float t[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) t[k] = (p0 + 8 * k < n_uparts) ? ubar[(int64_t)(p0 + 8 * k) * ubar_pstride + ee] : 0.f;
    ub += (t[0] + t[1]) + (t[2] + t[3]);
  }
  pr = fmaf(ub, duv, pr);
  float ys0 = (ya[0] + ya[1]) + (ya[2] + ya[3]), ys1 = (yc[0] + yc[1]) + (yc[2] + yc[3]);
  for (int p0 = 4; p0 < nparts; p0 += 4) {
    float a[4], b[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const float* yp = Ybar + (int64_t)(p0 + k) * ybar_pstride + ee * Denv;
      a[k] = (p0 + k < nparts && q < Denv) ? yp[q] : 0.f;
      b[k] = (p0 + k < nparts && q + 8 < Denv) ? yp[q + 8] : 0.f;
    }
    ys0 += (a[0] + a[1]) + (a[2] + a[3]);
    ys1 += (b[0] + b[1]) + (b[2] + b[3]);
  }
#pragma unroll
  for (int o = 1; o < 8; o <<= 1) pr += __shfl_xor_sync(FULLMASK, pr, o);   // r-bar (all 8 lanes of the edge hold it)
  float yb[16];
#pragma unroll
  for (int b = 0; b < 16; ++b) yb[b] = __shfl_sync(FULLMASK, (b < 8) ? ys0 : ys1, (lane & ~7) + (b & 7));
  float gx = 0.f, gy = 0.f, gz = 0.f;
  if (q == 0) {
    float4 g4 = geo[ee];
    float vx, vy, vz;
    sph_harm_vjp(g4.x, g4.y, g4.z, lmax, yb, vx, vy, vz);
    float dot = vx * g4.x + vy * g4.y + vz * g4.z;
    float ir = 1.0f / g4.w;
    gx = pr * g4.x + (vx - dot * g4.x) * ir;
    gy = pr * g4.y + (vy - dot * g4.y) * ir;
    gz = pr * g4.z + (vz - dot * g4.z) * ir;
    if (ge && live) { ge[3 * e] = gx; ge[3 * e + 1] = gy; ge[3 * e + 2] = gz; }
  }
  // lanes 0-2: F_i[k] += g[k] ; lanes 3-5: F_j[k] -= g[k]   (summing the centre part per run of equal centres in
  // shared memory first, three atomics per run instead of per edge, measured slower: 0.139 -> 0.163 ms at config 1)
  const int src = lane & ~7;
  gx = __shfl_sync(FULLMASK, gx, src); gy = __shfl_sync(FULLMASK, gy, src); gz = __shfl_sync(FULLMASK, gz, src);
  if (live && q < 6) {
    const int k = (q < 3) ? q : q - 3;
    const float g = (k == 0) ? gx : (k == 1) ? gy : gz;
    const int atom = (q < 3) ? ei[e] : ej[e];
    atomicAdd(&force[3 * (int64_t)atom + k], (q < 3) ? (double)g : -(double)g);
  }
}

__global__ void k_zero_check(double* force, int64_t n3, const int32_t* __restrict__ species, int64_t n, int S, int* flags) {
  int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (force && i < n3) force[i] = 0.0;
  if (i < n && (unsigned)species[i] >= (unsigned)S) atomicOr(&flags[1], 2);
}
__global__ void k_zero_f64(double* p, int64_t n) {
  int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i < n) p[i] = 0.0;
}

// ---- NVE ---------------------------------------------------------------------------------
#define ACC_CONV 9.648533212e-3
__global__ void k_nve(double* pos, double* vel, const double* force, const int32_t* species, const double* mass, int S,
                      int64_t n, double dt, int drift) {
  int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= n) return;
  double im = ACC_CONV / mass[zc(species[i], S)];
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    double v = vel[3 * i + k] + (0.5 * dt) * (force[3 * i + k] * im);
    vel[3 * i + k] = v;
    if (drift) pos[3 * i + k] += dt * v;
  }
}

// ---- ZBL pair repulsion (reading in DESIGN.md section 2) -------------------------------------------
// phi_ij(r) = k_e Z_i Z_j / r * Phi(r / a_ij) * u(r / r_c) at the FLAT cutoff; E_i += 1/2 sum_j phi_ij and, since the
// list holds both orders of every pair, F_i = sum_j phi'(r_ij) rhat_ij is a pure gather over the centre's own row.
__global__ void k_zbl(EdgeGeomArgs a, const double* __restrict__ zn, double* __restrict__ e_atom, double* __restrict__ force) {
  int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (warp >= a.nc) return;
  int i = (int)(a.c0 + warp);
  int64_t b = a.row_ptr[i], e = a.row_ptr[i + 1];
  const double zi = zn[zc(a.species[i], a.S)], p = (double)a.p;
  double es = 0.0, fx = 0.0, fy = 0.0, fz = 0.0;
  for (int64_t k = b + lane; k < e; k += 32) {
    int j = a.j[k];
    double dx = (a.pos[3 * (int64_t)j + 0] - a.pos[3 * (int64_t)i + 0]) + (double)a.shift[3 * k + 0] * a.box[0];
    double dy = (a.pos[3 * (int64_t)j + 1] - a.pos[3 * (int64_t)i + 1]) + (double)a.shift[3 * k + 1] * a.box[1];
    double dz = (a.pos[3 * (int64_t)j + 2] - a.pos[3 * (int64_t)i + 2]) + (double)a.shift[3 * k + 2] * a.box[2];
    double r2 = dx * dx + dy * dy + dz * dz;
    if (!(r2 < a.rc * a.rc) || !(r2 > 0.0)) continue;
    double r = sqrt(r2), inv = 1.0 / r;
    double zj = zn[zc(a.species[j], a.S)];
    double ia = (pow(zi, 0.23) + pow(zj, 0.23)) / 0.46850, xs = r * ia;
    double e1 = 0.18175 * exp(-3.19980 * xs), e2 = 0.50986 * exp(-0.94229 * xs), e3 = 0.28022 * exp(-0.40290 * xs),
           e4 = 0.02817 * exp(-0.20162 * xs);
    double Phi = e1 + e2 + e3 + e4;
    double dPhi = -(3.19980 * e1 + 0.94229 * e2 + 0.40290 * e3 + 0.20162 * e4) * ia;
    double x = r / a.rc;
    double xp1 = ipow_d(x, a.p - 1), xp = xp1 * x;
    double uu = 1.0 - 0.5 * (p + 1.0) * (p + 2.0) * xp + p * (p + 2.0) * xp * x - 0.5 * p * (p + 1.0) * xp * x * x;
    double dud = -0.5 * p * (p + 1.0) * (p + 2.0) * xp1 * (1.0 - x) * (1.0 - x) / a.rc;
    double c = 14.399645478425668 * zi * zj;
    double phi = c * inv * Phi * uu;
    double dphi = c * (-inv * inv * Phi * uu + inv * dPhi * uu + inv * Phi * dud);
    es += 0.5 * phi;
    fx += dphi * dx * inv; fy += dphi * dy * inv; fz += dphi * dz * inv;
  }
  es = warp_sum_d(es); fx = warp_sum_d(fx); fy = warp_sum_d(fy); fz = warp_sum_d(fz);
  if (lane == 0) {
    e_atom[i] += es;                     // this warp is the only writer of atom i in this kernel
    if (force) { force[3 * (int64_t)i] += fx; force[3 * (int64_t)i + 1] += fy; force[3 * (int64_t)i + 2] += fz; }
  }
}

// ---- per-edge energies in candidate order: redo the compaction walk of k_geom_fill, E_ij = sum of the fp64 partials
__global__ void k_edge_energy_out(EdgeGeomArgs a, const int64_t* __restrict__ rowa, const double* __restrict__ epart,
                                  int nparts, int64_t pstride, const float* __restrict__ xf, int d,
                                  const double* __restrict__ w_eff, double* __restrict__ e_edge) {
  int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (warp >= a.nc) return;
  int i = (int)(a.c0 + warp);
  int64_t b = a.row_ptr[i], e = a.row_ptr[i + 1];
  int64_t out0 = rowa[warp];
  int cnt = 0;
  for (int64_t kb = b; kb < e; kb += 32) {
    int64_t k = kb + lane;
    int j = 0; double dx = 0, dy = 0, dz = 0, r2 = 0, rc = a.rc;
    bool ok = (k < e) && edge_vec(a, i, k, j, dx, dy, dz, r2, rc);
    unsigned mask = __ballot_sync(FULLMASK, ok);
    if (k < e) {
      double v = 0.0;
      if (ok) {
        int64_t o = out0 + cnt + __popc(mask & ((1u << lane) - 1u));
        if (nparts > 0) for (int q = 0; q < nparts; ++q) v += epart[(int64_t)q * pstride + o];
        else for (int q = 0; q < d; ++q) v += (double)xf[o * d + q] * w_eff[q];
      }
      e_edge[k] = v;
    }
    cnt += __popc(mask);
  }
}

// ---- Nose-Hoover thermostat half step (reading in DESIGN.md section 2) ----------------------------
// st = {xi, eta}; scratch[0] receives the velocity scale s = exp(-xi dt/2); e_kin *= s^2.
__global__ void k_nh_scalar(double* st, double* e_kin, double n_dof, double t0, double tau, double dt, double* scratch) {
  const double gkt = n_dof * 8.617333262e-5 * t0, Q = gkt * tau * tau;
  double xi = st[0], K = *e_kin;
  xi = xi + 0.25 * dt * (2.0 * K - gkt) / Q;
  double s = exp(-xi * 0.5 * dt);
  st[1] = st[1] + xi * 0.5 * dt;
  K = K * s * s;
  xi = xi + 0.25 * dt * (2.0 * K - gkt) / Q;
  st[0] = xi; *e_kin = K; scratch[0] = s;
}
__global__ void k_scale_vel(double* vel, int64_t n3, const double* __restrict__ s) {
  int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i < n3) vel[i] *= s[0];
}

__global__ void k_kin(const double* vel, const int32_t* species, const double* mass, int S, int64_t n, double* out) {
  int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= n) return;
  double m = mass[zc(species[i], S)];
  out[i] = 0.5 * m * (vel[3 * i] * vel[3 * i] + vel[3 * i + 1] * vel[3 * i + 1] + vel[3 * i + 2] * vel[3 * i + 2]) / ACC_CONV;
}

}  // namespace

#define LAUNCH_CHECK(m)              \
  do {                               \
    (m)->launches++;                 \
    AL_CUDA(m, cudaGetLastError());  \
  } while (0)

int k_launch_active_count(allegro_model* m, const EdgeGeomArgs& a, int* deg) {
  ProfScope _ps(m, PC_GEOM);
  if (a.nc <= 0) return ALLEGRO_OK;
  k_active_count<<<(a.nc * 32 + 255) / 256, 256, 0, m->stream>>>(a, deg);
  LAUNCH_CHECK(m);
  return ALLEGRO_OK;
}

int k_launch_set_mact(allegro_model* m, const int64_t* rowa, int nc, int* m_act) {
  ProfScope _ps(m, PC_GEOM);
  k_set_mact<<<1, 1, 0, m->stream>>>(rowa, nc, m_act);
  LAUNCH_CHECK(m);
  return ALLEGRO_OK;
}

int k_launch_geom_fill(allegro_model* m, const EdgeGeomArgs& a, const int64_t* rowa, Work& w) {
  ProfScope _ps(m, PC_GEOM);
  if (a.nc <= 0) return ALLEGRO_OK;
  k_geom_fill<<<(a.nc * 32 + 255) / 256, 256, 0, m->stream>>>(a, rowa, (int*)w.ei.p, (int*)w.ej.p, (float4*)w.geo.p,
                                                           (float*)w.u.p, (float*)w.du.p, (float*)w.B.p, (float*)w.dB.p,
                                                           (float*)w.Y.p, m->Denv, m->ldY, (int*)w.m_act.p, (float*)w.sig.p, m->sigma);
  LAUNCH_CHECK(m);
  return ALLEGRO_OK;
}

int k_launch_twobody0(allegro_model* m, Work& w, const int32_t* species, const Dense& L0, bool single, int m_cap) {
  ProfScope _ps(m, PC_TWOBODY0);
  if (m_cap <= 0) return ALLEGRO_OK;
  float* act = single ? (float*)w.XS[0].p : (float*)w.tb_a[0].p;
  int ld = single ? (m->d + m->n) : L0.fo;
  k_twobody0<<<(m_cap + TB0_EDGES - 1) / TB0_EDGES, 256, 0, m->stream>>>((int*)w.m_act.p, (int*)w.ei.p, (int*)w.ej.p, species,
                                                                    (float*)w.B.p, (float*)w.u.p, L0.W, m->S, m->NB, L0.fo,
                                                                    (float*)w.tb_z[0].p, act, ld, single ? 1 : 0, m->hfmt,
                                                                    (m->hp.precision == 1 || m->hfmt >= 0) ? 1 : 0);
  LAUNCH_CHECK(m);
  return ALLEGRO_OK;
}

static size_t tp_smem(const allegro_model* m, int L) { return (size_t)(m->Denv + m->tp[L - 1].npairs) * m->n * sizeof(float); }

static void tp_common(allegro_model* m, Work& w, int L, TPArgs& a, const float* om, int ldo, const float* Vin,
                      const float* w0, int ldw) {
  a.rowa = (const int64_t*)w.rowa.p;
  a.om = om; a.ldo = ldo; a.Y = (const float*)w.Y.p; a.Denv = m->Denv; a.ldy = m->ldY;
  a.Vin = Vin; a.w0 = w0; a.ldw = ldw;
  a.v0_l = m->d_v0_l; a.v0_y = m->d_v0_y; a.env_l = m->d_env_l;
  a.t = m->tp[L - 1]; a.n = m->n; a.lmax = m->lmax; a.c_env = m->c_env;
}

int tpw_fwd(allegro_model* m, Work& w, int L, int nc, const float* om, int ldo, const float* Vin, const float* w0, int ldw,
            float* Tout, float* xs, int ldx);
int tpw_bwd(allegro_model* m, Work& w, int L, int nc, const float* om, int ldo, const float* Vin, const float* w0, int ldw,
            const float* VbarL, const float* sbar, int lds, float* Vbar_prev, float* ombar, int ldob, float* w0bar);

int tpc_fwd(allegro_model* m, Work& w, int L, int nc, const float* om, int ldo, const float* w0, int ldw, float* xs, int ldx);
int tpc_bwd(allegro_model* m, Work& w, int L, int nc, const float* om, int ldo, const float* w0, int ldw, float* ombar, int ldob,
            float* w0bar);
int tp2_fwd(allegro_model* m, Work& w, int L, int nc, const float* om, int ldo, const float* Vin, const float* w0, int ldw,
            float* Tout, float* xs, int ldx);
int tp2_bwd(allegro_model* m, Work& w, int L, int nc, const float* om, int ldo, const float* Vin, const float* w0, int ldw,
            const float* VbarL, const float* sbar, int lds, float* Vbar_prev, float* ombar, int ldob, float* w0bar);

int k_launch_tp_fwd(allegro_model* m, Work& w, int L, int nc, const float* om, int ldo, const float* Vin,
                    const float* w0, int ldw, float* Tout, float* xs, int ldx) {
  ProfScope _ps(m, PC_TP_FWD);
  if (nc <= 0) return ALLEGRO_OK;
  {
    int rc = tpc_fwd(m, w, L, nc, om, ldo, w0, ldw, xs, ldx);              // contracted per centre (tpc_kernels.cu): the default
    if (rc != ALLEGRO_ERR_UNIMPLEMENTED) return rc;
    rc = tp2_fwd(m, w, L, nc, om, ldo, Vin, w0, ldw, Tout, xs, ldx);       // per-edge products: cp.async ring + FFMA2 / mma.sync
    if (rc != ALLEGRO_ERR_UNIMPLEMENTED) return rc;
    rc = tpw_fwd(m, w, L, nc, om, ldo, Vin, w0, ldw, Tout, xs, ldx);       // warp-per-(center, channel group) fallback
    if (rc != ALLEGRO_ERR_UNIMPLEMENTED) return rc;
  }
  TPArgs a{};
  tp_common(m, w, L, a, om, ldo, Vin, w0, ldw);
  a.Tout = Tout; a.xs = xs; a.ldx = ldx; a.gamma_out = (float*)w.gamma.p;
  size_t sm = tp_smem(m, L);
  if (Vin == nullptr) {
    AL_CUDA(m, cudaFuncSetAttribute(k_tp_fwd<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
    k_tp_fwd<true><<<nc, 256, sm, m->stream>>>(a);
  } else {
    AL_CUDA(m, cudaFuncSetAttribute(k_tp_fwd<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
    k_tp_fwd<false><<<nc, 256, sm, m->stream>>>(a);
  }
  LAUNCH_CHECK(m);
  return ALLEGRO_OK;
}

int k_launch_tp_bwd(allegro_model* m, Work& w, int L, int nc, const float* om, int ldo, const float* Vin,
                    const float* w0, int ldw, const float* VbarL, const float* sbar, int lds, float* Vbar_prev,
                    float* ombar, int ldob, float* w0bar) {
  ProfScope _ps(m, PC_TP_BWD);
  if (nc <= 0) return ALLEGRO_OK;
  {
    int rc = tpc_bwd(m, w, L, nc, om, ldo, w0, ldw, ombar, ldob, w0bar);
    if (rc != ALLEGRO_ERR_UNIMPLEMENTED) return rc;
    rc = tp2_bwd(m, w, L, nc, om, ldo, Vin, w0, ldw, VbarL, sbar, lds, Vbar_prev, ombar, ldob, w0bar);
    if (rc != ALLEGRO_ERR_UNIMPLEMENTED) return rc;
    rc = tpw_bwd(m, w, L, nc, om, ldo, Vin, w0, ldw, VbarL, sbar, lds, Vbar_prev, ombar, ldob, w0bar);
    if (rc != ALLEGRO_ERR_UNIMPLEMENTED) return rc;
  }
  TPArgs a{};
  tp_common(m, w, L, a, om, ldo, Vin, w0, ldw);
  a.VbarL = VbarL; a.sbar = sbar; a.lds = lds; a.Vbar_prev = Vbar_prev; a.ombar = ombar; a.ldob = ldob;
  a.w0bar = w0bar; a.Ybar = (float*)w.Ybar.p;
  size_t sm = tp_smem(m, L);
  if (Vin == nullptr) {
    AL_CUDA(m, cudaFuncSetAttribute(k_tp_bwd<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
    k_tp_bwd<true><<<nc, 256, sm, m->stream>>>(a);
  } else {
    AL_CUDA(m, cudaFuncSetAttribute(k_tp_bwd<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
    k_tp_bwd<false><<<nc, 256, sm, m->stream>>>(a);
  }
  LAUNCH_CHECK(m);
  return ALLEGRO_OK;
}

int k_launch_energy(allegro_model* m, Work& w, const int32_t* species, int64_t c0, int nc, const float* xf, double* e_atom) {
  ProfScope _ps(m, PC_ENERGY);
  if (nc <= 0) return ALLEGRO_OK;
  if (w.n_eparts > 0 && xf != nullptr)
    k_energy_parts<<<(nc * 32 + 255) / 256, 256, 0, m->stream>>>((const int64_t*)w.rowa.p, nc, c0, (const double*)w.epart.p,
                                                                w.n_eparts, (int64_t)w.cap_edges, species, m->S, m->sigma, m->mu, e_atom);
  else
    k_energy<<<(nc * 32 + 255) / 256, 256, 0, m->stream>>>((const int64_t*)w.rowa.p, nc, c0, xf, m->d, m->w_eff_d, species,
                                                          m->S, m->sigma, m->mu, e_atom);
  LAUNCH_CHECK(m);
  return ALLEGRO_OK;
}

int k_launch_sum_f64(allegro_model* m, const double* x, int64_t n, double* out) {
  ProfScope _ps(m, PC_ENERGY);
  k_sum_f64<<<1, 1024, 0, m->stream>>>(x, n, out);
  LAUNCH_CHECK(m);
  return ALLEGRO_OK;
}

int k_launch_bwd_prep(allegro_model* m, Work& w, const float* xbar, int ldx, const float* z, int ldz, float c, float* zb,
                      int ldzb, int width, int m_cap) {
  ProfScope _ps(m, PC_BWD_ELEM);
  if (m_cap <= 0) return ALLEGRO_OK;
  k_bwd_prep<<<(unsigned)(((int64_t)m_cap * 32 + 255) / 256), 256, 0, m->stream>>>((int*)w.m_act.p, xbar, ldx, z, ldz,
                                                                                  (float*)w.u.p, c, zb, ldzb, width,
                                                                                  (float*)w.ubar.p + (size_t)(w.n_uparts - 1) * w.cap_edges, (float*)w.sig.p, m->w_eff_f);
  LAUNCH_CHECK(m);
  return ALLEGRO_OK;
}

int k_launch_edge_bwd(allegro_model* m, Work& w, const float* zb1, int ldz, const Dense& L0, bool single, double* force,
                      int m_cap) {
  ProfScope _ps(m, PC_EDGE_BWD);
  if (m_cap <= 0) return ALLEGRO_OK;
  (void)single;
  const int H = L0.fo;
  size_t sm = (size_t)(m->NB + EB_EDGES) * (H + 4) * sizeof(float);
  // per device: the opt-in is a property of the kernel on one device, and the size depends on the model (largest seen so far)
  static std::atomic<size_t> sm_set[64];
  std::atomic<size_t>& cur = sm_set[m->device & 63];
  if (sm > cur.load(std::memory_order_acquire)) {
    AL_CUDA(m, cudaFuncSetAttribute(k_edge_bwd, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
    cur.store(sm, std::memory_order_release);
  }
  int ypart0[AL_MAX_LAYERS + 1];
  const int n_yparts = al_ybar_layout(m, ypart0);
  k_edge_bwd<<<(unsigned)((m_cap + EB_EDGES - 1) / EB_EDGES), 256, sm, m->stream>>>(
      (int*)w.m_act.p, zb1, ldz, L0.W, m->S, m->NB, H, (float4*)w.geo.p, (float*)w.du.p, (float*)w.dB.p, (float*)w.ubar.p,
      w.n_uparts, (int64_t)w.cap_edges, (float*)w.Ybar.p, n_yparts, (int64_t)w.cap_edges * m->Denv,
      m->Denv, m->lmax, (int*)w.ei.p, (int*)w.ej.p, (float*)w.ge.p, force);
  LAUNCH_CHECK(m);
  return ALLEGRO_OK;
}

// Start of a compute call: zero the force array (may be null) and validate every atom's species; an out-of-range value
// raises status bit 2 (ALLEGRO_ERR_BAD_ARG at the next host synchronisation); table look-ups clamp (zc()).
int k_launch_begin_compute(allegro_model* m, double* force, const int32_t* species, int64_t n, int* flags) {
  ProfScope _ps(m, PC_EDGE_BWD);
  if (n <= 0) return ALLEGRO_OK;
  k_zero_check<<<(unsigned)((3 * n + 255) / 256), 256, 0, m->stream>>>(force, 3 * n, species, n, m->S, flags);
  LAUNCH_CHECK(m);
  return ALLEGRO_OK;
}

int k_launch_zero_f64(allegro_model* m, double* p, int64_t n) {
  ProfScope _ps(m, PC_EDGE_BWD);
  if (n <= 0) return ALLEGRO_OK;
  k_zero_f64<<<(unsigned)((n + 255) / 256), 256, 0, m->stream>>>(p, n);
  LAUNCH_CHECK(m);
  return ALLEGRO_OK;
}

int k_launch_nve_kick_drift(allegro_model* m, double* pos, double* vel, const double* force, const int32_t* species,
                            const double* mass, int64_t n, double dt, bool drift) {
  ProfScope _ps(m, PC_NVE);
  if (n <= 0) return ALLEGRO_OK;
  k_nve<<<(unsigned)((n + 255) / 256), 256, 0, m->stream>>>(pos, vel, force, species, mass, m->S, n, dt, drift ? 1 : 0);
  LAUNCH_CHECK(m);
  return ALLEGRO_OK;
}

int k_launch_kinetic(allegro_model* m, const double* vel, const int32_t* species, const double* mass, int64_t n,
                     double* e_kin, DevBuf& tmp) {
  ProfScope _ps(m, PC_NVE);
  AL_CHECK(al_reserve(m, tmp, (size_t)n * 8 + 16));
  if (n > 0) {
    k_kin<<<(unsigned)((n + 255) / 256), 256, 0, m->stream>>>(vel, species, mass, m->S, n, (double*)tmp.p);
    LAUNCH_CHECK(m);
  }
  return k_launch_sum_f64(m, (double*)tmp.p, n, e_kin);
}


int k_launch_zbl(allegro_model* m, const EdgeGeomArgs& a, const double* zbl_Z, double* e_atom, double* force) {
  ProfScope _ps(m, PC_ENERGY);
  if (a.nc <= 0) return ALLEGRO_OK;
  k_zbl<<<(a.nc * 32 + 255) / 256, 256, 0, m->stream>>>(a, zbl_Z, e_atom, force);
  LAUNCH_CHECK(m);
  return ALLEGRO_OK;
}

int k_launch_edge_energy_out(allegro_model* m, const EdgeGeomArgs& a, Work& w, const float* xf, double* e_edge) {
  ProfScope _ps(m, PC_ENERGY);
  if (a.nc <= 0) return ALLEGRO_OK;
  k_edge_energy_out<<<(a.nc * 32 + 255) / 256, 256, 0, m->stream>>>(a, (const int64_t*)w.rowa.p, (const double*)w.epart.p,
                                                                 w.n_eparts, (int64_t)w.cap_edges, xf, m->d, m->w_eff_d, e_edge);
  LAUNCH_CHECK(m);
  return ALLEGRO_OK;
}

int k_launch_nh_half(allegro_model* m, double* vel, int64_t n, double* nh_state, double* e_kin, double n_dof, double t0_K,
                     double tau_fs, double dt_fs, double* scratch) {
  ProfScope _ps(m, PC_NVE);
  k_nh_scalar<<<1, 1, 0, m->stream>>>(nh_state, e_kin, n_dof, t0_K, tau_fs, dt_fs, scratch);
  LAUNCH_CHECK(m);
  if (n > 0) {
    k_scale_vel<<<(unsigned)((3 * n + 255) / 256), 256, 0, m->stream>>>(vel, 3 * n, scratch);
    LAUNCH_CHECK(m);
  }
  return ALLEGRO_OK;
}
