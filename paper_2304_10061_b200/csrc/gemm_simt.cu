// fp32 FFMA GEMM with fused epilogues (precision mode 0: "F32" matmuls of PAPER.md Table IV, needed
// for the 1e-5 force tolerance).  128x64x16 tiles, 256 threads, 8x4 outputs per thread, float4 I/O.
#include <cstdlib>

#include "gemm.h"
#include "internal.h"

int al_gemm_tc(allegro_model* m, const GemmArgs& g);   // gemm_tc.cu (tcgen05)

namespace {

__device__ __forceinline__ float silu_f(float z) { return z / (1.0f + expf(-z)); }
__device__ __forceinline__ float dsilu_f(float z) {
  float s = 1.0f / (1.0f + expf(-z));
  return s * (1.0f + z * (1.0f - s));
}

constexpr int BM = 128, BN = 64, BK = 16, TM = 8, TN = 4, NT = 256;

__global__ void __launch_bounds__(NT) k_gemm_simt(GemmArgs g) {
  const int M = *g.m_ptr;
  const int row0 = blockIdx.x * BM, col0 = blockIdx.y * BN;
  if (row0 >= M) return;
  __shared__ __align__(16) float As[BK][BM + 4];
  __shared__ __align__(16) float Bs[BK][BN + 4];
  const int tid = threadIdx.x;
  const int ty = tid / (BN / TN), tx = tid % (BN / TN);
  float acc[TM][TN];
#pragma unroll
  for (int i = 0; i < TM; ++i)
#pragma unroll
    for (int j = 0; j < TN; ++j) acc[i][j] = 0.f;

  for (int k0 = 0; k0 < g.K; k0 += BK) {
    // A tile: BM rows x 4 float4
#pragma unroll
    for (int t = 0; t < (BM * BK / 4) / NT; ++t) {
      int idx = tid + t * NT;
      int r = idx >> 2, kq = (idx & 3) * 4;
      float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
      if (row0 + r < M && k0 + kq < g.K) v = *reinterpret_cast<const float4*>(g.A + (size_t)(row0 + r) * g.lda + k0 + kq);
      As[kq + 0][r] = v.x; As[kq + 1][r] = v.y; As[kq + 2][r] = v.z; As[kq + 3][r] = v.w;
    }
#pragma unroll
    for (int t = 0; t < (BN * BK / 4) / NT; ++t) {
      int idx = tid + t * NT;
      int r = idx >> 2, kq = (idx & 3) * 4;
      float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
      if (col0 + r < g.N && k0 + kq < g.K) v = *reinterpret_cast<const float4*>(g.Bt + (size_t)(col0 + r) * g.ldb + k0 + kq);
      Bs[kq + 0][r] = v.x; Bs[kq + 1][r] = v.y; Bs[kq + 2][r] = v.z; Bs[kq + 3][r] = v.w;
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < BK; ++k) {
      float4 a0 = *reinterpret_cast<const float4*>(&As[k][ty * TM]);
      float4 a1 = *reinterpret_cast<const float4*>(&As[k][ty * TM + 4]);
      float4 b = *reinterpret_cast<const float4*>(&Bs[k][tx * TN]);
      float a[TM] = {a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w};
      float bb[TN] = {b.x, b.y, b.z, b.w};
#pragma unroll
      for (int i = 0; i < TM; ++i)
#pragma unroll
        for (int j = 0; j < TN; ++j) acc[i][j] = fmaf(a[i], bb[j], acc[i][j]);
    }
    __syncthreads();
  }
  int col = col0 + tx * TN;
  // EPI_LATENT_LAST reduces over lanes with full-warp shuffles: no lane may exit early there; out-of-range
  // lanes compute on clamped coordinates and store nothing.
  const bool cok = col < g.N;
  const bool shf = (g.epi == EPI_LATENT_LAST) || g.prep;   // epilogues with warp shuffles
  if (!cok) {
    if (!shf) return;
    col = 0;
  }
#pragma unroll
  for (int i = 0; i < TM; ++i) {
    int row = row0 + ty * TM + i;
    const bool rok = row < M;
    if (!rok) {
      if (!shf) break;
      row = M - 1;   // keep the lanes alive for the shuffles below; nothing is stored for this row
    }
    float v[4] = {acc[i][0], acc[i][1], acc[i][2], acc[i][3]};
    float o[4];
    switch (g.epi) {
      case EPI_PLAIN:
#pragma unroll
        for (int j = 0; j < 4; ++j) o[j] = v[j];
        break;
      case EPI_SILU_BOTH:
      case EPI_SILU_U:
      case EPI_LATENT: {
        *reinterpret_cast<float4*>(g.out2 + (size_t)row * g.ldo2 + col) = make_float4(v[0], v[1], v[2], v[3]);
        float us = (g.epi == EPI_SILU_BOTH) ? 1.0f : g.u[row];
        if (g.epi == EPI_LATENT) {
          float4 x = *reinterpret_cast<const float4*>(g.aux1 + (size_t)row * g.ld1 + col);
          float xo[4] = {x.x, x.y, x.z, x.w};
#pragma unroll
          for (int j = 0; j < 4; ++j) o[j] = g.c0 * xo[j] + g.c1 * us * silu_f(v[j]);
        } else {
#pragma unroll
          for (int j = 0; j < 4; ++j) o[j] = us * silu_f(v[j]);
        }
      } break;
      case EPI_MUL_DSILU: {
        float4 z = *reinterpret_cast<const float4*>(g.aux1 + (size_t)row * g.ld1 + col);
        float zz[4] = {z.x, z.y, z.z, z.w};
#pragma unroll
        for (int j = 0; j < 4; ++j) o[j] = v[j] * dsilu_f(zz[j]);
      } break;
      case EPI_ADD2: {
        float4 x = *reinterpret_cast<const float4*>(g.aux1 + (size_t)row * g.ld1 + col);
        float4 y = *reinterpret_cast<const float4*>(g.aux2 + (size_t)row * g.ld2 + col);
        o[0] = v[0] + g.c0 * x.x + y.x; o[1] = v[1] + g.c0 * x.y + y.y;
        o[2] = v[2] + g.c0 * x.z + y.z; o[3] = v[3] + g.c0 * x.w + y.w;
      } break;
      case EPI_ADD2R: {
        float4 x = *reinterpret_cast<const float4*>(g.aux3 + col);
        float4 y = *reinterpret_cast<const float4*>(g.aux2 + (size_t)row * g.ld2 + col);
        float cs = g.c0 * g.u[row];
        o[0] = v[0] + cs * x.x + y.x; o[1] = v[1] + cs * x.y + y.y;
        o[2] = v[2] + cs * x.z + y.z; o[3] = v[3] + cs * x.w + y.w;
      } break;
      case EPI_LATENT_LAST: {
        float4 x = *reinterpret_cast<const float4*>(g.aux1 + (size_t)row * g.ld1 + col);
        float4 w = *reinterpret_cast<const float4*>(g.aux3 + col);
        float xo[4] = {x.x, x.y, x.z, x.w}, we[4] = {w.x, w.y, w.z, w.w}, zb[4];
        const float us = g.u[row], sg = g.sig[row];
        float up = 0.f; double ep = 0.0;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          const float sgm = 1.0f / (1.0f + expf(-v[j]));   // one sigmoid serves silu and silu'
          const float sl = v[j] * sgm;
          o[j] = g.c0 * xo[j] + g.c1 * us * sl;
          zb[j] = g.c1 * us * sg * we[j] * (sgm * (1.0f + v[j] * (1.0f - sgm)));
          up = fmaf(we[j], sl, up);
          ep += (double)o[j] * g.w_eff_d[col + j];
        }
        if (!cok) { up = 0.f; ep = 0.0; }
        if (rok && cok) *reinterpret_cast<float4*>(g.out2 + (size_t)row * g.ldo2 + col) = make_float4(zb[0], zb[1], zb[2], zb[3]);
        // 8 consecutive lanes (tx = 8p .. 8p+7) hold the 32 columns of one chunk of this row
#pragma unroll
        for (int off = 1; off < 8; off <<= 1) {
          up += __shfl_xor_sync(0xffffffffu, up, off);
          ep += __shfl_xor_sync(0xffffffffu, ep, off);
        }
        if ((tx & 7) == 0 && rok && cok) {
          const int p = col >> 5;
          g.upart[(int64_t)p * g.part_stride + row] = g.c1 * sg * up;
          g.epart[(int64_t)p * g.part_stride + row] = ep;
        }
      } break;
      default:
#pragma unroll
        for (int j = 0; j < 4; ++j) o[j] = v[j];
    }
    if (g.prep) {
      float4 zq = *reinterpret_cast<const float4*>(g.zp + (size_t)row * g.ldzp + col);
      const float zz[4] = {zq.x, zq.y, zq.z, zq.w};
      const float cu = g.cp * g.pu[row];
      float zb[4], up = 0.f;
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const float sgm = 1.0f / (1.0f + expf(-zz[j]));
        up = fmaf(o[j], zz[j] * sgm, up);
        zb[j] = cu * o[j] * (sgm * (1.0f + zz[j] * (1.0f - sgm)));
      }
      if (!cok) up = 0.f;
      if (rok && cok) *reinterpret_cast<float4*>(g.zbp + (size_t)row * g.ldzbp + col) = make_float4(zb[0], zb[1], zb[2], zb[3]);
#pragma unroll
      for (int off = 1; off < 8; off <<= 1) up += __shfl_xor_sync(0xffffffffu, up, off);
      if ((tx & 7) == 0 && rok && cok) g.upart[(int64_t)(g.pbase + (col >> 5)) * g.part_stride + row] = g.cp * up;
    }
    if (g.C && rok && cok) *reinterpret_cast<float4*>(g.C + (size_t)row * g.ldc + col) = make_float4(o[0], o[1], o[2], o[3]);
  }
}

}  // namespace

int al_gemm_tc3(allegro_model* m, const GemmArgs& g);  // gemm_tc.cu (tcgen05, 3xTF32 split operands)
int al_gemm_h16(allegro_model* m, const GemmArgs& g);  // gemm_tc.cu (tcgen05 kind::f16, 16-bit operands: precision 2 / 4)
int al_gemm_tc_row_parts(int N, bool split);

// precision 0 runs on the tensor cores as 3xTF32; precision 3 runs the plain FFMA kernel below
static bool fp32_simt(const allegro_model* m) { return m->hp.precision == 3; }

int al_gemm_row_parts(const allegro_model* m, int N) {
  if (fp32_simt(m)) return (N + 31) / 32;
  return al_gemm_tc_row_parts(N, m->hp.precision == 0);
}

bool al_gemm_supports_kcat(const allegro_model* m) { return !fp32_simt(m); }

int al_gemm(allegro_model* m, const GemmArgs& g) {
  ProfScope _ps(m, PC_GEMM);
  if (g.m_cap <= 0) return ALLEGRO_OK;
  if (g.A2 && (fp32_simt(m) || (g.K1 & 31) || g.K1 <= 0 || g.K1 >= g.K || (g.lda2 & 3))) {
    al_set_error(m, "gemm: K-concatenated A needs a tensor-core mode and K1 % 32 == 0");
    return ALLEGRO_ERR_BAD_HPARAMS;
  }
  if ((g.K & 3) || (g.N & 3) || (g.lda & 3) || (g.ldb & 3) || (g.ldc & 3)) {
    al_set_error(m, "gemm: dimensions must be multiples of 4");
    return ALLEGRO_ERR_BAD_HPARAMS;
  }
  if (m->hfmt >= 0) return al_gemm_h16(m, g);
  if (!fp32_simt(m)) return (m->hp.precision == 0) ? al_gemm_tc3(m, g) : al_gemm_tc(m, g);
  dim3 grid((g.m_cap + BM - 1) / BM, (g.N + BN - 1) / BN);
  k_gemm_simt<<<grid, NT, 0, m->stream>>>(g);
  m->launches++;
  AL_CUDA(m, cudaGetLastError());
  return ALLEGRO_OK;
}
