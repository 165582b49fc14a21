// Edge-batched MLP GEMMs with fused epilogues.
//   C[M,N] = epi( A[M,K] * Bt[N,K]^T )      A, Bt K-contiguous (row-major), fp32 in HBM
// M is read from device memory (*m_ptr): the number of active edges of the chunk is only known on
// the device; grids are sized for m_cap rows and blocks beyond *m_ptr exit.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

enum GemmEpi {
  EPI_PLAIN = 0,      // C = acc
  EPI_SILU_BOTH = 1,  // out2 = acc (pre-activation z) ; C = silu(acc)
  EPI_SILU_U = 2,     // out2 = acc ; C = u[m] * silu(acc)                              (two-body output x^0)
  EPI_LATENT = 3,     // out2 = acc ; C = c0 * aux1[m,n] + c1 * u[m] * silu(acc)        (x^L residual update)
  EPI_MUL_DSILU = 4,  // C = acc * silu'(aux1[m,n])                                    (backward through SiLU)
  EPI_ADD2 = 5,       // C = acc + c0 * aux1[m,n] + aux2[m,n]                           (x-bar accumulation)
  EPI_ADD2R = 6,      // C = acc + c0 * u[m] * aux3[n] + aux2[m,n]   (rank-1 incoming gradient sigma_e * w_eff)
  // Last latent layer, forward and the start of the backward in one epilogue (x-bar^{NL} = sigma_e w_eff is
  // known a priori): with x = c0 * aux1 + c1 * u * silu(acc),
  //   out2  = c1 * u[m] * sig[m] * aux3[n] * silu'(acc)                     (z-bar of this layer; replaces z)
  //   upart[p][m] = c1 * sig[m] * sum_{n in chunk p} aux3[n] * silu(acc)     (u-bar partial, fp32)
  //   epart[p][m] = sum_{n in chunk p} x * w_eff_d[n]                        (edge-energy partial, fp64)
  //   C = x only if C != nullptr (debug tap); chunks are 32 columns, see al_gemm_row_parts()
  EPI_LATENT_LAST = 7
};

struct GemmArgs {
  const float* A; int lda;
  // Optional K-concatenation of two activation tensors (tensor-core kernels only): columns [0, K1) of the A operand
  // come from A, columns [K1, K) from A2 (row stride lda2); K1 must be a multiple of 32.  A2 = null: plain A.
  const float* A2; int lda2; int K1;
  const float* Bt; int ldb;       // fp32 weights [N][K]
  const float *Bt_hi, *Bt_lo;     // TF32-exact / remainder split of Bt (precision 0 on tensor cores) or null
  float* C; int ldc;
  int N, K;
  int m_cap; const int* m_ptr;
  int epi;
  const float* aux1; int ld1;
  const float* aux2; int ld2;
  const float* aux3; int ld3;
  float* out2; int ldo2;
  const float* u;                 // per-row scalar
  const float* sig;               // per-row sigma_{Z_i(e)} (EPI_LATENT_LAST)
  const double* w_eff_d;          // [N] fp64 folded edge-MLP vector (EPI_LATENT_LAST)
  double* epart; float* upart; int64_t part_stride;   // [parts][part_stride] row partials (EPI_LATENT_LAST, prep)
  // Optional second stage of EPI_ADD2 / EPI_ADD2R (replaces k_bwd_prep): with xb = the epilogue's result (x-bar),
  //   zbp[m,n] = cp * pu[m] * xb * silu'(zp[m,n])          (z-bar entering the next MLP to differentiate)
  //   upart[pbase + chunk][m] = cp * sum_{n in chunk} xb * silu(zp[m,n])     (u-bar partial)
  // C may be NULL when x-bar itself is not needed afterwards.
  int prep; const float* zp; int ldzp; float* zbp; int ldzbp; const float* pu; float cp; int pbase;
  float c0, c1;
  // 1: the kernel walks its row tiles from the last to the first (set by the launcher, see al_next_rev(): consecutive
  // edge-ordered kernels alternate direction so each starts on the rows its producer left in L2)
  int rev;
  // precision 4 / 2 (16-bit operand storage): hfmt = element format of A / B and of every epilogue tensor (aux1, aux2, out2,
  // zp, zbp), 0 fp16, 1 bf16; io16 bit 0 (gemm_tc.cu IO16_C): C is 16-bit too, else fp32.  A, A2, Bt then point to 16-bit
  // data (Bt16); lda / lda2 / ldb and the epilogue strides count elements.
  int hfmt, io16;
  const void* Bt16;
};

// dispatch by allegro_hparams.precision: 0 3xTF32 tcgen05, 1 TF32 tcgen05, 3 fp32 FFMA (2 is refused at create time)
int al_gemm(struct allegro_model* m, const GemmArgs& g);
// number of 32-column row partials the EPI_LATENT_LAST epilogue of the active GEMM kernel writes for N columns
int al_gemm_row_parts(const struct allegro_model* m, int N);
// true when al_gemm runs a kernel that honours GemmArgs::A2 (the tcgen05 kernels)
bool al_gemm_supports_kcat(const struct allegro_model* m);
