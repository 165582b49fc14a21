// l_max = 3 forward instantiations: lane-split kernels (tp3_impl.cuh) for the wide layers, the 32-channel
// kernel of tp2_impl.cuh for the scalar-output last layer.
#include "tp3m_impl.cuh"

int tp2_l3_fwd(allegro_model* m, const TP2Common& q, int pat) {
  // TF32 mode (precision 1; the paper runs the tensor product in TF32): mma.sync kernels of tp3m_impl.cuh
  if (m->hp.precision == 1 && m->d % 8 == 0) {   // (32-byte rows of the scalar output need d % 8 == 0)
    // software-pipelined chunks, 2 warps per block (8 warps per SM at 238 / 255 registers); without the pipeline
    // (166 registers, 10 warps per SM) 3 % slower, 3 warps per block 25 % slower
    if (pat == P_16_16_31) { TP2<Pat<P_16_16_31>::NNZ> a{}; AL_CHECK(fill2(m, q, a)); return launch_fwd3m<P_16_16_31, true, 2, true>(m, a); }
    if (pat == P_16_31_16) { TP2<Pat<P_16_31_16>::NNZ> a{}; AL_CHECK(fill2(m, q, a)); return launch_fwd3m<P_16_31_16, false, 2, true>(m, a); }
  }
  if (pat == P_16_16_31) { TP2<Pat<P_16_16_31>::NNZ> a{}; AL_CHECK(fill2(m, q, a)); return launch_fwd3<P_16_16_31, true, 8, 4>(m, a); }
  if (pat == P_16_31_16) { TP2<Pat<P_16_31_16>::NNZ> a{}; AL_CHECK(fill2(m, q, a)); return launch_fwd3<P_16_31_16, false, 4, 4>(m, a); }
  if (pat == P_16_16_1) { TP2<Pat<P_16_16_1>::NNZ> a{}; AL_CHECK(fill2(m, q, a)); return launch_fwd2<P_16_16_1, 1, false, 3, 4>(m, a); }
  return ALLEGRO_ERR_UNIMPLEMENTED;
}
