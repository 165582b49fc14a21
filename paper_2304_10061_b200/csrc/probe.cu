// Peak probes for the roofline denominators bench.py reports ("TF32 tensor and fp32 FFMA peaks are
// not in MEASURED_PEAKS.json -- measure them").  Not on the hot path: called by bench.py once per run.
//
//   allegro_probe_ffma : fp32 FMA issue rate of the SIMT pipes -- every thread runs 16 independent FMA chains (no memory
//                        traffic), 8 blocks of 256 threads per SM; TFLOP/s = 2 * FMAs / time.
//   allegro_probe_tf32 : tcgen05.mma kind::tf32 issue rate -- one CTA per SM issues 128 x 256 x 8 MMAs back to back on
//                        operand tiles that stay in shared memory (no TMA, no epilogue): what the tensor pipe can do when
//                        nothing else limits it.
#include "internal.h"

namespace {

__global__ void __launch_bounds__(256) k_probe_ffma(float* out, int iters, float b, float c) {
  float a[16];
#pragma unroll
  for (int k = 0; k < 16; ++k) a[k] = (float)(threadIdx.x + k) * 1e-3f;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int r = 0; r < 4; ++r)
#pragma unroll
      for (int k = 0; k < 16; ++k) a[k] = fmaf(a[k], b, c);
  }
  float s = 0.f;
#pragma unroll
  for (int k = 0; k < 16; ++k) s += a[k];
  if (s == 12345.678f) out[0] = s;   // keeps the chains alive, never true in practice
}

__device__ __forceinline__ uint32_t p_smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

// K-major SWIZZLE_128B descriptor as in gemm_tc.cu (the operand values do not matter for the probe)
__device__ __forceinline__ uint64_t p_desc(uint32_t saddr) {
  uint64_t d = 0;
  d |= (uint64_t)((saddr & 0x3FFFF) >> 4);
  d |= (uint64_t)1 << 16;
  d |= (uint64_t)(1024 >> 4) << 32;
  d |= (uint64_t)1 << 46;
  d |= (uint64_t)2 << 61;
  return d;
}

__global__ void __launch_bounds__(128, 1) k_probe_tf32(int iters) {
  extern __shared__ uint8_t praw[];
  uint8_t* smem = (uint8_t*)(((uintptr_t)praw + 1023) & ~(uintptr_t)1023);
  // A: 128 rows x 32 floats (16 KB), B: 256 rows x 32 floats (32 KB), both zero
  for (int i = threadIdx.x; i < (16384 + 32768) / 4; i += blockDim.x) reinterpret_cast<float*>(smem)[i] = 0.f;
  __shared__ uint32_t tslot;
  __shared__ __align__(8) uint64_t bar;
  const int warp = threadIdx.x >> 5;
  if (threadIdx.x == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(p_smem_u32(&bar)));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 256;" ::"r"(p_smem_u32(&tslot)) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t tmem = tslot;
  if (threadIdx.x == 0) {
    const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(256 >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
    const uint64_t da = p_desc(p_smem_u32(smem)), db = p_desc(p_smem_u32(smem + 16384));
    for (int it = 0; it < iters; ++it) {
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const uint32_t acc = (it | k) ? 1u : 0u;
        asm volatile(
            "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
            "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}" ::"r"(tmem),
            "l"(da + 2 * k), "l"(db + 2 * k), "r"(idesc), "r"(acc)
            : "memory");
      }
    }
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(p_smem_u32(&bar)) : "memory");
    uint32_t done;
    do {
      asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                   : "=r"(done) : "r"(p_smem_u32(&bar)), "r"(0u) : "memory");
    } while (!done);
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (warp == 0) {
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 256;" ::"r"(tmem) : "memory");
  }
}

// run `launch` repeatedly: best single launch (burst) and the average over ~sustain_s seconds back to back (sustained)
template <class F>
int timed(allegro_model* m, F launch, double work_per_launch, double sustain_s, double* burst, double* sustained) {
  cudaEvent_t a, b;
  AL_CUDA(m, cudaEventCreate(&a)); AL_CUDA(m, cudaEventCreate(&b));
  for (int w = 0; w < 3; ++w) launch();
  AL_CUDA(m, cudaStreamSynchronize(m->stream));
  float best = 1e30f;
  for (int r = 0; r < 10; ++r) {
    cudaEventRecord(a, m->stream); launch(); cudaEventRecord(b, m->stream);
    AL_CUDA(m, cudaEventSynchronize(b));
    float t; cudaEventElapsedTime(&t, a, b);
    best = t < best ? t : best;
  }
  *burst = work_per_launch / (best * 1e-3) / 1e12;
  int n = (int)(sustain_s * 1e3 / best) + 1;
  cudaEventRecord(a, m->stream);
  for (int r = 0; r < n; ++r) launch();
  cudaEventRecord(b, m->stream);
  AL_CUDA(m, cudaEventSynchronize(b));
  float t; cudaEventElapsedTime(&t, a, b);
  *sustained = work_per_launch * n / (t * 1e-3) / 1e12;
  cudaEventDestroy(a); cudaEventDestroy(b);
  AL_CUDA(m, cudaGetLastError());
  return ALLEGRO_OK;
}

}  // namespace

extern "C" int allegro_probe_ffma(allegro_model* m, double sustain_s, double* burst_tflops, double* sustained_tflops) {
  if (!m || !burst_tflops || !sustained_tflops) return ALLEGRO_ERR_BAD_ARG;
  float* out = nullptr;
  AL_CHECK(al_alloc(m, (void**)&out, 64));
  const int iters = 4096, blocks = m->sm_count * 8;
  const double flops = 2.0 * 64.0 * iters * 256.0 * blocks;
  int rc = timed(m, [&] { k_probe_ffma<<<blocks, 256, 0, m->stream>>>(out, iters, 0.999f, 1e-3f); }, flops, sustain_s,
                 burst_tflops, sustained_tflops);
  cudaStreamSynchronize(m->stream);
  al_free(m, out);
  return rc;
}

extern "C" int allegro_probe_tf32(allegro_model* m, double sustain_s, double* burst_tflops, double* sustained_tflops) {
  if (!m || !burst_tflops || !sustained_tflops) return ALLEGRO_ERR_BAD_ARG;
  const int iters = 8192, smem = 16384 + 32768 + 1024;
  static AttrOnce once;
  if (once.need(m->device)) {
    AL_CUDA(m, cudaFuncSetAttribute(k_probe_tf32, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    once.done(m->device);
  }
  const double flops = 2.0 * 128.0 * 256.0 * 8.0 * 4.0 * iters * m->sm_count;
  return timed(m, [&] { k_probe_tf32<<<m->sm_count, 128, smem, m->stream>>>(iters); }, flops, sustain_s, burst_tflops,
               sustained_tflops);
}
