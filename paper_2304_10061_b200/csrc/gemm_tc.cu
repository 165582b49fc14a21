// tcgen05 tensor-core GEMM for the edge-batched MLPs (precision modes 0 / 1 / 2 / 4; "TF32 for matrix
// multiplications", Table IV).  sm_100a only: TMA (cp.async.bulk.tensor) stages K-major 128B-swizzled operand tiles in shared
// memory (two rings: A = activations from HBM, B = weights from L2), one elected thread issues tcgen05.mma (kind::tf32, or
// kind::f16 for 16-bit operand storage) with the fp32 accumulator in TMEM (double-buffered, 2 x 256 columns), sixteen epilogue
// warps read it back with tcgen05.ld, transpose 32 x 32 blocks through shared memory into a coalesced domain and apply one of
// the fused epilogues (SiLU / envelope / residual / SiLU' / energy and z-bar of the last layer / x-bar accumulation with the
// next layer's z-bar) before storing.
//
//   C[M,N] = epi( A[M,K] * Bt[N,K]^T ),  A and Bt row-major (K contiguous) in HBM; K may be the concatenation of two A tensors.
//
// Warp roles: warp 0 = TMA producer of A, warp 2 = TMA producer of B, warp 1 = MMA issuer (+ TMEM alloc), (3xTF32: warps 3-6
// split every landed A stage into hi / lo parts,) the remaining warps = epilogue (TMEM lane quarter = warp_id % 4, EPI_WARPS / 4
// warps per quarter taking alternate 32-column chunks).  Persistent CTAs, static tile schedule, n fastest.  Large launches run
// on CTA pairs (clusters of two, cta_group::2, 256-row tiles): see the comment above the kernel.
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cstdlib>

#include <map>
#include <tuple>
#include <type_traits>

#include "gemm.h"
#include "internal.h"

namespace {

constexpr int BM = 128;          // UMMA M (cta_group::1)
constexpr int BKF = 32;          // K floats per stage = one 128-byte swizzle atom
constexpr uint32_t A_STAGE_BYTES = BM * BKF * 4;           // 16 KB
// SPLIT = 3xTF32 (precision 0 on tensor cores): every operand is carried as hi + lo, hi = rn_tf32(x),
// lo = rn_tf32(x - hi), and  A*B ~= A_hi*B_hi + A_hi*B_lo + A_lo*B_hi  (the dropped lo*lo term and the rounding of
// the lo parts are each <= 2^-24 relative: the same order as one fp32 rounding).  B_hi / B_lo are prepared at create time; four "splitter" warps turn each landed A
// stage into A_hi (in place) and A_lo (second buffer) before the MMA warp may read it.
// widest column tile: the accumulator is double-buffered in 512 TMEM columns -> 256; the 3xTF32 mode on single CTAs keeps
// 128 (its weight stage holds B_hi and B_lo); on CTA pairs each CTA holds half a weight stage and 256 fits there too
__host__ __device__ constexpr int bn_max(bool split, int cg = 1) { return (split && cg == 1) ? 128 : 256; }
// CG = 2 (cta_group::2): a pair of CTAs works on one 256-row tile; each loads its own 128 rows of A and HALF of the B tile
__host__ __device__ constexpr uint32_t b_stage_bytes(bool split, int cg = 1) { return bn_max(split, cg) / cg * BKF * 4; }   // allocated for the largest BN
__host__ __device__ constexpr uint32_t a_ring_stage(bool split) { return (split ? 2 : 1) * A_STAGE_BYTES; }
__host__ __device__ constexpr uint32_t b_ring_stage(bool split, int cg = 1) { return (split ? 2 : 1) * b_stage_bytes(split, cg); }
// epilogue transpose staging: one 32x32 fp32 tile per warp, float4-granular XOR swizzle (conflict-free both ways)
constexpr uint32_t smem_bytes(int ast, int bst, int epi_warps, bool split, int cg = 1) {
  return ast * a_ring_stage(split) + bst * b_ring_stage(split, cg) + 1024 /*align*/ + 256 /*barriers*/ + epi_warps * 32 * 32 * 4;
}

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  uint32_t done, addr = smem_u32(bar);
  do {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t"
        "}"
        : "=r"(done)
        : "r"(addr), "r"(parity)
        : "memory");
  } while (!done);
}
__device__ __forceinline__ void tma_load_2d(void* smem_dst, const CUtensorMap* tm, uint64_t* bar, int c0, int c1) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];" ::"r"(
          smem_u32(smem_dst)),
      "l"(tm), "r"(smem_u32(bar)), "r"(c0), "r"(c1)
      : "memory");
}
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint64_t* bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tc_mma_tf32(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t"
      "}" ::"r"(tmem_d),
      "l"(da), "l"(db), "r"(idesc), "r"(accumulate)
      : "memory");
}
__device__ __forceinline__ void tc_mma_f16(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t"
      "}" ::"r"(tmem_d),
      "l"(da), "l"(db), "r"(idesc), "r"(accumulate)
      : "memory");
}
// ---- cta_group::2: two CTAs of a cluster (one TPC) run one MMA of M = 256.  Only the leader (cluster rank 0) issues MMAs and
// commits; its full barriers collect the TMA bytes of both CTAs; commits arrive on the barriers of both (multicast).
__device__ __forceinline__ uint32_t cluster_rank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
__device__ __forceinline__ uint32_t mapa_leader(uint32_t addr) {     // the same shared-memory offset in the CTA of rank 0
  uint32_t r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(0));
  return r;
}
__device__ __forceinline__ void cluster_sync_all() {
  asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx_cluster(uint32_t cluster_addr, uint32_t bytes) {
  // (default .release.cta semantics: with .release.cluster every arrive costs a MEMBAR + ERRBAR in the producer's loop)
  asm volatile("mbarrier.arrive.expect_tx.shared::cluster.b64 _, [%0], %1;" ::"r"(cluster_addr), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive_cluster(uint32_t cluster_addr) {
  asm volatile("mbarrier.arrive.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr) : "memory");
}
__device__ __forceinline__ void tma_load_2d_cg2(void* smem_dst, const CUtensorMap* tm, uint32_t bar_cluster_addr, int c0, int c1) {
  asm volatile(
      "cp.async.bulk.tensor.2d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];" ::"r"(
          smem_u32(smem_dst)),
      "l"(tm), "r"(bar_cluster_addr), "r"(c0), "r"(c1)
      : "memory");
}
__device__ __forceinline__ void tc_commit_cg2(uint64_t* bar) {   // arrives on `bar` at the same offset in both CTAs
  asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;" ::"r"(
                   smem_u32(bar)),
               "h"((uint16_t)3)
               : "memory");
}
__device__ __forceinline__ void tc_mma_tf32_cg2(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::2.kind::tf32 [%0], %1, %2, %3, p;\n\t"
      "}" ::"r"(tmem_d),
      "l"(da), "l"(db), "r"(idesc), "r"(accumulate)
      : "memory");
}
__device__ __forceinline__ void tc_mma_f16_cg2(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n\t"
      "}" ::"r"(tmem_d),
      "l"(da), "l"(db), "r"(idesc), "r"(accumulate)
      : "memory");
}
__device__ __forceinline__ void tc_ld32(uint32_t taddr, uint32_t* r) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
      "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
      "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
        "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]),
        "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]),
        "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
      : "r"(taddr));
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}

// K-major, SWIZZLE_128B shared-memory matrix descriptor (sm100 format): start>>4 | LBO | SBO=1024B | version=1 | layout=2
__device__ __forceinline__ uint64_t make_desc(uint32_t saddr) {
  uint64_t d = 0;
  d |= (uint64_t)((saddr & 0x3FFFF) >> 4);
  d |= (uint64_t)1 << 16;                 // LBO (unused for swizzled K-major)
  d |= (uint64_t)(1024 >> 4) << 32;       // SBO: 8 rows x 128 B
  d |= (uint64_t)1 << 46;                 // descriptor version (sm100)
  d |= (uint64_t)2 << 61;                 // SWIZZLE_128B
  return d;
}

// ---- epilogue memory operations -------------------------------------------------------------------------
// Epilogue operands are streamed (read or written once per launch): L1::no_allocate.  Every access is PREDICATED inside the
// asm statement and carries no "memory" clobber, so the 16-row half of a chunk is one basic block: with `if (ok) store`
// branches and clobbering stores the four row groups of a half ran one after the other, each exposing its own shared-memory
// load and MUFU chain (ncu r2m: 24 % `wait`, issue slots half idle at 4 epilogue warps per scheduler).
// HF = 0: four fp32 (16 bytes); HF = 1 / 2: four IEEE fp16 / bfloat16 values (8 bytes), converted where they are used.
enum { IO16_C = 1 };   // GemmArgs::io16: in the 16-bit kernels every epilogue tensor is 16-bit; C is, only if this bit is set
template <int HF>
__device__ __forceinline__ uint4 ep_load(const char* p, bool pred) {
  uint4 v = make_uint4(0u, 0u, 0u, 0u);
  if (HF)
    asm volatile("{\n\t.reg .pred q;\n\tsetp.ne.b32 q, %3, 0;\n\t@q ld.global.nc.L1::no_allocate.v2.u32 {%0,%1}, [%2];\n\t}"
                 : "+r"(v.x), "+r"(v.y) : "l"(p), "r"((int)pred));
  else
    asm volatile("{\n\t.reg .pred q;\n\tsetp.ne.b32 q, %5, 0;\n\t@q ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];\n\t}"
                 : "+r"(v.x), "+r"(v.y), "+r"(v.z), "+r"(v.w) : "l"(p), "r"((int)pred));
  return v;
}
template <int HF>
__device__ __forceinline__ float4 ep_cvt(const uint4 v) {
  if (HF == 1) {
    const float2 a = __half22float2(*reinterpret_cast<const __half2*>(&v.x));
    const float2 b = __half22float2(*reinterpret_cast<const __half2*>(&v.y));
    return make_float4(a.x, a.y, b.x, b.y);
  }
  if (HF == 2)
    return make_float4(__uint_as_float(v.x << 16), __uint_as_float(v.x & 0xFFFF0000u),
                       __uint_as_float(v.y << 16), __uint_as_float(v.y & 0xFFFF0000u));
  return make_float4(__uint_as_float(v.x), __uint_as_float(v.y), __uint_as_float(v.z), __uint_as_float(v.w));
}
template <int HF>
__device__ __forceinline__ void ep_store(char* p, const float4 v, bool pred) {
  if (HF) {
    uint2 o;
    if (HF == 1) {
      __half2 a = __floats2half2_rn(v.x, v.y), b = __floats2half2_rn(v.z, v.w);
      o.x = *reinterpret_cast<uint32_t*>(&a); o.y = *reinterpret_cast<uint32_t*>(&b);
    } else {
      __nv_bfloat162 a = __floats2bfloat162_rn(v.x, v.y), b = __floats2bfloat162_rn(v.z, v.w);
      o.x = *reinterpret_cast<uint32_t*>(&a); o.y = *reinterpret_cast<uint32_t*>(&b);
    }
    asm volatile("{\n\t.reg .pred q;\n\tsetp.ne.b32 q, %3, 0;\n\t@q st.global.L1::no_allocate.v2.u32 [%0], {%1,%2};\n\t}"
                 ::"l"(p), "r"(o.x), "r"(o.y), "r"((int)pred));
  } else {
    asm volatile("{\n\t.reg .pred q;\n\tsetp.ne.b32 q, %5, 0;\n\t@q st.global.L1::no_allocate.v4.f32 [%0], {%1,%2,%3,%4};\n\t}"
                 ::"l"(p), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w), "r"((int)pred));
  }
}
// C of a 16-bit kernel: 16-bit or fp32 by a launch-uniform flag -> two complementary predicated stores, no branch
template <int HF>
__device__ __forceinline__ void ep_store_c(char* p, const float4 v, bool pred, bool c16) {
  if (HF) { ep_store<HF>(p, v, pred && c16); ep_store<0>(p, v, pred && !c16); }
  else ep_store<0>(p, v, pred);
}
__device__ __forceinline__ void ep_st_f32(float* p, float v, bool pred) {
  asm volatile("{\n\t.reg .pred q;\n\tsetp.ne.b32 q, %2, 0;\n\t@q st.global.f32 [%0], %1;\n\t}" ::"l"(p), "f"(v), "r"((int)pred));
}
__device__ __forceinline__ void ep_st_f64(double* p, double v, bool pred) {
  asm volatile("{\n\t.reg .pred q;\n\tsetp.ne.b32 q, %2, 0;\n\t@q st.global.f64 [%0], %1;\n\t}" ::"l"(p), "d"(v), "r"((int)pred));
}
// staging tile of the TMEM -> coalesced-domain transposition, addressed as shared memory (a generic pointer costs LD.E / ST.E)
__device__ __forceinline__ void sts128(uint32_t a, uint32_t x, uint32_t y, uint32_t z, uint32_t w) {
  asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(a), "r"(x), "r"(y), "r"(z), "r"(w) : "memory");
}
// Not volatile: the compiler may hoist it above the (volatile) global stores of the previous row group.  What keeps it behind
// the warp barrier that follows the tile's st.shared is its address: derived from stg_fence()'s opaque result.
__device__ __forceinline__ float4 lds128(uint32_t a) {
  float4 v;
  asm("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a));
  return v;
}
__device__ __forceinline__ uint32_t stg_fence(uint32_t a) {
  uint32_t r;
  asm volatile("mov.u32 %0, %1;" : "=r"(r) : "r"(a) : "memory");
  return r;
}

// sigmoid = rcp.approx(1 + ex2.approx(-z log2 e)): the two MUFU operations and nothing else (__fdividef adds a range test and
// two scaling multiplies per element that 1 + e^-z in [1, inf] never needs); error ~1e-7 << TF32 rounding.
// Packed fp32 pairs (FMUL2 / FADD2 / FFMA2 of sm_100): the epilogue of the fused kernels is bound by issue slots, not by the
// fp32 pipe (ncu r2n: selected + not_selected 45 % of the warp samples, 13.5 scalar FMUL / FADD / FFMA per output element);
// a packed instruction takes one slot for two elements.  Roundings are those of the scalar code (IEEE rn per operation).
__device__ __forceinline__ float2 f2(float a) { return make_float2(a, a); }
__device__ __forceinline__ float2 sigm2(float2 z) {
  const float2 t = __fmul2_rn(z, f2(-1.4426950408889634f));
  float2 e, r;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(e.x) : "f"(t.x));
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(e.y) : "f"(t.y));
  const float2 d = __fadd2_rn(e, f2(1.0f));
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r.x) : "f"(d.x));
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r.y) : "f"(d.y));
  return r;
}
// silu'(z) = s + silu(z) (1 - s) from s = sigmoid(z) and sl = z s
__device__ __forceinline__ float2 dsilu2(float2 s, float2 sl) { return __ffma2_rn(sl, __ffma2_rn(s, f2(-1.0f), f2(1.0f)), s); }

// round to the nearest TF32 value (10 explicit mantissa bits; ties away from zero), result exact in TF32 so the
// MMA's own truncation of the operand is a no-op
__device__ __forceinline__ float tf32_rn(float x) { return __uint_as_float((__float_as_uint(x) + 0x1000u) & 0xFFFFE000u); }

// EPI (GemmEpi) and PREP (the z-bar / u-bar stage of EPI_ADD2 / EPI_ADD2R) are compile-time: one kernel per epilogue,
// so the epilogue carries no run-time dispatch, no dead operands and no re-loaded argument fields.
// HF = 1 / 2 (precision 4 / 2): A and B operands are fp16 / bf16 in HBM, one stage = 64 K-elements (the same
// 128-byte rows), tcgen05.mma.kind::f16 with fp32 accumulation; every epilogue tensor is 16-bit too, C only if GemmArgs::io16 has IO16_C.
// CG = 2: the kernel is launched in clusters of two CTAs (cta_group::2).  A pair owns 256-row tiles: CTA rank r loads rows
// [256 t + 128 r, +128) of A and rows [BN r / 2, +BN / 2) of the B tile, the leader issues one M = 256 MMA per k-slice, each
// CTA's TMEM receives its own 128 rows of the accumulator and each CTA runs the epilogue of its rows.  The weights cross the
// L2 -> SM fabric once per 256 rows instead of once per 128: with 128-row tiles the 13 GEMM launches of a config-3 chunk moved
// 62 GB from L2 to the SMs (weights = 2 x the activation bytes per k-slice) for 32 GB of DRAM traffic, the two heaviest at the
// ~12 TB/s the fabric delivers; pairs move 47 GB (profiles/r2r_summary.md).
template <int AST, int BST, int EPI_WARPS, bool SPLIT, int EPI, bool PREP, bool AUX2, int HF = 0, int CG = 1>
__global__ void __launch_bounds__(96 + (SPLIT ? 128 : 0) + 32 * EPI_WARPS, 1)
k_gemm_tf32(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmA2,
            const __grid_constant__ CUtensorMap tmB, const __grid_constant__ CUtensorMap tmB2, GemmArgs g, int BN, int ntn) {
  static_assert(CG == 1 || CG == 2, "CTA group size");
  constexpr int BN_MAX = bn_max(SPLIT, CG);
  constexpr uint32_t A_RING_STAGE = a_ring_stage(SPLIT), B_RING_STAGE = b_ring_stage(SPLIT, CG);
  constexpr uint32_t B_STAGE_BYTES = b_stage_bytes(SPLIT, CG);
  constexpr int EW0 = SPLIT ? 7 : 3;     // first epilogue warp (warps 3..6 are the splitter in SPLIT mode)
  constexpr bool H16 = HF != 0;              // HF = 1: IEEE fp16, 2: bfloat16 operands and epilogue tensors
  constexpr int BKE = H16 ? 2 * BKF : BKF;   // K elements per stage
  static_assert(!(SPLIT && H16), "3xTF32 and 16-bit operands exclude each other");
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  // Two independent rings: A (activations, from HBM: deep, AST stages of [A | (A_lo)]) and B (weights, from L2:
  // shallow, BST stages of [B (B_hi) | (B_lo)]).  The bytes of A in flight set the achieved HBM bandwidth (a probe
  // with the same tile-shaped access pattern reaches 2.5 TB/s with 16 KB in flight per SM and 6.1 TB/s with 64 KB).
  auto sA = [&](int s) { return smem + s * A_RING_STAGE; };
  auto sAlo = [&](int s) { return smem + s * A_RING_STAGE + A_STAGE_BYTES; };
  auto sB = [&](int s) { return smem + AST * A_RING_STAGE + s * B_RING_STAGE; };
  auto sBlo = [&](int s) { return smem + AST * A_RING_STAGE + s * B_RING_STAGE + B_STAGE_BYTES; };
  uint64_t* bars = (uint64_t*)(smem + AST * A_RING_STAGE + BST * B_RING_STAGE);
  uint64_t* fullA = bars;                    // [AST]  TMA -> (splitter | MMA)
  uint64_t* emptyA = bars + AST;             // [AST]  MMA -> TMA
  uint64_t* readyA = bars + 2 * AST;         // [AST]  splitter -> MMA (SPLIT only)
  uint64_t* fullB = bars + 3 * AST;          // [BST]
  uint64_t* emptyB = bars + 3 * AST + BST;   // [BST]
  uint64_t* tfull = bars + 3 * AST + 2 * BST;        // [2]
  uint64_t* tempty = bars + 3 * AST + 2 * BST + 2;   // [2]
  uint32_t* tmem_slot = (uint32_t*)(bars + 3 * AST + 2 * BST + 4);
  static_assert((3 * AST + 2 * BST + 5) * 8 <= 256, "barrier block");
  float* stage_buf = (float*)(smem + AST * A_RING_STAGE + BST * B_RING_STAGE + 256);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int M = *g.m_ptr;
  const int rank = (CG == 2) ? (int)cluster_rank() : 0;       // position in the CTA pair
  const int num_mt = (M + BM * CG - 1) / (BM * CG);           // row blocks of 128 CG rows
  const int num_tiles = num_mt * ntn;
  const int num_kb = (g.K + BKE - 1) / BKE;
  const int tile0 = blockIdx.x / CG, tile_step = gridDim.x / CG;   // both CTAs of a pair walk the same tiles

  if (threadIdx.x == 0) {
    // CG = 2: the leader's full barriers take one expect_tx arrival per CTA, its accumulator-empty barriers one arrival
    // per epilogue warp of both CTAs; the empty / accumulator-full barriers of each CTA are hit by the multicast commits
    // (3xTF32 on pairs: A lands on the CTA's own full barrier, its splitter warps hand the stage to the leader's ready barrier)
    for (int s = 0; s < AST; ++s) { mbar_init(&fullA[s], SPLIT ? 1 : CG); mbar_init(&emptyA[s], 1); mbar_init(&readyA[s], 4 * CG); }
    for (int s = 0; s < BST; ++s) { mbar_init(&fullB[s], CG); mbar_init(&emptyB[s], 1); }
    for (int s = 0; s < 2; ++s) { mbar_init(&tfull[s], 1); mbar_init(&tempty[s], EPI_WARPS * CG); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 1) {
    if (CG == 2) {
      asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(tmem_slot)) : "memory");
      asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
    } else {
      asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(tmem_slot)) : "memory");
      asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
  }
  tc_fence_before();
  __syncthreads();
  if (CG == 2) cluster_sync_all();     // the peer's barriers are initialised before anything arrives on them
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;

  if (warp == 0) {
    // ===== TMA producer, A ring =====
    if (lane == 0) {
      int stage = 0; uint32_t phase = 0;
      const int kb1 = g.A2 ? g.K1 / BKE : num_kb;   // k-blocks [kb1, num_kb) come from the second activation tensor
      for (int tile = tile0; tile < num_tiles; tile += tile_step) {
        int mt = tile / ntn;
        if (g.rev) mt = num_mt - 1 - mt;
        const int row = (mt * CG + rank) * BM;      // (past M for the odd last block of a pair: TMA fills zeros)
        for (int kb = 0; kb < num_kb; ++kb) {
          mbar_wait(&emptyA[stage], phase ^ 1);
          if (CG == 2 && !SPLIT) {
            const uint32_t fb = mapa_leader(smem_u32(&fullA[stage]));
            mbar_expect_tx_cluster(fb, A_STAGE_BYTES);
            if (kb < kb1) tma_load_2d_cg2(sA(stage), &tmA, fb, kb * BKE, row);
            else tma_load_2d_cg2(sA(stage), &tmA2, fb, (kb - kb1) * BKE, row);
          } else {
            mbar_expect_tx(&fullA[stage], A_STAGE_BYTES);
            if (kb < kb1) tma_load_2d(sA(stage), &tmA, &fullA[stage], kb * BKE, row);
            else tma_load_2d(sA(stage), &tmA2, &fullA[stage], (kb - kb1) * BKE, row);
          }
          if (++stage == AST) { stage = 0; phase ^= 1; }
        }
      }
    }
  } else if (warp == 2) {
    // ===== TMA producer, B ring =====
    if (lane == 0) {
      int stage = 0; uint32_t phase = 0;
      const uint32_t bytes = (SPLIT ? 2u : 1u) * (uint32_t)(BN / CG) * BKF * 4;
      for (int tile = tile0; tile < num_tiles; tile += tile_step) {
        int mt = tile / ntn, nt = tile - mt * ntn;
        for (int kb = 0; kb < num_kb; ++kb) {
          mbar_wait(&emptyB[stage], phase ^ 1);
          if (CG == 2) {
            const uint32_t fb = mapa_leader(smem_u32(&fullB[stage]));
            mbar_expect_tx_cluster(fb, bytes);
            tma_load_2d_cg2(sB(stage), &tmB, fb, kb * BKE, nt * BN + rank * (BN / 2));
            if (SPLIT) tma_load_2d_cg2(sBlo(stage), &tmB2, fb, kb * BKE, nt * BN + rank * (BN / 2));
          } else {
            mbar_expect_tx(&fullB[stage], bytes);
            tma_load_2d(sB(stage), &tmB, &fullB[stage], kb * BKE, nt * BN);
            if (SPLIT) tma_load_2d(sBlo(stage), &tmB2, &fullB[stage], kb * BKE, nt * BN);
          }
          if (++stage == BST) { stage = 0; phase ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    // ===== MMA issuer =====
    if (lane == 0 && rank == 0) {     // (CG = 2: the leader issues for the pair)
      // instruction descriptor: D=f32, A=B=tf32, K-major both, N>>3, M>>4 (M = 256 across the pair for CG = 2)
      // (A / B format field: 2 = tf32 for kind::tf32; kind::f16: 0 = f16, 1 = bf16)
      const uint32_t ofmt = H16 ? (uint32_t)(HF - 1) : 2u;
      const uint32_t idesc = (1u << 4) | (ofmt << 7) | (ofmt << 10) | ((uint32_t)(BN >> 3) << 17) | ((uint32_t)((BM * CG) >> 4) << 24);
      int sa = 0, sb = 0; uint32_t pa = 0, pb = 0; int it = 0;
      for (int tile = tile0; tile < num_tiles; tile += tile_step, ++it) {
        int acc = it & 1;
        mbar_wait(&tempty[acc], ((it >> 1) & 1) ^ 1);
        tc_fence_after();
        uint32_t d_tmem = tmem_base + acc * BN_MAX;
        for (int kb = 0; kb < num_kb; ++kb) {
          mbar_wait(SPLIT ? &readyA[sa] : &fullA[sa], pa);
          mbar_wait(&fullB[sb], pb);
          tc_fence_after();
          uint64_t da = make_desc(smem_u32(sA(sa)));
          uint64_t db = make_desc(smem_u32(sB(sb)));
#pragma unroll
          for (int k = 0; k < BKF / 8; ++k) {   // UMMA_K = 8 tf32 or 16 halves = 32 bytes -> +2 in the (addr >> 4) field
            if (CG == 2) {
              if (H16) tc_mma_f16_cg2(d_tmem, da + 2 * k, db + 2 * k, idesc, (kb | k) ? 1u : 0u);
              else tc_mma_tf32_cg2(d_tmem, da + 2 * k, db + 2 * k, idesc, (kb | k) ? 1u : 0u);
            } else {
              if (H16) tc_mma_f16(d_tmem, da + 2 * k, db + 2 * k, idesc, (kb | k) ? 1u : 0u);
              else tc_mma_tf32(d_tmem, da + 2 * k, db + 2 * k, idesc, (kb | k) ? 1u : 0u);
            }
          }
          if (SPLIT) {
            uint64_t dal = make_desc(smem_u32(sAlo(sa)));
            uint64_t dbl = make_desc(smem_u32(sBlo(sb)));
#pragma unroll
            for (int k = 0; k < BKF / 8; ++k) {
              if (CG == 2) {
                tc_mma_tf32_cg2(d_tmem, da + 2 * k, dbl + 2 * k, idesc, 1u);    // A_hi * B_lo
                tc_mma_tf32_cg2(d_tmem, dal + 2 * k, db + 2 * k, idesc, 1u);    // A_lo * B_hi
              } else {
                tc_mma_tf32(d_tmem, da + 2 * k, dbl + 2 * k, idesc, 1u);    // A_hi * B_lo
                tc_mma_tf32(d_tmem, dal + 2 * k, db + 2 * k, idesc, 1u);    // A_lo * B_hi
              }
            }
          }
          if (CG == 2) { tc_commit_cg2(&emptyA[sa]); tc_commit_cg2(&emptyB[sb]); }
          else { tc_commit(&emptyA[sa]); tc_commit(&emptyB[sb]); }
          if (++sa == AST) { sa = 0; pa ^= 1; }
          if (++sb == BST) { sb = 0; pb ^= 1; }
        }
        if (CG == 2) tc_commit_cg2(&tfull[acc]); else tc_commit(&tfull[acc]);
      }
    }
  } else if (SPLIT && warp < EW0) {
    // ===== splitter warps (3xTF32): A -> A_hi (in place, low 13 mantissa bits cleared) and A_lo = A - A_hi =====
    const int t = threadIdx.x - 96;       // 0..127
    int stage = 0; uint32_t phase = 0;
    for (int tile = tile0; tile < num_tiles; tile += tile_step) {
      for (int kb = 0; kb < num_kb; ++kb) {
        mbar_wait(&fullA[stage], phase);
        float4* pa = reinterpret_cast<float4*>(sA(stage));
        float4* pl = reinterpret_cast<float4*>(sAlo(stage));
#pragma unroll
        for (int i = 0; i < (int)(A_STAGE_BYTES / 16) / 128; ++i) {
          float4 v = pa[t + i * 128];
          float4 h = make_float4(tf32_rn(v.x), tf32_rn(v.y), tf32_rn(v.z), tf32_rn(v.w));
          pa[t + i * 128] = h;
          pl[t + i * 128] = make_float4(tf32_rn(v.x - h.x), tf32_rn(v.y - h.y), tf32_rn(v.z - h.z), tf32_rn(v.w - h.w));
        }
        // generic-proxy writes -> visible to the async proxy (tcgen05.mma reads shared memory through it)
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncwarp();
        if (lane == 0) {
          if (CG == 2) mbar_arrive_cluster(mapa_leader(smem_u32(&readyA[stage])));
          else mbar_arrive(&readyA[stage]);
        }
        if (++stage == AST) { stage = 0; phase ^= 1; }
      }
    }
  } else {
    // ===== epilogue warps =====
    const int q = warp & 3;   // TMEM lane quarter
    int it = 0;
    for (int tile = tile0; tile < num_tiles; tile += tile_step, ++it) {
      int mt = tile / ntn, nt = tile - mt * ntn;
      if (g.rev) mt = num_mt - 1 - mt;
      mt = mt * CG + rank;                 // this CTA's 128-row block
      int acc = it & 1;
      mbar_wait(&tfull[acc], (it >> 1) & 1);
      tc_fence_after();
      // Each 32-column chunk: TMEM -> registers (lane = row) -> padded smem -> registers in the
      // "coalesced domain" (8 lanes x float4 cover one row's 128 B, 4 rows per warp instruction), so
      // every global load/store of the epilogue touches 4 lines per instruction instead of 32.
      const uint32_t stg_s = smem_u32(stage_buf) + (uint32_t)(warp - EW0) * (32 * 8 * 16);
      const int chunk0 = (warp - EW0) >> 2;   // this warp takes chunks chunk0, chunk0 + EPI_WARPS/4, ...
      const int rsub = lane >> 3, c4 = (lane & 7) * 4;
      const int rbase = mt * BM + q * 32;
      const bool c16 = H16 && (g.io16 & IO16_C);
      const bool haveC = g.C != nullptr;
      for (int c0 = chunk0 * 32; c0 < BN; c0 += 32 * (EPI_WARPS / 4)) {
        {
          uint32_t r[32];
          tc_ld32(tmem_base + ((uint32_t)(q * 32) << 16) + acc * BN_MAX + c0, r);
#pragma unroll
          for (int gq = 0; gq < 8; ++gq)
            sts128(stg_s + (uint32_t)(lane * 8 + (gq ^ (lane & 7))) * 16, r[4 * gq], r[4 * gq + 1], r[4 * gq + 2], r[4 * gq + 3]);
        }
        __syncwarp();
        const uint32_t stg = stg_fence(stg_s);
        const int col = nt * BN + c0 + c4;
        const bool col_ok = (col < g.N) && (c0 + c4 < BN);
        // Two halves of 16 rows: issue every aux load of a half up front, then process it.  Halving keeps the register
        // count low enough for 16 epilogue warps.
        constexpr bool need1 = (EPI == EPI_LATENT || EPI == EPI_LATENT_LAST || EPI == EPI_MUL_DSILU || EPI == EPI_ADD2);
        constexpr bool need2 = (EPI == EPI_ADD2 || EPI == EPI_ADD2R) && AUX2;   // no aux2: the term is in the K-concatenation
        constexpr bool out2 = (EPI == EPI_SILU_BOTH || EPI == EPI_SILU_U || EPI == EPI_LATENT || EPI == EPI_LATENT_LAST);
        // the column vector of the rank-1 / energy epilogues is the same for all 32 rows of the chunk: one load per chunk
        float4 w3 = make_float4(0.f, 0.f, 0.f, 0.f);
        if (EPI == EPI_LATENT_LAST || EPI == EPI_ADD2R) w3 = *reinterpret_cast<const float4*>(g.aux3 + (col_ok ? col : 0));
        // row pointers of this lane for the chunk (row rbase + rsub, column col); rows advance by 4 per visit
        const int row0 = rbase + rsub;
        const size_t cco = col_ok ? (size_t)col : 0;
        constexpr size_t EH = H16 ? 2 : 4;        // element size of the aux / out2 / prep tensors
        const size_t ec = c16 ? 2 : 4;            // element size of C
#pragma unroll 1
        for (int h = 0; h < 2; ++h) {
          const int rowh = row0 + h * 16;
          const char* p1 = need1 ? reinterpret_cast<const char*>(g.aux1) + ((size_t)rowh * g.ld1 + cco) * EH : nullptr;
          const char* p2 = need2 ? reinterpret_cast<const char*>(g.aux2) + ((size_t)rowh * g.ld2 + cco) * EH : nullptr;
          const char* pz = PREP ? reinterpret_cast<const char*>(g.zp) + ((size_t)rowh * g.ldzp + cco) * EH : nullptr;
          const size_t st1 = (size_t)4 * g.ld1 * EH, st2 = (size_t)4 * g.ld2 * EH, stz = (size_t)4 * g.ldzp * EH;
          uint4 ax1[4], ax2[4], ax3[4];   // raw bits (fp32 x 4, or 16-bit x 4 in .x .y)
          // per-row scalars (u, sigma, u of the prep stage) are prefetched with the aux rows: loaded at their point of use they
          // were the top stall of the EPI_LATENT_LAST epilogue (ncu: long_scoreboard on the first multiply by u)
          constexpr bool need_u = (EPI == EPI_SILU_U || EPI == EPI_LATENT || EPI == EPI_LATENT_LAST || EPI == EPI_ADD2R);
          float ru[4], rs[4], rp[4];
#pragma unroll
          for (int ii = 0; ii < 4; ++ii) {
            const int row = rowh + ii * 4;
            const bool ok = row < M && col_ok;
            const int rowc = (row < M) ? row : M - 1;
            ru[ii] = need_u ? g.u[rowc] : 0.f;
            rs[ii] = (EPI == EPI_LATENT_LAST) ? g.sig[rowc] : 0.f;
            rp[ii] = PREP ? g.pu[rowc] : 0.f;
            ax1[ii] = need1 ? ep_load<HF>(p1 + ii * st1, ok) : make_uint4(0u, 0u, 0u, 0u);
            ax2[ii] = need2 ? ep_load<HF>(p2 + ii * st2, ok) : make_uint4(0u, 0u, 0u, 0u);
            ax3[ii] = PREP ? ep_load<HF>(pz + ii * stz, ok) : make_uint4(0u, 0u, 0u, 0u);
          }
          char* qo = out2 ? reinterpret_cast<char*>(g.out2) + ((size_t)rowh * g.ldo2 + cco) * EH : nullptr;
          char* qc = reinterpret_cast<char*>(g.C) + ((size_t)rowh * g.ldc + cco) * ec;
          char* qz = PREP ? reinterpret_cast<char*>(g.zbp) + ((size_t)rowh * g.ldzbp + cco) * EH : nullptr;
          const size_t sto = (size_t)4 * g.ldo2 * EH, stc = (size_t)4 * g.ldc * ec, stzb = (size_t)4 * g.ldzbp * EH;
#pragma unroll
          for (int ii = 0; ii < 4; ++ii) {
            const int rl = (h * 4 + ii) * 4 + rsub;
            const int row = rbase + rl;
            const bool ok = row < M && col_ok;          // out-of-range lanes compute on zeros and store nothing
            const float4 v4 = lds128(stg + (uint32_t)(rl * 8 + ((lane & 7) ^ (rl & 7))) * 16);
            float o[4];
            if (EPI == EPI_LATENT_LAST) {
              const float4 x = ep_cvt<HF>(ax1[ii]);
              const float us = ru[ii], sg = rs[ii];
              const float cu = g.c1 * us, cus = cu * sg;
              const float2 vv[2] = {make_float2(v4.x, v4.y), make_float2(v4.z, v4.w)};
              const float2 xx[2] = {make_float2(x.x, x.y), make_float2(x.z, x.w)};
              const float2 ww[2] = {make_float2(w3.x, w3.y), make_float2(w3.z, w3.w)};
              float2 oo[2], zz2[2], up2 = f2(0.f), ep2 = f2(0.f);
#pragma unroll
              for (int j = 0; j < 2; ++j) {
                // one sigmoid serves silu and silu'
                const float2 sgm = sigm2(vv[j]);
                const float2 sl = __fmul2_rn(vv[j], sgm);
                oo[j] = __ffma2_rn(f2(g.c0), xx[j], __fmul2_rn(f2(cu), sl));
                zz2[j] = __fmul2_rn(__fmul2_rn(f2(cus), ww[j]), dsilu2(sgm, sl));
                up2 = __ffma2_rn(ww[j], sl, up2);
                ep2 = __ffma2_rn(oo[j], ww[j], ep2);     // 4 terms in fp32 (w_eff rounded to fp32), the rest of the sum in fp64
              }
              o[0] = oo[0].x; o[1] = oo[0].y; o[2] = oo[1].x; o[3] = oo[1].y;
              const float zb[4] = {zz2[0].x, zz2[0].y, zz2[1].x, zz2[1].y};
              float up = up2.x + up2.y;
              const float ep4 = ep2.x + ep2.y;
              // 3xTF32 (fp32-accurate mode): the 8-lane sum of the 32-column energy partial runs in fp64; TF32 mode: in fp32
              // (32 terms, error ~1e-7 relative, far below the TF32 operand rounding) -- the fp64 shuffles and adds were the
              // heaviest part of this epilogue (ncu: 794 us at 3.0 TB/s, 3.8e8 warp instructions per launch at config 3)
              typedef typename std::conditional<SPLIT, double, float>::type ep_t;
              ep_t ep = ok ? (ep_t)ep4 : (ep_t)0;
              if (!ok) up = 0.f;
#pragma unroll
              for (int off = 1; off < 8; off <<= 1) {
                up += __shfl_xor_sync(0xffffffffu, up, off);
                ep += __shfl_xor_sync(0xffffffffu, ep, off);
              }
              ep_store<HF>(qo + ii * sto, make_float4(zb[0], zb[1], zb[2], zb[3]), ok);
              ep_store_c<HF>(qc + ii * stc, make_float4(o[0], o[1], o[2], o[3]), ok && haveC, c16);
              const int64_t pi = ((int64_t)nt * ((BN + 31) >> 5) + (c0 >> 5)) * g.part_stride + (ok ? row : 0);
              ep_st_f32(g.upart + pi, g.c1 * sg * up, ok && (lane & 7) == 0);
              ep_st_f64(g.epart + pi, (double)ep, ok && (lane & 7) == 0);
            } else if (PREP) {
              // EPI_ADD2 / EPI_ADD2R followed by the z-bar / u-bar stage of the next MLP
              const float2 vv[2] = {make_float2(v4.x, v4.y), make_float2(v4.z, v4.w)};
              float2 oo[2];
              if (EPI == EPI_ADD2) {
                const float4 x = ep_cvt<HF>(ax1[ii]);
                oo[0] = __ffma2_rn(f2(g.c0), make_float2(x.x, x.y), vv[0]);
                oo[1] = __ffma2_rn(f2(g.c0), make_float2(x.z, x.w), vv[1]);
              } else {
                const float cs = g.c0 * ru[ii];
                oo[0] = __ffma2_rn(f2(cs), make_float2(w3.x, w3.y), vv[0]);
                oo[1] = __ffma2_rn(f2(cs), make_float2(w3.z, w3.w), vv[1]);
              }
              if (need2) {
                const float4 y = ep_cvt<HF>(ax2[ii]);
                oo[0] = __fadd2_rn(oo[0], make_float2(y.x, y.y));
                oo[1] = __fadd2_rn(oo[1], make_float2(y.z, y.w));
              }
              const float4 zq = ep_cvt<HF>(ax3[ii]);
              const float2 zq2[2] = {make_float2(zq.x, zq.y), make_float2(zq.z, zq.w)};
              const float cu = g.cp * rp[ii];
              float2 zz2[2], up2 = f2(0.f);
#pragma unroll
              for (int j = 0; j < 2; ++j) {
                const float2 sgm = sigm2(zq2[j]);
                const float2 sl = __fmul2_rn(zq2[j], sgm);
                up2 = __ffma2_rn(oo[j], sl, up2);
                zz2[j] = __fmul2_rn(__fmul2_rn(f2(cu), oo[j]), dsilu2(sgm, sl));
              }
              o[0] = oo[0].x; o[1] = oo[0].y; o[2] = oo[1].x; o[3] = oo[1].y;
              const float zb[4] = {zz2[0].x, zz2[0].y, zz2[1].x, zz2[1].y};
              float up = up2.x + up2.y;
              if (!ok) up = 0.f;
#pragma unroll
              for (int off = 1; off < 8; off <<= 1) up += __shfl_xor_sync(0xffffffffu, up, off);
              ep_store<HF>(qz + ii * stzb, make_float4(zb[0], zb[1], zb[2], zb[3]), ok);
              ep_store_c<HF>(qc + ii * stc, make_float4(o[0], o[1], o[2], o[3]), ok && haveC, c16);
              const int64_t pi = (g.pbase + (int64_t)nt * ((BN + 31) >> 5) + (c0 >> 5)) * g.part_stride + (ok ? row : 0);
              ep_st_f32(g.upart + pi, g.cp * up, ok && (lane & 7) == 0);
            } else {
              const float2 vv[2] = {make_float2(v4.x, v4.y), make_float2(v4.z, v4.w)};
              float2 oo[2];
              switch (EPI) {
                case EPI_SILU_BOTH:
                case EPI_SILU_U:
                case EPI_LATENT: {
                  ep_store<HF>(qo + ii * sto, v4, ok);
                  const float us = (EPI == EPI_SILU_BOTH) ? 1.0f : ru[ii];
                  if (EPI == EPI_LATENT) {
                    const float4 x = ep_cvt<HF>(ax1[ii]);
                    const float2 xx[2] = {make_float2(x.x, x.y), make_float2(x.z, x.w)};
                    const float cu = g.c1 * us;
#pragma unroll
                    for (int j = 0; j < 2; ++j)
                      oo[j] = __ffma2_rn(f2(g.c0), xx[j], __fmul2_rn(f2(cu), __fmul2_rn(vv[j], sigm2(vv[j]))));
                  } else if (EPI == EPI_SILU_U) {
#pragma unroll
                    for (int j = 0; j < 2; ++j) oo[j] = __fmul2_rn(f2(us), __fmul2_rn(vv[j], sigm2(vv[j])));
                  } else {
#pragma unroll
                    for (int j = 0; j < 2; ++j) oo[j] = __fmul2_rn(vv[j], sigm2(vv[j]));
                  }
                } break;
                case EPI_MUL_DSILU: {
                  const float4 z = ep_cvt<HF>(ax1[ii]);
                  const float2 zq2[2] = {make_float2(z.x, z.y), make_float2(z.z, z.w)};
#pragma unroll
                  for (int j = 0; j < 2; ++j) {
                    const float2 sgm = sigm2(zq2[j]);
                    oo[j] = __fmul2_rn(vv[j], dsilu2(sgm, __fmul2_rn(zq2[j], sgm)));
                  }
                } break;
                case EPI_ADD2: {
                  const float4 x = ep_cvt<HF>(ax1[ii]);
                  const float4 y = ep_cvt<HF>(ax2[ii]);
                  oo[0] = __fadd2_rn(__ffma2_rn(f2(g.c0), make_float2(x.x, x.y), vv[0]), make_float2(y.x, y.y));
                  oo[1] = __fadd2_rn(__ffma2_rn(f2(g.c0), make_float2(x.z, x.w), vv[1]), make_float2(y.z, y.w));
                } break;
                case EPI_ADD2R: {
                  const float4 y = ep_cvt<HF>(ax2[ii]);
                  const float cs = g.c0 * ru[ii];
                  oo[0] = __fadd2_rn(__ffma2_rn(f2(cs), make_float2(w3.x, w3.y), vv[0]), make_float2(y.x, y.y));
                  oo[1] = __fadd2_rn(__ffma2_rn(f2(cs), make_float2(w3.z, w3.w), vv[1]), make_float2(y.z, y.w));
                } break;
                default:
                  oo[0] = vv[0]; oo[1] = vv[1];
              }
              o[0] = oo[0].x; o[1] = oo[0].y; o[2] = oo[1].x; o[3] = oo[1].y;
              ep_store_c<HF>(qc + ii * stc, make_float4(o[0], o[1], o[2], o[3]), ok, c16);
            }
          }
        }   // halves
        __syncwarp();
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) {
        if (CG == 2) mbar_arrive_cluster(mapa_leader(smem_u32(&tempty[acc])));
        else mbar_arrive(&tempty[acc]);
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (CG == 2) cluster_sync_all();     // both CTAs are done with the pair's TMEM and with each other's barriers
  if (warp == 1) {
    tc_fence_after();
    if (CG == 2) asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, 512;" ::"r"(tmem_base) : "memory");
    else asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem_base) : "memory");
  }
}

// ---- host side: tensor maps -----------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn g_encode = nullptr;

typedef std::tuple<const void*, long long, long long, long long, int, int> TmKey;   // ptr, rows, K, ld, box_rows, exact
typedef std::map<TmKey, CUtensorMap> TmCache;
// one cache per model (allegro_model::tmaps): the maps describe that model's work buffers and weights on its device and die
// with it (al_gemm_tc_free); keyed by (pointer, shape), so a buffer that is re-allocated at another address gets a new map
TmCache& tm_cache(allegro_model* m) {
  if (!m->tmaps) m->tmaps = new TmCache();
  return *static_cast<TmCache*>(m->tmaps);
}

// exact = true: plain fp32 load (the 3xTF32 path splits the operand itself); false: TFLOAT32 map, i.e. the load
// rounds to nearest TF32 (the MMA alone would truncate: measured 2-3x larger error)
// kind 2 / 3: fp16 / bf16 operands of precision 2 (2-byte elements, 64 of them per 128-byte box row)
int get_tmap(allegro_model* m, const void* ptr, long long rows, long long K, long long ld, int box_rows, int kind, CUtensorMap* out) {
  TmKey key(ptr, rows, K, ld, box_rows, kind);
  auto& c = tm_cache(m);
  auto it = c.find(key);
  if (it != c.end()) { *out = it->second; return ALLEGRO_OK; }
  if (!g_encode) {
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    AL_CUDA(m, cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres));
    if (!fn || qres != cudaDriverEntryPointSuccess) { al_set_error(m, "cuTensorMapEncodeTiled not available"); return ALLEGRO_ERR_CUDA; }
    g_encode = (EncodeTiledFn)fn;
  }
  cuuint64_t gdim[2] = {(cuuint64_t)K, (cuuint64_t)rows};
  const int esz = kind >= 2 ? 2 : 4;
  cuuint64_t gstr[1] = {(cuuint64_t)ld * esz};
  cuuint32_t box[2] = {(cuuint32_t)(128 / esz), (cuuint32_t)box_rows};
  const CUtensorMapDataType dt = kind == 0 ? CU_TENSOR_MAP_DATA_TYPE_TFLOAT32 : kind == 1 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32
                               : kind == 2 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT16 : CU_TENSOR_MAP_DATA_TYPE_BFLOAT16;
  cuuint32_t estr[2] = {1, 1};
  CUtensorMap tm;
  CUresult r = g_encode(&tm, dt, 2, const_cast<void*>(ptr), gdim, gstr, box, estr,
                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) { al_set_error(m, "cuTensorMapEncodeTiled failed, code " + std::to_string((int)r)); return ALLEGRO_ERR_CUDA; }
  if (c.size() > 4096) c.clear();
  c[key] = tm;
  *out = tm;
  return ALLEGRO_OK;
}

}  // namespace

#define GEMM_LAUNCH(AS, BS, EW, SP, EP, PR, A2, H6, CG_)                                                                  \
  {                                                                                                                      \
    static_assert(smem_bytes(AS, BS, EW, SP, CG_) <= 232448, "shared memory budget (227 KB)");                           \
    static AttrOnce once;                                                                                                \
    if (once.need(m->device)) {                                                                                          \
      AL_CUDA(m, cudaFuncSetAttribute(k_gemm_tf32<AS, BS, EW, SP, EP, PR, A2, H6, CG_>,                                  \
                                      cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes(AS, BS, EW, SP, CG_))); \
      once.done(m->device);                                                                                              \
    }                                                                                                                    \
    cudaLaunchConfig_t lc = {};                                                                                          \
    lc.gridDim = dim3((unsigned)grid); lc.blockDim = dim3(96 + (SP ? 128 : 0) + 32 * EW);                                \
    lc.dynamicSmemBytes = smem_bytes(AS, BS, EW, SP, CG_); lc.stream = m->stream;                                        \
    cudaLaunchAttribute la[1];                                                                                           \
    la[0].id = cudaLaunchAttributeClusterDimension;                                                                      \
    la[0].val.clusterDim.x = CG_; la[0].val.clusterDim.y = 1; la[0].val.clusterDim.z = 1;                                \
    lc.attrs = la; lc.numAttrs = 1;                                                                                      \
    if (CG_ == 2) {                                                                                                      \
      /* persistent pairs: never more clusters than the device can hold at once (a GPC with an odd SM count leaves one   \
         SM without a partner), or the tiles of the late clusters would run as a second wave */                          \
      static std::atomic<int> max_pairs[64];                                                                             \
      int mp = max_pairs[m->device & 63].load(std::memory_order_acquire);                                                \
      if (mp == 0) {                                                                                                     \
        int nc = 0;                                                                                                      \
        AL_CUDA(m, cudaOccupancyMaxActiveClusters(&nc, k_gemm_tf32<AS, BS, EW, SP, EP, PR, A2, H6, CG_>, &lc));          \
        mp = nc > 0 ? nc : -1;                                                                                           \
        max_pairs[m->device & 63].store(mp, std::memory_order_release);                                                  \
      }                                                                                                                  \
      if (mp < 0) { al_set_error(m, "gemm: no CTA pair fits on this device"); return ALLEGRO_ERR_CUDA; }                 \
      if (grid > 2 * mp) lc.gridDim = dim3((unsigned)(2 * mp));                                                          \
    }                                                                                                                    \
    AL_CUDA(m, cudaLaunchKernelEx(&lc, k_gemm_tf32<AS, BS, EW, SP, EP, PR, A2, H6, CG_>, tmA, tmA2, tmB, tmB2, g, BN, ntn)); \
  }
// one instantiation per epilogue (PREP only exists for the two x-bar epilogues)
#define GEMM_DISPATCH(AS, BS, EW, SP, H6, CG_)                                                                            \
  switch (g.epi) {                                                                                                       \
    case EPI_PLAIN: GEMM_LAUNCH(AS, BS, EW, SP, EPI_PLAIN, false, false, H6, CG_) break;                                 \
    case EPI_SILU_BOTH: GEMM_LAUNCH(AS, BS, EW, SP, EPI_SILU_BOTH, false, false, H6, CG_) break;                         \
    case EPI_SILU_U: GEMM_LAUNCH(AS, BS, EW, SP, EPI_SILU_U, false, false, H6, CG_) break;                               \
    case EPI_LATENT: GEMM_LAUNCH(AS, BS, EW, SP, EPI_LATENT, false, false, H6, CG_) break;                               \
    case EPI_MUL_DSILU: GEMM_LAUNCH(AS, BS, EW, SP, EPI_MUL_DSILU, false, false, H6, CG_) break;                         \
    case EPI_LATENT_LAST: GEMM_LAUNCH(AS, BS, EW, SP, EPI_LATENT_LAST, false, false, H6, CG_) break;                     \
    case EPI_ADD2:                                                                                                       \
      if (g.prep && g.aux2) GEMM_LAUNCH(AS, BS, EW, SP, EPI_ADD2, true, true, H6, CG_)                                   \
      else if (g.prep) GEMM_LAUNCH(AS, BS, EW, SP, EPI_ADD2, true, false, H6, CG_)                                       \
      else if (g.aux2) GEMM_LAUNCH(AS, BS, EW, SP, EPI_ADD2, false, true, H6, CG_)                                       \
      else GEMM_LAUNCH(AS, BS, EW, SP, EPI_ADD2, false, false, H6, CG_)                                                  \
      break;                                                                                                             \
    case EPI_ADD2R:                                                                                                      \
      if (g.prep && g.aux2) GEMM_LAUNCH(AS, BS, EW, SP, EPI_ADD2R, true, true, H6, CG_)                                  \
      else if (g.prep) GEMM_LAUNCH(AS, BS, EW, SP, EPI_ADD2R, true, false, H6, CG_)                                      \
      else if (g.aux2) GEMM_LAUNCH(AS, BS, EW, SP, EPI_ADD2R, false, true, H6, CG_)                                      \
      else GEMM_LAUNCH(AS, BS, EW, SP, EPI_ADD2R, false, false, H6, CG_)                                                 \
      break;                                                                                                             \
    default: al_set_error(m, "gemm: unknown epilogue"); return ALLEGRO_ERR_BAD_ARG;                                      \
  }

// Tile geometry shared by the non-split launchers.  CTA pairs (cta_group::2, 256-row tiles) whenever the problem has at least
// one pair tile per pair of SMs; small problems keep 128-row tiles (twice as many tiles to spread over the SMs).
struct TileGeom { int ntn, BN, cg, grid; };
static void tile_cols(int N, int bnmax, int* ntn, int* BN) {
  *ntn = (N + bnmax - 1) / bnmax;
  *BN = ((N + *ntn - 1) / *ntn + 15) & ~15;
}
static TileGeom tile_geom(const allegro_model* m, const GemmArgs& g, bool split = false) {
  TileGeom t;
  const int sms = m->sm_count & ~1;
  tile_cols(g.N, bn_max(split, 2), &t.ntn, &t.BN);
  const int pair_tiles = ((g.m_cap + 2 * BM - 1) / (2 * BM)) * t.ntn;
  t.cg = (m->gemm_cta_pairs && pair_tiles * 2 >= sms && sms >= 2) ? 2 : 1;
  if (split && t.cg == 2) {
    // the row-partial buffers of the fused epilogues are indexed by 32-column chunk and sized for the single-CTA tiling
    // (al_gemm_tc_row_parts): the pair tiling may be used only where both tilings number the chunks alike
    int n1, b1;
    tile_cols(g.N, bn_max(true, 1), &n1, &b1);
    if ((b1 & 31) || (t.BN & 31)) t.cg = 1;
  }
  if (t.cg == 2) t.grid = sms;
  else {
    tile_cols(g.N, bn_max(split, 1), &t.ntn, &t.BN);
    const int tiles_cap = ((g.m_cap + BM - 1) / BM) * t.ntn;
    t.grid = tiles_cap < m->sm_count ? tiles_cap : m->sm_count;
  }
  return t;
}

// precision 1: TF32 operands (rounded to nearest by the TMA load), fp32 accumulation
int al_gemm_tc(allegro_model* m, const GemmArgs& g_in) {
  GemmArgs g = g_in;
  g.rev = al_next_rev(m);
  const TileGeom t = tile_geom(m, g);
  const int ntn = t.ntn, BN = t.BN, grid = t.grid;
  CUtensorMap tmA, tmA2, tmB, tmB2;
  AL_CHECK(get_tmap(m, g.A, g.m_cap, g.A2 ? g.K1 : g.K, g.lda, BM, 0, &tmA));
  if (g.A2) AL_CHECK(get_tmap(m, g.A2, g.m_cap, g.K - g.K1, g.lda2, BM, 0, &tmA2));
  else tmA2 = tmA;
  AL_CHECK(get_tmap(m, g.Bt, g.N, g.K, g.ldb, BN / t.cg, 0, &tmB));
  tmB2 = tmB;
  // Ring depths, 128-row tiles: A 4 x 16 KB, B 3 x 32 KB (6/2 and 3/3 within 1 %; round 2, config 2, GEMM group per step,
  // A stages / B stages / epilogue warps: 4/3/16 32.5 ms, 5/3/12 33.9 ms, 6/3/8 37.3 ms, 6/2/16 35.4 ms; L2 prefetch of the A
  // tiles 4-12 k-blocks ahead 33.3 ms; B stages multicast inside 2-CTA clusters (still cta_group::1) 32.8 ms: the multicast
  // does not cut L2 traffic below cluster size 8).  CTA pairs: each CTA holds half of every B stage (16 KB), the shared
  // memory that frees deepens the rings to A 6 / B 4.
  if (t.cg == 2) { GEMM_DISPATCH(6, 4, 16, false, 0, 2) }
  else { GEMM_DISPATCH(4, 3, 16, false, 0, 1) }
  m->launches++;
  return ALLEGRO_OK;
}

// precision 2 / 4: 16-bit operands (fp16 or bf16, g.hfmt) in HBM, tcgen05.mma.kind::f16, fp32 accumulation
int al_gemm_h16(allegro_model* m, const GemmArgs& g_in) {
  GemmArgs g = g_in;
  g.rev = al_next_rev(m);
  if (!g.Bt16) { al_set_error(m, "16-bit GEMM: 16-bit weights missing"); return ALLEGRO_ERR_BAD_ARG; }
  if ((g.K & 7) || (g.lda & 7) || (g.ldb & 7) || (g.A2 && ((g.lda2 & 7) || (g.K1 & 63)))) {
    al_set_error(m, "16-bit GEMM: K and the row strides must be multiples of 8 elements (K1 of 64)");
    return ALLEGRO_ERR_BAD_HPARAMS;
  }
  const int kind = 2 + (g.hfmt ? 1 : 0);
  const TileGeom t = tile_geom(m, g);
  const int ntn = t.ntn, BN = t.BN, grid = t.grid;
  CUtensorMap tmA, tmA2, tmB, tmB2;
  AL_CHECK(get_tmap(m, g.A, g.m_cap, g.A2 ? g.K1 : g.K, g.lda, BM, kind, &tmA));
  if (g.A2) AL_CHECK(get_tmap(m, g.A2, g.m_cap, g.K - g.K1, g.lda2, BM, kind, &tmA2));
  else tmA2 = tmA;
  AL_CHECK(get_tmap(m, g.Bt16, g.N, g.K, g.ldb, BN / t.cg, kind, &tmB));
  tmB2 = tmB;
  if (t.cg == 2) {
    if (g.hfmt == 0) { GEMM_DISPATCH(6, 4, 16, false, 1, 2) } else { GEMM_DISPATCH(6, 4, 16, false, 2, 2) }
  } else {
    if (g.hfmt == 0) { GEMM_DISPATCH(4, 3, 16, false, 1, 1) } else { GEMM_DISPATCH(4, 3, 16, false, 2, 1) }
  }
  m->launches++;
  return ALLEGRO_OK;
}

// precision 0 on tensor cores: 3xTF32 split operands (fp32-level accuracy), tiles 128 x <=128
int al_gemm_tc3(allegro_model* m, const GemmArgs& g_in) {
  GemmArgs g = g_in;
  g.rev = al_next_rev(m);
  if (!g.Bt_hi || !g.Bt_lo) { al_set_error(m, "3xTF32 GEMM: split weights missing"); return ALLEGRO_ERR_BAD_ARG; }
  const TileGeom t = tile_geom(m, g, true);
  const int ntn = t.ntn, BN = t.BN, grid = t.grid;
  CUtensorMap tmA, tmA2, tmB, tmB2;
  AL_CHECK(get_tmap(m, g.A, g.m_cap, g.A2 ? g.K1 : g.K, g.lda, BM, 1, &tmA));
  if (g.A2) AL_CHECK(get_tmap(m, g.A2, g.m_cap, g.K - g.K1, g.lda2, BM, 1, &tmA2));
  else tmA2 = tmA;
  AL_CHECK(get_tmap(m, g.Bt_hi, g.N, g.K, g.ldb, BN / t.cg, 1, &tmB));
  AL_CHECK(get_tmap(m, g.Bt_lo, g.N, g.K, g.ldb, BN / t.cg, 1, &tmB2));
  // pairs: 256-column tiles (each CTA holds 128 rows of B_hi and of B_lo per stage: the shared-memory layout of the single-CTA
  // kernel), weights cross L2 -> SM once per 256 rows and the activations twice instead of four times
  if (t.cg == 2) { GEMM_DISPATCH(4, 2, 8, true, 0, 2) }
  else { GEMM_DISPATCH(4, 2, 8, true, 0, 1) }
  m->launches++;
  return ALLEGRO_OK;
}
#undef GEMM_DISPATCH
#undef GEMM_LAUNCH

int al_gemm_tc_row_parts(int N, bool split) {
  int ntn = (N + bn_max(split) - 1) / bn_max(split);
  int BN = ((N + ntn - 1) / ntn + 15) & ~15;
  return ntn * ((BN + 31) >> 5);
}

void al_gemm_tc_free(allegro_model* m) {
  delete static_cast<TmCache*>(m->tmaps);
  m->tmaps = nullptr;
}
