// a5 -- the A.W contraction of the CROWN backward recursion (A <- A.Lambda_i W_i)
// on the 5th-generation tensor cores, fp32-accurate via 3xTF32:
//     D = A_hi.W_hi + A_hi.W_lo + A_lo.W_hi          (a = a_hi + a_lo, both exactly TF32-representable)
// The dropped A_lo.W_lo term and the TF32 rounding of the lo parts are O(2^-22) relative per product.
//
// Design (sm_100a):
//   * operands K-major in global memory: A_hi/A_lo [M,K], Wt_hi/Wt_lo [N,K] (weights are transposed and
//     split once at crown_init); TMA (cp.async.bulk.tensor, 128B swizzle) stages 4 operand tiles per
//     pipeline stage into shared memory; one elected thread issues tcgen05.mma.kind::tf32 (UMMA 128 x BN x 8)
//     with the accumulator in TMEM;
//   * warp roles: warp 0 TMA producer, warp 1 MMA issuer, warp 2 TMEM allocator, warps 4-11 epilogue
//     (two warps per TMEM lane quadrant, 64 columns each, one tcgen05.ld.32x32b.x64 per drain);
//   * measured on B200: the tensor core's fp32 accumulation truncates, ~0.5 ulp of the running sum per MMA,
//     so the error grows linearly with the length of an accumulation chain.  Two measures keep the result at
//     CUDA-core FFMA accuracy: (1) two accumulators in TMEM, "big" for hi.hi and "small" for lo.hi + hi.lo
//     (2^-11 of big), so big sees one MMA per k-step and small's truncation is 2^-11 smaller; (2) K is cut into
//     drain chunks of k_drain elements (default 128 = 16 MMAs on big): each chunk of big is accumulated in
//     TMEM, then added into an fp32 register running sum by the epilogue warps (round-to-nearest) while the
//     tensor core fills the other buffer; small is drained every 16384 elements of K.  All four accumulators
//     (big/small x double buffer) use the full 512 TMEM columns;
//   * persistent grid (one CTA per SM), static tile order grouped along M for L2 reuse of W.
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include "common.cuh"
#include "kernels.h"

namespace crownb200 {

namespace tc {

constexpr int BM = 128;
constexpr int BK = 32;               // 32 fp32 = 128 B = one swizzle row
constexpr int UMMA_K = 8;            // kind::tf32: 32 bytes of K per instruction
constexpr int GROUP_M = 8;           // m-blocks per raster group

template <int BN>
struct Cfg {
  static constexpr int STAGES = (BN == 128) ? 3 : 2;
  static constexpr int A_BYTES = BM * BK * 4;
  static constexpr int B_BYTES = BN * BK * 4;
  static constexpr int STAGE_BYTES = 2 * A_BYTES + 2 * B_BYTES;
  static constexpr int EPI_WARPS = 8;                // 4 lane quadrants x 2 column halves of BN/2
  static constexpr int EPI_COLS = BN / 2;            // columns drained by one epilogue warp
  static constexpr int THREADS = 128 + EPI_WARPS * 32;
  static constexpr int TMEM_COLS = 4 * BN;           // {big, small} accumulators, each double-buffered
  static constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + 1024 /*align slack*/ + 256 /*barriers*/;
};

// ---------------------------------------------------------------- PTX wrappers
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" :: "r"(bar) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
      "selp.u32 %0, 1, 0, p;\n\t}"
      : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
  return ok != 0;
}
__device__ __forceinline__ uint64_t globaltimer_ns() {
  uint64_t t;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
  return t;
}
// Bounded wait: a protocol bug must trap, not hang the GPU.
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  if (mbar_try_wait(bar, parity)) return;
  uint64_t t0 = globaltimer_ns();
  uint32_t spins = 0;
  while (!mbar_try_wait(bar, parity)) {
    if ((++spins & 1023u) == 0 && globaltimer_ns() - t0 > 4000000000ull) {
      printf("crownb200 gemm_tc: mbarrier wait timed out (block %d thread %d bar %u parity %u)\n",
             blockIdx.x, threadIdx.x, bar, parity);
      __trap();
    }
  }
}
__device__ __forceinline__ void fence_barrier_init() {
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void fence_proxy_async() {
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* map, int x, int y, uint32_t bar) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
      :: "r"(dst), "l"(map), "r"(x), "r"(y), "r"(bar) : "memory");
}
__device__ __forceinline__ void prefetch_tmap(const CUtensorMap* map) {
  asm volatile("prefetch.tensormap [%0];" :: "l"(map) : "memory");
}
__device__ __forceinline__ void tcgen05_fence_after() {
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
}
__device__ __forceinline__ void tcgen05_fence_before() {
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
}
__device__ __forceinline__ void tmem_alloc(uint32_t dst_smem, uint32_t ncols) {
  asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" :: "r"(dst_smem), "r"(ncols) : "memory");
}
__device__ __forceinline__ void tmem_relinquish() {
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t addr, uint32_t ncols) {
  asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(addr), "r"(ncols) : "memory");
}
__device__ __forceinline__ void umma_tf32(uint32_t tmem_d, uint64_t desc_a, uint64_t desc_b, uint32_t idesc,
                                          uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}"
      :: "r"(tmem_d), "l"(desc_a), "l"(desc_b), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void umma_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" :: "r"(bar) : "memory");
}
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&v)[32]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
      "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,"
      "%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
      : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
        "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]),
        "=r"(v[16]), "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]),
        "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
      : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_ld64(uint32_t taddr, uint32_t (&v)[64]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x64.b32 "
      "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,"
      "%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31,"
      "%32,%33,%34,%35,%36,%37,%38,%39,%40,%41,%42,%43,%44,%45,%46,%47,"
      "%48,%49,%50,%51,%52,%53,%54,%55,%56,%57,%58,%59,%60,%61,%62,%63}, [%64];"
      : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
        "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]),
        "=r"(v[16]), "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]),
        "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31]),
        "=r"(v[32]), "=r"(v[33]), "=r"(v[34]), "=r"(v[35]), "=r"(v[36]), "=r"(v[37]), "=r"(v[38]), "=r"(v[39]),
        "=r"(v[40]), "=r"(v[41]), "=r"(v[42]), "=r"(v[43]), "=r"(v[44]), "=r"(v[45]), "=r"(v[46]), "=r"(v[47]),
        "=r"(v[48]), "=r"(v[49]), "=r"(v[50]), "=r"(v[51]), "=r"(v[52]), "=r"(v[53]), "=r"(v[54]), "=r"(v[55]),
        "=r"(v[56]), "=r"(v[57]), "=r"(v[58]), "=r"(v[59]), "=r"(v[60]), "=r"(v[61]), "=r"(v[62]), "=r"(v[63])
      : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_ld_wait() {
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}

// Shared-memory matrix descriptor, K-major operand tile with 128-byte swizzle (rows of 128 B, 8-row groups
// 1024 B apart): start address (>>4) | SBO = 1024 B (>>4) at bit 32 | version 1 at bit 46 | SWIZZLE_128B (2) at bit 61.
__device__ __forceinline__ uint64_t make_kmajor_sw128_desc(uint32_t smem_addr) {
  uint64_t d = 0;
  d |= (uint64_t)((smem_addr & 0x3FFFFu) >> 4);
  d |= (uint64_t)(1024u >> 4) << 32;
  d |= (uint64_t)1 << 46;
  d |= (uint64_t)2 << 61;
  return d;
}
// Instruction descriptor for kind::tf32, fp32 accumulate, both operands K-major, M = 128, N = BN.
__host__ __device__ constexpr uint32_t make_idesc_tf32(int m, int n) {
  return (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(m >> 4) << 24);
}

__device__ __forceinline__ void tile_coords(int t, int m_tiles, int n_tiles, int& mb, int& nb) {
  // groups of GROUP_M m-blocks sweep all n-blocks: concurrently running CTAs share W tiles in L2
  int per_group = GROUP_M * n_tiles;
  int g = t / per_group;
  int first_m = g * GROUP_M;
  int gm = min(GROUP_M, m_tiles - first_m);
  int in_g = t - g * per_group;
  mb = first_m + in_g % gm;
  nb = in_g / gm;
}

template <int BN>
__global__ void __launch_bounds__(Cfg<BN>::THREADS, 1)
gemm_tf32x3_kernel(const __grid_constant__ CUtensorMap tmA_hi, const __grid_constant__ CUtensorMap tmA_lo,
                   const __grid_constant__ CUtensorMap tmB_hi, const __grid_constant__ CUtensorMap tmB_lo,
                   float* __restrict__ D, long long ldd, int M, int N, int K, int kb_per_chunk,
                   int chunks_per_small) {
  using C = Cfg<BN>;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t raw = smem_u32(smem_raw);
  const uint32_t base = (raw + 1023u) & ~1023u;
  const uint32_t bar_base = base + C::STAGES * C::STAGE_BYTES;
  // barriers: full[STAGES], empty[STAGES], bfull[2], bempty[2] (big accumulator), sfull[2], sempty[2] (small
  // accumulator); then the TMEM base address slot
  auto full_bar = [&](int s) { return bar_base + 8u * s; };
  auto empty_bar = [&](int s) { return bar_base + 8u * (C::STAGES + s); };
  auto bfull_bar = [&](int b) { return bar_base + 8u * (2 * C::STAGES + b); };
  auto bempty_bar = [&](int b) { return bar_base + 8u * (2 * C::STAGES + 2 + b); };
  auto sfull_bar = [&](int b) { return bar_base + 8u * (2 * C::STAGES + 4 + b); };
  auto sempty_bar = [&](int b) { return bar_base + 8u * (2 * C::STAGES + 6 + b); };
  const uint32_t tmem_slot = bar_base + 8u * (2 * C::STAGES + 8);
  volatile uint32_t* tmem_slot_ptr =
      reinterpret_cast<volatile uint32_t*>(smem_raw + (tmem_slot - raw));

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int m_tiles = (M + BM - 1) / BM, n_tiles = (N + BN - 1) / BN;
  const int num_tiles = m_tiles * n_tiles;
  const int num_kb = (K + BK - 1) / BK;
  const int num_chunks = (num_kb + kb_per_chunk - 1) / kb_per_chunk;

  if (warp == 0 && lane == 0) {
    prefetch_tmap(&tmA_hi); prefetch_tmap(&tmA_lo); prefetch_tmap(&tmB_hi); prefetch_tmap(&tmB_lo);
  }
  if (warp == 1 && lane == 0) {
    for (int s = 0; s < C::STAGES; ++s) { mbar_init(full_bar(s), 1); mbar_init(empty_bar(s), 1); }
    for (int b = 0; b < 2; ++b) {
      mbar_init(bfull_bar(b), 1); mbar_init(bempty_bar(b), C::EPI_WARPS);
      mbar_init(sfull_bar(b), 1); mbar_init(sempty_bar(b), C::EPI_WARPS);
    }
    fence_barrier_init();
  }
  if (warp == 2) {
    tmem_alloc(tmem_slot, C::TMEM_COLS);
    tmem_relinquish();
  }
  tcgen05_fence_before();
  __syncthreads();
  tcgen05_fence_after();
  const uint32_t tmem_base = *tmem_slot_ptr;
  // TMEM columns: big[b] at b*BN, small[b] at 2*BN + b*BN

  if (warp == 0) {
    // ===================== TMA producer =====================
    if (lane == 0) {
      int stage = 0; uint32_t parity = 0;
      for (int t = blockIdx.x; t < num_tiles; t += gridDim.x) {
        int mb, nb; tile_coords(t, m_tiles, n_tiles, mb, nb);
        const int m0 = mb * BM, n0 = nb * BN;
        for (int kb = 0; kb < num_kb; ++kb) {
          mbar_wait(empty_bar(stage), parity ^ 1u);
          const uint32_t sA_hi = base + stage * C::STAGE_BYTES;
          const uint32_t sA_lo = sA_hi + C::A_BYTES;
          const uint32_t sB_hi = sA_lo + C::A_BYTES;
          const uint32_t sB_lo = sB_hi + C::B_BYTES;
          mbar_expect_tx(full_bar(stage), C::STAGE_BYTES);
          tma_load_2d(sA_hi, &tmA_hi, kb * BK, m0, full_bar(stage));
          tma_load_2d(sA_lo, &tmA_lo, kb * BK, m0, full_bar(stage));
          tma_load_2d(sB_hi, &tmB_hi, kb * BK, n0, full_bar(stage));
          tma_load_2d(sB_lo, &tmB_lo, kb * BK, n0, full_bar(stage));
          if (++stage == C::STAGES) { stage = 0; parity ^= 1u; }
        }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer =====================
    // Two accumulators of different magnitude: "big" takes hi.hi (one MMA per k-step, drained to the CUDA-core
    // running sum every chunk), "small" takes lo.hi + hi.lo (2^-11 of big; drained every chunks_per_small chunks).
    // The tensor core's fp32 accumulation truncates, ~0.5 ulp of the accumulator per MMA: keeping the two apart
    // means big sees a third of the MMAs and small's truncation is 2^-11 smaller in absolute terms.
    if (lane == 0) {
      constexpr uint32_t idesc = make_idesc_tf32(BM, BN);
      int stage = 0; uint32_t parity = 0;
      uint32_t big_cnt = 0, small_cnt = 0;
      for (int t = blockIdx.x; t < num_tiles; t += gridDim.x) {
        uint32_t acc_small = 0;
        for (int c = 0; c < num_chunks; ++c) {
          const uint32_t bbuf = big_cnt & 1u, sbuf = small_cnt & 1u;
          mbar_wait(bempty_bar(bbuf), ((big_cnt >> 1) & 1u) ^ 1u);
          if (acc_small == 0) mbar_wait(sempty_bar(sbuf), ((small_cnt >> 1) & 1u) ^ 1u);
          tcgen05_fence_after();
          const uint32_t tmem_big = tmem_base + bbuf * BN;
          const uint32_t tmem_small = tmem_base + 2 * BN + sbuf * BN;
          const int kb_end = min(num_kb, (c + 1) * kb_per_chunk);
          uint32_t acc_big = 0;
          for (int kb = c * kb_per_chunk; kb < kb_end; ++kb) {
            mbar_wait(full_bar(stage), parity);
            tcgen05_fence_after();
            const uint32_t sA_hi = base + stage * C::STAGE_BYTES;
            const uint32_t sA_lo = sA_hi + C::A_BYTES;
            const uint32_t sB_hi = sA_lo + C::A_BYTES;
            const uint32_t sB_lo = sB_hi + C::B_BYTES;
#pragma unroll
            for (int k = 0; k < BK / UMMA_K; ++k) {
              const uint32_t koff = k * UMMA_K * 4;  // bytes inside the 128 B swizzle row
              const uint64_t dA_hi = make_kmajor_sw128_desc(sA_hi + koff);
              const uint64_t dA_lo = make_kmajor_sw128_desc(sA_lo + koff);
              const uint64_t dB_hi = make_kmajor_sw128_desc(sB_hi + koff);
              const uint64_t dB_lo = make_kmajor_sw128_desc(sB_lo + koff);
              umma_tf32(tmem_small, dA_lo, dB_hi, idesc, acc_small);
              umma_tf32(tmem_small, dA_hi, dB_lo, idesc, 1u);
              umma_tf32(tmem_big, dA_hi, dB_hi, idesc, acc_big);
              acc_small = 1u; acc_big = 1u;
            }
            umma_commit(empty_bar(stage));   // frees the smem stage once these MMAs have read it
            if (++stage == C::STAGES) { stage = 0; parity ^= 1u; }
          }
          umma_commit(bfull_bar(bbuf));      // big chunk complete
          ++big_cnt;
          if ((c + 1) % chunks_per_small == 0 || c == num_chunks - 1) {
            umma_commit(sfull_bar(sbuf));    // small accumulator complete
            ++small_cnt; acc_small = 0;
          }
        }
      }
    }
  } else if (warp >= 4) {
    // ===================== epilogue: TMEM -> fp32 running sum -> global =====================
    const int ew = warp - 4;
    const int quad = warp & 3;               // TMEM lane quadrant this warp may access
    const int chalf = ew >> 2;               // which half of the BN columns
    constexpr int EC = C::EPI_COLS;
    uint32_t big_cnt = 0, small_cnt = 0;
    for (int t = blockIdx.x; t < num_tiles; t += gridDim.x) {
      int mb, nb; tile_coords(t, m_tiles, n_tiles, mb, nb);
      float acc[EC];
#pragma unroll
      for (int i = 0; i < EC; ++i) acc[i] = 0.f;
      for (int c = 0; c < num_chunks; ++c) {
        {
          const uint32_t buf = big_cnt & 1u;
          mbar_wait(bfull_bar(buf), (big_cnt >> 1) & 1u);
          tcgen05_fence_after();
          const uint32_t taddr = tmem_base + ((uint32_t)(quad * 32) << 16) + buf * BN + chalf * EC;
          static_assert(EC == 64, "epilogue drains 64 columns per warp");
          uint32_t v[64];
          tmem_ld64(taddr, v);
          tmem_ld_wait();
#pragma unroll
          for (int i = 0; i < 64; ++i) acc[i] += __uint_as_float(v[i]);
          tcgen05_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(bempty_bar(buf));
          ++big_cnt;
        }
        if ((c + 1) % chunks_per_small == 0 || c == num_chunks - 1) {
          const uint32_t buf = small_cnt & 1u;
          mbar_wait(sfull_bar(buf), (small_cnt >> 1) & 1u);
          tcgen05_fence_after();
          const uint32_t taddr = tmem_base + ((uint32_t)(quad * 32) << 16) + 2 * BN + buf * BN + chalf * EC;
          static_assert(EC == 64, "epilogue drains 64 columns per warp");
          uint32_t v[64];
          tmem_ld64(taddr, v);
          tmem_ld_wait();
#pragma unroll
          for (int i = 0; i < 64; ++i) acc[i] += __uint_as_float(v[i]);
          tcgen05_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(sempty_bar(buf));
          ++small_cnt;
        }
      }
      const int row = mb * BM + quad * 32 + lane;
      const int col0 = nb * BN + chalf * EC;
      if (row < M) {
        float* drow = D + (long long)row * ldd + col0;
#pragma unroll
        for (int i = 0; i < EC; i += 4) {
          if (col0 + i + 3 < N) {
            *reinterpret_cast<float4*>(drow + i) = make_float4(acc[i], acc[i + 1], acc[i + 2], acc[i + 3]);
          } else {
#pragma unroll
            for (int e = 0; e < 4; ++e)
              if (col0 + i + e < N) drow[i + e] = acc[i + e];
          }
        }
      }
    }
  }

  tcgen05_fence_before();
  __syncthreads();
  if (warp == 2) {
    tcgen05_fence_after();
    tmem_dealloc(tmem_base, C::TMEM_COLS);
  }
}

// ---------------------------------------------------------------- host side
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*,
                                  CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                  CUtensorMapFloatOOBfill);

static EncodeTiledFn get_encode_fn() {
  static EncodeTiledFn fn = nullptr;
  if (fn) return fn;
  void* p = nullptr;
  cudaDriverEntryPointQueryResult q;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess ||
      q != cudaDriverEntryPointSuccess)
    return nullptr;
  fn = reinterpret_cast<EncodeTiledFn>(p);
  return fn;
}

// [rows, K] fp32 row-major, box = 32 (K) x box_rows, 128B swizzle, zero fill out of bounds.
static bool make_tmap(CUtensorMap* m, const float* ptr, int rows, int K, int box_rows) {
  EncodeTiledFn fn = get_encode_fn();
  if (!fn) return false;
  cuuint64_t dims[2] = {(cuuint64_t)K, (cuuint64_t)rows};
  cuuint64_t strides[1] = {(cuuint64_t)K * 4};
  cuuint32_t box[2] = {(cuuint32_t)BK, (cuuint32_t)box_rows};
  cuuint32_t estr[2] = {1, 1};
  CUresult r = fn(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<float*>(ptr), dims, strides, box, estr,
                  CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                  CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS;
}

template <int BN>
static int launch_bn(const float* A_hi, const float* A_lo, const float* Wt_hi, const float* Wt_lo, float* D,
                     long long ldd, int M, int N, int K, int k_drain, int num_sms, cudaStream_t s,
                     const char** err) {
  using C = Cfg<BN>;
  CUtensorMap ta, tb, tc_, td;
  if (!make_tmap(&ta, A_hi, M, K, BM) || !make_tmap(&tb, A_lo, M, K, BM) ||
      !make_tmap(&tc_, Wt_hi, N, K, BN) || !make_tmap(&td, Wt_lo, N, K, BN)) {
    if (err) *err = "cuTensorMapEncodeTiled failed";
    return -1;
  }
  static bool attr_set = false;
  if (!attr_set) {
    cudaError_t e = cudaFuncSetAttribute(gemm_tf32x3_kernel<BN>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         C::SMEM_BYTES);
    if (e != cudaSuccess) { if (err) *err = cudaGetErrorString(e); return -1; }
    attr_set = true;
  }
  int m_tiles = (M + BM - 1) / BM, n_tiles = (N + BN - 1) / BN;
  long long tiles = (long long)m_tiles * n_tiles;
  int grid = (int)(tiles < num_sms ? tiles : num_sms);
  if (k_drain <= 0) k_drain = 128;   // 16 hi.hi MMAs per TMEM chain: truncation bias ~4e-7 rel
  int kb_per_chunk = (k_drain + BK - 1) / BK;
  if (kb_per_chunk < 1) kb_per_chunk = 1;
  int chunks_per_small = 16384 / (kb_per_chunk * BK);   // small accumulator drained every 16384 elements of K
  if (chunks_per_small < 1) chunks_per_small = 1;
  gemm_tf32x3_kernel<BN><<<grid, C::THREADS, C::SMEM_BYTES, s>>>(ta, tb, tc_, td, D, ldd, M, N, K, kb_per_chunk,
                                                                 chunks_per_small);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) { if (err) *err = cudaGetErrorString(e); return -1; }
  return 0;
}

}  // namespace tc

int gemm_tc_supported(int M, int N, int K) {
  // TMA needs 16-byte row pitches (K % 4) and the epilogue stores float4 (N % 4).  M below one tile is fine (TMA
  // zero-fills the missing rows) and still beats the CUDA-core kernel; N < 128 or K < 32 is left to that kernel.
  return M >= 1 && N >= 128 && K >= 32 && (K % 4 == 0) && (N % 4 == 0);
}

int launch_gemm_tc(const float* A_hi, const float* A_lo, const float* Wt_hi, const float* Wt_lo, float* D,
                   long long ldd, int M, int N, int K, int k_drain, int num_sms, cudaStream_t s,
                   const char** err) {
  auto mis = [](const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15) != 0; };
  if (!gemm_tc_supported(M, N, K) || mis(A_hi) || mis(A_lo) || mis(Wt_hi) || mis(Wt_lo) || mis(D) ||
      (ldd % 4) != 0) {
    if (err) *err = "gemm_tc: unsupported shape or misaligned operand";
    return -1;
  }
  return tc::launch_bn<128>(A_hi, A_lo, Wt_hi, Wt_lo, D, ldd, M, N, K, k_drain, num_sms, s, err);
}

}  // namespace crownb200
