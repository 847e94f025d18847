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
#include "tc_common.cuh"

namespace crownb200 {

namespace tc {


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
  static constexpr int EPI_STAGE_BYTES = EPI_WARPS * 4096;   // one 32 x 32 fp32 slab per epilogue warp (TMA store)
  static constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + EPI_STAGE_BYTES + 1024 /*align slack*/ + 256 /*barriers*/;
};

template <int BN>
__global__ void __launch_bounds__(Cfg<BN>::THREADS, 1)
gemm_tf32x3_kernel(const __grid_constant__ CUtensorMap tmA_hi, const __grid_constant__ CUtensorMap tmA_lo,
                   const __grid_constant__ CUtensorMap tmB_hi, const __grid_constant__ CUtensorMap tmB_lo,
                   const __grid_constant__ CUtensorMap tmD, int M, int N, int K, int kb_per_chunk,
                   int chunks_per_small, int accumulate, const ConcArgs conc) {
  using C = Cfg<BN>;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t raw = smem_u32(smem_raw);
  const uint32_t base = (raw + 1023u) & ~1023u;
  const uint32_t epi_base = base + C::STAGES * C::STAGE_BYTES;           // 1024-aligned: swizzled store slabs
  const uint32_t bar_base = epi_base + C::EPI_STAGE_BYTES;
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
      if (conc.part != nullptr) {
        // a8 fused: this warp's 64 columns of row `row` against the box of the row's property; A_0 is never stored
        const int row = mb * BM + quad * 32 + lane;
        const int col0 = nb * BN + chalf * EC;
        if (row < M) {
          const int b = (row / conc.R) % conc.B;
          const float* xl = conc.x_lo + (long long)b * conc.ldx + conc.col_off + col0;
          const float* xh = conc.x_hi + (long long)b * conc.ldx + conc.col_off + col0;
          float dot = 0.f, ab = 0.f;
#pragma unroll
          for (int i = 0; i < EC; i += 4) {
            if (col0 + i < N) {                      // N % 4 == 0: whole float4 in range
              const float4 lo = __ldg(reinterpret_cast<const float4*>(xl + i));
              const float4 hi = __ldg(reinterpret_cast<const float4*>(xh + i));
              dot = fmaf(acc[i], 0.5f * (lo.x + hi.x), dot);     ab = fmaf(fabsf(acc[i]), 0.5f * (hi.x - lo.x), ab);
              dot = fmaf(acc[i + 1], 0.5f * (lo.y + hi.y), dot); ab = fmaf(fabsf(acc[i + 1]), 0.5f * (hi.y - lo.y), ab);
              dot = fmaf(acc[i + 2], 0.5f * (lo.z + hi.z), dot); ab = fmaf(fabsf(acc[i + 2]), 0.5f * (hi.z - lo.z), ab);
              dot = fmaf(acc[i + 3], 0.5f * (lo.w + hi.w), dot); ab = fmaf(fabsf(acc[i + 3]), 0.5f * (hi.w - lo.w), ab);
            }
          }
          float2* dst = reinterpret_cast<float2*>(conc.part) + (long long)row * conc.parts + (conc.piece0 + nb * 2 + chalf);
          *dst = make_float2(dot, ab);
        }
        continue;
      }
      // tile -> global through shared memory and the TMA: lane = row writes its 32 columns (128 B) of a slab in the
      // 128B-swizzled layout (conflict-free), one lane issues the bulk tensor store, which also clips the M / N edges
      const uint32_t slab = epi_base + (uint32_t)ew * 4096u + (uint32_t)lane * 128u;
      const uint32_t sw = (uint32_t)(lane & 7);
#pragma unroll
      for (int sl = 0; sl < EC / 32; ++sl) {
        if (lane == 0) bulk_wait_read0();          // the previous store has finished reading this warp's slab
        __syncwarp();
#pragma unroll
        for (int c = 0; c < 8; ++c) {
          const int i = sl * 32 + c * 4;
          asm volatile("st.shared.v4.f32 [%0], {%1,%2,%3,%4};"
                       :: "r"(slab + (((uint32_t)c ^ sw) << 4)), "f"(acc[i]), "f"(acc[i + 1]), "f"(acc[i + 2]), "f"(acc[i + 3]) : "memory");
        }
        fence_proxy_async();
        __syncwarp();
        if (lane == 0) {
          if (accumulate) tma_reduce_add_2d(&tmD, epi_base + (uint32_t)ew * 4096u, nb * BN + chalf * EC + sl * 32, mb * BM + quad * 32);
          else tma_store_2d(&tmD, epi_base + (uint32_t)ew * 4096u, nb * BN + chalf * EC + sl * 32, mb * BM + quad * 32);
          bulk_commit();
        }
      }
    }
    if (lane == 0) bulk_wait0();
  }

  tcgen05_fence_before();
  __syncthreads();
  if (warp == 2) {
    tcgen05_fence_after();
    tmem_dealloc(tmem_base, C::TMEM_COLS);
  }
}

// ---------------------------------------------------------------- host side
template <int BN>
static int launch_bn(const float* A_hi, const float* A_lo, const float* Wt_hi, const float* Wt_lo, float* D,
                     long long ldd, int M, int N, int K, int k_drain, int num_sms, cudaStream_t s,
                     const char** err, const ConcArgs* conc) {
  using C = Cfg<BN>;
  CUtensorMap tout;
  const bool fused_conc = conc && conc->part;
  // fused concretisation stores no D: the output map is a placeholder over the partial-sum buffer
  if (!(fused_conc ? make_tmap_out(&tout, conc->part, M, 4, 4) : make_tmap_out(&tout, D, M, N, ldd))) {
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
  // K panels.  One wave of 148 tiles shares ~8 m-blocks of A and ~19 n-blocks of W; streamed over the whole K their
  // hi/lo limbs are (8 + 19) * 128 rows * K * 8 B, which for K = 16384 is 450 MB: far beyond the 126 MB L2, and
  // measured (profiles/r1_gemm_tf32x3_cfg3.md) as DRAM traffic above the kernel's own request volume.  Cutting K
  // into panels whose per-wave working set fits L2 makes operand re-use independent of how far CTAs drift apart;
  // panels after the first add into D with the TMA's fp32 reduce-add (fixed order: deterministic).
  const long long share_blocks = (long long)(m_tiles < GROUP_M ? m_tiles : GROUP_M) +
                                 (long long)(n_tiles < 19 ? n_tiles : 19);
  const long long bytes_per_k = share_blocks * 128 * 8;
  int kp = K;
  if (bytes_per_k * K > (96LL << 20)) {
    kp = (int)((64LL << 20) / bytes_per_k) / 512 * 512;
    if (kp < 1024) kp = 1024;
  }
  if (fused_conc && kp != K) { if (err) *err = "gemm_tc: fused concretisation needs a single K panel"; return -1; }
  const ConcArgs cargs = fused_conc ? *conc : ConcArgs();
  for (int k0 = 0; k0 < K; k0 += kp) {
    const int kk = K - k0 < kp ? K - k0 : kp;
    CUtensorMap ta, tb, tc_, td;
    if (!make_tmap(&ta, A_hi + k0, M, kk, BM, K) || !make_tmap(&tb, A_lo + k0, M, kk, BM, K) ||
        !make_tmap(&tc_, Wt_hi + k0, N, kk, BN, K) || !make_tmap(&td, Wt_lo + k0, N, kk, BN, K)) {
      if (err) *err = "cuTensorMapEncodeTiled failed";
      return -1;
    }
    gemm_tf32x3_kernel<BN><<<grid, C::THREADS, C::SMEM_BYTES, s>>>(ta, tb, tc_, td, tout, M, N, kk, kb_per_chunk,
                                                                   chunks_per_small, k0 > 0 ? 1 : 0, cargs);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { if (err) *err = cudaGetErrorString(e); return -1; }
  }
  return 0;
}

}  // namespace tc

int gemm_tc_supported(int M, int N, int K) {
  // TMA needs 16-byte row pitches (K % 4) and the epilogue stores float4 (N % 4).  M below one tile is fine (TMA
  // zero-fills the missing rows) and still beats the CUDA-core kernel; N < 128 or K < 32 is left to that kernel.
  return M >= 1 && N >= 128 && K >= 32 && (K % 4 == 0) && (N % 4 == 0);
}

int gemm_tc_conc_parts(int N) { return 2 * ((N + 127) / 128); }

int gemm_tc_conc_supported(int M, int N, int K) {
  // single K panel (see launch_bn): the working-set rule only cuts K above ~3000 for >= 27 shared blocks
  return gemm_tc_supported(M, N, K) && K <= 2048;
}

int launch_gemm_tc(const float* A_hi, const float* A_lo, const float* Wt_hi, const float* Wt_lo, float* D,
                   long long ldd, int M, int N, int K, int k_drain, int num_sms, cudaStream_t s,
                   const char** err, const ConcArgs* conc) {
  auto mis = [](const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15) != 0; };
  const bool fc = conc && conc->part;
  if (!gemm_tc_supported(M, N, K) || mis(A_hi) || mis(A_lo) || mis(Wt_hi) || mis(Wt_lo) || (!fc && (mis(D) || (ldd % 4) != 0)) ||
      (fc && (mis(conc->x_lo) || mis(conc->x_hi) || mis(conc->part)))) {
    if (err) *err = "gemm_tc: unsupported shape or misaligned operand";
    return -1;
  }
  return tc::launch_bn<128>(A_hi, A_lo, Wt_hi, Wt_lo, D, ldd, M, N, K, k_drain, num_sms, s, err, conc);
}

}  // namespace crownb200
