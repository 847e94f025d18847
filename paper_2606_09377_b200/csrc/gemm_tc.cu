// a5 -- the A.W contraction of the CROWN backward recursion (A <- A.Lambda_i W_i)
// on the 5th-generation tensor cores, fp32-accurate via 3xTF32:
//     D = A_hi.W_hi + A_hi.W_lo + A_lo.W_hi          (a = a_hi + a_lo, both exactly TF32-representable)
// The dropped A_lo.W_lo term and the TF32 rounding of the lo parts are O(2^-22) relative per product.
// The epilogue optionally applies the NEXT step of the recursion, so that `A <- A.Lambda_i W_i` is one kernel:
//   a4 fused: relaxation of the product through the ReLU below (sign split, slopes, d += A-/+ . bU, d += Abar . b)
//             and the TF32 hi/lo split of Abar, which is written as the next contraction's operand;
//   a8 fused: concretisation of the product against the input box (the last contraction of a pass).
//
// Design (sm_100a), round 2: a CTA PAIR per output tile (tcgen05 cta_group::2).
//   * Round 1's 128x128 single-CTA tile moved 64 KB of operand limbs from L2 into shared memory per 768 tensor
//     cycles (83 B/cycle/SM); its three measured operating points (cfg2 165, cfg3 192, cfg4 153 useful TFLOP/s)
//     all sit at 10-12 TB/s of L2->SM traffic, the chip's L2 throughput.  A pair tile of
//     256 x BN (BN <= 256): each CTA stages ITS 128 rows of A and HALF of the W tile (BN/2 rows), one UMMA
//     256 x BN x 8 reads both halves, so the same 64 KB per stage feed twice the tensor work (32 flop/B).
//   * operands K-major in global memory: A_hi/A_lo [M,K], Wt_hi/Wt_lo [N,K] (weights transposed and split once at
//     crown_init); TMA (cp.async.bulk.tensor, 128B swizzle) stages 4 tiles per pipeline stage; both CTAs' loads
//     signal the LEADER CTA's full barrier; one thread of the leader issues tcgen05.mma.cta_group::2.kind::tf32 and
//     releases stages / publishes accumulators with multicast commits to both CTAs;
//   * warp roles per CTA: warp 0 TMA producer, warp 1 MMA issuer (leader CTA only), warp 2 TMEM allocator, warps 4-11
//     epilogue (two warps per TMEM lane quadrant, 128 columns each).  setmaxnreg moves registers from warps 0-3 to
//     the epilogue warps, which keep a 128-column fp32 running sum per thread;
//   * measured on B200 (round 1): the tensor core's fp32 accumulation truncates, ~0.5 ulp of the running sum per MMA,
//     so the error grows linearly with the length of an accumulation chain.  K is therefore cut into drain chunks of
//     k_drain elements (default 64 = 24 MMAs; 128 when K <= 256): each chunk is accumulated in TMEM (two 256-column buffers = all 512
//     columns), then added into the fp32 register running sum by the epilogue warps (round-to-nearest) while the
//     tensor core fills the other buffer;
//   * persistent grid (one CTA pair per TPC), static tile order grouped along M for L2 reuse of W; K is cut into
//     panels whose per-wave working set fits L2, later panels add into D with the TMA's fp32 reduce-add.
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include "common.cuh"
#include "kernels.h"
#include "tc_common.cuh"

namespace crownb200 {

namespace tc {

constexpr int PAIR_M = 2 * BM;                       // rows of a pair tile
constexpr int BN_MAX = 256;
constexpr int STAGES = 3;
constexpr int A_BYTES = BM * BK * 4;                 // 16 KB: one limb of this CTA's 128 rows
constexpr int B_BYTES = (BN_MAX / 2) * BK * 4;       // 16 KB: one limb of this CTA's half of the W tile
constexpr int STAGE_BYTES = 2 * A_BYTES + 2 * B_BYTES;
constexpr int EPI_WARPS = 8;                         // 4 lane quadrants x 2 column halves of 128
constexpr int EC = 128;                              // columns owned by one epilogue warp
constexpr int THREADS = 128 + EPI_WARPS * 32;
constexpr int TMEM_COLS = 512;                       // two accumulator buffers of 256 columns
constexpr int EPI_STAGE_BYTES = EPI_WARPS * 4096;    // one 32 x 32 fp32 slab per epilogue warp (TMA store)
constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + EPI_STAGE_BYTES + 1024 /*align slack*/ + 256 /*barriers*/;

enum { EPI_STORE = 0, EPI_ADD = 1, EPI_RELAX = 2, EPI_CONC = 3 };

// round-to-nearest (ties away) to TF32 on the bit pattern: the arithmetic of cvt.rna.tf32.f32 for finite inputs in
// two integer instructions (the PTX conversion compiles to a longer sequence that also handles NaN payloads)
__device__ __forceinline__ float tf32_rn_bits(float x) {
  return __uint_as_float((__float_as_uint(x) + 0x1000u) & 0xffffe000u);
}

// streaming 128-bit store under a predicate, without a branch around it (a branch per store keeps ptxas from moving the
// shared-memory reads of the following stores above it)
__device__ __forceinline__ void stg_stream4_if(bool on, float* p, const float4& v) {
  asm volatile("{\n\t.reg .pred q;\n\tsetp.ne.s32 q, %5, 0;\n\t@q st.global.L1::no_allocate.v4.f32 [%0], {%1,%2,%3,%4};\n\t}"
               :: "l"(p), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w), "r"((int)on) : "memory");
}

struct EpiArgs {
  int mode = EPI_STORE;
  int B = 0, R = 0;              // row m -> branch m / (B*R), property (m / R) % B
  int col_off = 0;               // first column of this launch inside the full row (N-slab of a streamed operand)
  int parts = 0;                 // 32-column pieces per full row
  float* part = nullptr;         // EPI_RELAX: [M, parts] floats; EPI_CONC: [M, parts] float2
  // EPI_RELAX
  const float4* coef = nullptr;  // [B, coef_ld] {dU, bU, dL, unstable}
  long long coef_ld = 0;
  const float* bias = nullptr;   // bias of the Linear below the ReLU, [coef_ld], or nullptr
  float* out_hi = nullptr; float* out_lo = nullptr; long long ldd = 0;   // limbs of the relaxed product (this launch's slab)
  // EPI_CONC
  const float* x_lo = nullptr; const float* x_hi = nullptr; int ldx = 0;
};

__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(THREADS, 1)
gemm2_tf32x3_kernel(const __grid_constant__ CUtensorMap tmA_hi, const __grid_constant__ CUtensorMap tmA_lo,
                    const __grid_constant__ CUtensorMap tmB_hi, const __grid_constant__ CUtensorMap tmB_lo,
                    const __grid_constant__ CUtensorMap tmD, const __grid_constant__ CUtensorMap tmD_lo,
                    int M, int N, int K, int BN, int kb_per_chunk, const EpiArgs ea) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t raw = smem_u32(smem_raw);
  const uint32_t base = (raw + 1023u) & ~1023u;
  const uint32_t epi_base = base + STAGES * STAGE_BYTES;           // 1024-aligned: swizzled store slabs
  const uint32_t bar_base = epi_base + EPI_STAGE_BYTES;
  // barriers (same offsets in both CTAs): full[STAGES] (leader's is used), empty[STAGES], accfull[2],
  // accempty[2] (leader's is used); then the TMEM base address slot
  auto full_bar = [&](int s) { return bar_base + 8u * s; };
  auto empty_bar = [&](int s) { return bar_base + 8u * (STAGES + s); };
  auto accfull_bar = [&](int b) { return bar_base + 8u * (2 * STAGES + b); };
  auto accempty_bar = [&](int b) { return bar_base + 8u * (2 * STAGES + 2 + b); };
  const uint32_t tmem_slot = bar_base + 8u * (2 * STAGES + 4);
  volatile uint32_t* tmem_slot_ptr = reinterpret_cast<volatile uint32_t*>(smem_raw + (tmem_slot - raw));

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = cluster_ctarank();             // 0 = leader
  const int cluster_id = blockIdx.x >> 1, num_clusters = gridDim.x >> 1;
  const int m_tiles = (M + PAIR_M - 1) / PAIR_M, n_tiles = (N + BN - 1) / BN;
  const int num_tiles = m_tiles * n_tiles;
  const int num_kb = (K + BK - 1) / BK;
  const int num_chunks = (num_kb + kb_per_chunk - 1) / kb_per_chunk;
  const int bh = BN >> 1;                              // rows of W this CTA stages

  if (warp == 0 && lane == 0) {
    prefetch_tmap(&tmA_hi); prefetch_tmap(&tmA_lo); prefetch_tmap(&tmB_hi); prefetch_tmap(&tmB_lo);
  }
  if (warp == 1 && lane == 0) {
    for (int s = 0; s < STAGES; ++s) { mbar_init(full_bar(s), 1); mbar_init(empty_bar(s), 1); }
    for (int b = 0; b < 2; ++b) { mbar_init(accfull_bar(b), 1); mbar_init(accempty_bar(b), 2 * EPI_WARPS); }
    fence_barrier_init();
  }
  if (warp == 2) {
    tmem_alloc_pair(tmem_slot, TMEM_COLS);
    tmem_relinquish_pair();
  }
  tcgen05_fence_before();
  __syncthreads();
  cluster_sync_all();          // both CTAs' barriers are initialised before any remote arrive / multicast commit
  tcgen05_fence_after();
  const uint32_t tmem_base = *tmem_slot_ptr;

  if (warp < 4) {
    setmaxnreg_dec<56>();
    if (warp == 0) {
      // ===================== TMA producer (both CTAs) =====================
      if (lane == 0) {
        int stage = 0; uint32_t parity = 0;
        const uint32_t stage_tx = 2u * (2u * A_BYTES + 2u * (uint32_t)bh * BK * 4u);   // both CTAs' bytes
        for (int t = cluster_id; t < num_tiles; t += num_clusters) {
          int mb, nb; tile_coords(t, m_tiles, n_tiles, mb, nb);
          const int m0 = mb * PAIR_M + (int)rank * BM, n0 = nb * BN + (int)rank * bh;
          for (int kb = 0; kb < num_kb; ++kb) {
            mbar_wait(empty_bar(stage), parity ^ 1u);
            const uint32_t sA_hi = base + stage * STAGE_BYTES;
            const uint32_t sA_lo = sA_hi + A_BYTES;
            const uint32_t sB_hi = sA_lo + A_BYTES;
            const uint32_t sB_lo = sB_hi + B_BYTES;
            const uint32_t fb = mapa_cluster(full_bar(stage), 0);
            if (rank == 0) mbar_expect_tx(full_bar(stage), stage_tx);
            tma_load_2d_pair(sA_hi, &tmA_hi, kb * BK, m0, fb);
            tma_load_2d_pair(sA_lo, &tmA_lo, kb * BK, m0, fb);
            tma_load_2d_pair(sB_hi, &tmB_hi, kb * BK, n0, fb);
            tma_load_2d_pair(sB_lo, &tmB_lo, kb * BK, n0, fb);
            if (++stage == STAGES) { stage = 0; parity ^= 1u; }
          }
        }
      }
    } else if (warp == 1 && rank == 0) {
      // ===================== MMA issuer (leader CTA) =====================
      if (lane == 0) {
        const uint32_t idesc = make_idesc_tf32(PAIR_M, BN);
        int stage = 0; uint32_t parity = 0;
        uint32_t cnt = 0;
        for (int t = cluster_id; t < num_tiles; t += num_clusters) {
          for (int c = 0; c < num_chunks; ++c) {
            const uint32_t buf = cnt & 1u;
            mbar_wait(accempty_bar(buf), ((cnt >> 1) & 1u) ^ 1u);
            tcgen05_fence_after();
            const uint32_t tmem_d = tmem_base + buf * BN_MAX;
            const int kb_end = min(num_kb, (c + 1) * kb_per_chunk);
            uint32_t acc = 0;
            for (int kb = c * kb_per_chunk; kb < kb_end; ++kb) {
              mbar_wait(full_bar(stage), parity);
              tcgen05_fence_after();
              const uint32_t sA_hi = base + stage * STAGE_BYTES;
              const uint32_t sA_lo = sA_hi + A_BYTES;
              const uint32_t sB_hi = sA_lo + A_BYTES;
              const uint32_t sB_lo = sB_hi + B_BYTES;
#pragma unroll
              for (int k = 0; k < BK / UMMA_K; ++k) {
                const uint32_t koff = k * UMMA_K * 4;  // bytes inside the 128 B swizzle row
                const uint64_t dA_hi = make_kmajor_sw128_desc(sA_hi + koff);
                const uint64_t dA_lo = make_kmajor_sw128_desc(sA_lo + koff);
                const uint64_t dB_hi = make_kmajor_sw128_desc(sB_hi + koff);
                const uint64_t dB_lo = make_kmajor_sw128_desc(sB_lo + koff);
                umma_tf32_pair(tmem_d, dA_lo, dB_hi, idesc, acc);      // the two small products first
                umma_tf32_pair(tmem_d, dA_hi, dB_lo, idesc, 1u);
                umma_tf32_pair(tmem_d, dA_hi, dB_hi, idesc, 1u);
                acc = 1u;
              }
              umma_commit_pair(empty_bar(stage), 3);   // frees the stage in both CTAs once these MMAs have read it
              if (++stage == STAGES) { stage = 0; parity ^= 1u; }
            }
            umma_commit_pair(accfull_bar(buf), 3);     // chunk complete: both CTAs' epilogues may drain
            ++cnt;
          }
        }
      }
    }
  } else {
    // ===================== epilogue: TMEM -> fp32 running sum -> fused step -> global =====================
    setmaxnreg_inc<224>();
    const int ew = warp - 4;
    const int quad = warp & 3;               // TMEM lane quadrant this warp may access
    const int chalf = ew >> 2;               // which 128 of the (up to) 256 tile columns
    const uint32_t accempty_remote[2] = {mapa_cluster(accempty_bar(0), 0), mapa_cluster(accempty_bar(1), 0)};
    const uint32_t slab_base = epi_base + (uint32_t)ew * 4096u;
    const uint32_t slab = slab_base + (uint32_t)lane * 128u;
    const uint32_t sw = (uint32_t)(lane & 7);
    const long long BR = (long long)ea.B * ea.R;
    uint32_t cnt = 0;
    for (int t = cluster_id; t < num_tiles; t += num_clusters) {
      int mb, nb; tile_coords(t, m_tiles, n_tiles, mb, nb);
      const int row = mb * PAIR_M + (int)rank * BM + quad * 32 + lane;       // this thread's output row
      const int row0 = mb * PAIR_M + (int)rank * BM + quad * 32;             // first row of the warp's slab
      const int tcol0 = nb * BN + chalf * EC;                                 // first column of the warp (in this launch)
      const bool rok = row < M;
      const int rr = rok ? row : 0;
      // EPI_RELAX: the warp's relaxation coefficients (lane = column) are requested before the tile's MMAs are waited
      // for, so their global-memory latency (4 dependent round trips per tile otherwise, 22 % of the epilogue's stall
      // samples in capture C of profiles/r2_gemm2.md) is hidden behind the drain.  The loaded values are kept raw; the
      // branch-dependent selection happens where they are used (a consumer placed here would wait for the loads here).
      float4 craw[EC / 32];
      float braw[EC / 32];
      if (ea.mode == EPI_RELAX) {
        const float4* crow = ea.coef + (long long)((rr / ea.R) % ea.B) * ea.coef_ld + ea.col_off;
#pragma unroll
        for (int sl = 0; sl < EC / 32; ++sl) {
          // columns past N take the last column's (finite) coefficients: their accumulators are exact zeros (the TMA
          // zero-fills the missing rows of W) and they are never stored, so d and the output do not see them; an
          // unconditional load leaves no select after it that would wait for the data here
          const int cc = min(tcol0 + sl * 32 + lane, N - 1);
          craw[sl] = __ldg(crow + cc);                                      // {dU, bU, dL, unstable}
          braw[sl] = 0.f;
          if (ea.bias) braw[sl] = __ldg(ea.bias + ea.col_off + cc);
        }
      }
      float acc[EC];
#pragma unroll
      for (int i = 0; i < EC; ++i) acc[i] = 0.f;
      for (int c = 0; c < num_chunks; ++c) {
        const uint32_t buf = cnt & 1u;
        mbar_wait(accfull_bar(buf), (cnt >> 1) & 1u);
        tcgen05_fence_after();
        const uint32_t taddr = tmem_base + ((uint32_t)(quad * 32) << 16) + buf * BN_MAX + chalf * EC;
#pragma unroll
        for (int h = 0; h < EC / 32; ++h) {
          if (chalf * EC + h * 32 < BN) {      // warp-uniform
            uint32_t v[32];
            tmem_ld32(taddr + h * 32, v);
            tmem_ld_wait();
#pragma unroll
            for (int i = 0; i < 32; ++i) acc[h * 32 + i] += __uint_as_float(v[i]);
          }
        }
        tcgen05_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive_cluster_relaxed(accempty_remote[buf]);
        ++cnt;
      }
      // do the warp's 32 rows share (branch, property)?  Always for identity passes with R % 32 == 0 (the hot case).
      const bool uni = (ea.R & 31) == 0;

      if (ea.mode == EPI_CONC) {
        // a8 fused: 32-column pieces of this row against the box of the row's property; A_0 is never stored
        const int b = (rr / ea.R) % ea.B;
        const float* xl = ea.x_lo + (long long)b * ea.ldx + ea.col_off;
        const float* xh = ea.x_hi + (long long)b * ea.ldx + ea.col_off;
        float2* prow = reinterpret_cast<float2*>(ea.part) + (long long)rr * ea.parts + (ea.col_off >> 5);
#pragma unroll
        for (int sl = 0; sl < EC / 32; ++sl) {
          const int col = tcol0 + sl * 32;
          if (chalf * EC + sl * 32 >= BN || col >= N) continue;            // warp-uniform
          float dot = 0.f, ab = 0.f;
          if (uni) {
            // box centre / radius of the 32 columns: loaded once per warp (lane = column), read back as broadcasts
            float2 cr = make_float2(0.f, 0.f);
            if (col + lane < N) { const float l = __ldg(xl + col + lane), h = __ldg(xh + col + lane); cr = make_float2(0.5f * (l + h), 0.5f * (h - l)); }
            __syncwarp();
            asm volatile("st.shared.v2.f32 [%0], {%1,%2};" :: "r"(slab_base + (uint32_t)lane * 8u), "f"(cr.x), "f"(cr.y) : "memory");
            __syncwarp();
#pragma unroll
            for (int i = 0; i < 32; ++i) {
              float2 c;
              asm volatile("ld.shared.v2.f32 {%0,%1}, [%2];" : "=f"(c.x), "=f"(c.y) : "r"(slab_base + (uint32_t)i * 8u));
              const float a = acc[sl * 32 + i];
              dot = fmaf(a, c.x, dot); ab = fmaf(fabsf(a), c.y, ab);
            }
          } else {
#pragma unroll
            for (int i = 0; i < 32; i += 4) {
              if (col + i < N) {                     // N % 4 == 0: whole float4 in range
                const float4 lo = __ldg(reinterpret_cast<const float4*>(xl + col + i));
                const float4 hi = __ldg(reinterpret_cast<const float4*>(xh + col + i));
                const float a0 = acc[sl * 32 + i], a1 = acc[sl * 32 + i + 1], a2 = acc[sl * 32 + i + 2], a3 = acc[sl * 32 + i + 3];
                dot = fmaf(a0, 0.5f * (lo.x + hi.x), dot); ab = fmaf(fabsf(a0), 0.5f * (hi.x - lo.x), ab);
                dot = fmaf(a1, 0.5f * (lo.y + hi.y), dot); ab = fmaf(fabsf(a1), 0.5f * (hi.y - lo.y), ab);
                dot = fmaf(a2, 0.5f * (lo.z + hi.z), dot); ab = fmaf(fabsf(a2), 0.5f * (hi.z - lo.z), ab);
                dot = fmaf(a3, 0.5f * (lo.w + hi.w), dot); ab = fmaf(fabsf(a3), 0.5f * (hi.w - lo.w), ab);
              }
            }
          }
          if (rok) prow[col >> 5] = make_float2(dot, ab);
        }
        continue;
      }

      if (ea.mode == EPI_RELAX) {
        // a4 fused: lower: Abar = A+ dL + A- dU, d += A- . bU; upper: Abar = A+ dU + A- dL,
        // d += A+ . bU; both: d += Abar . b.  One fp32 partial per (row, 32-column piece), summed in index order later.
        // Host side guarantees R % 32 == 0: the warp's 32 rows share (branch, property).  The warp's 4 KB slab is used
        // three times in turn: (1) the 32 columns' {slope for a > 0, slope for a <= 0, bU, bias}, loaded once per warp
        // (lane = column) and read back as broadcasts; (2) the hi limbs and (3) the lo limbs, written row-per-lane
        // (swizzled, conflict-free) and read back four rows per warp instruction, so the global stores are full
        // 128-byte row segments.
        // The slab loop is NOT unrolled: fully unrolled the fused epilogue is 55 KB of straight-line code that eight warps
        // walk through at eight different places (24 % of its stall samples were instruction-fetch stalls, one every 48
        // instructions, capture C of profiles/r2_gemm2.md).  The body always works on acc[0..31] / craw[0]; the registers
        // of the remaining slabs are moved down by one slab after each iteration.
        const bool upper = rr >= BR;
#pragma unroll 1
        for (int sl = 0; sl < EC / 32; ++sl) {
          const int col = tcol0 + sl * 32;
          if (chalf * EC + sl * 32 >= BN || col >= N) break;               // warp-uniform; later slabs are further out
          // {slope for a > 0, slope for a <= 0, bU, bias}
          const float4 cf = make_float4(upper ? craw[0].x : craw[0].z, upper ? craw[0].z : craw[0].x, craw[0].y, braw[0]);
          __syncwarp();
          asm volatile("st.shared.v4.f32 [%0], {%1,%2,%3,%4};"
                       :: "r"(slab_base + (uint32_t)lane * 16u), "f"(cf.x), "f"(cf.y), "f"(cf.z), "f"(cf.w) : "memory");
          __syncwarp();
          float hi[32], dsum = 0.f;
#pragma unroll
          for (int i = 0; i < 32; ++i) {
            float4 c;
            asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(c.x), "=f"(c.y), "=f"(c.z), "=f"(c.w) : "r"(slab_base + (uint32_t)i * 16u));
            const float a = acc[i];
            const float o = a * (a > 0.f ? c.x : c.y);     // == A+ s_pos + A- s_neg (one of the two terms is +-0)
            dsum = fmaf(upper ? fmaxf(a, 0.f) : fminf(a, 0.f), c.z, dsum);
            dsum = fmaf(o, c.w, dsum);
            hi[i] = tf32_rn_bits(o);
            acc[i] = tf32_rn_bits(o - hi[i]);    // lo limb, kept in the accumulator registers
          }
          if (rok) ea.part[(long long)row * ea.parts + ((ea.col_off + col) >> 5)] = dsum;
#pragma unroll
          for (int limb = 0; limb < 2; ++limb) {
            __syncwarp();                                   // the slab's previous contents have been read by every lane
#pragma unroll
            for (int c4 = 0; c4 < 8; ++c4) {
              const int i = c4 * 4;
              if (limb == 0)
                asm volatile("st.shared.v4.f32 [%0], {%1,%2,%3,%4};"
                             :: "r"(slab + (((uint32_t)c4 ^ sw) << 4)), "f"(hi[c4 * 4]), "f"(hi[c4 * 4 + 1]), "f"(hi[c4 * 4 + 2]), "f"(hi[c4 * 4 + 3]) : "memory");
              else
                asm volatile("st.shared.v4.f32 [%0], {%1,%2,%3,%4};"
                             :: "r"(slab + (((uint32_t)c4 ^ sw) << 4)), "f"(acc[i]), "f"(acc[i + 1]), "f"(acc[i + 2]), "f"(acc[i + 3]) : "memory");
            }
            __syncwarp();
            const int c4 = lane & 7, r0 = lane >> 3;
            // one pointer per lane, advanced by four rows per store (no per-store 64-bit index arithmetic)
            float* outp = (limb == 0 ? ea.out_hi : ea.out_lo) + (long long)(row0 + r0) * ea.ldd + col + c4 * 4;
            const long long step = 4 * ea.ldd;
            const int rows_left = col + c4 * 4 < N ? M - row0 - r0 : 0;     // store row r0 + 4 it while 4 it < rows_left
            // four shared-memory reads, then their four stores, twice (paired up one by one, every store would wait for
            // its own read's latency; eight at once do not fit the register budget next to the 128 accumulators)
#pragma unroll
            for (int half = 0; half < 2; ++half) {
              float4 v[4];
#pragma unroll
              for (int q = 0; q < 4; ++q) {
                const int r = (half * 4 + q) * 4 + r0;
                asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v[q].x), "=f"(v[q].y), "=f"(v[q].z), "=f"(v[q].w)
                             : "r"(slab_base + (uint32_t)r * 128u + (((uint32_t)c4 ^ (uint32_t)(r & 7)) << 4)));
              }
#pragma unroll
              for (int q = 0; q < 4; ++q) {
                stg_stream4_if((half * 4 + q) * 4 < rows_left, outp, v[q]);
                outp += step;
              }
            }
          }
          if (sl + 1 < EC / 32) {
#pragma unroll
            for (int i = 0; i < EC - 32; ++i) acc[i] = acc[i + 32];
#pragma unroll
            for (int q = 0; q + 1 < EC / 32; ++q) { craw[q] = craw[q + 1]; braw[q] = braw[q + 1]; }
          }
        }
        continue;
      }

      if (ea.mode == EPI_STORE) {
        // product -> global: row-per-lane into the swizzled slab, read back four rows per warp instruction, stored as
        // full 128-byte row segments (no asynchronous store to wait for: short-K tiles stay MMA-bound)
#pragma unroll
        for (int sl = 0; sl < EC / 32; ++sl) {
          const int col = tcol0 + sl * 32;
          if (chalf * EC + sl * 32 >= BN || col >= N) continue;            // warp-uniform
          __syncwarp();
#pragma unroll
          for (int c4 = 0; c4 < 8; ++c4) {
            const int i = sl * 32 + c4 * 4;
            asm volatile("st.shared.v4.f32 [%0], {%1,%2,%3,%4};"
                         :: "r"(slab + (((uint32_t)c4 ^ sw) << 4)), "f"(acc[i]), "f"(acc[i + 1]), "f"(acc[i + 2]), "f"(acc[i + 3]) : "memory");
          }
          __syncwarp();
          // as in the fused epilogue: one pointer per lane, four reads then their four predicated stores, twice
          const int c4 = lane & 7, r0 = lane >> 3;
          float* outp = ea.out_hi + (long long)(row0 + r0) * ea.ldd + col + c4 * 4;
          const long long step = 4 * ea.ldd;
          const int rows_left = col + c4 * 4 < N ? M - row0 - r0 : 0;
#pragma unroll
          for (int half = 0; half < 2; ++half) {
            float4 v[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) {
              const int r = (half * 4 + q) * 4 + r0;
              asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v[q].x), "=f"(v[q].y), "=f"(v[q].z), "=f"(v[q].w)
                           : "r"(slab_base + (uint32_t)r * 128u + (((uint32_t)c4 ^ (uint32_t)(r & 7)) << 4)));
            }
#pragma unroll
            for (int q = 0; q < 4; ++q) {
              stg_stream4_if((half * 4 + q) * 4 < rows_left, outp, v[q]);
              outp += step;
            }
          }
        }
        continue;
      }

      // EPI_ADD (K panels after the first): D += tile through shared memory and the TMA's fp32 reduce-add; lane = row
      // writes its 32 columns of a slab in the 128B-swizzled layout, one lane issues the bulk tensor reduction, which
      // also clips the M / N edges
#pragma unroll
      for (int sl = 0; sl < EC / 32; ++sl) {
        const int col = tcol0 + sl * 32;
        if (chalf * EC + sl * 32 >= BN || col >= N) continue;              // warp-uniform
        if (lane == 0) bulk_wait_read0();          // the previous reduction has finished reading this warp's slab
        __syncwarp();
#pragma unroll
        for (int c4 = 0; c4 < 8; ++c4) {
          const int i = sl * 32 + c4 * 4;
          asm volatile("st.shared.v4.f32 [%0], {%1,%2,%3,%4};"
                       :: "r"(slab + (((uint32_t)c4 ^ sw) << 4)), "f"(acc[i]), "f"(acc[i + 1]), "f"(acc[i + 2]), "f"(acc[i + 3]) : "memory");
        }
        fence_proxy_async();
        __syncwarp();
        if (lane == 0) { tma_reduce_add_2d(&tmD, slab_base, col, row0); bulk_commit(); }
      }
    }
    if (lane == 0) bulk_wait0();
  }

  tcgen05_fence_before();
  __syncthreads();
  cluster_sync_all();          // the peer may still multicast into / arrive on this CTA's barriers until here
  if (warp == 2) {
    tcgen05_fence_after();
    tmem_dealloc_pair(tmem_base, TMEM_COLS);
  }
}

// ---------------------------------------------------------------- host side
static int g_max_clusters = 0;     // per process AND device-independent upper bound is not assumed: see gemm_tc_init_device

static int launch_pair(const float* A_hi, const float* A_lo, const float* Wt_hi, const float* Wt_lo, float* D, float* D_lo,
                       long long ldd, int M, int N, int K, int k_drain, int num_sms, cudaStream_t s,
                       const char** err, const EpiArgs& epi_in) {
  EpiArgs epi = epi_in;
  // tile width: the fewest 256-wide column blocks, evened out to a multiple of 32 (784 -> 4 x 224, not 3 x 256 + 16)
  const int n_blocks = (N + BN_MAX - 1) / BN_MAX;
  int BN = ((N + n_blocks - 1) / n_blocks + 31) / 32 * 32;
  if (BN > BN_MAX) BN = BN_MAX;
  if (BN < 32) BN = 32;
  int clusters = num_sms / 2;
  if (g_max_clusters > 0 && clusters > g_max_clusters) clusters = g_max_clusters;
  const int m_tiles = (M + PAIR_M - 1) / PAIR_M;
  // small problems (cfg1: M = 512, latency-bound): narrower tiles put more CTA pairs to work and shorten the
  // per-tile MMA chain; the per-element summation order does not depend on BN
  while (BN > 32 && (long long)m_tiles * ((N + BN - 1) / BN) * 2 <= clusters) BN = (BN / 2 + 31) / 32 * 32;
  const int n_tiles = (N + BN - 1) / BN;
  const long long tiles = (long long)m_tiles * n_tiles;
  if (tiles < clusters) clusters = (int)tiles;
  if (clusters < 1) clusters = 1;
  // 24 MMAs per TMEM chain: truncation bias <= ~7e-7 of the chunk's magnitude.  Short contractions (K <= 256,
  // the MNIST-FC-sized layers) take two chunks of 128 instead: the whole tile then fits the two TMEM buffers, so the NEXT
  // tile's MMAs run during this tile's epilogue instead of stalling after two of four chunks -- the fused-relaxation
  // epilogue is what paces these launches (cfg2: 2.68 -> 2.28 ms/step); the total bias stays at the level of an fp32 FFMA
  // loop over K = 256 (~1e-6 relative, two chains of 48 MMAs)
  if (k_drain <= 0) k_drain = (K <= 256) ? 128 : 64;
  int kb_per_chunk = (k_drain + BK - 1) / BK;
  if (kb_per_chunk < 1) kb_per_chunk = 1;
  // K panels.  One wave of 74 pair tiles shares ~8 m-blocks of A and ~10 n-blocks of W; streamed over the whole K their
  // hi/lo limbs are 18 * 256 rows * K * 8 B, far beyond the 126 MB L2 for K = 16384 (measured in round 1 as DRAM traffic
  // above the kernel's own request volume, profiles/r1_gemm_tf32x3_cfg3.md).  Cutting K into panels whose per-wave
  // working set fits L2 makes operand re-use independent of how far CTAs drift apart; panels after the first add
  // into D with the TMA's fp32 reduce-add (fixed order: deterministic).  The panel length depends on K only (not on
  // M or N), so row-chunked and N-slabbed (streamed) runs sum in the same order: bitwise equal results.
  const long long bytes_per_k = 18LL * 256 * 8;
  int kp = K;
  if (bytes_per_k * K > (96LL << 20)) {
    kp = (int)((64LL << 20) / bytes_per_k) / 512 * 512;
    if (kp < 1024) kp = 1024;
  }
  if (epi.mode != EPI_STORE && kp != K) { if (err) *err = "gemm_tc: fused epilogues need a single K panel"; return -1; }
  CUtensorMap tout, tout_lo;
  bool ok = true;
  if (epi.mode == EPI_CONC) {
    // no D is stored: the output maps are placeholders over the partial-sum buffer
    ok = make_tmap_out(&tout, epi.part, M, 4, 4) && make_tmap_out(&tout_lo, epi.part, M, 4, 4);
  } else if (epi.mode == EPI_RELAX) {
    epi.out_hi = D; epi.out_lo = D_lo; epi.ldd = ldd;       // written with plain coalesced stores, no output maps
    ok = make_tmap_out(&tout, epi.part, M, 4, 4) && make_tmap_out(&tout_lo, epi.part, M, 4, 4);
  } else {
    epi.out_hi = D; epi.ldd = ldd;                          // first panel: plain coalesced stores; later panels: TMA reduce-add
    ok = make_tmap_out(&tout, D, M, N, ldd) && make_tmap_out(&tout_lo, D, M, N, ldd);
  }
  if (!ok) { if (err) *err = "cuTensorMapEncodeTiled failed"; return -1; }
  for (int k0 = 0; k0 < K; k0 += kp) {
    const int kk = K - k0 < kp ? K - k0 : kp;
    CUtensorMap ta, tb, tc_, td;
    if (!make_tmap(&ta, A_hi + k0, M, kk, BM, K) || !make_tmap(&tb, A_lo + k0, M, kk, BM, K) ||
        !make_tmap(&tc_, Wt_hi + k0, N, kk, BN / 2, K) || !make_tmap(&td, Wt_lo + k0, N, kk, BN / 2, K)) {
      if (err) *err = "cuTensorMapEncodeTiled failed";
      return -1;
    }
    if (epi.mode == EPI_STORE || epi.mode == EPI_ADD) epi.mode = k0 > 0 ? EPI_ADD : EPI_STORE;
    gemm2_tf32x3_kernel<<<2 * clusters, THREADS, SMEM_BYTES, s>>>(ta, tb, tc_, td, tout, tout_lo, M, N, kk, BN, kb_per_chunk, epi);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { if (err) *err = cudaGetErrorString(e); return -1; }
  }
  return 0;
}

}  // namespace tc

int gemm_tc_init_device() {
  if (cudaFuncSetAttribute(tc::gemm2_tf32x3_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, tc::SMEM_BYTES) != cudaSuccess)
    return -1;
  // how many CTA pairs can be resident at once (one per TPC when every SM is available)
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(2, 1, 1); cfg.blockDim = dim3(tc::THREADS, 1, 1); cfg.dynamicSmemBytes = tc::SMEM_BYTES;
  cudaLaunchAttribute at; at.id = cudaLaunchAttributeClusterDimension; at.val.clusterDim.x = 2; at.val.clusterDim.y = 1; at.val.clusterDim.z = 1;
  cfg.attrs = &at; cfg.numAttrs = 1;
  int n = 0;
  if (cudaOccupancyMaxActiveClusters(&n, tc::gemm2_tf32x3_kernel, &cfg) == cudaSuccess && n > 0) tc::g_max_clusters = n;
  else (void)cudaGetLastError();
  return 0;
}

int gemm_tc_supported(int M, int N, int K) {
  // TMA needs 16-byte row pitches (K % 4) and the epilogue handles columns in float4 groups (N % 4).  M below one tile
  // is fine (TMA zero-fills the missing rows) and still beats the CUDA-core kernel; N < 128 or K < 32 is left to that kernel.
  return M >= 1 && N >= 128 && K >= 32 && (K % 4 == 0) && (N % 4 == 0);
}

int gemm_tc_parts(int N_total) { return (N_total + 31) / 32; }

int gemm_tc_single_panel(int K) { return 18LL * 256 * 8 * K <= (96LL << 20); }

int gemm_tc_num_panels(int K) {     // kernel launches of one contraction (same rule as launch_pair)
  if (gemm_tc_single_panel(K)) return 1;
  int kp = (int)((64LL << 20) / (18LL * 256 * 8)) / 512 * 512;
  if (kp < 1024) kp = 1024;
  return (K + kp - 1) / kp;
}

static bool mis16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15) != 0; }

int launch_gemm_tc(const float* A_hi, const float* A_lo, const float* Wt_hi, const float* Wt_lo, float* D,
                   long long ldd, int M, int N, int K, int k_drain, int num_sms, cudaStream_t s,
                   const char** err, const ConcArgs* conc, const RelaxEpiArgs* rel) {
  const bool fc = conc && conc->part;
  const bool fr = rel && rel->part;
  if (!gemm_tc_supported(M, N, K) || mis16(A_hi) || mis16(A_lo) || mis16(Wt_hi) || mis16(Wt_lo) ||
      (!fc && (mis16(D) || (ldd % 4) != 0)) || (fc && fr) ||
      (fc && (mis16(conc->x_lo) || mis16(conc->x_hi) || mis16(conc->part) || (conc->col_off % 32) != 0)) ||
      (fr && (mis16(rel->out_lo) || mis16(rel->coef) || (rel->col_off % 32) != 0))) {
    if (err) *err = "gemm_tc: unsupported shape or misaligned operand";
    return -1;
  }
  tc::EpiArgs e;
  float* D_lo = nullptr;
  if (fc) {
    e.mode = tc::EPI_CONC; e.B = conc->B; e.R = conc->R; e.col_off = conc->col_off; e.parts = conc->parts;
    e.part = conc->part; e.x_lo = conc->x_lo; e.x_hi = conc->x_hi; e.ldx = conc->ldx;
  } else if (fr) {
    e.mode = tc::EPI_RELAX; e.B = rel->B; e.R = rel->R; e.col_off = rel->col_off; e.parts = rel->parts;
    e.part = rel->part; e.coef = rel->coef; e.coef_ld = rel->coef_ld; e.bias = rel->bias;
    D_lo = rel->out_lo;
  } else {
    e.mode = tc::EPI_STORE; e.B = 1; e.R = M > 0 ? M : 1;
  }
  return tc::launch_pair(A_hi, A_lo, Wt_hi, Wt_lo, D, D_lo, ldd, M, N, K, k_drain, num_sms, s, err, e);
}

}  // namespace crownb200
