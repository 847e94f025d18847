// a4 + a5 fused -- ReLU relaxation of A, both bias accumulations and the A.W contraction
// (A <- A.Lambda_i W_i) in ONE kernel.  The relaxed matrix Abar and its TF32 hi/lo limbs
// never exist in HBM: per layer step the kernel reads A (fp32) once and writes the product once.
//
// Same tcgen05/TMEM/TMA pipeline as gemm_tc.cu (3xTF32, split big/small accumulators, K drain chunks) plus a
// TRANSFORM warpgroup between TMA and the MMA issuer:
//   TMA      : raw fp32 A tile [128 x 32] + prepacked W tiles (hi, lo) -> shared memory stage, 128B swizzle
//   transform: thread t owns row t of the tile: reads its 128 bytes, applies the relaxation of its branch
//              (lower: a>0 ? a*dL : a*dU, upper: a>0 ? a*dU : a*dL), accumulates d += A-/+ . bU and
//              d += Abar . b in registers over the whole K loop, splits Abar into TF32 hi (written in place)
//              and lo (second tile), in the swizzled layout the UMMA descriptors expect;
//              fence.proxy.async + mbarrier hand the stage to the MMA issuer
//   MMA      : lo.hi + hi.lo -> small accumulator, hi.hi -> big accumulator (TMEM)
//   epilogue : TMEM -> fp32 running sum -> global, as in gemm_tc.cu
// Row addressing is grouped: GEMM row m = g*Rg + r, g = br*B + b; the source tile of (g, r0) starts at source row
// base(g) + r0, which lets the first step of a pass read rows of W_k in place (shared by all properties and both
// branches) with no identity matrix and no broadcast copy.
#include "common.cuh"
#include "kernels.h"
#include "tc_common.cuh"

namespace crownb200 {
namespace tcf {

using namespace tc;

constexpr int BN = 128;
constexpr int STAGES = 3;
constexpr int A_BYTES = BM * BK * 4;
constexpr int B_BYTES = BN * BK * 4;
constexpr int COEF_OFF = 2 * A_BYTES + 2 * B_BYTES;      // per stage: 4 x 128 B {dU, bU, dL, bias} of the k-block
constexpr int STAGE_BYTES = COEF_OFF + 1024;             // raw/hi A, lo A, W hi, W lo, coefficients (1 KB keeps alignment)
constexpr int EPI_WARPS = 8;
constexpr int XF_WARPS = 8;            // two threads per tile row, 16 of the 32 k-elements each
constexpr int THREADS = 128 + EPI_WARPS * 32 + XF_WARPS * 32;
constexpr int TMEM_COLS = 4 * BN;
constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + 1024 + 256 + 2 * BM * 4;   // + d exchange slots

struct Params {
  float* D; long long ldd;
  int M, N, K;
  int n_groups, Rg, tiles_per_group;   // row groups (flat mode: 1 group of M rows)
  long long base_br, base_b;           // source row of group g = (g / B) * base_br + (g % B) * base_b
  int B, R;                            // m -> (br, b, r) for the coefficient lookup
  const float* planes;                 // relaxation coefficients {dU, bU, dL} as planes [3][plane_stride], row b at
  long long plane_stride;              //   b*K; nullptr = split only
  const float* bias;                   // [K] or nullptr
  float* d;                            // [2, B, R] in/out or nullptr
  int kb_per_chunk, chunks_per_small;
};

// 1-D bulk copy global -> shared, completion counted on an mbarrier (bytes % 16 == 0, 16-byte aligned addresses)
__device__ __forceinline__ void bulk_load(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               :: "r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ float4 lds128(uint32_t addr) {
  float4 v;
  asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
  return v;
}
__device__ __forceinline__ void sts128(uint32_t addr, const float4& v) {
  asm volatile("st.shared.v4.f32 [%0], {%1,%2,%3,%4};" :: "r"(addr), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}

template <bool RELAX>
__global__ void __launch_bounds__(THREADS, 1)
gemm_fused_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB_hi,
                  const __grid_constant__ CUtensorMap tmB_lo, const Params p) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t raw = smem_u32(smem_raw);
  const uint32_t base = (raw + 1023u) & ~1023u;
  const uint32_t bar_base = base + STAGES * STAGE_BYTES;
  auto full_bar = [&](int s) { return bar_base + 8u * s; };                    // TMA landed
  auto empty_bar = [&](int s) { return bar_base + 8u * (STAGES + s); };        // MMAs have read the stage
  auto ready_bar = [&](int s) { return bar_base + 8u * (2 * STAGES + s); };    // transform done
  auto bfull_bar = [&](int b) { return bar_base + 8u * (3 * STAGES + b); };
  auto bempty_bar = [&](int b) { return bar_base + 8u * (3 * STAGES + 2 + b); };
  auto sfull_bar = [&](int b) { return bar_base + 8u * (3 * STAGES + 4 + b); };
  auto sempty_bar = [&](int b) { return bar_base + 8u * (3 * STAGES + 6 + b); };
  const uint32_t tmem_slot = bar_base + 8u * (3 * STAGES + 8);
  volatile uint32_t* tmem_slot_ptr = reinterpret_cast<volatile uint32_t*>(smem_raw + (tmem_slot - raw));

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int m_tiles = p.n_groups * p.tiles_per_group, n_tiles = (p.N + BN - 1) / BN;
  const int num_tiles = m_tiles * n_tiles;
  const int num_kb = (p.K + BK - 1) / BK;
  const int num_chunks = (num_kb + p.kb_per_chunk - 1) / p.kb_per_chunk;

  if (warp == 0 && lane == 0) { prefetch_tmap(&tmA); prefetch_tmap(&tmB_hi); prefetch_tmap(&tmB_lo); }
  if (warp == 1 && lane == 0) {
    for (int s = 0; s < STAGES; ++s) { mbar_init(full_bar(s), 1); mbar_init(empty_bar(s), 1); mbar_init(ready_bar(s), XF_WARPS * 32); }
    for (int b = 0; b < 2; ++b) {
      mbar_init(bfull_bar(b), 1); mbar_init(bempty_bar(b), EPI_WARPS);
      mbar_init(sfull_bar(b), 1); mbar_init(sempty_bar(b), EPI_WARPS);
    }
    fence_barrier_init();
  }
  if (warp == 2) { tmem_alloc(tmem_slot, TMEM_COLS); tmem_relinquish(); }
  tcgen05_fence_before();
  __syncthreads();
  tcgen05_fence_after();
  const uint32_t tmem_base = *tmem_slot_ptr;

  // tile -> (group, first row in group, source row, n block)
  auto tile_info = [&](int t, int& g, int& r0, int& nb) {
    int mb; tile_coords(t, m_tiles, n_tiles, mb, nb);
    g = mb / p.tiles_per_group;
    r0 = (mb - g * p.tiles_per_group) * BM;
  };

  if (warp == 0) {
    // ===================== TMA producer =====================
    if (lane == 0) {
      int stage = 0; uint32_t parity = 0;
      for (int t = blockIdx.x; t < num_tiles; t += gridDim.x) {
        int g, r0, nb; tile_info(t, g, r0, nb);
        const int src_row = (int)((g / p.B) * p.base_br + (g % p.B) * p.base_b) + r0;
        const int n0 = nb * BN;
        const int b = (int)((((long long)g * p.Rg + r0) / p.R) % p.B);   // the tile's rows share one property
        for (int kb = 0; kb < num_kb; ++kb) {
          mbar_wait(empty_bar(stage), parity ^ 1u);
          const uint32_t sA = base + stage * STAGE_BYTES;
          const uint32_t sB_hi = sA + 2 * A_BYTES, sB_lo = sB_hi + B_BYTES;
          const int k0 = kb * BK;
          const uint32_t cbytes = (uint32_t)min(BK, p.K - k0) * 4u;
          mbar_expect_tx(full_bar(stage), A_BYTES + 2 * B_BYTES + (RELAX ? 3u * cbytes : 0u) + (p.bias ? cbytes : 0u));
          if (RELAX) {
            const float* pl = p.planes + (long long)b * p.K + k0;
            bulk_load(sA + COEF_OFF, pl, cbytes, full_bar(stage));
            bulk_load(sA + COEF_OFF + 128, pl + p.plane_stride, cbytes, full_bar(stage));
            bulk_load(sA + COEF_OFF + 256, pl + 2 * p.plane_stride, cbytes, full_bar(stage));
          }
          if (p.bias) bulk_load(sA + COEF_OFF + 384, p.bias + k0, cbytes, full_bar(stage));
          tma_load_2d(sA, &tmA, kb * BK, src_row, full_bar(stage));
          tma_load_2d(sB_hi, &tmB_hi, kb * BK, n0, full_bar(stage));
          tma_load_2d(sB_lo, &tmB_lo, kb * BK, n0, full_bar(stage));
          if (++stage == STAGES) { stage = 0; parity ^= 1u; }
        }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer =====================
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
          const int kb_end = min(num_kb, (c + 1) * p.kb_per_chunk);
          uint32_t acc_big = 0;
          for (int kb = c * p.kb_per_chunk; kb < kb_end; ++kb) {
            mbar_wait(full_bar(stage), parity);      // W tiles landed (async proxy)
            mbar_wait(ready_bar(stage), parity);     // A hi/lo written by the transform warps
            tcgen05_fence_after();
            const uint32_t sA_hi = base + stage * STAGE_BYTES;
            const uint32_t sA_lo = sA_hi + A_BYTES;
            const uint32_t sB_hi = sA_lo + A_BYTES;
            const uint32_t sB_lo = sB_hi + B_BYTES;
#pragma unroll
            for (int k = 0; k < BK / UMMA_K; ++k) {
              const uint32_t koff = k * UMMA_K * 4;
              const uint64_t dA_hi = make_kmajor_sw128_desc(sA_hi + koff);
              const uint64_t dA_lo = make_kmajor_sw128_desc(sA_lo + koff);
              const uint64_t dB_hi = make_kmajor_sw128_desc(sB_hi + koff);
              const uint64_t dB_lo = make_kmajor_sw128_desc(sB_lo + koff);
              umma_tf32(tmem_small, dA_lo, dB_hi, idesc, acc_small);
              umma_tf32(tmem_small, dA_hi, dB_lo, idesc, 1u);
              umma_tf32(tmem_big, dA_hi, dB_hi, idesc, acc_big);
              acc_small = 1u; acc_big = 1u;
            }
            umma_commit(empty_bar(stage));
            if (++stage == STAGES) { stage = 0; parity ^= 1u; }
          }
          umma_commit(bfull_bar(bbuf));
          ++big_cnt;
          if ((c + 1) % p.chunks_per_small == 0 || c == num_chunks - 1) {
            umma_commit(sfull_bar(sbuf));
            ++small_cnt; acc_small = 0;
          }
        }
      }
    }
  } else if (warp >= 4 + EPI_WARPS) {
    // ===================== transform: relaxation + bias accumulation + TF32 split =====================
    const int xt = threadIdx.x - (4 + EPI_WARPS) * 32;       // 0..255
    const int row = xt & (BM - 1), half = xt >> 7;           // tile row, which 16 of the 32 k-elements
    const uint32_t sw = (uint32_t)(row & 7);
    float* dx = reinterpret_cast<float*>(smem_raw + (bar_base + 256u - raw));   // [2][BM] exchange slots
    int stage = 0; uint32_t parity = 0;
    uint32_t tile_cnt = 0;
    for (int t = blockIdx.x; t < num_tiles; t += gridDim.x, ++tile_cnt) {
      int g, r0, nb; tile_info(t, g, r0, nb);
      const bool row_ok = r0 + row < p.Rg;
      const long long m = (long long)g * p.Rg + (row_ok ? r0 + row : 0);
      const bool upper = m >= (long long)p.B * p.R;
      // per-stage coefficient slots {dU, bU, dL, bias}; the lower branch multiplies a>0 by dL and a<0 by dU, the
      // upper branch swaps them
      const int pos_slot = upper ? 0 : 2, neg_slot = upper ? 2 : 0;
      float dacc = 0.f;
      for (int kb = 0; kb < num_kb; ++kb) {
        mbar_wait(full_bar(stage), parity);
        float4* srow = reinterpret_cast<float4*>(smem_raw + (base + stage * STAGE_BYTES - raw) + row * 128);
        float4* srow_lo = srow + A_BYTES / 16;
        const float4* cslot = reinterpret_cast<const float4*>(smem_raw + (base + stage * STAGE_BYTES + COEF_OFF - raw));
        float4 x[4];
#pragma unroll
        for (int c = 0; c < 4; ++c) x[c] = srow[(half * 4 + c) ^ sw];
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          const int k = kb * BK + (half * 4 + c) * 4;
          float v[4] = {x[c].x, x[c].y, x[c].z, x[c].w};
          if (k < p.K) {
            float bs[4] = {0.f, 0.f, 0.f, 0.f};
            if (p.bias) { const float4 b4 = cslot[24 + half * 4 + c]; bs[0] = b4.x; bs[1] = b4.y; bs[2] = b4.z; bs[3] = b4.w; }
            if (RELAX) {
              const float4 sp4 = cslot[pos_slot * 8 + half * 4 + c];
              const float4 sn4 = cslot[neg_slot * 8 + half * 4 + c];
              const float4 bu4 = cslot[8 + half * 4 + c];
              const float sp[4] = {sp4.x, sp4.y, sp4.z, sp4.w}, sn[4] = {sn4.x, sn4.y, sn4.z, sn4.w};
              const float bu[4] = {bu4.x, bu4.y, bu4.z, bu4.w};
#pragma unroll
              for (int j = 0; j < 4; ++j) {
                const float a = v[j];
                const float pos = fmaxf(a, 0.f), neg = fminf(a, 0.f);
                const float o = pos * sp[j] + neg * sn[j];      // one term is +-0: o == a * slope exactly
                dacc = fmaf(upper ? pos : neg, bu[j], dacc);
                dacc = fmaf(o, bs[j], dacc);
                v[j] = o;
              }
            } else {
#pragma unroll
              for (int j = 0; j < 4; ++j) dacc = fmaf(v[j], bs[j], dacc);
            }
          }
          float4 hi, lo;
          tf32_split(v[0], hi.x, lo.x); tf32_split(v[1], hi.y, lo.y);
          tf32_split(v[2], hi.z, lo.z); tf32_split(v[3], hi.w, lo.w);
          srow[(half * 4 + c) ^ sw] = hi;
          srow_lo[(half * 4 + c) ^ sw] = lo;
        }
        fence_proxy_async();                 // generic-proxy smem writes -> visible to the tensor core (async proxy)
        mbar_arrive(ready_bar(stage));
        if (++stage == STAGES) { stage = 0; parity ^= 1u; }
      }
      // d[m] += (first half) + (second half), always in that order: deterministic
      if (p.d && nb == 0) {
        float* slot = dx + (tile_cnt & 1u) * BM;
        if (half == 1) slot[row] = dacc;
        asm volatile("bar.sync 1, %0;" :: "n"(XF_WARPS * 32) : "memory");
        if (half == 0 && row_ok) p.d[m] += dacc + slot[row];
      }
    }
  } else if (warp >= 4) {
    // ===================== epilogue: TMEM -> fp32 running sum -> global =====================
    const int ew = warp - 4;
    const int quad = warp & 3;
    const int chalf = ew >> 2;
    constexpr int EC = BN / 2;
    uint32_t big_cnt = 0, small_cnt = 0;
    for (int t = blockIdx.x; t < num_tiles; t += gridDim.x) {
      int g, r0, nb; tile_info(t, g, r0, nb);
      float acc[EC];
#pragma unroll
      for (int i = 0; i < EC; ++i) acc[i] = 0.f;
      for (int c = 0; c < num_chunks; ++c) {
        {
          const uint32_t buf = big_cnt & 1u;
          mbar_wait(bfull_bar(buf), (big_cnt >> 1) & 1u);
          tcgen05_fence_after();
          const uint32_t taddr = tmem_base + ((uint32_t)(quad * 32) << 16) + buf * BN + chalf * EC;
#pragma unroll
          for (int h = 0; h < EC / 16; ++h) {
            uint32_t v[16];
            tmem_ld16(taddr + h * 16, v);
            tmem_ld_wait();
#pragma unroll
            for (int i = 0; i < 16; ++i) acc[h * 16 + i] += __uint_as_float(v[i]);
          }
          tcgen05_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(bempty_bar(buf));
          ++big_cnt;
        }
        if ((c + 1) % p.chunks_per_small == 0 || c == num_chunks - 1) {
          const uint32_t buf = small_cnt & 1u;
          mbar_wait(sfull_bar(buf), (small_cnt >> 1) & 1u);
          tcgen05_fence_after();
          const uint32_t taddr = tmem_base + ((uint32_t)(quad * 32) << 16) + 2 * BN + buf * BN + chalf * EC;
#pragma unroll
          for (int h = 0; h < EC / 16; ++h) {
            uint32_t v[16];
            tmem_ld16(taddr + h * 16, v);
            tmem_ld_wait();
#pragma unroll
            for (int i = 0; i < 16; ++i) acc[h * 16 + i] += __uint_as_float(v[i]);
          }
          tcgen05_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(sempty_bar(buf));
          ++small_cnt;
        }
      }
      const int r = r0 + quad * 32 + lane;
      const int col0 = nb * BN + chalf * EC;
      if (r < p.Rg) {
        float* drow = p.D + ((long long)g * p.Rg + r) * p.ldd + col0;
#pragma unroll
        for (int i = 0; i < EC; i += 4) {
          if (col0 + i + 3 < p.N) {
            *reinterpret_cast<float4*>(drow + i) = make_float4(acc[i], acc[i + 1], acc[i + 2], acc[i + 3]);
          } else {
#pragma unroll
            for (int e = 0; e < 4; ++e)
              if (col0 + i + e < p.N) drow[i + e] = acc[i + e];
          }
        }
      }
    }
  }

  tcgen05_fence_before();
  __syncthreads();
  if (warp == 2) { tcgen05_fence_after(); tmem_dealloc(tmem_base, TMEM_COLS); }
}

}  // namespace tcf

int gemm_fused_supported(const AView& A, int B, int R, int N, int K) {
  if (!gemm_tc_supported(2 * B * R, N, K)) return 0;
  if (A.lo != nullptr || A.ld != K || A.n != K) return 0;
  if ((A.sB % K) != 0 || (A.sBr % K) != 0) return 0;
  if ((reinterpret_cast<uintptr_t>(A.p) & 15) != 0) return 0;
  if (B > 1 && R < 64) return 0;     // grouped tiling (one property per tile) would be mostly padding
  return 1;
}

int launch_gemm_fused(const AView& A, int B, int R, const float* planes, long long plane_stride, const float* bias,
                      float* d,
                      const float* Wt_hi, const float* Wt_lo, float* D, long long ldd, int N, int K, int k_drain,
                      int num_sms, cudaStream_t s, const char** err) {
  using namespace tcf;
  if (!gemm_fused_supported(A, B, R, N, K)) { if (err) *err = "gemm_fused: unsupported view or shape"; return -1; }
  Params p;
  p.D = D; p.ldd = ldd; p.M = 2 * B * R; p.N = N; p.K = K;
  p.B = B; p.R = R; p.planes = planes; p.plane_stride = plane_stride; p.bias = bias; p.d = d;
  // flat tiling only when every 128-row tile stays inside one (branch, property) group
  const bool flat = A.sB == (long long)R * K && A.sBr == (long long)B * R * K && (R % BM == 0);
  long long src_rows;
  if (flat) { p.n_groups = 1; p.Rg = p.M; p.base_br = 0; p.base_b = 0; src_rows = p.M; }
  else {
    p.n_groups = 2 * B; p.Rg = R; p.base_br = A.sBr / K; p.base_b = A.sB / K;
    src_rows = p.base_br + (long long)(B - 1) * p.base_b + R;
  }
  p.tiles_per_group = (p.Rg + BM - 1) / BM;
  if (k_drain <= 0) k_drain = 128;
  p.kb_per_chunk = (k_drain + BK - 1) / BK;
  p.chunks_per_small = 16384 / (p.kb_per_chunk * BK);
  if (p.chunks_per_small < 1) p.chunks_per_small = 1;
  CUtensorMap ta, tb, tc_;
  if (src_rows > 0x7fffffffLL || !make_tmap(&ta, A.p, (int)src_rows, K, BM) || !make_tmap(&tb, Wt_hi, N, K, BN) ||
      !make_tmap(&tc_, Wt_lo, N, K, BN)) { if (err) *err = "cuTensorMapEncodeTiled failed"; return -1; }
  static bool attr_set = false;
  if (!attr_set) {
    cudaError_t e1 = cudaFuncSetAttribute(gemm_fused_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
    cudaError_t e2 = cudaFuncSetAttribute(gemm_fused_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
    if (e1 != cudaSuccess || e2 != cudaSuccess) { if (err) *err = cudaGetErrorString(e1 != cudaSuccess ? e1 : e2); return -1; }
    attr_set = true;
  }
  const long long tiles = (long long)p.n_groups * p.tiles_per_group * ((N + BN - 1) / BN);
  const int grid = (int)(tiles < num_sms ? tiles : num_sms);
  if (planes) gemm_fused_kernel<true><<<grid, THREADS, SMEM_BYTES, s>>>(ta, tb, tc_, p);
  else gemm_fused_kernel<false><<<grid, THREADS, SMEM_BYTES, s>>>(ta, tb, tc_, p);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) { if (err) *err = cudaGetErrorString(e); return -1; }
  return 0;
}

}  // namespace crownb200
