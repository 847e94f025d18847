// a6 on the tensor cores -- BoundConv backward A_in = conv^T(A_out, W) for the 3x3 / stride 1 /
// pad 1 convolutions of a ResNet as a per-tap implicit GEMM on tcgen05 (3xTF32, fp32-accurate):
//     A_in[m, ci, y, x] = sum_{tap (i,j)} sum_co  A_out[m, co, y+1-i, x+1-j] * W[co, ci, i, j]
// For one spec row m and a band of TR image rows (TR * W = 128 output pixels) every tap is one small GEMM
//     D[128 pixels, C_in] += Aop_tap[128 pixels, C_out] . W_tap[C_out, C_in]
// whose A operand is a SHIFTED WINDOW of one staged tile: no im2col expansion.  The tile is staged K-major (C_out
// contiguous, 128-byte swizzled rows = 32 output channels) by transform warps that read A_out in its NCHW layout
// (coalesced along x), split it into TF32 hi / lo limbs and write both; one tile per horizontal shift dx (a 4-byte
// shift cannot be expressed in a 16-byte-granular shared-memory descriptor), the three vertical taps of a dx are
// descriptor offsets of W rows (multiples of 1024 B).  The 9 x C_in x 32 weight tiles stay resident in shared memory.
//   warp 0      : MMA issuer (up to 36 tcgen05.mma.kind::tf32 per dx: 3 dy x 4 k-steps x {lo.hi, hi.lo, hi.hi}),
//                 dealt round robin to 8 accumulators
//   warp 1      : TMEM allocator;  warp 2: signaller (named barrier of the transform warps -> mbarrier of the issuer)
//   warps 4-7   : epilogue, lane = output pixel: adds up the item's 8 independent TMEM accumulators (each a chain of
//                 <= 14 MMAs: round 1 measured that long TMEM accumulation chains truncate), adds the residual fork's
//                 other contribution (addend) and stores A_in coalesced along x
//   warps 8-15  : transform (NCHW fp32 -> K-major swizzled hi / lo tiles), one dx tile ahead of the tensor core
// Layers outside this shape (stride 2, 1x1, 8x8 maps, C > 32) stay on the CUDA-core kernel of conv.cu.
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "common.cuh"
#include "kernels.h"
#include "tc_common.cuh"

namespace crownb200 {
namespace ctc {

using namespace tc;

// round-to-nearest (ties away) to TF32 on the bit pattern: cvt.rna.tf32.f32 for finite inputs in two integer ops
__device__ __forceinline__ float tf32_rn_bits(float x) {
  return __uint_as_float((__float_as_uint(x) + 0x1000u) & 0xffffe000u);
}

constexpr int KC = 32;                     // output channels per K chunk = one 128-byte swizzle row
constexpr int XF_WARPS = 8;
constexpr int THREADS = 32 * (8 + XF_WARPS);
constexpr int MAXROWS = 192;               // (TR + 2) * W rows of a dx tile: W = 32 -> 6 * 32, W = 16 -> 10 * 16
constexpr int TILE_BYTES = MAXROWS * 128;  // one limb of one dx tile
constexpr int NBUF = 3;                    // dx tiles in flight
constexpr int NACC = 8;                    // independent TMEM accumulators per item (see the MMA issuer)

template <int NPAD>
struct Smem {
  static constexpr int W_BYTES = 9 * NPAD * 128;             // one limb of the 9 weight tiles [tap][ci][32 co]
  static constexpr int A_OFF = 2 * W_BYTES;
  static constexpr int BAR_OFF = A_OFF + NBUF * 2 * TILE_BYTES;
  static constexpr int TOTAL = BAR_OFF + 256 + 1024;         // + barriers + alignment slack
};

struct Params {
  const float* A; long long sBr, sB, ld;                       // A_out view [2, B, R, c_out * H * W] (fp32, no lo limb)
  const float* Wgt;                                             // [c_out, c_in, 3, 3]
  const float* addend; float* out;                              // [rows, c_in * H * W] contiguous
  int B, R; long long rows;
  int c_in, c_out, H, W, TR, bands;                             // TR image rows per tile (TR * W = 128), bands = H / TR
};

template <int NPAD>
__global__ void __launch_bounds__(THREADS, 1) conv_bwd_tc_kernel(const Params p) {
  using S = Smem<NPAD>;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t raw = smem_u32(smem_raw);
  const uint32_t base = (raw + 1023u) & ~1023u;
  uint8_t* gbase = smem_raw + (base - raw);
  const uint32_t bar_base = base + S::BAR_OFF;
  auto full_bar = [&](int b) { return bar_base + 8u * b; };                 // dx tile written
  auto empty_bar = [&](int b) { return bar_base + 8u * (NBUF + b); };       // MMAs have read the dx tile
  auto accfull_bar = [&](int b) { return bar_base + 8u * (2 * NBUF + b); };
  auto accempty_bar = [&](int b) { return bar_base + 8u * (2 * NBUF + 2 + b); };
  const uint32_t tmem_slot = bar_base + 8u * (2 * NBUF + 4);
  volatile uint32_t* tmem_slot_ptr = reinterpret_cast<volatile uint32_t*>(gbase + S::BAR_OFF + 8 * (2 * NBUF + 4));

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int HW = p.H * p.W;
  const long long items = p.rows * p.bands;
  const int tile_rows = (p.TR + 2) * p.W;

  // ---- weights: [tap][ci (NPAD rows)][32 co] K-major, 128B-swizzled, hi and lo limbs; resident for the whole kernel
  for (int idx = threadIdx.x; idx < 9 * NPAD * (KC / 4); idx += blockDim.x) {
    const int c4 = idx % (KC / 4), n = (idx / (KC / 4)) % NPAD, tap = idx / ((KC / 4) * NPAD);
    float4 hi, lo;
    float v[4];
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      const int co = c4 * 4 + e;
      v[e] = (n < p.c_in && co < p.c_out) ? __ldg(p.Wgt + ((long long)co * p.c_in + n) * 9 + tap) : 0.f;
    }
    tf32_split(v[0], hi.x, lo.x); tf32_split(v[1], hi.y, lo.y); tf32_split(v[2], hi.z, lo.z); tf32_split(v[3], hi.w, lo.w);
    const uint32_t off = (uint32_t)(tap * NPAD + n) * 128u + (((uint32_t)c4 ^ (uint32_t)(n & 7)) << 4);
    *reinterpret_cast<float4*>(gbase + off) = hi;
    *reinterpret_cast<float4*>(gbase + S::W_BYTES + off) = lo;
  }
  if (warp == 0 && lane == 0) {
    for (int b = 0; b < NBUF; ++b) { mbar_init(full_bar(b), 1); mbar_init(empty_bar(b), 1); }
    for (int b = 0; b < 2; ++b) { mbar_init(accfull_bar(b), 1); mbar_init(accempty_bar(b), 4); }
    fence_barrier_init();
  }
  if (warp == 1) { tmem_alloc(tmem_slot, 2 * NACC * NPAD); tmem_relinquish(); }
  fence_proxy_async();                       // the weight tiles were written through the generic proxy
  tcgen05_fence_before();
  __syncthreads();
  tcgen05_fence_after();
  const uint32_t tmem_base = *tmem_slot_ptr;

  if (warp == 0) {
    // ===================== MMA issuer =====================
    // A 128 x NPAD accumulator tile is small: back-to-back MMAs into the SAME tile serialise on the tensor core's
    // accumulate latency (measured: ~250 cycles per MMA with one accumulator, against ~32 cycles of operand reads).
    // The MMAs of an item are therefore dealt round robin to NACC independent accumulators, which the epilogue adds
    // up; every TMEM chain is then at most 14 MMAs long, so no intermediate drains are needed for fp32 accuracy.
    if (lane == 0) {
      constexpr uint32_t idesc = make_idesc_tf32(128, NPAD);
      const int ksteps = (p.c_out + UMMA_K - 1) / UMMA_K;   // channels >= c_out are zero padding: not multiplied
      uint32_t seq = 0, item = 0;
      for (long long it = blockIdx.x; it < items; it += gridDim.x, ++item) {
        const int ab = item & 1u; const uint32_t apar = (item >> 1) & 1u;
        mbar_wait(accempty_bar(ab), apar ^ 1u);
        uint32_t cnt = 0;
        for (int dxb = 0; dxb < 3; ++dxb, ++seq) {
          const int buf = seq % NBUF; const uint32_t bpar = (seq / NBUF) & 1u;
          mbar_wait(full_bar(buf), bpar);
          tcgen05_fence_after();
          const uint32_t sA_hi = base + S::A_OFF + buf * 2 * TILE_BYTES, sA_lo = sA_hi + TILE_BYTES;
          const int j = 2 - dxb;                         // tile dxb holds A_out shifted by s = dxb - 1 = 1 - j
#pragma unroll
          for (int i = 0; i < 3; ++i) {
            const uint32_t roff = (uint32_t)((2 - i) * p.W) * 128u;     // vertical tap = window offset of (2 - i) image rows
            const uint32_t sB_hi = base + (uint32_t)((i * 3 + j) * NPAD) * 128u, sB_lo = sB_hi + S::W_BYTES;
#pragma unroll
            for (int k = 0; k < KC / UMMA_K; ++k) {
              if (k >= ksteps) break;
              const uint32_t koff = k * UMMA_K * 4;
              const uint64_t dA_hi = make_kmajor_sw128_desc(sA_hi + roff + koff);
              const uint64_t dA_lo = make_kmajor_sw128_desc(sA_lo + roff + koff);
              const uint64_t dB_hi = make_kmajor_sw128_desc(sB_hi + koff);
              const uint64_t dB_lo = make_kmajor_sw128_desc(sB_lo + koff);
              const uint32_t t0 = tmem_base + (ab * NACC + (cnt % NACC)) * NPAD; const uint32_t f0 = cnt >= NACC; ++cnt;
              const uint32_t t1 = tmem_base + (ab * NACC + (cnt % NACC)) * NPAD; const uint32_t f1 = cnt >= NACC; ++cnt;
              const uint32_t t2 = tmem_base + (ab * NACC + (cnt % NACC)) * NPAD; const uint32_t f2 = cnt >= NACC; ++cnt;
              umma_tf32(t0, dA_lo, dB_hi, idesc, f0);
              umma_tf32(t1, dA_hi, dB_lo, idesc, f1);
              umma_tf32(t2, dA_hi, dB_hi, idesc, f2);
            }
          }
          umma_commit(empty_bar(buf));
        }
        umma_commit(accfull_bar(ab));
      }
    }
  } else if (warp == 2) {
    // ===================== signaller: 256 named-barrier arrivals of the transform threads -> one mbarrier arrive ======
    uint32_t seq = 0;
    for (long long it = blockIdx.x; it < items; it += gridDim.x) {
      for (int dxb = 0; dxb < 3; ++dxb, ++seq) {
        const int buf = seq % NBUF;
        asm volatile("bar.sync %0, %1;" :: "r"(1 + buf), "n"(XF_WARPS * 32 + 32) : "memory");
        if (lane == 0) { fence_proxy_async(); mbar_arrive(full_bar(buf)); }
      }
    }
  } else if (warp >= 8) {
    // ===================== transform: NCHW fp32 -> K-major swizzled TF32 hi / lo tiles =====================
    // A warp task = (group of 4 output channels, 32 consecutive tile rows); tasks are dealt round robin to the 8
    // warps and everything about a task that does not depend on the item (tile offset, source offset, edge flags) is
    // computed once.  Per item every element of the haloed band is loaded ONCE: all of a thread's loads are issued
    // back to back with no dependent instruction in between (a use right after a load stalls the in-order warp and
    // serialises the remaining loads: measured 15k cycles per item), and the NEXT item's loads are issued before this
    // item's tiles are written, so their latency hides behind the shuffle / store phase.  The three horizontally
    // shifted tiles are produced from registers with warp shuffles along x.
    const int xw = warp - 8;
    const int wshift = p.W == 32 ? 5 : 4;
    const int G = 2 * ((p.c_out + UMMA_K - 1) / UMMA_K);    // groups of 4 channels that are multiplied
    const int ntask = G * (tile_rows >> 5);
    constexpr int NT = 6;                                   // tasks per warp (8 groups x 6 chunks / 8 warps)
    uint32_t toff[NT];                                      // byte offset of the task's 16-byte chunk in a tile
    int soff[NT], tyy[NT];                                  // source offset (first of the 4 channels) at y0 = 1; tile row yy
    bool tval[NT], okl[NT], okr[NT];                        // task exists; left / right neighbour inside the image row
    int cval[NT];                                           // channels of the group below c_out (0..4)
#pragma unroll
    for (int t = 0; t < NT; ++t) {
      const int id = xw + 8 * t;
      const int co4 = id % G, rch = id / G;
      const int r = rch * 32 + lane;
      const int x = r & (p.W - 1);
      tval[t] = id < ntask;
      tyy[t] = r >> wshift;
      toff[t] = (uint32_t)r * 128u + (((uint32_t)co4 ^ (uint32_t)(r & 7)) << 4);
      soff[t] = co4 * 4 * HW + (tyy[t] - 1) * p.W + x;
      okl[t] = x >= 1; okr[t] = x + 1 < p.W;
      cval[t] = min(4, max(0, p.c_out - co4 * 4));
    }
    auto load_item = [&](long long it, float (&v)[NT][4]) {
      const long long m = it / p.bands;
      const int y0 = (int)(it % p.bands) * p.TR;
      const int r_ = (int)(m % p.R);
      const long long tt = m / p.R;
      const float* src = p.A + (tt / p.B) * p.sBr + (tt % p.B) * p.sB + (long long)r_ * p.ld + y0 * p.W;
#pragma unroll
      for (int t = 0; t < NT; ++t) {
        const int y = y0 - 1 + tyy[t];
        const bool in = tval[t] && y >= 0 && y < p.H;
        const float* q = src + soff[t];
#pragma unroll
        for (int e = 0; e < 4; ++e) v[t][e] = (in && e < cval[t]) ? __ldg(q + e * HW) : 0.f;
      }
    };
    uint32_t seq = 0;
    float v[NT][4];
    if ((long long)blockIdx.x < items) load_item(blockIdx.x, v);
    for (long long it = blockIdx.x; it < items; it += gridDim.x) {
      float vn[NT][4];
      if (it + gridDim.x < items) load_item(it + gridDim.x, vn);
      for (int dxb = 0; dxb < 3; ++dxb, ++seq) {
        const int buf = seq % NBUF; const uint32_t bpar = (seq / NBUF) & 1u;
        mbar_wait(empty_bar(buf), bpar ^ 1u);
        uint8_t* t_hi = gbase + S::A_OFF + buf * 2 * TILE_BYTES;
        uint8_t* t_lo = t_hi + TILE_BYTES;
        const int s = dxb - 1;                              // tile[yy][x] = A_out[y0 - 1 + yy][x + s]
#pragma unroll
        for (int t = 0; t < NT; ++t) {
          if (!tval[t]) continue;                           // warp-uniform
          const bool ok = s == 0 || (s < 0 ? okl[t] : okr[t]);   // neighbour inside the image row (else zero padding)
          float4 hi, lo;
          float w[4];
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            const float nb = s == 0 ? v[t][e] : __shfl_sync(0xffffffffu, v[t][e], (lane + s) & 31);
            w[e] = ok ? nb : 0.f;
          }
          hi.x = tf32_rn_bits(w[0]); lo.x = tf32_rn_bits(w[0] - hi.x);
          hi.y = tf32_rn_bits(w[1]); lo.y = tf32_rn_bits(w[1] - hi.y);
          hi.z = tf32_rn_bits(w[2]); lo.z = tf32_rn_bits(w[2] - hi.z);
          hi.w = tf32_rn_bits(w[3]); lo.w = tf32_rn_bits(w[3] - hi.w);
          *reinterpret_cast<float4*>(t_hi + toff[t]) = hi;
          *reinterpret_cast<float4*>(t_lo + toff[t]) = lo;
        }
        fence_proxy_async();                 // generic-proxy smem writes -> visible to the tensor core (async proxy)
        // hand-off through a named barrier and the signaller warp: an mbarrier arrive (release) by THIS thread would
        // first wait for its prefetched global loads of the next item and expose their latency on every pass
        asm volatile("bar.arrive %0, %1;" :: "r"(1 + buf), "n"(XF_WARPS * 32 + 32) : "memory");
      }
#pragma unroll
      for (int t = 0; t < NT; ++t)
#pragma unroll
        for (int e = 0; e < 4; ++e) v[t][e] = vn[t][e];
    }
  } else if (warp >= 4) {
    // ===================== epilogue: lane = output pixel =====================
    const int quad = warp & 3;
    const int pix = quad * 32 + lane;                    // pixel of the band
    const int ty = pix / p.W, x = pix % p.W;
    uint32_t seq = 0;
    for (long long it = blockIdx.x; it < items; it += gridDim.x) {
      const long long m = it / p.bands;
      const int y0 = (int)(it % p.bands) * p.TR;
      float sum[NPAD];
      // the residual fork's other contribution: all loads issued up front (they complete while the MMAs still run)
      const float* arow = p.addend ? p.addend + (m * p.c_in) * (long long)HW + (long long)(y0 + ty) * p.W + x : nullptr;
#pragma unroll
      for (int c = 0; c < NPAD; ++c) sum[c] = (arow && c < p.c_in) ? __ldg(arow + (long long)c * HW) : 0.f;
      {
        const int ab = seq & 1u; const uint32_t apar = (seq >> 1) & 1u;
        ++seq;
        mbar_wait(accfull_bar(ab), apar);
        tcgen05_fence_after();
#pragma unroll
        for (int a = 0; a < NACC; ++a) {
          const uint32_t taddr = tmem_base + ((uint32_t)(quad * 32) << 16) + (ab * NACC + a) * NPAD;
          if constexpr (NPAD == 32) {
            uint32_t v[32]; tmem_ld32(taddr, v); tmem_ld_wait();
#pragma unroll
            for (int c = 0; c < 32; ++c) sum[c] += __uint_as_float(v[c]);
          } else {
            uint32_t v[16]; tmem_ld16(taddr, v); tmem_ld_wait();
#pragma unroll
            for (int c = 0; c < 16; ++c) sum[c] += __uint_as_float(v[c]);
          }
        }
        tcgen05_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(accempty_bar(ab));
      }
      float* orow = p.out + (m * p.c_in) * (long long)HW + (long long)(y0 + ty) * p.W + x;
#pragma unroll
      for (int c = 0; c < NPAD; ++c) {
        if (c < p.c_in) {
          const float o = sum[c];
          orow[(long long)c * HW] = o;
        }
      }
    }
  }

  tcgen05_fence_before();
  __syncthreads();
  if (warp == 1) { tcgen05_fence_after(); tmem_dealloc(tmem_base, 2 * NACC * NPAD); }
}

}  // namespace ctc

int conv_tc_init_device() {
  cudaError_t e1 = cudaFuncSetAttribute(ctc::conv_bwd_tc_kernel<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, ctc::Smem<16>::TOTAL);
  cudaError_t e2 = cudaFuncSetAttribute(ctc::conv_bwd_tc_kernel<32>, cudaFuncAttributeMaxDynamicSharedMemorySize, ctc::Smem<32>::TOTAL);
  return (e1 == cudaSuccess && e2 == cudaSuccess) ? 0 : -1;
}

int conv_tc_supported(int c_in, int h, int w, int c_out, int kh, int kw, int stride, int pad, int ho, int wo) {
  // Measured per layer on B200 (profiles/r2_conv_tc_vs_ffma.md): a 128 x N x 8 MMA costs ~105 cycles whatever N <= 32 is,
  // so the tensor-core kernel wins 2.2x at 32 channels (16 x 16 maps: 135 vs 295 us) and loses at 16 channels
  // (32 x 32 maps: 300 vs 280 us; the 3-channel stem: 299 vs 164 us).  It is used where it wins.
  return kh == 3 && kw == 3 && stride == 1 && pad == 1 && ho == h && wo == w && (w == 16 || w == 32) &&
         (h * w) % 128 == 0 && c_in > 16 && c_in <= 32 && c_out > 16 && c_out <= 32;
}

int launch_conv_transpose_tc(const AView& A, const float* W, const float* addend, float* out, int B, int R,
                             int c_in, int h, int w, int c_out, int num_sms, cudaStream_t s) {
  ctc::Params p;
  if (A.lo) return -1;                   // split views go to the CUDA-core kernel (none reaches a conv node today)
  p.A = A.p; p.sBr = A.sBr; p.sB = A.sB; p.ld = A.ld;
  p.Wgt = W; p.addend = addend; p.out = out; p.B = B; p.R = R; p.rows = 2LL * B * R;
  p.c_in = c_in; p.c_out = c_out; p.H = h; p.W = w; p.TR = 128 / w; p.bands = h / p.TR;
  const long long items = p.rows * p.bands;
  if (items <= 0) return 0;
  const int grid = (int)(items < num_sms ? items : num_sms);
  if (c_in <= 16) ctc::conv_bwd_tc_kernel<16><<<grid, ctc::THREADS, ctc::Smem<16>::TOTAL, s>>>(p);
  else ctc::conv_bwd_tc_kernel<32><<<grid, ctc::THREADS, ctc::Smem<32>::TOTAL, s>>>(p);
  return cudaGetLastError() == cudaSuccess ? 0 : -1;
}

}  // namespace crownb200
