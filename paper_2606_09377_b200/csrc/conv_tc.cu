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
//   warp 0      : MMA issuer (36 tcgen05.mma.kind::tf32 per dx: 3 dy x 4 k-steps x {lo.hi, hi.lo, hi.hi})
//   warp 1      : TMEM allocator
//   warps 4-7   : epilogue, lane = output pixel: drains the TMEM accumulator after every dx into an fp32 register sum
//                 (round 1 measured that long TMEM accumulation chains truncate: 36 MMAs per chain keeps fp32 accuracy),
//                 adds the residual fork's other contribution (addend) and stores A_in coalesced along x
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

constexpr int KC = 32;                     // output channels per K chunk = one 128-byte swizzle row
constexpr int XF_WARPS = 8;
constexpr int THREADS = 32 * (8 + XF_WARPS);
constexpr int MAXROWS = 192;               // (TR + 2) * W rows of a dx tile: W = 32 -> 6 * 32, W = 16 -> 10 * 16
constexpr int TILE_BYTES = MAXROWS * 128;  // one limb of one dx tile
constexpr int NBUF = 3;                    // dx tiles in flight

template <int NPAD>
struct Smem {
  static constexpr int W_BYTES = 9 * NPAD * 128;             // one limb of the 9 weight tiles [tap][ci][32 co]
  static constexpr int A_OFF = 2 * W_BYTES;
  static constexpr int BAR_OFF = A_OFF + NBUF * 2 * TILE_BYTES;
  static constexpr int TOTAL = BAR_OFF + 256 + 1024;         // + barriers + alignment slack
};

struct Params {
  const float* A; const float* A_lo; long long sBr, sB, ld;   // A_out view [2, B, R, c_out * H * W]
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
    for (int b = 0; b < NBUF; ++b) { mbar_init(full_bar(b), XF_WARPS * 32); mbar_init(empty_bar(b), 1); }
    for (int b = 0; b < 2; ++b) { mbar_init(accfull_bar(b), 1); mbar_init(accempty_bar(b), 4); }
    fence_barrier_init();
  }
  if (warp == 1) { tmem_alloc(tmem_slot, 2 * NPAD < 32 ? 32 : 2 * NPAD); tmem_relinquish(); }
  fence_proxy_async();                       // the weight tiles were written through the generic proxy
  tcgen05_fence_before();
  __syncthreads();
  tcgen05_fence_after();
  const uint32_t tmem_base = *tmem_slot_ptr;

  if (warp == 0) {
    // ===================== MMA issuer =====================
    if (lane == 0) {
      constexpr uint32_t idesc = make_idesc_tf32(128, NPAD);
      uint32_t seq = 0;                                 // dx passes issued so far
      for (long long it = blockIdx.x; it < items; it += gridDim.x) {
        for (int dxb = 0; dxb < 3; ++dxb, ++seq) {
          const int buf = seq % NBUF; const uint32_t bpar = (seq / NBUF) & 1u;
          const int ab = seq & 1u; const uint32_t apar = (seq >> 1) & 1u;
          mbar_wait(full_bar(buf), bpar);
          mbar_wait(accempty_bar(ab), apar ^ 1u);
          tcgen05_fence_after();
          const uint32_t sA_hi = base + S::A_OFF + buf * 2 * TILE_BYTES, sA_lo = sA_hi + TILE_BYTES;
          const uint32_t tmem_d = tmem_base + ab * NPAD;
          const int j = 2 - dxb;                         // tile dxb holds A_out shifted by s = dxb - 1 = 1 - j
          const int ksteps = (p.c_out + UMMA_K - 1) / UMMA_K;   // channels >= c_out are zero padding: not multiplied
          uint32_t acc = 0;
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
              umma_tf32(tmem_d, dA_lo, dB_hi, idesc, acc);
              umma_tf32(tmem_d, dA_hi, dB_lo, idesc, 1u);
              umma_tf32(tmem_d, dA_hi, dB_hi, idesc, 1u);
              acc = 1u;
            }
          }
          umma_commit(empty_bar(buf));
          umma_commit(accfull_bar(ab));
        }
      }
    }
  } else if (warp >= 8) {
    // ===================== transform: NCHW fp32 -> K-major swizzled TF32 hi / lo tiles =====================
    const int xw = warp - 8;                             // 0..7 = group of 4 output channels (co4)
    uint32_t seq = 0;
    for (long long it = blockIdx.x; it < items; it += gridDim.x) {
      const long long m = it / p.bands;
      const int y0 = (int)(it % p.bands) * p.TR;
      const int r_ = (int)(m % p.R);
      const long long tt = m / p.R;
      const long long roff = (tt / p.B) * p.sBr + (tt % p.B) * p.sB + (long long)r_ * p.ld;
      const float* src = p.A + roff;
      const float* src_lo = p.A_lo ? p.A_lo + roff : nullptr;
      for (int dxb = 0; dxb < 3; ++dxb, ++seq) {
        const int buf = seq % NBUF; const uint32_t bpar = (seq / NBUF) & 1u;
        mbar_wait(empty_bar(buf), bpar ^ 1u);
        uint8_t* t_hi = gbase + S::A_OFF + buf * 2 * TILE_BYTES;
        uint8_t* t_lo = t_hi + TILE_BYTES;
        const int s = dxb - 1;
        const bool used = xw * 4 < ((p.c_out + UMMA_K - 1) / UMMA_K) * UMMA_K;     // this warp's channels are multiplied
        for (int r = lane; used && r < tile_rows; r += 32) {     // tile row = (yy, x): lanes run along x (coalesced loads)
          const int yy = r / p.W, x = r % p.W;
          const int y = y0 - 1 + yy, xs = x + s;
          const bool in = y >= 0 && y < p.H && xs >= 0 && xs < p.W;
          float v[4];
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            const int co = xw * 4 + e;
            float val = 0.f;
            if (in && co < p.c_out) {
              const long long o = (long long)co * HW + y * p.W + xs;
              val = src[o];
              if (src_lo) val += src_lo[o];
            }
            v[e] = val;
          }
          float4 hi, lo;
          tf32_split(v[0], hi.x, lo.x); tf32_split(v[1], hi.y, lo.y); tf32_split(v[2], hi.z, lo.z); tf32_split(v[3], hi.w, lo.w);
          const uint32_t off = (uint32_t)r * 128u + (((uint32_t)xw ^ (uint32_t)(r & 7)) << 4);
          *reinterpret_cast<float4*>(t_hi + off) = hi;
          *reinterpret_cast<float4*>(t_lo + off) = lo;
        }
        fence_proxy_async();                 // generic-proxy smem writes -> visible to the tensor core (async proxy)
        mbar_arrive(full_bar(buf));
      }
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
#pragma unroll
      for (int c = 0; c < NPAD; ++c) sum[c] = 0.f;
      for (int dxb = 0; dxb < 3; ++dxb, ++seq) {
        const int ab = seq & 1u; const uint32_t apar = (seq >> 1) & 1u;
        mbar_wait(accfull_bar(ab), apar);
        tcgen05_fence_after();
        const uint32_t taddr = tmem_base + ((uint32_t)(quad * 32) << 16) + ab * NPAD;
        if constexpr (NPAD == 32) {
          uint32_t v[32]; tmem_ld32(taddr, v); tmem_ld_wait();
#pragma unroll
          for (int c = 0; c < 32; ++c) sum[c] += __uint_as_float(v[c]);
        } else {
          uint32_t v[16]; tmem_ld16(taddr, v); tmem_ld_wait();
#pragma unroll
          for (int c = 0; c < 16; ++c) sum[c] += __uint_as_float(v[c]);
        }
        tcgen05_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(accempty_bar(ab));
      }
      float* orow = p.out + (m * p.c_in) * (long long)HW + (long long)(y0 + ty) * p.W + x;
      const float* arow = p.addend ? p.addend + (m * p.c_in) * (long long)HW + (long long)(y0 + ty) * p.W + x : nullptr;
#pragma unroll
      for (int c = 0; c < NPAD; ++c) {
        if (c < p.c_in) {
          float o = sum[c];
          if (arow) o += arow[(long long)c * HW];
          orow[(long long)c * HW] = o;
        }
      }
    }
  }

  tcgen05_fence_before();
  __syncthreads();
  if (warp == 1) { tcgen05_fence_after(); tmem_dealloc(tmem_base, 2 * NPAD < 32 ? 32 : 2 * NPAD); }
}

}  // namespace ctc

int conv_tc_init_device() {
  cudaError_t e1 = cudaFuncSetAttribute(ctc::conv_bwd_tc_kernel<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, ctc::Smem<16>::TOTAL);
  cudaError_t e2 = cudaFuncSetAttribute(ctc::conv_bwd_tc_kernel<32>, cudaFuncAttributeMaxDynamicSharedMemorySize, ctc::Smem<32>::TOTAL);
  return (e1 == cudaSuccess && e2 == cudaSuccess) ? 0 : -1;
}

int conv_tc_supported(int c_in, int h, int w, int c_out, int kh, int kw, int stride, int pad, int ho, int wo) {
  return kh == 3 && kw == 3 && stride == 1 && pad == 1 && ho == h && wo == w && (w == 16 || w == 32) &&
         (h * w) % 128 == 0 && c_in >= 1 && c_in <= 32 && c_out >= 1 && c_out <= 32;
}

int launch_conv_transpose_tc(const AView& A, const float* W, const float* addend, float* out, int B, int R,
                             int c_in, int h, int w, int c_out, int num_sms, cudaStream_t s) {
  ctc::Params p;
  p.A = A.p; p.A_lo = A.lo; p.sBr = A.sBr; p.sB = A.sB; p.ld = A.ld;
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
