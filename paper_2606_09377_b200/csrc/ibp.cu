// a1 -- IBP through a Linear layer, centre/radius form (l' = W+ l + W- u + b,
// u' = W+ u + W- l + b, which equals c' -+ r' with c' = W c + b, r' = |W| r).
//
// The kernel is bound by the single read of W (4 n_out n_in bytes per batch tile): every warp streams
// RW rows of W with 128-bit coalesced loads (each 512 B segment of a row is one warp request) and
// multiplies them against the centre / radius vectors of BT properties staged in shared memory.
// RW rows per warp re-use every shared-memory operand RW times, so the LDS traffic stays below the
// FMA rate; BT accumulator pairs per row live in registers.
#include "common.cuh"
#include "kernels.h"

namespace crownb200 {

constexpr int kIbpKC = 512;      // K chunk staged in shared memory (floats)
constexpr int kIbpWarps = 8;

template <int BT, int RW>
__global__ void __launch_bounds__(kIbpWarps * 32, 2)
ibp_linear_kernel(const float* __restrict__ W, const float* __restrict__ bias,
                  const float* __restrict__ l_in, const float* __restrict__ u_in, int relu_in,
                  float* __restrict__ l_out, float* __restrict__ u_out, int B, int n_out, int n_in, int ldo) {
  __shared__ __align__(16) float sc[BT][kIbpKC];
  __shared__ __align__(16) float sr[BT][kIbpKC];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int row0 = (blockIdx.x * kIbpWarps + warp) * RW;
  const int b0 = blockIdx.y * BT;
  const bool vec = (n_in % 4 == 0) && ((reinterpret_cast<uintptr_t>(W) & 15) == 0);

  float accC[RW][BT], accR[RW][BT];
#pragma unroll
  for (int i = 0; i < RW; ++i)
#pragma unroll
    for (int b = 0; b < BT; ++b) { accC[i][b] = 0.f; accR[i][b] = 0.f; }

  for (int k0 = 0; k0 < n_in; k0 += kIbpKC) {
    const int kc = min(kIbpKC, n_in - k0);
    __syncthreads();
    for (int idx = threadIdx.x; idx < BT * kIbpKC; idx += blockDim.x) {
      int b = idx / kIbpKC, j = idx % kIbpKC;
      float c = 0.f, r = 0.f;
      if (b0 + b < B && j < kc) {
        float lo = l_in[(long long)(b0 + b) * n_in + k0 + j];
        float hi = u_in[(long long)(b0 + b) * n_in + k0 + j];
        if (relu_in) { lo = fmaxf(lo, 0.f); hi = fmaxf(hi, 0.f); }
        c = 0.5f * (lo + hi);
        r = 0.5f * (hi - lo);
      }
      sc[b][j] = c;
      sr[b][j] = r;
    }
    __syncthreads();
    if (vec) {
      for (int j = lane * 4; j < kc; j += 128) {
        float4 w[RW];
#pragma unroll
        for (int i = 0; i < RW; ++i) {
          int row = row0 + i;
          w[i] = row < n_out ? ldg_stream4(W + (long long)row * n_in + k0 + j) : make_float4(0, 0, 0, 0);
        }
#pragma unroll
        for (int b = 0; b < BT; ++b) {
          float4 c = *reinterpret_cast<const float4*>(&sc[b][j]);
          float4 r = *reinterpret_cast<const float4*>(&sr[b][j]);
#pragma unroll
          for (int i = 0; i < RW; ++i) {
            accC[i][b] = fmaf(w[i].x, c.x, accC[i][b]);
            accC[i][b] = fmaf(w[i].y, c.y, accC[i][b]);
            accC[i][b] = fmaf(w[i].z, c.z, accC[i][b]);
            accC[i][b] = fmaf(w[i].w, c.w, accC[i][b]);
            accR[i][b] = fmaf(fabsf(w[i].x), r.x, accR[i][b]);
            accR[i][b] = fmaf(fabsf(w[i].y), r.y, accR[i][b]);
            accR[i][b] = fmaf(fabsf(w[i].z), r.z, accR[i][b]);
            accR[i][b] = fmaf(fabsf(w[i].w), r.w, accR[i][b]);
          }
        }
      }
    } else {
      for (int j = lane; j < kc; j += 32) {
#pragma unroll
        for (int i = 0; i < RW; ++i) {
          int row = row0 + i;
          float w = row < n_out ? W[(long long)row * n_in + k0 + j] : 0.f;
#pragma unroll
          for (int b = 0; b < BT; ++b) {
            accC[i][b] = fmaf(w, sc[b][j], accC[i][b]);
            accR[i][b] = fmaf(fabsf(w), sr[b][j], accR[i][b]);
          }
        }
      }
    }
  }
#pragma unroll
  for (int i = 0; i < RW; ++i) {
    int row = row0 + i;
#pragma unroll
    for (int b = 0; b < BT; ++b) {
      float c = warp_sum(accC[i][b]);
      float r = warp_sum(accR[i][b]);
      if (lane == 0 && row < n_out && b0 + b < B) {
        c += bias ? bias[row] : 0.f;
        l_out[(long long)(b0 + b) * ldo + row] = c - r;
        u_out[(long long)(b0 + b) * ldo + row] = c + r;
      }
    }
  }
}

void launch_ibp_linear(const float* W, const float* bias, const float* l_in, const float* u_in,
                       int relu_in, float* l_out, float* u_out, int B, int n_out, int n_in, int ldo,
                       cudaStream_t s) {
  if (B <= 0 || n_out <= 0) return;
  constexpr int RW = 4;
  dim3 block(kIbpWarps * 32);
  int gx = ceil_div(n_out, kIbpWarps * RW);
  if (B <= 1) {
    ibp_linear_kernel<1, RW><<<dim3(gx, 1), block, 0, s>>>(W, bias, l_in, u_in, relu_in, l_out, u_out, B, n_out, n_in, ldo);
  } else if (B <= 2) {
    ibp_linear_kernel<2, RW><<<dim3(gx, 1), block, 0, s>>>(W, bias, l_in, u_in, relu_in, l_out, u_out, B, n_out, n_in, ldo);
  } else if (B <= 4) {
    ibp_linear_kernel<4, RW><<<dim3(gx, 1), block, 0, s>>>(W, bias, l_in, u_in, relu_in, l_out, u_out, B, n_out, n_in, ldo);
  } else {
    ibp_linear_kernel<8, RW><<<dim3(gx, ceil_div(B, 8)), block, 0, s>>>(W, bias, l_in, u_in, relu_in, l_out, u_out, B, n_out, n_in, ldo);
  }
}

}  // namespace crownb200
