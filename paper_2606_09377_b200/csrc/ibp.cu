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

constexpr int kIbpWarps = 8;
constexpr int kIbpSmemMax = 160 * 1024;   // centre/radius staging budget (dynamic shared memory)

// KC (runtime, multiple of 512): elements of K staged per pass; the whole K when it fits kIbpSmemMax, so that W is
// streamed with one barrier per block and 4 x RW independent 128-bit loads in flight per thread.
template <int BT, int RW>
__global__ void __launch_bounds__(kIbpWarps * 32, 1)
ibp_linear_kernel(const float* __restrict__ W, const float* __restrict__ bias,
                  const float* __restrict__ l_in, const float* __restrict__ u_in, int relu_in,
                  float* __restrict__ l_out, float* __restrict__ u_out, int B, int n_out, int n_in, int ldo, int KC) {
  extern __shared__ __align__(16) float ibp_smem[];
  float* sc = ibp_smem;                      // [BT][KC]
  float* sr = ibp_smem + (size_t)BT * KC;    // [BT][KC]
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int b0 = blockIdx.y * BT;
  const bool vec = (n_in % 4 == 0) && ((reinterpret_cast<uintptr_t>(W) & 15) == 0);
  const bool single = KC >= n_in;     // whole K staged once: the block is persistent over row groups

  auto stage = [&](int k0, int kc) {
    for (int idx = threadIdx.x; idx < BT * KC; idx += blockDim.x) {
      int b = idx / KC, j = idx % KC;
      float c = 0.f, r = 0.f;
      if (b0 + b < B && j < kc) {
        float lo = l_in[(long long)(b0 + b) * n_in + k0 + j];
        float hi = u_in[(long long)(b0 + b) * n_in + k0 + j];
        if (relu_in) { lo = fmaxf(lo, 0.f); hi = fmaxf(hi, 0.f); }
        c = 0.5f * (lo + hi);
        r = 0.5f * (hi - lo);
      }
      sc[idx] = c;
      sr[idx] = r;
    }
  };
  if (single) { stage(0, n_in); __syncthreads(); }

  for (int rb = blockIdx.x; rb * kIbpWarps * RW < n_out; rb += gridDim.x) {
  const int row0 = (rb * kIbpWarps + warp) * RW;
  float accC[RW][BT], accR[RW][BT];
#pragma unroll
  for (int i = 0; i < RW; ++i)
#pragma unroll
    for (int b = 0; b < BT; ++b) { accC[i][b] = 0.f; accR[i][b] = 0.f; }

  for (int k0 = 0; k0 < n_in; k0 += KC) {
    const int kc = min(KC, n_in - k0);
    if (!single) { __syncthreads(); stage(k0, kc); __syncthreads(); }
    if (vec) {
      // 4 strips of 128 columns per iteration: 4 * RW loads are issued before the first FMA needs one
      for (int j0 = lane * 4; j0 < kc; j0 += 512) {
        float4 w[4][RW];
#pragma unroll
        for (int u = 0; u < 4; ++u)
#pragma unroll
          for (int i = 0; i < RW; ++i) {
            const int row = row0 + i, j = j0 + u * 128;
            w[u][i] = (row < n_out && j < kc) ? ldg_stream4(W + (long long)row * n_in + k0 + j) : make_float4(0, 0, 0, 0);
          }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          const int j = j0 + u * 128;
          if (j >= kc) break;
#pragma unroll
          for (int b = 0; b < BT; ++b) {
            float4 c = *reinterpret_cast<const float4*>(&sc[b * KC + j]);
            float4 r = *reinterpret_cast<const float4*>(&sr[b * KC + j]);
#pragma unroll
            for (int i = 0; i < RW; ++i) {
              accC[i][b] = fmaf(w[u][i].x, c.x, accC[i][b]);
              accC[i][b] = fmaf(w[u][i].y, c.y, accC[i][b]);
              accC[i][b] = fmaf(w[u][i].z, c.z, accC[i][b]);
              accC[i][b] = fmaf(w[u][i].w, c.w, accC[i][b]);
              accR[i][b] = fmaf(fabsf(w[u][i].x), r.x, accR[i][b]);
              accR[i][b] = fmaf(fabsf(w[u][i].y), r.y, accR[i][b]);
              accR[i][b] = fmaf(fabsf(w[u][i].z), r.z, accR[i][b]);
              accR[i][b] = fmaf(fabsf(w[u][i].w), r.w, accR[i][b]);
            }
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
            accC[i][b] = fmaf(w, sc[b * KC + j], accC[i][b]);
            accR[i][b] = fmaf(fabsf(w), sr[b * KC + j], accR[i][b]);
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
  }   // row groups
}

template <int BT, int RW>
static void ibp_launch(const float* W, const float* bias, const float* l_in, const float* u_in, int relu_in,
                       float* l_out, float* u_out, int B, int n_out, int n_in, int ldo, cudaStream_t s) {
  int KC = (n_in + 511) / 512 * 512;
  const int kc_max = kIbpSmemMax / (2 * BT * 4) / 512 * 512;
  if (KC > kc_max) KC = kc_max;
  const size_t smem = (size_t)2 * BT * KC * 4;
  int gx = ceil_div(n_out, kIbpWarps * RW);
  if (KC >= n_in) {                                // persistent: stage c/r once per block, then stream row groups
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int per = ceil_div(sms, ceil_div(B, BT));
    if (gx > per) gx = per;
  }
  dim3 grid(gx, ceil_div(B, BT));
  ibp_linear_kernel<BT, RW><<<grid, kIbpWarps * 32, smem, s>>>(W, bias, l_in, u_in, relu_in, l_out, u_out, B, n_out, n_in, ldo, KC);
}

int ibp_init_device() {
  cudaError_t e1 = cudaFuncSetAttribute(ibp_linear_kernel<1, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize, kIbpSmemMax);
  cudaError_t e2 = cudaFuncSetAttribute(ibp_linear_kernel<2, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize, kIbpSmemMax);
  cudaError_t e3 = cudaFuncSetAttribute(ibp_linear_kernel<4, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize, kIbpSmemMax);
  return (e1 == cudaSuccess && e2 == cudaSuccess && e3 == cudaSuccess) ? 0 : -1;
}

void launch_ibp_linear(const float* W, const float* bias, const float* l_in, const float* u_in,
                       int relu_in, float* l_out, float* u_out, int B, int n_out, int n_in, int ldo,
                       cudaStream_t s) {
  if (B <= 0 || n_out <= 0) return;
  if (B <= 1) ibp_launch<1, 4>(W, bias, l_in, u_in, relu_in, l_out, u_out, B, n_out, n_in, ldo, s);
  else if (B <= 2) ibp_launch<2, 4>(W, bias, l_in, u_in, relu_in, l_out, u_out, B, n_out, n_in, ldo, s);
  else if (B <= 4) ibp_launch<4, 4>(W, bias, l_in, u_in, relu_in, l_out, u_out, B, n_out, n_in, ldo, s);
  else ibp_launch<4, 4>(W, bias, l_in, u_in, relu_in, l_out, u_out, B, n_out, n_in, ldo, s);   // W re-read per 4 properties
}

}  // namespace crownb200
