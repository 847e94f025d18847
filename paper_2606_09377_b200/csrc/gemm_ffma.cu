// a5 (fallback) -- plain fp32 contraction D[M,N] = A[M,K] . W[K,N] on the CUDA cores.
// Used where tensor-core tiles would be mostly padding or TMA cannot address the operand
// (K = 10 / 100 spec rows, tiny test networks, K % 4 != 0) and as the on-device cross-check of the
// tcgen05 kernel.  64x64x16 tiles, 256 threads, 4x4 outputs per thread, every access bounds-checked.
#include "common.cuh"
#include "kernels.h"

namespace crownb200 {

constexpr int FBM = 64, FBN = 64, FBK = 16;

__global__ void __launch_bounds__(256)
gemm_ffma_kernel(const float* __restrict__ A, long long lda, const float* __restrict__ W, long long ldw,
                 float* __restrict__ D, long long ldd, int M, int N, int K) {
  __shared__ float sA[FBK][FBM + 4];   // transposed: sA[k][m]
  __shared__ float sW[FBK][FBN + 4];
  const int tid = threadIdx.x;
  const int tx = tid % 16, ty = tid / 16;       // 16 x 16 threads, 4x4 each
  const int m0 = blockIdx.y * FBM, n0 = blockIdx.x * FBN;
  float acc[4][4];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j] = 0.f;

  for (int k0 = 0; k0 < K; k0 += FBK) {
    // A tile: 64 x 16 -> 1024 elements, 4 per thread; k fastest for coalescing
#pragma unroll
    for (int t = 0; t < 4; ++t) {
      int idx = tid + t * 256;
      int mm = idx / FBK, kk = idx % FBK;
      int gm = m0 + mm, gk = k0 + kk;
      sA[kk][mm] = (gm < M && gk < K) ? A[(long long)gm * lda + gk] : 0.f;
    }
    // W tile: 16 x 64, n fastest
#pragma unroll
    for (int t = 0; t < 4; ++t) {
      int idx = tid + t * 256;
      int kk = idx / FBN, nn = idx % FBN;
      int gk = k0 + kk, gn = n0 + nn;
      sW[kk][nn] = (gk < K && gn < N) ? W[(long long)gk * ldw + gn] : 0.f;
    }
    __syncthreads();
#pragma unroll
    for (int kk = 0; kk < FBK; ++kk) {
      float a[4], w[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) a[i] = sA[kk][ty * 4 + i];
#pragma unroll
      for (int j = 0; j < 4; ++j) w[j] = sW[kk][tx * 4 + j];
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(a[i], w[j], acc[i][j]);
    }
    __syncthreads();
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    int gm = m0 + ty * 4 + i;
    if (gm >= M) continue;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      int gn = n0 + tx * 4 + j;
      if (gn < N) D[(long long)gm * ldd + gn] = acc[i][j];
    }
  }
}

void launch_gemm_ffma(const float* A, long long lda, const float* W, long long ldw, float* D,
                      long long ldd, int M, int N, int K, cudaStream_t s) {
  if (M <= 0 || N <= 0) return;
  dim3 grid(ceil_div(N, FBN), ceil_div(M, FBM));
  gemm_ffma_kernel<<<grid, 256, 0, s>>>(A, lda, W, ldw, D, ldd, M, N, K);
}

}  // namespace crownb200
