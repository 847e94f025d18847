// a2 / a6 -- Conv2d steps of the hot path; a conv layer is linear, so IBP uses the
// conv itself in centre/radius form and the CROWN backward recursion uses its transpose
// (PAPER.md:144, :289).  Channel counts here are 3..64 and maps are 8..32 wide: tensor-core tiles would be
// mostly padding, the work is L2/HBM-bound, so these are CUDA-core gather kernels with the (tiny) filter
// bank staged in shared memory and the spatial index fastest across a warp (coalesced A reads/writes).
#include "common.cuh"
#include "kernels.h"

namespace crownb200 {

// ---- a2: IBP through Conv2d.  c' = conv(c, W) + b, r' = conv(r, |W|);  l' = c' - r', u' = c' + r'.
// grid: (spatial tiles, c_out, B); one thread per output pixel of one output channel.
__global__ void __launch_bounds__(256)
ibp_conv_kernel(const float* __restrict__ W, const float* __restrict__ bias, const float* __restrict__ l_in,
                const float* __restrict__ u_in, int relu_in, float* __restrict__ l_out,
                float* __restrict__ u_out, int c_in, int h, int w, int c_out, int kh, int kw, int stride,
                int pad, int ho, int wo) {
  extern __shared__ float sw[];   // [c_in*kh*kw] filter of this output channel
  const int co = blockIdx.y, b = blockIdx.z;
  const int fsz = c_in * kh * kw;
  for (int i = threadIdx.x; i < fsz; i += blockDim.x) sw[i] = W[(long long)co * fsz + i];
  __syncthreads();
  const int pix = blockIdx.x * blockDim.x + threadIdx.x;
  if (pix >= ho * wo) return;
  const int p = pix / wo, q = pix % wo;
  const float* lb = l_in + (long long)b * c_in * h * w;
  const float* ub = u_in + (long long)b * c_in * h * w;
  float c = 0.f, r = 0.f;
  for (int ci = 0; ci < c_in; ++ci)
    for (int i = 0; i < kh; ++i) {
      const int y = p * stride + i - pad;
      if (y < 0 || y >= h) continue;
      for (int j = 0; j < kw; ++j) {
        const int x = q * stride + j - pad;
        if (x < 0 || x >= w) continue;
        float lo = lb[(ci * h + y) * w + x], hi = ub[(ci * h + y) * w + x];
        if (relu_in) { lo = fmaxf(lo, 0.f); hi = fmaxf(hi, 0.f); }
        const float wv = sw[(ci * kh + i) * kw + j];
        c = fmaf(wv, 0.5f * (lo + hi), c);
        r = fmaf(fabsf(wv), 0.5f * (hi - lo), r);
      }
    }
  c += bias ? bias[co] : 0.f;
  const long long o = ((long long)b * c_out + co) * ho * wo + pix;
  l_out[o] = c - r;
  u_out[o] = c + r;
}

void launch_ibp_conv(const float* W, const float* bias, const float* l_in, const float* u_in, int relu_in,
                     float* l_out, float* u_out, int B, int c_in, int h, int w, int c_out, int kh, int kw,
                     int stride, int pad, int ho, int wo, cudaStream_t s) {
  if (B <= 0) return;
  int threads = 256;
  while (threads > 32 && threads / 2 >= ho * wo) threads /= 2;
  dim3 grid(ceil_div(ho * wo, threads), c_out, B);
  size_t smem = (size_t)c_in * kh * kw * sizeof(float);
  ibp_conv_kernel<<<grid, threads, smem, s>>>(W, bias, l_in, u_in, relu_in, l_out, u_out, c_in, h, w, c_out,
                                              kh, kw, stride, pad, ho, wo);
}

// ---- a6: A_in = conv^T(A_out, W) (+ addend: the other incoming A of a residual fork).
// A_in[m, ci, y, x] = sum_{co,i,j : y = p*stride + i - pad, x = q*stride + j - pad} W[co,ci,i,j] * A_out[m,co,p,q].
// grid: (spatial tiles, c_in, rows); the filter slice W[:, ci, :, :] sits in shared memory.
__global__ void __launch_bounds__(256)
conv_transpose_kernel(const float* __restrict__ A, long long sBr, long long sB, long long ld, int B, int R,
                      const float* __restrict__ W, const float* __restrict__ addend, float* __restrict__ out,
                      int c_in, int h, int w, int c_out, int kh, int kw, int stride, int pad, int ho, int wo) {
  extern __shared__ float sw[];   // [c_out*kh*kw]
  const int ci = blockIdx.y;
  const int ksz = kh * kw;
  for (int i = threadIdx.x; i < c_out * ksz; i += blockDim.x) {
    const int co = i / ksz, k = i % ksz;
    sw[i] = W[((long long)co * c_in + ci) * ksz + k];
  }
  __syncthreads();
  const int pix = blockIdx.x * blockDim.x + threadIdx.x;
  if (pix >= h * w) return;
  const int y = pix / w, x = pix % w;
  for (long long m = blockIdx.z; m < 2LL * B * R; m += gridDim.z) {
    const int r = (int)(m % R);
    const long long t = m / R;
    const int b = (int)(t % B), br = (int)(t / B);
    const float* a = A + br * sBr + b * sB + (long long)r * ld;
    float acc = 0.f;
    for (int i = 0; i < kh; ++i) {
      const int py = y + pad - i;
      if (py < 0 || py % stride) continue;
      const int p = py / stride;
      if (p >= ho) continue;
      for (int j = 0; j < kw; ++j) {
        const int qx = x + pad - j;
        if (qx < 0 || qx % stride) continue;
        const int q = qx / stride;
        if (q >= wo) continue;
        const float* ap = a + p * wo + q;
        const float* wp = sw + i * kw + j;
        for (int co = 0; co < c_out; ++co) acc = fmaf(wp[co * ksz], ap[(long long)co * ho * wo], acc);
      }
    }
    const long long o = (m * c_in + ci) * (long long)(h * w) + pix;
    out[o] = addend ? acc + addend[o] : acc;
  }
}

void launch_conv_transpose(const AView& A, const float* W, const float* addend, float* out, int B, int R,
                           int c_in, int h, int w, int c_out, int kh, int kw, int stride, int pad, int ho,
                           int wo, cudaStream_t s) {
  long long rows = 2LL * B * R;
  if (rows <= 0) return;
  int threads = 256;
  while (threads > 32 && threads / 2 >= h * w) threads /= 2;
  dim3 grid(ceil_div(h * w, threads), c_in, (unsigned)(rows < 32768 ? rows : 32768));
  size_t smem = (size_t)c_out * kh * kw * sizeof(float);
  conv_transpose_kernel<<<grid, threads, smem, s>>>(A.p, A.sBr, A.sB, A.ld, B, R, W, addend, out, c_in, h, w,
                                                    c_out, kh, kw, stride, pad, ho, wo);
}

}  // namespace crownb200
