// NEXT-1 -- alpha optimisation of alpha-CROWN ("gradient ascent over alpha tightens the lower bound (or
// lowers the upper bound)"; alpha tensors [layers x specs x batch x neurons]).
//
// The derivative of the final bound with respect to the slopes is the transpose of the backward pass O3 (DESIGN.md
// sec. 11): with G_i = d bound / d A_i (one vector per (branch, property, spec row)),
//   input   : G = x_c -/+ sign(A_0) * x_r                    (the corner of the box that attains the bound)
//   Linear i: G_i = G_in . W_i^T + b_i      Conv i: G_i = conv(G_in, W_i) + b_i      Add: G_i = G_a + G_b
//   ReLU   i: lower  G_i = [A_i>0] dL G_in + [A_i<0] (dU G_in + bU),   d lb / d alpha_i = A_i^+ * G_in  (unstable only)
//             upper  G_i = [A_i>0] (dU G_in + bU) + [A_i<0] dL G_in,   d ub / d alpha_i = A_i^- * G_in
// i.e. a forward sweep of 2*B*S "points" through the network, every ReLU replaced by the line the sign of the saved
// A_i selects.  Kernels of that sweep; the host side is in backward.cu (crown_alpha_grad / crown_alpha_ascent).
#include "common.cuh"
#include "kernels.h"

namespace crownb200 {

// ---- corner of the box: G[br,b,s,:] = x_c - sign(A0[0,b,s,:]) x_r (br 0), x_c + sign(A0[1,b,s,:]) x_r (br 1) -------
__global__ void __launch_bounds__(256)
alpha_corner_kernel(const float* __restrict__ A0, const float* __restrict__ x_lo, const float* __restrict__ x_hi,
                    float* __restrict__ G, int B, int S, int n0) {
  const long long per_br = (long long)B * S * n0;
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= 2 * per_br) return;
  const int br = (int)(i / per_br);
  const long long r = i % per_br;
  const int b = (int)(r / ((long long)S * n0)), j = (int)(r % n0);
  const float lo = x_lo[(long long)b * n0 + j], hi = x_hi[(long long)b * n0 + j];
  const float xc = 0.5f * (lo + hi), xr = 0.5f * (hi - lo);
  const float a = A0[i];
  const float sg = a > 0.f ? 1.f : (a < 0.f ? -1.f : 0.f);        // one-sided derivative 0 at the kink (reading G23)
  G[i] = br == 0 ? xc - sg * xr : xc + sg * xr;
}

// the same, one block per (branch, property, spec) row and four columns per thread: no 64-bit division per element (the scalar
// kernel above spends ~100 instructions per element on them: 287 us for the 231 MB of cfg2's 4096 sub-domains).  G_lo != nullptr:
// G / G_lo receive the TF32 limbs of the corner (the operand of the first Linear's contraction, no split pass).
__global__ void __launch_bounds__(256)
alpha_corner_rows_kernel(const float* __restrict__ A0, const float* __restrict__ x_lo, const float* __restrict__ x_hi,
                         float* __restrict__ G, float* __restrict__ G_lo, int B, int S, int n0) {
  const long long row = blockIdx.x;                      // (br * B + b) * S + s
  const int br = (int)(row / ((long long)B * S));
  const int b = (int)((row / S) % B);
  const float4* l4 = reinterpret_cast<const float4*>(x_lo + (long long)b * n0);
  const float4* h4 = reinterpret_cast<const float4*>(x_hi + (long long)b * n0);
  float4* g4 = reinterpret_cast<float4*>(G + row * n0);
  float4* gl4 = G_lo ? reinterpret_cast<float4*>(G_lo + row * n0) : nullptr;
  const float sgn = br == 0 ? -1.f : 1.f;
  for (int j = threadIdx.x; j < (n0 >> 2); j += blockDim.x) {
    const float4 a = ldg_stream4(A0 + row * n0 + 4 * j), lo = __ldg(l4 + j), hi = __ldg(h4 + j);
    float4 g;
    // x_c -/+ sign(a) x_r; sign(0) = 0: one-sided derivative 0 at the kink (reading G23)
    g.x = fmaf(sgn * (a.x > 0.f ? 1.f : (a.x < 0.f ? -1.f : 0.f)), 0.5f * (hi.x - lo.x), 0.5f * (lo.x + hi.x));
    g.y = fmaf(sgn * (a.y > 0.f ? 1.f : (a.y < 0.f ? -1.f : 0.f)), 0.5f * (hi.y - lo.y), 0.5f * (lo.y + hi.y));
    g.z = fmaf(sgn * (a.z > 0.f ? 1.f : (a.z < 0.f ? -1.f : 0.f)), 0.5f * (hi.z - lo.z), 0.5f * (lo.z + hi.z));
    g.w = fmaf(sgn * (a.w > 0.f ? 1.f : (a.w < 0.f ? -1.f : 0.f)), 0.5f * (hi.w - lo.w), 0.5f * (lo.w + hi.w));
    if (gl4) {
      float4 h, l;
      tf32_split(g.x, h.x, l.x); tf32_split(g.y, h.y, l.y); tf32_split(g.z, h.z, l.z); tf32_split(g.w, h.w, l.w);
      g4[j] = h; gl4[j] = l;
    } else {
      g4[j] = g;
    }
  }
}

void launch_alpha_corner(const float* A0, const float* x_lo, const float* x_hi, float* G, int B, int S, int n0,
                         cudaStream_t s, float* G_lo) {
  const long long cnt = 2LL * B * S * n0;
  if (cnt <= 0) return;
  auto mis = [](const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15) != 0; };
  if ((n0 & 3) == 0 && !mis(A0) && !mis(x_lo) && !mis(x_hi) && !mis(G) && !(G_lo && mis(G_lo))) {
    alpha_corner_rows_kernel<<<(unsigned)(2LL * B * S), 256, 0, s>>>(A0, x_lo, x_hi, G, G_lo, B, S, n0);
    return;
  }
  // G_lo is only offered by the caller when the vector path applies (alpha_corner_limbs_ok)
  alpha_corner_kernel<<<ceil_div(cnt, 256), 256, 0, s>>>(A0, x_lo, x_hi, G, B, S, n0);
}

bool alpha_corner_limbs_ok(const float* A0, const float* x_lo, const float* x_hi, const float* G, const float* G_lo, int n0) {
  auto mis = [](const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15) != 0; };
  return (n0 & 3) == 0 && !mis(A0) && !mis(x_lo) && !mis(x_hi) && !mis(G) && !mis(G_lo);
}

// ---- Linear: D[M,N] = G[M,K] . W[N,K]^T + bias[N]  (W row-major [n_out, n_in] as the network stores it) ------------
// CUDA-core FFMA, 64x64x16 tiles, 256 threads x (4x4) outputs, both operands K-contiguous (128-bit loads when K % 4 == 0).
constexpr int ABM = 64, ABN = 64, ABK = 16;

template <bool VEC>
__global__ void __launch_bounds__(256)
alpha_linear_kernel(const float* __restrict__ G, const float* __restrict__ W, const float* __restrict__ bias,
                    float* __restrict__ D, int M, int N, int K) {
  __shared__ float sG[ABK][ABM + 4];   // [k][m]
  __shared__ float sW[ABK][ABN + 4];   // [k][n]
  const int tid = threadIdx.x;
  const int tx = tid % 16, ty = tid / 16;
  const int m0 = blockIdx.y * ABM, n0 = blockIdx.x * ABN;
  float acc[4][4];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j] = 0.f;
  const int lr = tid / 4, lk = (tid % 4) * 4;    // this thread's row of the tile and first k of its 4
  for (int k0 = 0; k0 < K; k0 += ABK) {
    const int gk = k0 + lk;
    float4 g = make_float4(0.f, 0.f, 0.f, 0.f), w = g;
    const int gm = m0 + lr, gn = n0 + lr;
    if (VEC) {
      if (gm < M && gk < K) g = *reinterpret_cast<const float4*>(G + (long long)gm * K + gk);
      if (gn < N && gk < K) w = __ldg(reinterpret_cast<const float4*>(W + (long long)gn * K + gk));
    } else {
      if (gm < M) {
        const float* q = G + (long long)gm * K;
        g.x = gk < K ? q[gk] : 0.f; g.y = gk + 1 < K ? q[gk + 1] : 0.f; g.z = gk + 2 < K ? q[gk + 2] : 0.f; g.w = gk + 3 < K ? q[gk + 3] : 0.f;
      }
      if (gn < N) {
        const float* q = W + (long long)gn * K;
        w.x = gk < K ? q[gk] : 0.f; w.y = gk + 1 < K ? q[gk + 1] : 0.f; w.z = gk + 2 < K ? q[gk + 2] : 0.f; w.w = gk + 3 < K ? q[gk + 3] : 0.f;
      }
    }
    sG[lk][lr] = g.x; sG[lk + 1][lr] = g.y; sG[lk + 2][lr] = g.z; sG[lk + 3][lr] = g.w;
    sW[lk][lr] = w.x; sW[lk + 1][lr] = w.y; sW[lk + 2][lr] = w.z; sW[lk + 3][lr] = w.w;
    __syncthreads();
#pragma unroll
    for (int kk = 0; kk < ABK; ++kk) {
      const float4 a = *reinterpret_cast<const float4*>(&sG[kk][ty * 4]);
      const float4 b = *reinterpret_cast<const float4*>(&sW[kk][tx * 4]);
      const float av[4] = {a.x, a.y, a.z, a.w}, bv[4] = {b.x, b.y, b.z, b.w};
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(av[i], bv[j], acc[i][j]);
    }
    __syncthreads();
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int gm = m0 + ty * 4 + i;
    if (gm >= M) continue;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int gn = n0 + tx * 4 + j;
      if (gn < N) D[(long long)gm * N + gn] = acc[i][j] + (bias ? __ldg(bias + gn) : 0.f);
    }
  }
}

void launch_alpha_linear(const float* G, const float* W, const float* bias, float* D, int M, int N, int K,
                         cudaStream_t s) {
  if (M <= 0 || N <= 0) return;
  dim3 grid(ceil_div(N, ABN), ceil_div(M, ABM));
  const bool vec = (K % 4 == 0) && ((reinterpret_cast<uintptr_t>(G) | reinterpret_cast<uintptr_t>(W)) & 15) == 0;
  if (vec) alpha_linear_kernel<true><<<grid, 256, 0, s>>>(G, W, bias, D, M, N, K);
  else alpha_linear_kernel<false><<<grid, 256, 0, s>>>(G, W, bias, D, M, N, K);
}

// ---- Conv2d forward of points: out[m, co, p, q] = bias[co] + sum W[co,ci,i,j] * in[m, ci, p*s+i-pad, q*s+j-pad] -----
// one thread per output pixel of four output channels (the gather of ibp_conv_kernel without the radius half)
constexpr int kPtConvCO = 4;
__global__ void __launch_bounds__(256)
alpha_conv_kernel(const float* __restrict__ W, const float* __restrict__ bias, const float* __restrict__ in,
                  float* __restrict__ out, int c_in, int h, int w, int c_out, int kh, int kw, int stride, int pad,
                  int ho, int wo) {
  extern __shared__ float sw[];   // [kPtConvCO][c_in*kh*kw]
  const int co0 = blockIdx.y * kPtConvCO;
  const long long m = blockIdx.z;
  const int fsz = c_in * kh * kw;
  for (int i = threadIdx.x; i < kPtConvCO * fsz; i += blockDim.x) {
    const int o = i / fsz, k = i % fsz;
    sw[i] = (co0 + o < c_out) ? W[(long long)(co0 + o) * fsz + k] : 0.f;
  }
  __syncthreads();
  const int pix = blockIdx.x * blockDim.x + threadIdx.x;
  if (pix >= ho * wo) return;
  const int p = pix / wo, q = pix % wo;
  const float* src = in + m * c_in * h * w;
  float c[kPtConvCO];
#pragma unroll
  for (int o = 0; o < kPtConvCO; ++o) c[o] = 0.f;
  for (int ci = 0; ci < c_in; ++ci)
    for (int i = 0; i < kh; ++i) {
      const int y = p * stride + i - pad;
      if (y < 0 || y >= h) continue;
      for (int j = 0; j < kw; ++j) {
        const int x = q * stride + j - pad;
        if (x < 0 || x >= w) continue;
        const float v = src[(ci * h + y) * w + x];
        const int k = (ci * kh + i) * kw + j;
#pragma unroll
        for (int o = 0; o < kPtConvCO; ++o) c[o] = fmaf(sw[o * fsz + k], v, c[o]);
      }
    }
#pragma unroll
  for (int o = 0; o < kPtConvCO; ++o) {
    const int co = co0 + o;
    if (co >= c_out) break;
    out[(m * c_out + co) * ho * wo + pix] = c[o] + (bias ? bias[co] : 0.f);
  }
}

void launch_alpha_conv(const float* W, const float* bias, const float* in, float* out, long long M, int c_in, int h,
                       int w, int c_out, int kh, int kw, int stride, int pad, int ho, int wo, cudaStream_t s) {
  if (M <= 0) return;
  int threads = 256;
  while (threads > 32 && threads / 2 >= ho * wo) threads /= 2;
  const size_t smem = (size_t)kPtConvCO * c_in * kh * kw * sizeof(float);
  for (long long m0 = 0; m0 < M; m0 += 65535) {       // gridDim.z limit
    const long long mz = M - m0 < 65535 ? M - m0 : 65535;
    dim3 grid(ceil_div(ho * wo, threads), ceil_div(c_out, kPtConvCO), (unsigned)mz);
    alpha_conv_kernel<<<grid, threads, smem, s>>>(W, bias, in + m0 * c_in * h * w, out + m0 * c_out * ho * wo, c_in, h,
                                                  w, c_out, kh, kw, stride, pad, ho, wo);
  }
}

// ---- Add: G = Ga + Gb ---------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
alpha_add_kernel(const float* __restrict__ a, const float* __restrict__ b, float* __restrict__ o, long long cnt) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < cnt) o[i] = a[i] + b[i];
}
void launch_alpha_add(const float* a, const float* b, float* o, long long cnt, cudaStream_t s) {
  if (cnt <= 0) return;
  alpha_add_kernel<<<ceil_div(cnt, 256), 256, 0, s>>>(a, b, o, cnt);
}

__global__ void __launch_bounds__(256) add_bias_rows_kernel(float* __restrict__ D, const float* __restrict__ bias, long long cnt, int N) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < cnt) D[i] += __ldg(bias + (int)(i % N));
}
void launch_add_bias_rows(float* D, const float* bias, long long M, int N, cudaStream_t s) {
  const long long cnt = M * N;
  if (cnt <= 0) return;
  add_bias_rows_kernel<<<ceil_div(cnt, 256), 256, 0, s>>>(D, bias, cnt, N);
}

__global__ void __launch_bounds__(256) add_bias_div_kernel(float* __restrict__ D, const float* __restrict__ bias, long long cnt, int N, int div) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < cnt) D[i] += __ldg(bias + (int)((i / div) % N));
}
void launch_add_bias_div(float* D, const float* bias, long long cnt, int N, int div, cudaStream_t s) {
  if (cnt <= 0) return;
  add_bias_div_kernel<<<ceil_div(cnt, 256), 256, 0, s>>>(D, bias, cnt, N, div);
}

// ---- ReLU: forward value through the selected line, gradient w.r.t. alpha, optional in-place projected step ---------
// element (b, s, j) for both branches.  A, Gin, Gout: [2, B, S, n]; coef [B, n] {dU, bU, dL_fixed, unstable};
// alpha_lo / alpha_up [B, S, n].  step != nullptr: alpha <- clip(clip(alpha) +/- step[0] * dir(g), 0, 1) with
// dir = g (mode 0, "plain") or sign(g) (mode 1, "sign"); else g_lo / g_up receive the gradients (may be nullptr).
__device__ __forceinline__ float clip01f(float a) { return fminf(fmaxf(a, 0.f), 1.f); }
__device__ __forceinline__ float sgnf(float a) { return a > 0.f ? 1.f : (a < 0.f ? -1.f : 0.f); }

__global__ void __launch_bounds__(256)
alpha_relu_kernel(const float* __restrict__ A, const float* __restrict__ Gin, const float4* __restrict__ coef,
                  float* alpha_lo, float* alpha_up, float* __restrict__ Gout, float* __restrict__ g_lo,
                  float* __restrict__ g_up, const float* __restrict__ step, int mode, int B, int S, int n,
                  const int8_t* __restrict__ split, float* beta_lo, float* beta_up, float* __restrict__ gb_lo,
                  float* __restrict__ gb_up, const float* __restrict__ gin_bias, float* __restrict__ Gout_lo) {
  const long long per_br = (long long)B * S * n;
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= per_br) return;
  const int b = (int)(i / ((long long)S * n)), j = (int)(i % n);
  const float4 c = __ldg(coef + (long long)b * n + j);
  const bool unstable = c.w != 0.f;
  const float aL = A[i], aU = A[per_br + i];
  // gin_bias: the bias of the Linear that produced Gin, added here instead of in a pass of its own over Gin
  const float gb = gin_bias ? __ldg(gin_bias + j) : 0.f;
  const float gL = Gin[i] + gb, gU = Gin[per_br + i] + gb;
  const float alL = alpha_lo[i], alU = alpha_up[i];
  const float sL = unstable ? clip01f(alL) : c.z, sU = unstable ? clip01f(alU) : c.z;
  const float dU = c.x, bU = c.y;
  const float oL = aL > 0.f ? sL * gL : (aL < 0.f ? fmaf(dU, gL, bU) : 0.f);
  const float oU = aU > 0.f ? fmaf(dU, gU, bU) : (aU < 0.f ? sU * gU : 0.f);
  if (Gout_lo) {        // the only consumer is a tensor-core Linear: its operand limbs are written here (no split pass)
    float h, l;
    tf32_split(oL, h, l); Gout[i] = h; Gout_lo[i] = l;
    tf32_split(oU, h, l); Gout[per_br + i] = h; Gout_lo[per_br + i] = l;
  } else {
    Gout[i] = oL;
    Gout[per_br + i] = oU;
  }
  const float dl = unstable ? fmaxf(aL, 0.f) * gL : 0.f;
  const float du = unstable ? fminf(aU, 0.f) * gU : 0.f;
  if (step) {
    const float eta = step[0];
    alpha_lo[i] = clip01f(clip01f(alL) + eta * (mode ? sgnf(dl) : dl));      // ascent on lb
    alpha_up[i] = clip01f(clip01f(alU) - eta * (mode ? sgnf(du) : du));      // descent on ub
  } else {
    if (g_lo) g_lo[i] = dl;
    if (g_up) g_up[i] = du;
  }
  if (split) {
    // NEXT-2 (reading G28): the split term -beta_lo * s (lower) / +beta_up * s (upper) is added to A w.r.t. this ReLU's
    // INPUT, whose derivative is Gin: d lb / d beta_lo = -s * Gin, d ub / d beta_up = +s * Gin
    const float sg = (float)split[(long long)b * n + j];
    const float bl = -sg * gL, bu = sg * gU;
    if (step) {
      const float eb = step[1];
      if (beta_lo) beta_lo[i] = fmaxf(fmaxf(beta_lo[i], 0.f) + eb * (mode ? sgnf(bl) : bl), 0.f);    // ascent on lb
      if (beta_up) beta_up[i] = fmaxf(fmaxf(beta_up[i], 0.f) - eb * (mode ? sgnf(bu) : bu), 0.f);    // descent on ub
    } else {
      if (gb_lo) gb_lo[i] = bl;
      if (gb_up) gb_up[i] = bu;
    }
  }
}

void launch_alpha_relu(const float* A, const float* Gin, const float4* coef, float* alpha_lo, float* alpha_up,
                       float* Gout, float* g_lo, float* g_up, const float* step, int mode, int B, int S, int n,
                       cudaStream_t s, const int8_t* split, float* beta_lo, float* beta_up, float* gb_lo, float* gb_up,
                       const float* gin_bias, float* Gout_lo) {
  const long long cnt = (long long)B * S * n;
  if (cnt <= 0) return;
  alpha_relu_kernel<<<ceil_div(cnt, 256), 256, 0, s>>>(A, Gin, coef, alpha_lo, alpha_up, Gout, g_lo, g_up, step, mode,
                                                      B, S, n, split, beta_lo, beta_up, gb_lo, gb_up, gin_bias, Gout_lo);
}

// ---- best-so-far bounds over the iterates (every iterate is sound): lb_best = max, ub_best = min; the step size
// decays for the next iteration.  first != 0: initialise instead of combine.
__global__ void __launch_bounds__(256)
alpha_best_kernel(const float* __restrict__ lb, const float* __restrict__ ub, float* __restrict__ lb_best,
                  float* __restrict__ ub_best, float* step, float decay, int first, int count) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < count) {
    // NaN-propagating on purpose: fmaxf / fminf would drop a NaN iterate and keep the (finite) best
    const float l = lb[i], u = ub[i];
    lb_best[i] = first ? l : ((l > lb_best[i] || l != l) ? l : lb_best[i]);
    ub_best[i] = first ? u : ((u < ub_best[i] || u != u) ? u : ub_best[i]);
  }
  if (i == 0 && step && !first) { step[0] *= decay; step[1] *= decay; }
}

void launch_alpha_best(const float* lb, const float* ub, float* lb_best, float* ub_best, float* step, float decay,
                       int first, int count, cudaStream_t s) {
  if (count <= 0) return;
  alpha_best_kernel<<<ceil_div(count, 256), 256, 0, s>>>(lb, ub, lb_best, ub_best, step, decay, first, count);
}

__global__ void alpha_set_step_kernel(float* step, float v, float vb) { step[0] = v; step[1] = vb; }
void launch_alpha_set_step(float* step, float v, cudaStream_t s, float v_beta) { alpha_set_step_kernel<<<1, 1, 0, s>>>(step, v, v_beta); }

}  // namespace crownb200
