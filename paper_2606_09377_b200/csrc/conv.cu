// a2 / a6 -- Conv2d steps of the hot path; a conv layer is linear, so IBP uses the
// conv itself in centre/radius form and the CROWN backward recursion uses its transpose
// (PAPER.md:144, :289).  Channel counts here are 3..64 and maps are 8..32 wide: tensor-core tiles would be
// mostly padding, the work is L2/HBM-bound, so these are CUDA-core gather kernels with the (tiny) filter
// bank staged in shared memory and the spatial index fastest across a warp (coalesced A reads/writes).
#include "common.cuh"
#include "kernels.h"

namespace crownb200 {

// ---- a2: IBP through Conv2d.  c' = conv(c, W) + b, r' = conv(r, |W|);  l' = c' - r', u' = c' + r'.
// grid: (spatial tiles, c_out / 4, B); block: (PIX output pixels) x (CS slices of the input channels).  A thread owns
// one output pixel of FOUR output channels for its slice of input channels, so every (l, u) pair read from global
// memory feeds 8 FMAs and the dependent tap loop is c_in / CS * kh * kw long instead of c_in * kh * kw (the maps here
// are 8..32 wide with 3..64 channels and B = 8 images: the kernel is latency-bound, parallelism is what it lacks);
// the CS partial sums are added in slice order through shared memory (deterministic).
constexpr int kIbpConvCO = 4;
// KS > 0: square KS x KS filter known at compile time (the tap loops unroll, same order of operations); KS = 0: any kh x kw
template <int KS>
__global__ void __launch_bounds__(512)
ibp_conv_kernel(const float* __restrict__ W, const float* __restrict__ bias, const float* __restrict__ l_in,
                const float* __restrict__ u_in, int relu_in, float* __restrict__ l_out,
                float* __restrict__ u_out, int c_in, int h, int w, int c_out, int kh_, int kw_, int stride,
                int pad, int ho, int wo) {
  const int kh = KS > 0 ? KS : kh_, kw = KS > 0 ? KS : kw_;
  extern __shared__ float sw[];   // [kIbpConvCO][c_in*kh*kw] filters, then [CS][PIX][2*kIbpConvCO] partial sums
  const int co0 = blockIdx.y * kIbpConvCO, b = blockIdx.z;
  const int fsz = c_in * kh * kw;
  const int PIX = blockDim.x, CS = blockDim.y;
  const int tid = threadIdx.y * PIX + threadIdx.x, nthr = PIX * CS;
  float* red = sw + kIbpConvCO * fsz;
  for (int i = tid; i < kIbpConvCO * fsz; i += nthr) {
    const int o = i / fsz, k = i % fsz;
    sw[i] = (co0 + o < c_out) ? W[(long long)(co0 + o) * fsz + k] : 0.f;
  }
  __syncthreads();
  const int pix = blockIdx.x * PIX + threadIdx.x;
  const bool live = pix < ho * wo;
  const int p = live ? pix / wo : 0, q = live ? pix % wo : 0;
  const float* lb = l_in + (long long)b * c_in * h * w;
  const float* ub = u_in + (long long)b * c_in * h * w;
  float c[kIbpConvCO], r[kIbpConvCO];
#pragma unroll
  for (int o = 0; o < kIbpConvCO; ++o) { c[o] = 0.f; r[o] = 0.f; }
  if (live)
    for (int ci = threadIdx.y; ci < c_in; ci += CS)
#pragma unroll
      for (int i = 0; i < kh; ++i) {
        const int y = p * stride + i - pad;
        if (y < 0 || y >= h) continue;
#pragma unroll
        for (int j = 0; j < kw; ++j) {
          const int x = q * stride + j - pad;
          if (x < 0 || x >= w) continue;
          float lo = lb[(ci * h + y) * w + x], hi = ub[(ci * h + y) * w + x];
          if (relu_in) { lo = fmaxf(lo, 0.f); hi = fmaxf(hi, 0.f); }
          const float xc = 0.5f * (lo + hi), xr = 0.5f * (hi - lo);
          const int k = (ci * kh + i) * kw + j;
#pragma unroll
          for (int o = 0; o < kIbpConvCO; ++o) {
            const float wv = sw[o * fsz + k];
            c[o] = fmaf(wv, xc, c[o]);
            r[o] = fmaf(fabsf(wv), xr, r[o]);
          }
        }
      }
  if (CS > 1) {
    float* mine = red + ((size_t)threadIdx.y * PIX + threadIdx.x) * (2 * kIbpConvCO);
#pragma unroll
    for (int o = 0; o < kIbpConvCO; ++o) { mine[o] = c[o]; mine[kIbpConvCO + o] = r[o]; }
    __syncthreads();
    if (threadIdx.y != 0) return;
    for (int sl = 1; sl < CS; ++sl) {
      const float* oth = red + ((size_t)sl * PIX + threadIdx.x) * (2 * kIbpConvCO);
#pragma unroll
      for (int o = 0; o < kIbpConvCO; ++o) { c[o] += oth[o]; r[o] += oth[kIbpConvCO + o]; }
    }
  }
  if (!live) return;
#pragma unroll
  for (int o = 0; o < kIbpConvCO; ++o) {
    const int co = co0 + o;
    if (co >= c_out) break;
    const float cc = c[o] + (bias ? bias[co] : 0.f);
    const long long idx = ((long long)b * c_out + co) * ho * wo + pix;
    l_out[idx] = cc - r[o];
    u_out[idx] = cc + r[o];
  }
}

void launch_ibp_conv(const float* W, const float* bias, const float* l_in, const float* u_in, int relu_in,
                     float* l_out, float* u_out, int B, int c_in, int h, int w, int c_out, int kh, int kw,
                     int stride, int pad, int ho, int wo, cudaStream_t s) {
  if (B <= 0) return;
  int pix = 128;
  while (pix > 32 && pix / 2 >= ho * wo) pix /= 2;
  int cs = 1;
  while (cs < 8 && cs * 2 <= c_in && pix * cs * 2 <= 512) cs *= 2;
  dim3 grid(ceil_div(ho * wo, pix), ceil_div(c_out, kIbpConvCO), B), block(pix, cs);
  size_t smem = ((size_t)kIbpConvCO * c_in * kh * kw + (cs > 1 ? (size_t)cs * pix * 2 * kIbpConvCO : 0)) * sizeof(float);
  if (kh == 3 && kw == 3)
    ibp_conv_kernel<3><<<grid, block, smem, s>>>(W, bias, l_in, u_in, relu_in, l_out, u_out, c_in, h, w, c_out, kh, kw, stride, pad, ho, wo);
  else if (kh == 1 && kw == 1)
    ibp_conv_kernel<1><<<grid, block, smem, s>>>(W, bias, l_in, u_in, relu_in, l_out, u_out, c_in, h, w, c_out, kh, kw, stride, pad, ho, wo);
  else
    ibp_conv_kernel<0><<<grid, block, smem, s>>>(W, bias, l_in, u_in, relu_in, l_out, u_out, c_in, h, w, c_out, kh, kw, stride, pad, ho, wo);
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

// ---- a6, fast path: register-tiled gather.  Block = RB rows x CG input-channel groups x PT pixel threads.
// A thread owns 4 output pixels of ONE stride-parity class (same valid filter taps for all four, spaced XQ apart
// in the class's x index so that a warp reads consecutive shared-memory words and writes consecutive outputs)
// times CT input channels: 4*CT accumulators.  Per (co, tap): 4 LDS of A, CT/4 broadcast LDS.128 of W, 4*CT FFMA.
// A_out of the block's rows is staged, zero-haloed, in shared memory COC output channels at a time together
// with the filter slice transposed to [co][tap][ci] (ci fastest).  Staging is asynchronous (cp.async, 4-byte
// copies because the halo shifts alignment) and double-buffered: chunk c+1 is in flight while chunk c is
// multiplied.  Each thread precomputes once which tile elements it copies (the tile geometry is the same for
// every (row, co)), so the copy loop has no divisions.
struct ConvBwdGeom {
  int c_in, h, w, c_out, ho, wo, pad;
  int NY, NX, XQ, PT, CG, RB, COC;      // per-class rows / cols / x-quads, thread split, co chunk
  int omin_y, omin_x, PH, PW;           // shared-memory tile origin and size
  int stage_floats;                     // floats per pipeline stage (filters + A tiles)
};

constexpr int kConvFillMax = 6;
constexpr size_t kConvBwdSmemBudget = 96 * 1024;         // tile elements per thread (tile <= 6 * blockDim)

__device__ __forceinline__ void cp_async4(float* dst_smem, const float* src) {
  const uint32_t d = static_cast<uint32_t>(__cvta_generic_to_shared(dst_smem));
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" :: "r"(d), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" :: "n"(N) : "memory"); }

template <int KH, int KW, int S, int CT>
__global__ void __launch_bounds__(256, 2)
conv_bwd_tiled_kernel(const float* __restrict__ A, long long sBr, long long sB, long long ld, int B, int R,
                      const float* __restrict__ W, const float* __restrict__ addend, float* __restrict__ out,
                      ConvBwdGeom g) {
  extern __shared__ __align__(16) float smem_f[];
  __shared__ const float* rowp[4];
  constexpr int KK = KH * KW;
  const int cgct = g.CG * CT;
  const int w_floats = g.COC * KK * cgct;              // stage layout: Ws [COC][KK][cgct], then As [RB][COC][PH][PW]
  const int tid = threadIdx.x;
  const int nthreads = g.PT * g.CG * g.RB;
  const int pt = tid % g.PT, cg = (tid / g.PT) % g.CG, rb = tid / (g.PT * g.CG);
  const long long rows = 2LL * B * R;
  const long long m_base = (long long)blockIdx.x * g.RB;
  const int ci_base = blockIdx.y * cgct;
  const int tile = g.PH * g.PW;
  // pixel thread -> (parity class, yy, xq)
  const int per_class = g.NY * g.XQ;
  const int cls = pt / per_class, rem = pt % per_class;
  const int cy = cls / S, cx = cls % S;
  const int yy = rem / g.XQ, xq = rem % g.XQ;
  const int y = cy + S * yy;
  const bool active = tid < nthreads;

  if (tid < g.RB) {
    const long long m = m_base + tid;
    const float* ptr = nullptr;
    if (m < rows) {
      const int r = (int)(m % R);
      const long long tt = m / R;
      ptr = A + (tt / B) * sBr + (tt % B) * sB + (long long)r * ld;
    }
    rowp[tid] = ptr;
  }
  // zero both stages once: the halo (and rows past the end) stay zero, the copies only touch the interior
  for (int i = tid; i < g.stage_floats / 2; i += blockDim.x) reinterpret_cast<float4*>(smem_f)[i] = make_float4(0.f, 0.f, 0.f, 0.f);   // stage_floats % 4 == 0
  // this thread's share of a tile: source offset inside one (row, co) map, or -1 for halo elements
  int soff[kConvFillMax], doff[kConvFillMax];
#pragma unroll
  for (int k = 0; k < kConvFillMax; ++k) {
    const int idx = tid + k * blockDim.x;
    const int p = idx / g.PW + g.omin_y, q = idx % g.PW + g.omin_x;
    const bool in = idx < tile && p >= 0 && p < g.ho && q >= 0 && q < g.wo;
    soff[k] = in ? p * g.wo + q : -1;
    doff[k] = idx;
  }
  __syncthreads();

  auto fill = [&](int co0, int stage) {
    float* Ws = smem_f + stage * g.stage_floats;
    float* As = Ws + w_floats;
    const int cc = min(g.COC, g.c_out - co0);
    for (int idx = tid; idx < cc * KK * cgct; idx += blockDim.x) {
      const int c = idx % cgct, t2 = idx / cgct;
      const int tap = t2 % KK, co = t2 / KK;
      const int ci = ci_base + c;
      if (ci < g.c_in) cp_async4(Ws + idx, W + ((long long)(co0 + co) * g.c_in + ci) * KK + tap);
    }
    for (int r_ = 0; r_ < g.RB; ++r_) {
      const float* base = rowp[r_];
      if (base == nullptr) continue;
      base += (long long)co0 * g.ho * g.wo;
      float* dst = As + r_ * g.COC * tile;
      if (tile <= (int)blockDim.x) {      // small maps (8x8: 100 elements): one slot per thread, not six predicated ones
        for (int co = 0; co < cc; ++co, base += g.ho * g.wo, dst += tile)
          if (soff[0] >= 0) cp_async4(dst + doff[0], base + soff[0]);
      } else {
        for (int co = 0; co < cc; ++co) {
#pragma unroll
          for (int k = 0; k < kConvFillMax; ++k)
            if (soff[k] >= 0) cp_async4(dst + doff[k], base + soff[k]);
          base += g.ho * g.wo;
          dst += tile;
        }
      }
    }
    cp_async_commit();
  };

  // tap table (loop-invariant): offset inside the tile, or -1 when the tap does not hit this parity class
  int toff[KK];
#pragma unroll
  for (int i = 0; i < KH; ++i)
#pragma unroll
    for (int j = 0; j < KW; ++j) {
      const int ny_ = cy + g.pad - i, nx_ = cx + g.pad - j;
      const bool ok = (((ny_ % S) + S) % S == 0) && (((nx_ % S) + S) % S == 0);
      const int oy = ok ? ny_ / S : 0, ox = ok ? nx_ / S : 0;
      toff[i * KW + j] = ok ? (yy + oy - g.omin_y) * g.PW + (ox - g.omin_x) : -1;
    }
  int u[4]; bool uv[4];
#pragma unroll
  for (int t = 0; t < 4; ++t) {
    const int ut = xq + t * g.XQ;
    uv[t] = active && ut < g.NX && (cx + S * ut) < g.w && y < g.h;
    u[t] = uv[t] ? ut : 0;
  }
  // accumulators start from the residual fork's other contribution (addend) when there is one: its loads are issued
  // here, all at once, and complete behind the first shared-memory fill
  const long long m_row = m_base + rb;
  float acc[4][CT];
#pragma unroll
  for (int t = 0; t < 4; ++t)
#pragma unroll
    for (int c = 0; c < CT; ++c) {
      const int ci = ci_base + cg * CT + c;
      float a0 = 0.f;
      if (addend != nullptr && active && m_row < rows && uv[t] && ci < g.c_in)
        a0 = __ldg(addend + ((m_row * g.c_in + ci) * g.h + y) * (long long)g.w + (cx + S * u[t]));
      acc[t][c] = a0;
    }

  const int nchunks = (g.c_out + g.COC - 1) / g.COC;
  fill(0, 0);
  for (int ch = 0; ch < nchunks; ++ch) {
    const int stage = ch & 1;
    if (ch + 1 < nchunks) { fill((ch + 1) * g.COC, stage ^ 1); cp_async_wait<1>(); }
    else cp_async_wait<0>();
    __syncthreads();
    if (active) {
      const int cc = min(g.COC, g.c_out - ch * g.COC);
      const float* Ws = smem_f + stage * g.stage_floats;
      const float* ap = Ws + w_floats + rb * g.COC * tile;
      const float* wp = Ws + cg * CT;
      for (int co = 0; co < cc; ++co, ap += tile, wp += KK * cgct) {
#pragma unroll
        for (int tap = 0; tap < KK; ++tap) {
          if (S > 1 && toff[tap] < 0) continue;
          float a[4];
#pragma unroll
          for (int t = 0; t < 4; ++t) a[t] = ap[toff[tap] + u[t]];
#pragma unroll
          for (int c4 = 0; c4 < CT; c4 += 4) {
            const float4 wv = *reinterpret_cast<const float4*>(wp + tap * cgct + c4);
#pragma unroll
            for (int t = 0; t < 4; ++t) {
              acc[t][c4 + 0] = fmaf(a[t], wv.x, acc[t][c4 + 0]);
              acc[t][c4 + 1] = fmaf(a[t], wv.y, acc[t][c4 + 1]);
              acc[t][c4 + 2] = fmaf(a[t], wv.z, acc[t][c4 + 2]);
              acc[t][c4 + 3] = fmaf(a[t], wv.w, acc[t][c4 + 3]);
            }
          }
        }
      }
    }
    __syncthreads();      // the stage is refilled by the next iteration's fill
  }
  const long long m = m_base + rb;
  if (!active || m >= rows) return;
#pragma unroll
  for (int c = 0; c < CT; ++c) {
    const int ci = ci_base + cg * CT + c;
    if (ci >= g.c_in) continue;
#pragma unroll
    for (int t = 0; t < 4; ++t) {
      if (!uv[t]) continue;
      const long long o = ((m * g.c_in + ci) * g.h + y) * (long long)g.w + (cx + S * u[t]);
      out[o] = acc[t][c];
    }
  }
}

template <int KH, int KW, int S, int CT>
static bool launch_conv_bwd_tiled(const AView& A, const float* W, const float* addend, float* out, int B, int R,
                                  int c_in, int h, int w, int c_out, int pad, int ho, int wo, cudaStream_t s) {
  ConvBwdGeom g;
  g.c_in = c_in; g.h = h; g.w = w; g.c_out = c_out; g.ho = ho; g.wo = wo; g.pad = pad;
  g.NY = (h + S - 1) / S; g.NX = (w + S - 1) / S; g.XQ = (g.NX + 3) / 4;
  g.PT = S * S * g.NY * g.XQ;
  if (g.PT > 256) return false;
  const int groups = (c_in + CT - 1) / CT;
  g.CG = 256 / g.PT < groups ? 256 / g.PT : groups;
  if (g.CG < 1) g.CG = 1;
  g.RB = 256 / (g.PT * g.CG);
  if (g.RB < 1) g.RB = 1;
  if (g.RB > 4) g.RB = 4;
  int omin_y = 0, omax_y = 0, omin_x = 0, omax_x = 0;
  for (int c = 0; c < S; ++c) {
    for (int i = 0; i < KH; ++i) { int n = c + pad - i; if (((n % S) + S) % S == 0) { omin_y = n / S < omin_y ? n / S : omin_y; omax_y = n / S > omax_y ? n / S : omax_y; } }
    for (int j = 0; j < KW; ++j) { int n = c + pad - j; if (((n % S) + S) % S == 0) { omin_x = n / S < omin_x ? n / S : omin_x; omax_x = n / S > omax_x ? n / S : omax_x; } }
  }
  g.omin_y = omin_y; g.omin_x = omin_x;
  g.PH = g.NY + omax_y - omin_y;
  g.PW = g.NX + omax_x - omin_x;
  const int threads = ((g.PT * g.CG * g.RB + 31) / 32) * 32;
  if (g.PH * g.PW > kConvFillMax * threads) return false;
  const int cgct = g.CG * CT;
  const size_t budget = kConvBwdSmemBudget;              // two stages; two blocks per SM still fit
  const size_t per_co = ((size_t)KH * KW * cgct + (size_t)g.RB * g.PH * g.PW) * sizeof(float);
  int coc = (int)(budget / 2 / per_co);
  if (coc < 1) return false;
  if (coc > c_out) coc = c_out;
  g.COC = coc;
  g.stage_floats = (int)(per_co * coc / sizeof(float));
  g.stage_floats = (g.stage_floats + 3) / 4 * 4;
  const size_t smem = (size_t)2 * g.stage_floats * sizeof(float);
  const long long rows = 2LL * B * R;
  dim3 grid((unsigned)((rows + g.RB - 1) / g.RB), (unsigned)((groups + g.CG - 1) / g.CG));
  conv_bwd_tiled_kernel<KH, KW, S, CT><<<grid, threads, smem, s>>>(A.p, A.sBr, A.sB, A.ld, B, R, W, addend, out, g);
  return true;
}

template <int KH, int KW, int S>
static bool launch_conv_bwd_ct(const AView& A, const float* W, const float* addend, float* out, int B, int R,
                               int c_in, int h, int w, int c_out, int pad, int ho, int wo, cudaStream_t s) {
  if (c_in % 16 == 0) return launch_conv_bwd_tiled<KH, KW, S, 16>(A, W, addend, out, B, R, c_in, h, w, c_out, pad, ho, wo, s);
  if (c_in > 4) return launch_conv_bwd_tiled<KH, KW, S, 8>(A, W, addend, out, B, R, c_in, h, w, c_out, pad, ho, wo, s);
  return launch_conv_bwd_tiled<KH, KW, S, 4>(A, W, addend, out, B, R, c_in, h, w, c_out, pad, ho, wo, s);
}

template <int KH, int KW, int S>
static bool conv_bwd_set_attr() {
  const int bytes = (int)kConvBwdSmemBudget + 64;
  return cudaFuncSetAttribute(conv_bwd_tiled_kernel<KH, KW, S, 16>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes) == cudaSuccess &&
         cudaFuncSetAttribute(conv_bwd_tiled_kernel<KH, KW, S, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes) == cudaSuccess &&
         cudaFuncSetAttribute(conv_bwd_tiled_kernel<KH, KW, S, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes) == cudaSuccess;
}

// ---- a6, 1x1 convolutions (the stride-2 skip connections of a ResNet; pad 0).  conv^T of a 1x1 kernel is a per-pixel
// matrix product: A_in[m, ci, s*p, s*q] = sum_co W[co, ci] * A_out[m, co, p, q], every other pixel a structural zero.
// Block = one spec row x PIX output pixels; A_out[m, :, tile] and W^T sit in shared memory; a thread owns one pixel x
// CIP input channels and writes its s x s block of the input map (value + zeros) so that the stores of a warp are contiguous.
// The generic tiled kernel walked the zero pixels as if they were work: 151 + 127 us for 0.84 GFLOP on cfg5 (profiles/r2_conv.md).
template <int CIP>
__global__ void __launch_bounds__(256)
conv_bwd_1x1_kernel(const float* __restrict__ A, long long sBr, long long sB, long long ld, int B, int R,
                    const float* __restrict__ W, const float* __restrict__ addend, float* __restrict__ out,
                    int c_in, int h, int w, int c_out, int stride, int ho, int wo, int PIX, int vec) {
  extern __shared__ __align__(16) float sm[];
  float* Ws = sm;                          // [c_out][c_in]  (c_out * c_in is a multiple of 4 when vec: As stays 16-byte aligned)
  float* As = sm + c_out * c_in;           // [c_out][PIX]
  const long long m = blockIdx.y;
  const int pix0 = blockIdx.x * PIX;
  const int npix = ho * wo;
  for (int i = threadIdx.x; i < c_out * c_in; i += blockDim.x) Ws[i] = __ldg(W + i);     // W [c_out, c_in, 1, 1]
  {
    const int r = (int)(m % R);
    const long long tt = m / R;
    const float* a = A + (tt / B) * sBr + (tt % B) * sB + (long long)r * ld;
    if (vec) {       // 16-byte asynchronous copies, all in flight at once (the tile is c_out contiguous runs of PIX floats)
      const int q4 = PIX >> 2;
      for (int i = threadIdx.x; i < c_out * q4; i += blockDim.x) {
        const int co = i / q4, p4 = (i % q4) << 2;
        float* dst = As + co * PIX + p4;
        if (pix0 + p4 < npix) {
          const uint32_t d = static_cast<uint32_t>(__cvta_generic_to_shared(dst));
          asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" :: "r"(d), "l"(a + (long long)co * npix + pix0 + p4) : "memory");
        } else {
          *reinterpret_cast<float4*>(dst) = make_float4(0.f, 0.f, 0.f, 0.f);
        }
      }
      cp_async_commit();
      cp_async_wait<0>();
    } else {
      for (int i = threadIdx.x; i < c_out * PIX; i += blockDim.x) {
        const int co = i / PIX, p = i % PIX;
        As[i] = (pix0 + p < npix) ? __ldg(a + (long long)co * npix + pix0 + p) : 0.f;
      }
    }
  }
  __syncthreads();
  const int p = threadIdx.x % PIX, cg = threadIdx.x / PIX;
  const int ci0 = cg * CIP;
  if (ci0 >= c_in || pix0 + p >= npix) return;
  float acc[CIP];
#pragma unroll
  for (int c = 0; c < CIP; ++c) acc[c] = 0.f;
  for (int co = 0; co < c_out; ++co) {
    const float a = As[co * PIX + p];
    const float* wr = Ws + co * c_in + ci0;
#pragma unroll
    for (int c = 0; c < CIP; ++c) acc[c] = fmaf(a, (ci0 + c < c_in) ? wr[c] : 0.f, acc[c]);
  }
  const int py = (pix0 + p) / wo, px = (pix0 + p) % wo;
#pragma unroll
  for (int c = 0; c < CIP; ++c) {
    const int ci = ci0 + c;
    if (ci >= c_in) break;
    const long long base = (m * c_in + ci) * (long long)(h * w);
    if (stride == 2 && (w & 1) == 0 && 2 * py + 1 < h &&
        ((reinterpret_cast<uintptr_t>(out) | reinterpret_cast<uintptr_t>(addend)) & 7) == 0) {
      // the 2 x 2 input block of this output pixel as two 8-byte stores: {value, 0} and {0, 0} (+ the addend); one
      // 4-byte store per input pixel left every second lane of a store instruction idle
      const long long o = base + (long long)(2 * py) * w + 2 * px;        // even: 8-byte aligned (h * w and w are even)
      float2 r0 = make_float2(acc[c], 0.f), r1 = make_float2(0.f, 0.f);
      if (addend) {
        const float2 e0 = __ldg(reinterpret_cast<const float2*>(addend + o)), e1 = __ldg(reinterpret_cast<const float2*>(addend + o + w));
        r0.x += e0.x; r0.y += e0.y; r1.x += e1.x; r1.y += e1.y;
      }
      *reinterpret_cast<float2*>(out + o) = r0;
      *reinterpret_cast<float2*>(out + o + w) = r1;
      continue;
    }
    for (int dy = 0; dy < stride; ++dy) {
      const int y = py * stride + dy;
      if (y >= h) break;
      for (int dx = 0; dx < stride; ++dx) {
        const int x = px * stride + dx;
        if (x >= w) break;
        const long long o = base + (long long)y * w + x;
        const float v = (dy == 0 && dx == 0) ? acc[c] : 0.f;
        out[o] = addend ? v + __ldg(addend + o) : v;
      }
    }
  }
}

// ---- a6, 3x3 / stride 2 / pad 1 (the down-sampling convolutions of a ResNet; h = 2 ho, w = 2 wo).
// A thread owns the 2 x 2 block of INPUT pixels (2p..2p+1, 2q..2q+1) x CT input channels, i.e. one pixel of each of the four
// stride-parity classes, so every thread runs the same 9 taps on the same 4 values of A_out:
//   in(2p  ,2q  ) += W11 a(p,q)                          in(2p  ,2q+1) += W10 a(p,q+1) + W12 a(p,q)
//   in(2p+1,2q  ) += W01 a(p+1,q) + W21 a(p,q)           in(2p+1,2q+1) += W00 a(p+1,q+1) + W02 a(p+1,q) + W20 a(p,q+1) + W22 a(p,q)
// (y = 2p' + i - 1).  The generic tiled kernel gives a thread four pixels of ONE class: classes need 1, 2, 2 and 4 taps, so
// with 16-thread classes half the lanes of every FFMA were idle (ncu: 16.0 active threads per FFMA on 32 -> 64 @ 8x8) and
// with warp-sized classes the block waited for its 4-tap warps (profiles/r2_conv.md: 8 and 12.6 TFLOP/s).
// Block = RB rows x CG channel groups x (ho * wo) pixel threads; A_out tiles (zero halo right / below) and the filter slice
// [co][tap][ci] are staged COC output channels at a time.
// P = 2: a thread owns TWO horizontally adjacent positions (p, q), (p, q + 1) of A_out, i.e. a 2 x 4 block of input pixels: every
// filter tap loaded from shared memory feeds two FFMAs instead of one (P = 1 runs 36 broadcast LDS.128 per 144 FFMAs, 40 % FMA pipe).
template <int CT, int P>
__global__ void __launch_bounds__(256, 2)
conv_bwd_3x3s2_kernel(const float* __restrict__ A, long long sBr, long long sB, long long ld, int B, int R,
                      const float* __restrict__ W, const float* __restrict__ addend, float* __restrict__ out,
                      int c_in, int c_out, int ho, int wo, int COC, int CG, int RB, int stage_floats) {
  extern __shared__ __align__(16) float sm[];
  __shared__ const float* rowp[4];
  const int cgct = CG * CT;
  const int wq = wo / P;                           // thread columns per row of A_out (wo % P == 0)
  const int PT = ho * wq, PW = wo + 1, tile = (ho + 1) * PW;
  const int w_floats = COC * 9 * cgct;             // stage layout: Ws [COC][9][cgct], then As [RB][COC][tile]
  const int tid = threadIdx.x;
  const int pt = tid % PT, cg = (tid / PT) % CG, rb = tid / (PT * CG);
  const bool active = rb < RB;
  const long long rows = 2LL * B * R;
  const long long m_base = (long long)blockIdx.x * RB;
  const int ci_base = blockIdx.y * cgct;
  const int p = pt / wq, q = (pt % wq) * P;
  const int a_off = p * PW + q;
  if (tid < RB) {
    const long long m = m_base + tid;
    const float* ptr = nullptr;
    if (m < rows) {
      const int r = (int)(m % R);
      const long long tt = m / R;
      ptr = A + (tt / B) * sBr + (tt % B) * sB + (long long)r * ld;
    }
    rowp[tid] = ptr;
  }
  // both stages zeroed once: the halo column / row (and rows past the end) stay zero, the copies touch the interior only
  for (int i = tid; i < stage_floats / 2; i += blockDim.x) reinterpret_cast<float4*>(sm)[i] = make_float4(0.f, 0.f, 0.f, 0.f);   // stage_floats % 4 == 0
  int soff[2];                                      // this thread's (up to two) elements of a (row, co) tile
#pragma unroll
  for (int k = 0; k < 2; ++k) {
    const int e = tid + k * (int)blockDim.x;
    const int y = e / PW, x = e % PW;
    soff[k] = (e < tile && y < ho && x < wo) ? y * wo + x : -1;
  }
  __syncthreads();
  // asynchronous staging (cp.async, 4-byte copies: the halo shifts alignment), double-buffered
  auto fill = [&](int co0, int stage) {
    float* Ws = sm + stage * stage_floats;
    float* As = Ws + w_floats;
    const int cc = min(COC, c_out - co0);
    for (int j = tid; j < 9 * cgct; j += blockDim.x) {     // (tap, c) fixed per thread, the loop walks the output channels: no division per copy
      const int c = j % cgct, tap = j / cgct;
      const int ci = ci_base + c;
      if (ci >= c_in) continue;
      const float* src = W + ((long long)co0 * c_in + ci) * 9 + tap;
      float* dst = Ws + j;
      for (int co = 0; co < cc; ++co, src += (long long)c_in * 9, dst += 9 * cgct) cp_async4(dst, src);
    }
    for (int r_ = 0; r_ < RB; ++r_) {
      const float* base = rowp[r_];
      if (base == nullptr) continue;
      base += (long long)co0 * (ho * wo);
      float* dst = As + r_ * COC * tile;
      for (int co = 0; co < cc; ++co, base += ho * wo, dst += tile) {
#pragma unroll
        for (int k = 0; k < 2; ++k)
          if (soff[k] >= 0) cp_async4(dst + tid + k * (int)blockDim.x, base + soff[k]);
      }
    }
    cp_async_commit();
  };
  float acc[4 * P][CT];
#pragma unroll
  for (int k = 0; k < 4 * P; ++k)
#pragma unroll
    for (int c = 0; c < CT; ++c) acc[k][c] = 0.f;
  const int nchunks = (c_out + COC - 1) / COC;
  fill(0, 0);
  for (int ch = 0; ch < nchunks; ++ch) {
    const int stage = ch & 1;
    if (ch + 1 < nchunks) { fill((ch + 1) * COC, stage ^ 1); cp_async_wait<1>(); }
    else cp_async_wait<0>();
    __syncthreads();
    if (active) {
      const int cc = min(COC, c_out - ch * COC);
      const float* Ws = sm + stage * stage_floats;
      const float* ap = Ws + w_floats + rb * COC * tile + a_off;
      const float* wp = Ws + cg * CT;
      for (int co = 0; co < cc; ++co, ap += tile, wp += 9 * cgct) {
        float a0[P + 1], a1[P + 1];                 // A_out rows p and p + 1, columns q .. q + P
#pragma unroll
        for (int u = 0; u <= P; ++u) { a0[u] = ap[u]; a1[u] = ap[PW + u]; }
#pragma unroll
        for (int c4 = 0; c4 < CT; c4 += 4) {
          float4 w[9];
#pragma unroll
          for (int t = 0; t < 9; ++t) w[t] = *reinterpret_cast<const float4*>(wp + t * cgct + c4);
#define CROWN_S2_STEP(C_, F_) \
          acc[4 * u + 0][c4 + C_] = fmaf(w[4].F_, a00, acc[4 * u + 0][c4 + C_]); \
          acc[4 * u + 1][c4 + C_] = fmaf(w[3].F_, a01, fmaf(w[5].F_, a00, acc[4 * u + 1][c4 + C_])); \
          acc[4 * u + 2][c4 + C_] = fmaf(w[1].F_, a10, fmaf(w[7].F_, a00, acc[4 * u + 2][c4 + C_])); \
          acc[4 * u + 3][c4 + C_] = fmaf(w[0].F_, a11, fmaf(w[2].F_, a10, fmaf(w[6].F_, a01, fmaf(w[8].F_, a00, acc[4 * u + 3][c4 + C_]))));
#pragma unroll
          for (int u = 0; u < P; ++u) {
            const float a00 = a0[u], a01 = a0[u + 1], a10 = a1[u], a11 = a1[u + 1];
            CROWN_S2_STEP(0, x) CROWN_S2_STEP(1, y) CROWN_S2_STEP(2, z) CROWN_S2_STEP(3, w)
          }
#undef CROWN_S2_STEP
        }
      }
    }
    __syncthreads();      // the stage is refilled by the next iteration's fill
  }
  const long long m = m_base + rb;
  if (!active || m >= rows) return;
  const int h = 2 * ho, w_ = 2 * wo;
  const long long plane = (long long)h * w_;
  const long long o0 = ((m * c_in + ci_base + cg * CT) * h + 2 * p) * (long long)w_ + 2 * q;     // even: 8-byte aligned (P = 2: 16)
  if (P == 2) {
    // a position pair is four adjacent input columns: one 16-byte store per input row; four channels' addends at a time
#pragma unroll
    for (int c0 = 0; c0 < CT; c0 += 4) {
      float4 e0[4], e1[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        e0[k] = make_float4(0.f, 0.f, 0.f, 0.f); e1[k] = e0[k];
        if (addend && ci_base + cg * CT + c0 + k < c_in) {
          const long long o = o0 + (c0 + k) * plane;
          e0[k] = __ldg(reinterpret_cast<const float4*>(addend + o)); e1[k] = __ldg(reinterpret_cast<const float4*>(addend + o + w_));
        }
      }
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const int c = c0 + k;
        if (ci_base + cg * CT + c >= c_in) continue;
        const long long o = o0 + c * plane;
        *reinterpret_cast<float4*>(out + o) = make_float4(acc[0][c] + e0[k].x, acc[1][c] + e0[k].y, acc[4 * (P - 1)][c] + e0[k].z, acc[4 * (P - 1) + 1][c] + e0[k].w);
        *reinterpret_cast<float4*>(out + o + w_) = make_float4(acc[2][c] + e1[k].x, acc[3][c] + e1[k].y, acc[4 * (P - 1) + 2][c] + e1[k].z, acc[4 * (P - 1) + 3][c] + e1[k].w);
      }
    }
    return;
  }
  // eight channels at a time: their sixteen addend loads are issued together, then added and stored (one channel at a time
  // every add waited for its own load: 23 - 45 % of this kernel's samples sat on those FADDs)
#pragma unroll
  for (int c0 = 0; c0 < CT; c0 += 8) {
    float2 e0[8], e1[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      e0[k] = make_float2(0.f, 0.f); e1[k] = make_float2(0.f, 0.f);
      if (addend && ci_base + cg * CT + c0 + k < c_in) {
        const long long o = o0 + (c0 + k) * plane;
        e0[k] = __ldg(reinterpret_cast<const float2*>(addend + o)); e1[k] = __ldg(reinterpret_cast<const float2*>(addend + o + w_));
      }
    }
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      const int c = c0 + k;
      if (ci_base + cg * CT + c >= c_in) continue;
      const long long o = o0 + c * plane;
      *reinterpret_cast<float2*>(out + o) = make_float2(acc[0][c] + e0[k].x, acc[1][c] + e0[k].y);
      *reinterpret_cast<float2*>(out + o + w_) = make_float2(acc[2][c] + e1[k].x, acc[3][c] + e1[k].y);
    }
  }
}

// ---- a6, 3x3 / stride 1 / pad 1 with w % 4 == 0 and h * w / 4 <= 256 (the 32x32, 16x16 and 8x8 maps of a ResNet).
// A thread owns a strip of FOUR ADJACENT pixels (y, 4q .. 4q+3) x CT input channels.  Per output channel it reads, for each
// of the three image rows y-1 .. y+1, one aligned float4 and the two neighbours left and right of it (the tile is stored with
// a 4-column left pad, so column 4q is 16-byte aligned) -- 9 shared-memory loads of A feed all 9 taps of all 4 pixels:
//   in(y, 4q+t) += sum_{i,j} W[i][j] * a[y+1-i][4q+t+1-j]
// The generic tiled kernel gives a thread four pixels that are XQ apart and loads every (tap, pixel) operand separately
// (36 loads per output channel, each with its own address arithmetic): ncu showed 42 % FFMA in its instruction mix.
template <int CT>
__global__ void __launch_bounds__(256, 2)
conv_bwd_3x3s1_kernel(const float* __restrict__ A, long long sBr, long long sB, long long ld, int B, int R,
                      const float* __restrict__ W, const float* __restrict__ addend, float* __restrict__ out,
                      int c_in, int c_out, int h, int w, int COC, int CG, int RB, int stage_floats) {
  extern __shared__ __align__(16) float sm[];
  __shared__ const float* rowp[4];
  const int cgct = CG * CT;
  const int wq = w >> 2;                           // strips per image row
  const int PT = h * wq, PW = w + 8, tile = (h + 2) * PW;
  const int w_floats = (COC * 9 * cgct + 3) & ~3;  // stage layout: Ws [COC][9][cgct], then As [RB][COC][tile] (16-byte aligned)
  const int tid = threadIdx.x;
  const int pt = tid % PT, cg = (tid / PT) % CG, rb = tid / (PT * CG);
  const bool active = rb < RB;
  const long long rows = 2LL * B * R;
  const long long m_base = (long long)blockIdx.x * RB;
  const int ci_base = blockIdx.y * cgct;
  const int y = pt / wq, q = pt % wq;
  const int a_off = y * PW + 4 + 4 * q;            // tile row y holds image row y - 1; image column x sits at tile column x + 4
  if (tid < RB) {
    const long long m = m_base + tid;
    const float* ptr = nullptr;
    if (m < rows) {
      const int r = (int)(m % R);
      const long long tt = m / R;
      ptr = A + (tt / B) * sBr + (tt % B) * sB + (long long)r * ld;
    }
    rowp[tid] = ptr;
  }
  // both stages zeroed once: the halo (and rows past the end) stay zero, the copies touch the interior only
  for (int i = tid; i < stage_floats / 2; i += blockDim.x) reinterpret_cast<float4*>(sm)[i] = make_float4(0.f, 0.f, 0.f, 0.f);   // stage_floats % 4 == 0
  __syncthreads();
  const int epp = PT;                              // float4 elements of one (row, co) map: h * w / 4 = PT
  // The fill loops carry no division: ncu's per-instruction samples had 44 % of this kernel's time in their index
  // arithmetic (idx % epp, / epp, % cc, / cc, ... once per 16 copied bytes) against 34 % in the FFMA loop.
  //   filters: element j of a [9][cgct] slab (tap, c) is fixed per thread; the loop walks the output channels;
  //   A tiles: with 256 % epp == 0 (the 32x32, 16x16 and 8x8 maps) a thread's float4 position e inside a map is fixed and
  //   its (row, co) pair advances by 256 / epp per step, carried as two counters; other map sizes take the general loop.
  const bool fixed_e = (blockDim.x % epp) == 0;
  const int fe = tid % epp, fpr0 = tid / epp, fstep = blockDim.x / epp;
  const int fyy = fe / wq, fxq = fe % wq;
  const long long fsrc_off = (long long)fyy * w + 4 * fxq;
  const int fdst_off = (fyy + 1) * PW + 4 + 4 * fxq;
  auto fill = [&](int co0, int stage) {
    float* Ws = sm + stage * stage_floats;
    float* As = Ws + w_floats;
    const int cc = min(COC, c_out - co0);
    for (int j = tid; j < 9 * cgct; j += blockDim.x) {
      const int c = j % cgct, tap = j / cgct;
      const int ci = ci_base + c;
      if (ci >= c_in) continue;
      const float* src = W + ((long long)co0 * c_in + ci) * 9 + tap;
      float* dst = Ws + j;
      for (int co = 0; co < cc; ++co, src += (long long)c_in * 9, dst += 9 * cgct) cp_async4(dst, src);
    }
    if (fixed_e) {
      int co = fpr0 % cc, r_ = fpr0 / cc;          // one division per fill and thread
      for (int pr = fpr0; pr < RB * cc; pr += fstep) {
        const float* base = rowp[r_];
        if (base != nullptr) {
          const float* src = base + (long long)(co0 + co) * h * w + fsrc_off;
          float* dst = As + ((long long)r_ * COC + co) * tile + fdst_off;
          const uint32_t d = static_cast<uint32_t>(__cvta_generic_to_shared(dst));
          asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" :: "r"(d), "l"(src) : "memory");
        }
        co += fstep;
        while (co >= cc) { co -= cc; ++r_; }
      }
    } else {
      for (int idx = tid; idx < RB * cc * epp; idx += blockDim.x) {
        const int e = idx % epp, pr = idx / epp;
        const int co = pr % cc, r_ = pr / cc;
        const float* base = rowp[r_];
        if (base == nullptr) continue;
        const int yy = e / wq, xq = e % wq;
        const float* src = base + ((long long)(co0 + co) * h + yy) * w + 4 * xq;
        float* dst = As + ((long long)r_ * COC + co) * tile + (yy + 1) * PW + 4 + 4 * xq;
        const uint32_t d = static_cast<uint32_t>(__cvta_generic_to_shared(dst));
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" :: "r"(d), "l"(src) : "memory");
      }
    }
    cp_async_commit();
  };
  float acc[4][CT];
#pragma unroll
  for (int t = 0; t < 4; ++t)
#pragma unroll
    for (int c = 0; c < CT; ++c) acc[t][c] = 0.f;
  const int nchunks = (c_out + COC - 1) / COC;
  fill(0, 0);
  for (int ch = 0; ch < nchunks; ++ch) {
    const int stage = ch & 1;
    if (ch + 1 < nchunks) { fill((ch + 1) * COC, stage ^ 1); cp_async_wait<1>(); }
    else cp_async_wait<0>();
    __syncthreads();
    if (active) {
      const int cc = min(COC, c_out - ch * COC);
      const float* Ws = sm + stage * stage_floats;
      const float* ap = Ws + w_floats + (long long)rb * COC * tile + a_off;
      const float* wp = Ws + cg * CT;
      for (int co = 0; co < cc; ++co, ap += tile, wp += 9 * cgct) {
        float a[3][6];                              // a[dy][k] = A_out[y - 1 + dy][4q - 1 + k]
#pragma unroll
        for (int dy = 0; dy < 3; ++dy) {
          const float4 v = *reinterpret_cast<const float4*>(ap + dy * PW);
          a[dy][0] = ap[dy * PW - 1]; a[dy][1] = v.x; a[dy][2] = v.y; a[dy][3] = v.z; a[dy][4] = v.w; a[dy][5] = ap[dy * PW + 4];
        }
#pragma unroll
        for (int c4 = 0; c4 < CT; c4 += 4) {
#pragma unroll
          for (int i = 0; i < 3; ++i) {
#pragma unroll
            for (int j = 0; j < 3; ++j) {
              const float4 wv = *reinterpret_cast<const float4*>(wp + (i * 3 + j) * cgct + c4);
              // image row y + 1 - i is tile row offset dy = 2 - i; pixel 4q + t reads column 4q + t + 1 - j = a[.][t + 2 - j]
#pragma unroll
              for (int t = 0; t < 4; ++t) {
                const float av = a[2 - i][t + 2 - j];
                acc[t][c4 + 0] = fmaf(av, wv.x, acc[t][c4 + 0]);
                acc[t][c4 + 1] = fmaf(av, wv.y, acc[t][c4 + 1]);
                acc[t][c4 + 2] = fmaf(av, wv.z, acc[t][c4 + 2]);
                acc[t][c4 + 3] = fmaf(av, wv.w, acc[t][c4 + 3]);
              }
            }
          }
        }
      }
    }
    __syncthreads();      // the stage is refilled by the next iteration's fill
  }
  const long long m = m_base + rb;
  if (!active || m >= rows) return;
  // four channels at a time: the addend loads are issued together, then added and stored
  const long long plane = (long long)h * w;
  const long long o0 = ((m * c_in + ci_base + cg * CT) * h + y) * (long long)w + 4 * q;
#pragma unroll
  for (int c0 = 0; c0 < CT; c0 += 4) {
    float4 e[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      e[k] = make_float4(0.f, 0.f, 0.f, 0.f);
      if (addend && ci_base + cg * CT + c0 + k < c_in) e[k] = __ldg(reinterpret_cast<const float4*>(addend + o0 + (c0 + k) * plane));
    }
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const int c = c0 + k;
      if (ci_base + cg * CT + c >= c_in) continue;
      *reinterpret_cast<float4*>(out + o0 + c * plane) =
          make_float4(acc[0][c] + e[k].x, acc[1][c] + e[k].y, acc[2][c] + e[k].z, acc[3][c] + e[k].w);
    }
  }
}

static bool launch_conv_bwd_3x3s1(const AView& A, const float* W, const float* addend, float* out, int B, int R,
                                  int c_in, int h, int w, int c_out, int pad, int ho, int wo, cudaStream_t s) {
  if (pad != 1 || ho != h || wo != w || (w & 3) || h * (w >> 2) > 256 || h * (w >> 2) < 16) return false;
  auto mis = [](const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15) != 0; };
  if (mis(A.p) || mis(out) || (addend && mis(addend)) || (A.ld & 3) || (A.sB & 3) || (A.sBr & 3)) return false;
  const int CT = (c_in % 16 == 0) ? 16 : (c_in > 4 ? 8 : 4);
  const int PT = h * (w >> 2);
  const int groups = (c_in + CT - 1) / CT;
  int CG = 256 / PT < groups ? 256 / PT : groups;
  if (CG < 1) CG = 1;
  int RB = 256 / (PT * CG);
  if (RB < 1) RB = 1;
  if (RB > 4) RB = 4;
  const int tile = (h + 2) * (w + 8);
  const size_t per_co = ((size_t)9 * CG * CT + (size_t)RB * tile) * sizeof(float);
  int COC = (int)((44 * 1024) / per_co);           // two stages of <= 44 KB, two blocks per SM
  if (COC < 1) return false;
  if (COC > c_out) COC = c_out;
  const int stage_floats = (int)(((((size_t)COC * 9 * CG * CT + 3) & ~(size_t)3) + (size_t)COC * RB * tile + 3) / 4 * 4);
  const size_t smem = (size_t)2 * stage_floats * sizeof(float);
  const long long rows = 2LL * B * R;
  dim3 grid((unsigned)((rows + RB - 1) / RB), (unsigned)((groups + CG - 1) / CG));
#define CROWN_S1_GO(CT_) conv_bwd_3x3s1_kernel<CT_><<<grid, 256, smem, s>>>(A.p, A.sBr, A.sB, A.ld, B, R, W, addend, out, c_in, c_out, h, w, COC, CG, RB, stage_floats)
  if (CT == 16) CROWN_S1_GO(16); else if (CT == 8) CROWN_S1_GO(8); else CROWN_S1_GO(4);
#undef CROWN_S1_GO
  return true;
}

// Forward 3x3 / stride 1 / pad 1 convolution of M points through the strip kernel (NEXT-1 forward sweep): conv(x, W) is the
// transpose kernel run with the filter bank flipped and its channel roles swapped,
//   out[m, co, y, x] = sum_ci sum_{i,j} Wk[ci][co][i][j] * in[m, ci, y+1-i, x+1-j],   Wk[ci][co][i][j] = W[co][ci][2-i][2-j]
// (Wk is made by launch_flip_conv_weights).  `in` / `out` are [M, c, h, w] contiguous; the bias is added by the caller.
int conv3x3s1_points_supported(int c_in, int h, int w, int c_out) {
  (void)c_in; (void)c_out;
  return (w & 3) == 0 && h * (w >> 2) <= 256 && h * (w >> 2) >= 16;
}
int launch_conv3x3s1_points(const float* in, const float* Wk, float* out, long long M, int c_in, int h, int w, int c_out,
                            cudaStream_t s) {
  if (M <= 0 || (M & 1)) return -1;
  AView v; v.p = in; v.ld = (long long)c_in * h * w; v.n = c_in * h * w; v.sB = 0; v.sBr = (M / 2) * v.ld;
  // rows m < M/2 as "branch 0", the rest as "branch 1" of a B = 1, R = M/2 problem; reduce channels = c_in, outputs = c_out
  return launch_conv_bwd_3x3s1(v, Wk, nullptr, out, 1, (int)(M / 2), c_out, h, w, c_in, 1, h, w, s) ? 0 : -1;
}
__global__ void flip_conv_weights_kernel(const float* __restrict__ W, float* __restrict__ Wk, int c_out, int c_in) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= c_out * c_in * 9) return;
  const int tap = i % 9, ci = (i / 9) % c_in, co = i / (9 * c_in);           // i indexes W[co][ci][tap]
  Wk[((long long)ci * c_out + co) * 9 + (8 - tap)] = W[i];
}
void launch_flip_conv_weights(const float* W, float* Wk, int c_out, int c_in, cudaStream_t s) {
  const int cnt = c_out * c_in * 9;
  if (cnt <= 0) return;
  flip_conv_weights_kernel<<<ceil_div(cnt, 256), 256, 0, s>>>(W, Wk, c_out, c_in);
}

int conv_s2_supported(int c_in, int h, int w, int c_out, int kh, int kw, int stride, int pad, int ho, int wo) {
  (void)c_in; (void)c_out;
  return kh == 3 && kw == 3 && stride == 2 && pad == 1 && h == 2 * ho && w == 2 * wo && ho * wo <= 256 && ho * wo >= 16 &&
         (ho + 1) * (wo + 1) <= 512;
}

static bool launch_conv_bwd_3x3s2(const AView& A, const float* W, const float* addend, float* out, int B, int R,
                                  int c_in, int h, int w, int c_out, int pad, int ho, int wo, cudaStream_t s) {
  if (!conv_s2_supported(c_in, h, w, c_out, 3, 3, 2, pad, ho, wo)) return false;
  if ((reinterpret_cast<uintptr_t>(out) & 7) || (addend && (reinterpret_cast<uintptr_t>(addend) & 7))) return false;
  // two positions per thread (P = 2) with 8 channels where the map is even-wide and the 16-byte stores are aligned; else one
  // position with 8 / 16 channels
  const bool p2 = (wo % 2 == 0) && ho * (wo / 2) >= 8 && !(reinterpret_cast<uintptr_t>(out) & 15) &&
                  !(addend && (reinterpret_cast<uintptr_t>(addend) & 15));
  const int CT = p2 ? 8 : ((c_in % 16 == 0) ? 16 : 8);
  const int PT = p2 ? ho * (wo / 2) : ho * wo;
  const int groups = (c_in + CT - 1) / CT;
  int CG = 256 / PT < groups ? 256 / PT : groups;
  if (CG < 1) CG = 1;
  int RB = 256 / (PT * CG);
  if (RB < 1) RB = 1;
  if (RB > 4) RB = 4;
  const int tile = (ho + 1) * (wo + 1);
  if (tile > 2 * 256) return false;
  const size_t per_co = ((size_t)9 * CG * CT + (size_t)RB * tile) * sizeof(float);
  int COC = (int)((44 * 1024) / per_co);           // two stages of <= 44 KB, two blocks per SM
  if (COC < 1) return false;
  if (COC > c_out) COC = c_out;
  const int stage_floats = (int)((per_co * COC / sizeof(float) + 3) / 4 * 4);
  const size_t smem = (size_t)2 * stage_floats * sizeof(float);
  const long long rows = 2LL * B * R;
  const int threads = 256;                          // the element -> thread map of the staging assumes blockDim = 256
  dim3 grid((unsigned)((rows + RB - 1) / RB), (unsigned)((groups + CG - 1) / CG));
  if (p2) conv_bwd_3x3s2_kernel<8, 2><<<grid, threads, smem, s>>>(A.p, A.sBr, A.sB, A.ld, B, R, W, addend, out, c_in, c_out, ho, wo, COC, CG, RB, stage_floats);
  else if (CT == 16) conv_bwd_3x3s2_kernel<16, 1><<<grid, threads, smem, s>>>(A.p, A.sBr, A.sB, A.ld, B, R, W, addend, out, c_in, c_out, ho, wo, COC, CG, RB, stage_floats);
  else conv_bwd_3x3s2_kernel<8, 1><<<grid, threads, smem, s>>>(A.p, A.sBr, A.sB, A.ld, B, R, W, addend, out, c_in, c_out, ho, wo, COC, CG, RB, stage_floats);
  return true;
}

// rows / columns of the input map that no output pixel reaches (h > stride * ho) are zero-filled by this launcher's caller
// contract: supported only when stride * ho >= h and stride * wo >= w, i.e. every input pixel belongs to some s x s block
static bool launch_conv_bwd_1x1(const AView& A, const float* W, const float* addend, float* out, int B, int R,
                                int c_in, int h, int w, int c_out, int stride, int pad, int ho, int wo, cudaStream_t s) {
  if (pad != 0 || stride < 1 || stride * ho < h || stride * wo < w || c_in > 64 || c_out > 64) return false;
  const long long rows = 2LL * B * R;
  if (rows > 65535) return false;
  const int npix = ho * wo;
  int PIX = 256;
  while (PIX > 32 && PIX / 2 >= npix) PIX /= 2;
  const int groups = 256 / PIX;                                   // channel groups per block
  int cip = (c_in + groups - 1) / groups;
  cip = cip <= 4 ? 4 : (cip <= 8 ? 8 : 16);
  if ((long long)cip * groups < c_in) return false;
  const size_t smem = ((size_t)c_out * c_in + (size_t)c_out * PIX) * sizeof(float);
  if (smem > 96 * 1024) return false;
  dim3 grid((unsigned)((npix + PIX - 1) / PIX), (unsigned)rows);
  const int vec = (npix % 4 == 0) && (PIX % 4 == 0) && ((c_out * c_in) % 4 == 0) && (A.ld % 4 == 0) && (A.sB % 4 == 0) &&
                  (A.sBr % 4 == 0) && ((reinterpret_cast<uintptr_t>(A.p) & 15) == 0);
  auto go = [&](auto kern) {
    kern<<<grid, 256, smem, s>>>(A.p, A.sBr, A.sB, A.ld, B, R, W, addend, out, c_in, h, w, c_out, stride, ho, wo, PIX, vec);
  };
  if (cip == 4) go(conv_bwd_1x1_kernel<4>);
  else if (cip == 8) go(conv_bwd_1x1_kernel<8>);
  else go(conv_bwd_1x1_kernel<16>);
  return true;
}

void launch_conv_transpose(const AView& A, const float* W, const float* addend, float* out, int B, int R,
                           int c_in, int h, int w, int c_out, int kh, int kw, int stride, int pad, int ho,
                           int wo, cudaStream_t s, int allow_tc, int num_sms) {
  long long rows = 2LL * B * R;
  if (rows <= 0) return;
  if (allow_tc && conv_tc_supported(c_in, h, w, c_out, kh, kw, stride, pad, ho, wo) &&
      launch_conv_transpose_tc(A, W, addend, out, B, R, c_in, h, w, c_out, num_sms, s) == 0) return;
  if ((A.sB % 1 == 0) && rows < (1LL << 31)) {
    bool done = false;
    if (kh == 1 && kw == 1 && launch_conv_bwd_1x1(A, W, addend, out, B, R, c_in, h, w, c_out, stride, pad, ho, wo, s)) return;
    if (kh == 3 && kw == 3 && stride == 1 && launch_conv_bwd_3x3s1(A, W, addend, out, B, R, c_in, h, w, c_out, pad, ho, wo, s)) done = true;
    else if (kh == 3 && kw == 3 && stride == 1) done = launch_conv_bwd_ct<3, 3, 1>(A, W, addend, out, B, R, c_in, h, w, c_out, pad, ho, wo, s);
    else if (kh == 3 && kw == 3 && stride == 2 && launch_conv_bwd_3x3s2(A, W, addend, out, B, R, c_in, h, w, c_out, pad, ho, wo, s)) done = true;
    else if (kh == 3 && kw == 3 && stride == 2) done = launch_conv_bwd_ct<3, 3, 2>(A, W, addend, out, B, R, c_in, h, w, c_out, pad, ho, wo, s);
    else if (kh == 1 && kw == 1 && stride == 1) done = launch_conv_bwd_ct<1, 1, 1>(A, W, addend, out, B, R, c_in, h, w, c_out, pad, ho, wo, s);
    else if (kh == 1 && kw == 1 && stride == 2) done = launch_conv_bwd_ct<1, 1, 2>(A, W, addend, out, B, R, c_in, h, w, c_out, pad, ho, wo, s);
    if (done) return;
  }
  int threads = 256;
  while (threads > 32 && threads / 2 >= h * w) threads /= 2;
  dim3 grid(ceil_div(h * w, threads), c_in, (unsigned)(rows < 32768 ? rows : 32768));
  size_t smem = (size_t)c_out * kh * kw * sizeof(float);
  conv_transpose_kernel<<<grid, threads, smem, s>>>(A.p, A.sBr, A.sB, A.ld, B, R, W, addend, out, c_in, h, w,
                                                    c_out, kh, kw, stride, pad, ho, wo);
}

int conv_init_device() {
  const int b1 = 96 * 1024;
  if (cudaFuncSetAttribute(conv_bwd_3x3s1_kernel<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, b1) != cudaSuccess ||
      cudaFuncSetAttribute(conv_bwd_3x3s1_kernel<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, b1) != cudaSuccess ||
      cudaFuncSetAttribute(conv_bwd_3x3s1_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, b1) != cudaSuccess) return -1;
  if (cudaFuncSetAttribute(conv_bwd_3x3s2_kernel<16, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, b1) != cudaSuccess ||
      cudaFuncSetAttribute(conv_bwd_3x3s2_kernel<8, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, b1) != cudaSuccess ||
      cudaFuncSetAttribute(conv_bwd_3x3s2_kernel<8, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, b1) != cudaSuccess) return -1;
  if (cudaFuncSetAttribute(conv_bwd_1x1_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, b1) != cudaSuccess ||
      cudaFuncSetAttribute(conv_bwd_1x1_kernel<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, b1) != cudaSuccess ||
      cudaFuncSetAttribute(conv_bwd_1x1_kernel<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, b1) != cudaSuccess) return -1;
  return (conv_bwd_set_attr<3, 3, 1>() && conv_bwd_set_attr<3, 3, 2>() && conv_bwd_set_attr<1, 1, 1>() &&
          conv_bwd_set_attr<1, 1, 2>()) ? 0 : -1;
}

}  // namespace crownb200
