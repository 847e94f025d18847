// HBM-bound kernels of the CROWN hot path (SURVEY.md sec. 8(a) rows a3, a4, a8, a9 and helpers).
// Every kernel here streams its operands once with 128-bit coalesced accesses; row reductions use
// warp shuffles (one warp owns a row pair, so bias accumulation needs no atomics).
#include "common.cuh"
#include "kernels.h"

namespace crownb200 {

// ------------------------------------------------------------------------------------------------
// a3 -- relaxation coefficients.  Classification order active -> inactive -> unstable
// (reading G3); adaptive rule lambda = 1 iff u > -l (reading G4).
// ------------------------------------------------------------------------------------------------
__global__ void relax_coeffs_kernel(const float* __restrict__ l, const float* __restrict__ u,
                                    float4* __restrict__ coef, long long count, int rule,
                                    const int8_t* __restrict__ split) {
  long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= count) return;
  float lo = l[i], hi = u[i];
  if (split) {                      // BaB sub-domain (reading G26): the fixed state clamps the interval
    const int sg = split[i];
    if (sg > 0) lo = fmaxf(lo, 0.f); else if (sg < 0) hi = fminf(hi, 0.f);
  }
  float4 c;
  if (lo >= 0.f) {
    c = make_float4(1.f, 0.f, 1.f, 0.f);
  } else if (hi <= 0.f) {
    c = make_float4(0.f, 0.f, 0.f, 0.f);
  } else {
    float den = hi - lo;
    float dU = hi / den;
    float bU = (-lo * hi) / den;
    float dL = rule == 0 ? (hi > -lo ? 1.f : 0.f) : (rule == 2 ? 1.f : 0.f);
    c = make_float4(dU, bU, dL, 1.f);
  }
  coef[i] = c;
}

void launch_relax_coeffs(const float* l, const float* u, float4* coef, long long count, int rule, cudaStream_t s,
                         const int8_t* split) {
  if (count <= 0) return;
  int threads = 256;
  relax_coeffs_kernel<<<ceil_div(count, threads), threads, 0, s>>>(l, u, coef, count, rule, split);
}

// ------------------------------------------------------------------------------------------------
// a4 -- fused relaxation.  One warp owns one (property b, row r) pair and walks the neuron axis for
// BOTH branches, so the coefficient vectors and alpha are read once per pair.
//   lower: Abar = A+ * dL + A- * dU,  d += A- . bU        (Eq. 1)
//   upper: Abar = A+ * dU + A- * dL,  d += A+ . bU
//   both : d += Abar . bias           (bias of the linear layer the contraction goes through next)
// ------------------------------------------------------------------------------------------------
struct RelaxDev {
  const float* A; long long sBr, sB, ld;
  const float4* coef;
  const float* alpha_lo; const float* alpha_up;
  const float* bias; int bias_div;
  float* out; float* out_lo; float* d;
  int B, R, n;
  const int8_t* split; const float* beta_lo; const float* beta_up;   // NEXT-2 (BETA instantiations only)
  int wpp;      // warps per (b, r) pair: 1, 2, 4 or 8 (all in one block); a function of n ONLY, so that the summation
                // order of d does not depend on how the rows are chunked (chunked == unchunked bitwise)
};

// long rows with few (b, r) pairs (cfg5: 792 pairs of 16384 neurons) leave most SMs idle with one warp per pair
static inline int warps_per_pair(int n) { return n >= 4096 ? 8 : (n >= 2048 ? 4 : (n >= 1024 ? 2 : 1)); }

__device__ __forceinline__ float clip01(float a) { return fminf(fmaxf(a, 0.f), 1.f); }

// one element, both branches.  Returns contributions to d.
// btL / btU: the beta-CROWN terms max(beta_lo, 0) * s and max(beta_up, 0) * s of this element (0 without a split)
template <bool RELU, bool ALPHA>
__device__ __forceinline__ void relax_elem(float aL, float aU, const float4& c, float alL, float alU,
                                           float bias, float& oL, float& oU, float& dLacc, float& dUacc,
                                           float btL = 0.f, float btU = 0.f) {
  if (RELU) {
    float dU = c.x, bU = c.y;
    float sL = c.z, sU = c.z;
    if (ALPHA) {
      if (c.w != 0.f) { sL = clip01(alL); sU = clip01(alU); }
    }
    float pL = fmaxf(aL, 0.f), mL = fminf(aL, 0.f);
    float pU = fmaxf(aU, 0.f), mU = fminf(aU, 0.f);
    oL = pL * sL + mL * dU - btL;
    oU = pU * dU + mU * sU + btU;
    dLacc = fmaf(mL, bU, dLacc);
    dUacc = fmaf(pU, bU, dUacc);
  } else {
    oL = aL; oU = aU;
  }
  dLacc = fmaf(oL, bias, dLacc);
  dUacc = fmaf(oU, bias, dUacc);
}

template <bool RELU, bool ALPHA, bool SPLIT, int VEC, bool BETA = false>
__global__ void __launch_bounds__(256) relax_kernel(RelaxDev p) {
  const int lane = threadIdx.x & 31;
  const int wpp = p.wpp;
  const long long warp = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const long long pair_raw = warp / wpp;
  const int wi = (int)(warp % wpp);                       // this warp's slice of the row
  const bool valid = pair_raw < (long long)p.B * p.R;
  const int n_eff = valid ? p.n : 0;
  // warps are dealt to (property, row) pairs property-major.  At the start of a pass the input rows are shared by all
  // properties (rows of W_k, zero-stride view) and come from DRAM once per property (ncu, cfg3: 10.4 GB read for 0.65 GB of
  // distinct input).  Two orders that remove those re-reads were measured and dropped: single rows round robin over the
  // properties (3-7 % slower: the writes scatter over B distant rows) and groups of rows small enough to stay in L2 with
  // every property writing a whole group (1-3 % slower).  The kernel is bound by its STORES -- 41.6 GB in 8.59 ms = 4.8 TB/s
  // of writes on cfg3 -- and the re-reads ride along for free.
  const long long pair = valid ? pair_raw : 0;
  const int b = (int)(pair / p.R), r = (int)(pair % p.R);
  const float* a0 = p.A + (long long)b * p.sB + (long long)r * p.ld;
  const float* a1 = a0 + p.sBr;
  const float4* cf = RELU ? p.coef + (long long)b * p.n : nullptr;
  const long long arow = ((long long)b * p.R + r) * p.n;
  const float* alL = ALPHA ? p.alpha_lo + arow : nullptr;
  const float* alU = ALPHA ? p.alpha_up + arow : nullptr;
  const int8_t* sp = BETA ? p.split + (long long)b * p.n : nullptr;
  const float* btL = (BETA && p.beta_lo) ? p.beta_lo + arow : nullptr;
  const float* btU = (BETA && p.beta_up) ? p.beta_up + arow : nullptr;
  const long long BR = (long long)p.B * p.R;
  float* o0 = p.out + (pair) * (long long)p.n;
  float* o1 = p.out + (BR + pair) * (long long)p.n;
  float* q0 = SPLIT ? p.out_lo + (pair) * (long long)p.n : nullptr;
  float* q1 = SPLIT ? p.out_lo + (BR + pair) * (long long)p.n : nullptr;
  float accL = 0.f, accU = 0.f;

  if (VEC == 4) {
    for (int j = (wi * 32 + lane) * 4; j < n_eff; j += wpp * 128) {
      float4 xL = ldg_stream4(a0 + j);
      float4 xU = ldg_stream4(a1 + j);
      float4 c0 = make_float4(0, 0, 0, 0), c1 = c0, c2 = c0, c3 = c0;
      if (RELU) { c0 = __ldg(cf + j); c1 = __ldg(cf + j + 1); c2 = __ldg(cf + j + 2); c3 = __ldg(cf + j + 3); }
      float4 tL = make_float4(0, 0, 0, 0), tU = tL;
      if (ALPHA) {
        tL = ldg_stream4(alL + j);
        tU = (alU == alL) ? tL : ldg_stream4(alU + j);
      }
      float4 bs = make_float4(0, 0, 0, 0);
      if (p.bias) {
        if (p.bias_div == 1) bs = __ldg(reinterpret_cast<const float4*>(p.bias + j));
        else { bs.x = __ldg(p.bias + (j) / p.bias_div); bs.y = __ldg(p.bias + (j + 1) / p.bias_div);
               bs.z = __ldg(p.bias + (j + 2) / p.bias_div); bs.w = __ldg(p.bias + (j + 3) / p.bias_div); }
      }
      float4 yL, yU;
      float4 eL = make_float4(0, 0, 0, 0), eU = eL;
      if (BETA) {
        const char4 sg = *reinterpret_cast<const char4*>(sp + j);
        if (btL) { const float4 v = ldg_stream4(btL + j);
                   eL = make_float4(fmaxf(v.x, 0.f) * sg.x, fmaxf(v.y, 0.f) * sg.y, fmaxf(v.z, 0.f) * sg.z, fmaxf(v.w, 0.f) * sg.w); }
        if (btU) { const float4 v = (btU == btL) ? ldg_stream4(btL + j) : ldg_stream4(btU + j);
                   eU = make_float4(fmaxf(v.x, 0.f) * sg.x, fmaxf(v.y, 0.f) * sg.y, fmaxf(v.z, 0.f) * sg.z, fmaxf(v.w, 0.f) * sg.w); }
      }
      relax_elem<RELU, ALPHA>(xL.x, xU.x, c0, tL.x, tU.x, bs.x, yL.x, yU.x, accL, accU, eL.x, eU.x);
      relax_elem<RELU, ALPHA>(xL.y, xU.y, c1, tL.y, tU.y, bs.y, yL.y, yU.y, accL, accU, eL.y, eU.y);
      relax_elem<RELU, ALPHA>(xL.z, xU.z, c2, tL.z, tU.z, bs.z, yL.z, yU.z, accL, accU, eL.z, eU.z);
      relax_elem<RELU, ALPHA>(xL.w, xU.w, c3, tL.w, tU.w, bs.w, yL.w, yU.w, accL, accU, eL.w, eU.w);
      if (SPLIT) {
        float4 hL, lL, hU, lU;
        tf32_split(yL.x, hL.x, lL.x); tf32_split(yL.y, hL.y, lL.y);
        tf32_split(yL.z, hL.z, lL.z); tf32_split(yL.w, hL.w, lL.w);
        tf32_split(yU.x, hU.x, lU.x); tf32_split(yU.y, hU.y, lU.y);
        tf32_split(yU.z, hU.z, lU.z); tf32_split(yU.w, hU.w, lU.w);
        stg_stream4(o0 + j, hL); stg_stream4(q0 + j, lL);
        stg_stream4(o1 + j, hU); stg_stream4(q1 + j, lU);
      } else {
        stg_stream4(o0 + j, yL);
        stg_stream4(o1 + j, yU);
      }
    }
  } else {
    for (int j = wi * 32 + lane; j < n_eff; j += wpp * 32) {
      float xL = a0[j], xU = a1[j];
      float4 c = RELU ? cf[j] : make_float4(0, 0, 0, 0);
      float tL = ALPHA ? alL[j] : 0.f, tU = ALPHA ? alU[j] : 0.f;
      float bs = p.bias ? p.bias[j / p.bias_div] : 0.f;
      float yL, yU;
      float eL = 0.f, eU = 0.f;
      if (BETA) {
        const float sg = (float)sp[j];
        if (btL) eL = fmaxf(btL[j], 0.f) * sg;
        if (btU) eU = fmaxf(btU[j], 0.f) * sg;
      }
      relax_elem<RELU, ALPHA>(xL, xU, c, tL, tU, bs, yL, yU, accL, accU, eL, eU);
      if (SPLIT) {
        float h, l2;
        tf32_split(yL, h, l2); o0[j] = h; q0[j] = l2;
        tf32_split(yU, h, l2); o1[j] = h; q1[j] = l2;
      } else { o0[j] = yL; o1[j] = yU; }
    }
  }
  accL = warp_sum(accL);
  accU = warp_sum(accU);
  if (wpp == 1) {
    if (valid && lane == 0 && p.d) {
      p.d[pair] += accL;
      p.d[BR + pair] += accU;
    }
    return;
  }
  __shared__ float red[8][2];
  const int w = threadIdx.x >> 5;
  if (lane == 0) { red[w][0] = accL; red[w][1] = accU; }
  __syncthreads();
  if (valid && wi == 0 && lane == 0 && p.d) {             // slices added in slice order: deterministic
    float sL = red[w][0], sU = red[w][1];
    for (int k = 1; k < wpp; ++k) { sL += red[w + k][0]; sU += red[w + k][1]; }
    p.d[pair] += sL;
    p.d[BR + pair] += sU;
  }
}

template <bool RELU, bool ALPHA, bool SPLIT>
static void relax_dispatch_vec(const RelaxDev& p, bool vec, int blocks, cudaStream_t s) {
  if (RELU && p.split) {          // beta-CROWN term (NEXT-2)
    if (vec) relax_kernel<RELU, ALPHA, SPLIT, 4, RELU><<<blocks, 256, 0, s>>>(p);
    else relax_kernel<RELU, ALPHA, SPLIT, 1, RELU><<<blocks, 256, 0, s>>>(p);
    return;
  }
  if (vec) relax_kernel<RELU, ALPHA, SPLIT, 4><<<blocks, 256, 0, s>>>(p);
  else relax_kernel<RELU, ALPHA, SPLIT, 1><<<blocks, 256, 0, s>>>(p);
}

void launch_relax(const RelaxArgs& a, cudaStream_t s) {
  RelaxDev p;
  p.A = a.A.p; p.sBr = a.A.sBr; p.sB = a.A.sB; p.ld = a.A.ld;
  p.coef = a.coef; p.alpha_lo = a.alpha_lo; p.alpha_up = a.alpha_up ? a.alpha_up : a.alpha_lo;
  if (!p.alpha_lo) p.alpha_lo = p.alpha_up;
  p.bias = a.bias; p.bias_div = a.bias_div > 0 ? a.bias_div : 1;
  p.out = a.out; p.out_lo = a.out_lo; p.d = a.d; p.B = a.B; p.R = a.R; p.n = a.n;
  p.split = (a.coef && (a.beta_lo || a.beta_up)) ? a.split : nullptr; p.beta_lo = a.beta_lo; p.beta_up = a.beta_up;
  long long pairs = (long long)a.B * a.R;
  if (pairs <= 0 || a.n <= 0) return;
  p.wpp = warps_per_pair(a.n);
  int blocks = ceil_div(pairs * p.wpp * 32, 256);
  auto al16 = [](const void* q) { return (reinterpret_cast<uintptr_t>(q) & 15) == 0; };
  bool vec = (a.n % 4 == 0) && (p.ld % 4 == 0) && (p.sB % 4 == 0) && (p.sBr % 4 == 0) && al16(p.A) &&
             al16(p.out) && (!p.out_lo || al16(p.out_lo)) && (!p.alpha_lo || al16(p.alpha_lo)) &&
             (!p.alpha_up || al16(p.alpha_up)) && (!p.bias || p.bias_div != 1 || al16(p.bias)) &&
             (!p.split || ((reinterpret_cast<uintptr_t>(p.split) & 3) == 0 && (!p.beta_lo || al16(p.beta_lo)) &&
                           (!p.beta_up || al16(p.beta_up))));
  bool relu = a.coef != nullptr, alpha = relu && p.alpha_lo != nullptr, split = a.out_lo != nullptr;
#define CROWN_RELAX_CASE(R_, A_, S_) relax_dispatch_vec<R_, A_, S_>(p, vec, blocks, s)
  if (relu) {
    if (alpha) { if (split) CROWN_RELAX_CASE(true, true, true); else CROWN_RELAX_CASE(true, true, false); }
    else       { if (split) CROWN_RELAX_CASE(true, false, true); else CROWN_RELAX_CASE(true, false, false); }
  } else {
    if (split) CROWN_RELAX_CASE(false, false, true); else CROWN_RELAX_CASE(false, false, false);
  }
#undef CROWN_RELAX_CASE
}

// ------------------------------------------------------------------------------------------------
// a8 -- concretisation.  One warp per (b, r) pair, both branches (x_c, x_r shared).
// ------------------------------------------------------------------------------------------------
template <int VEC>
__global__ void __launch_bounds__(256) concretize_kernel(const float* __restrict__ A, long long sBr,
                                                         long long sB, long long ld, int n,
                                                         const float* __restrict__ d,
                                                         const float* __restrict__ x_lo,
                                                         const float* __restrict__ x_hi,
                                                         float* __restrict__ lb, float* __restrict__ ub,
                                                         int out_stride, int B, int R) {
  const int lane = threadIdx.x & 31;
  const long long pair = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (pair >= (long long)B * R) return;
  const int b = (int)(pair / R), r = (int)(pair % R);
  const float* a0 = A + (long long)b * sB + (long long)r * ld;
  const float* a1 = a0 + sBr;
  const float* xl = x_lo + (long long)b * n;
  const float* xh = x_hi + (long long)b * n;
  float dotL = 0.f, absL = 0.f, dotU = 0.f, absU = 0.f;
  if (VEC == 4) {
    for (int j = lane * 4; j < n; j += 128) {
      float4 vL = ldg_stream4(a0 + j), vU = ldg_stream4(a1 + j);
      float4 lo = __ldg(reinterpret_cast<const float4*>(xl + j));
      float4 hi = __ldg(reinterpret_cast<const float4*>(xh + j));
      float cx = 0.5f * (lo.x + hi.x), rx = 0.5f * (hi.x - lo.x);
      float cy = 0.5f * (lo.y + hi.y), ry = 0.5f * (hi.y - lo.y);
      float cz = 0.5f * (lo.z + hi.z), rz = 0.5f * (hi.z - lo.z);
      float cw = 0.5f * (lo.w + hi.w), rw = 0.5f * (hi.w - lo.w);
      dotL = fmaf(vL.x, cx, dotL); absL = fmaf(fabsf(vL.x), rx, absL);
      dotL = fmaf(vL.y, cy, dotL); absL = fmaf(fabsf(vL.y), ry, absL);
      dotL = fmaf(vL.z, cz, dotL); absL = fmaf(fabsf(vL.z), rz, absL);
      dotL = fmaf(vL.w, cw, dotL); absL = fmaf(fabsf(vL.w), rw, absL);
      dotU = fmaf(vU.x, cx, dotU); absU = fmaf(fabsf(vU.x), rx, absU);
      dotU = fmaf(vU.y, cy, dotU); absU = fmaf(fabsf(vU.y), ry, absU);
      dotU = fmaf(vU.z, cz, dotU); absU = fmaf(fabsf(vU.z), rz, absU);
      dotU = fmaf(vU.w, cw, dotU); absU = fmaf(fabsf(vU.w), rw, absU);
    }
  } else {
    for (int j = lane; j < n; j += 32) {
      float vL = a0[j], vU = a1[j];
      float c = 0.5f * (xl[j] + xh[j]), rr = 0.5f * (xh[j] - xl[j]);
      dotL = fmaf(vL, c, dotL); absL = fmaf(fabsf(vL), rr, absL);
      dotU = fmaf(vU, c, dotU); absU = fmaf(fabsf(vU), rr, absU);
    }
  }
  dotL = warp_sum(dotL); absL = warp_sum(absL);
  dotU = warp_sum(dotU); absU = warp_sum(absU);
  if (lane == 0) {
    const long long BR = (long long)B * R;
    float dl = d ? d[pair] : 0.f, du = d ? d[BR + pair] : 0.f;
    lb[(long long)b * out_stride + r] = (dotL - absL) + dl;
    ub[(long long)b * out_stride + r] = (dotU + absU) + du;
  }
}

void launch_concretize(const AView& A, const float* d, const float* x_lo, const float* x_hi,
                       float* lb, float* ub, int out_stride, int B, int R, cudaStream_t s) {
  long long pairs = (long long)B * R;
  if (pairs <= 0) return;
  int blocks = ceil_div(pairs * 32, 256);
  auto al16 = [](const void* q) { return (reinterpret_cast<uintptr_t>(q) & 15) == 0; };
  bool vec = (A.n % 4 == 0) && (A.ld % 4 == 0) && (A.sB % 4 == 0) && (A.sBr % 4 == 0) && al16(A.p) &&
             al16(x_lo) && al16(x_hi);
  if (vec) concretize_kernel<4><<<blocks, 256, 0, s>>>(A.p, A.sBr, A.sB, A.ld, A.n, d, x_lo, x_hi, lb, ub, out_stride, B, R);
  else concretize_kernel<1><<<blocks, 256, 0, s>>>(A.p, A.sBr, A.sB, A.ld, A.n, d, x_lo, x_hi, lb, ub, out_stride, B, R);
}

// a8, second half of the fused form: add the per-piece (dot, |.|) pairs written by the contraction epilogue in
// index order and finish lb = dot - ab + d (branch 0), ub = dot + ab + d (branch 1).
__global__ void concretize_parts_kernel(const float2* __restrict__ part, int parts, const float* __restrict__ d,
                                        float* __restrict__ lb, float* __restrict__ ub, int out_stride, int B, int R) {
  const long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long BR = (long long)B * R;
  if (m >= 2 * BR) return;
  float dot = 0.f, ab = 0.f;
  for (int i = 0; i < parts; ++i) { const float2 v = part[m * parts + i]; dot += v.x; ab += v.y; }
  const int br = (int)(m / BR);
  const long long pair = m % BR;
  const int b = (int)(pair / R), r = (int)(pair % R);
  const float dd = d ? d[m] : 0.f;
  if (br == 0) lb[(long long)b * out_stride + r] = (dot - ab) + dd;
  else ub[(long long)b * out_stride + r] = (dot + ab) + dd;
}
void launch_concretize_parts(const float* part, int parts, const float* d, float* lb, float* ub, int out_stride,
                             int B, int R, cudaStream_t s) {
  const long long rows = 2LL * B * R;
  if (rows <= 0) return;
  concretize_parts_kernel<<<ceil_div(rows, 256), 256, 0, s>>>(reinterpret_cast<const float2*>(part), parts, d, lb, ub,
                                                             out_stride, B, R);
}

// d[m] += sum_i part[m*parts + i], i ascending: the per-piece d contributions written by the relaxing epilogue of the
// contraction (a4 fused).  One thread per row; fixed order, so the result does not depend on the tiling.
__global__ void reduce_parts_kernel(const float* __restrict__ part, int parts, float* __restrict__ d, long long rows) {
  const long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (m >= rows) return;
  const float* p = part + m * parts;
  float acc = 0.f;
  for (int i = 0; i < parts; ++i) acc += p[i];
  d[m] += acc;
}
void launch_reduce_parts(const float* part, int parts, float* d, long long rows, cudaStream_t s) {
  if (rows <= 0 || parts <= 0) return;
  reduce_parts_kernel<<<ceil_div(rows, 128), 128, 0, s>>>(part, parts, d, rows);
}

// ------------------------------------------------------------------------------------------------
// helpers
// ------------------------------------------------------------------------------------------------
__global__ void init_d_kernel(float* d, const float* bias, int row0, int B, int R) {
  long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  long long tot = 2LL * B * R;
  if (i >= tot) return;
  int r = (int)(i % R);
  d[i] = bias ? bias[row0 + r] : 0.f;
}
void launch_init_d(float* d, const float* bias, int row0, int B, int R, cudaStream_t s) {
  long long tot = 2LL * B * R;
  if (tot <= 0) return;
  init_d_kernel<<<ceil_div(tot, 256), 256, 0, s>>>(d, bias, row0, B, R);
}

__global__ void __launch_bounds__(256) rowdot_bias_kernel(const float* __restrict__ A, const float* __restrict__ Alo,
                                                          long long sBr, long long sB, long long ld, int n,
                                                          const float* __restrict__ bias, int bias_div,
                                                          float* d, int B, int R, int wpp) {
  const int lane = threadIdx.x & 31;
  const long long warp = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const long long m_raw = warp / wpp;
  const int wi = (int)(warp % wpp);
  const long long BR = (long long)B * R;
  const bool valid = m_raw < 2 * BR;
  const long long m = valid ? m_raw : 0;
  if (!valid) n = 0;
  int br = (int)(m / BR);
  long long pair = m % BR;
  int b = (int)(pair / R), r = (int)(pair % R);
  const long long off = br * sBr + (long long)b * sB + (long long)r * ld;
  const float* a = A + off;
  float acc = 0.f;
  if (Alo) {            // view carries a TF32 lo limb: the value is hi + lo
    const float* al = Alo + off;
    for (int j = wi * 32 + lane; j < n; j += wpp * 32) acc = fmaf(a[j] + al[j], bias[j / bias_div], acc);
  } else {
    for (int j = wi * 32 + lane; j < n; j += wpp * 32) acc = fmaf(a[j], bias[j / bias_div], acc);
  }
  acc = warp_sum(acc);
  if (wpp == 1) { if (valid && lane == 0) d[m] += acc; return; }
  __shared__ float red[8];
  const int w = threadIdx.x >> 5;
  if (lane == 0) red[w] = acc;
  __syncthreads();
  if (valid && wi == 0 && lane == 0) {
    float sacc = red[w];
    for (int k = 1; k < wpp; ++k) sacc += red[w + k];
    d[m] += sacc;
  }
}
void launch_rowdot_bias(const AView& A, const float* bias, int bias_div, float* d, int B, int R,
                        cudaStream_t s) {
  long long rows = 2LL * B * R;
  if (rows <= 0 || !bias) return;
  const int wpp = warps_per_pair(A.n);
  rowdot_bias_kernel<<<ceil_div(rows * wpp * 32, 256), 256, 0, s>>>(A.p, A.lo, A.sBr, A.sB, A.ld, A.n, bias,
                                                                   bias_div > 0 ? bias_div : 1, d, B, R, wpp);
}

// out[m, :] = a[m, :] (+ b[m, :]) for the 2*B*R rows of two strided views; blockIdx.y = row, threads walk the row
// with 128-bit accesses when everything is 16-byte aligned (no per-element index arithmetic).
template <int VEC>
__global__ void __launch_bounds__(256) view_add_kernel(const float* __restrict__ a, const float* __restrict__ a_lo,
                                                       long long aBr, long long aB, long long ald,
                                                       const float* __restrict__ b2, const float* __restrict__ b_lo,
                                                       long long bBr, long long bB, long long bld,
                                                       float* __restrict__ out, int B, int R, int n, long long row_base) {
  const long long m = row_base + blockIdx.y;
  const int r = (int)(m % R);
  const long long t = m / R;
  const int b = (int)(t % B), br = (int)(t / B);
  const long long offa = br * aBr + b * aB + (long long)r * ald;
  const long long offb = br * bBr + b * bB + (long long)r * bld;
  const float* pa = a + offa;
  const float* pal = a_lo ? a_lo + offa : nullptr;        // TF32 lo limbs: the value of a view is hi + lo
  const float* pb = b2 ? b2 + offb : nullptr;
  const float* pbl = (b2 && b_lo) ? b_lo + offb : nullptr;
  float* po = out + m * (long long)n;
  if (VEC == 4) {
    for (int j = (blockIdx.x * blockDim.x + threadIdx.x) * 4; j < n; j += gridDim.x * blockDim.x * 4) {
      float4 v = ldg_stream4(pa + j);
      if (pal) { const float4 w = ldg_stream4(pal + j); v.x += w.x; v.y += w.y; v.z += w.z; v.w += w.w; }
      if (pb) {
        float4 w = ldg_stream4(pb + j);
        if (pbl) { const float4 w2 = ldg_stream4(pbl + j); w.x += w2.x; w.y += w2.y; w.z += w2.z; w.w += w2.w; }
        v.x += w.x; v.y += w.y; v.z += w.z; v.w += w.w;
      }
      stg_stream4(po + j, v);
    }
  } else {
    for (int j = blockIdx.x * blockDim.x + threadIdx.x; j < n; j += gridDim.x * blockDim.x) {
      float v = pa[j];
      if (pal) v += pal[j];
      if (pb) v += pbl ? pb[j] + pbl[j] : pb[j];
      po[j] = v;
    }
  }
}
void launch_view_add(const AView& a, const AView* b, float* out, int B, int R, cudaStream_t s) {
  const long long rows = 2LL * B * R;
  if (rows <= 0 || a.n <= 0) return;
  auto al16 = [](const void* q) { return (reinterpret_cast<uintptr_t>(q) & 15) == 0; };
  auto view_ok = [&](const AView& v) { return al16(v.p) && (!v.lo || al16(v.lo)) && v.ld % 4 == 0 && v.sB % 4 == 0 && v.sBr % 4 == 0; };
  const bool vec = a.n % 4 == 0 && al16(out) && view_ok(a) && (!b || view_ok(*b));
  const int per = vec ? 1024 : 256;                       // elements per block pass
  int gx = ceil_div(a.n, per);
  if (gx > 16) gx = 16;
  for (long long r0 = 0; r0 < rows; r0 += 65535) {        // gridDim.y limit
    const int ny = (int)(rows - r0 < 65535 ? rows - r0 : 65535);
    dim3 grid(gx, ny);
    if (vec) view_add_kernel<4><<<grid, 256, 0, s>>>(a.p, a.lo, a.sBr, a.sB, a.ld, b ? b->p : nullptr, b ? b->lo : nullptr,
                                                   b ? b->sBr : 0, b ? b->sB : 0, b ? b->ld : 0, out, B, R, a.n, r0);
    else view_add_kernel<1><<<grid, 256, 0, s>>>(a.p, a.lo, a.sBr, a.sB, a.ld, b ? b->p : nullptr, b ? b->lo : nullptr,
                                                b ? b->sBr : 0, b ? b->sB : 0, b ? b->ld : 0, out, B, R, a.n, r0);
  }
}

__global__ void verdict_kernel(const float* __restrict__ lb, uint8_t* __restrict__ v, int B, int S) {
  int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= B) return;
  // fail closed: a NaN lower bound compares false, so the property is NOT verified (fminf would drop the NaN)
  bool ok = S > 0;
  for (int s = 0; s < S; ++s) ok = ok && (lb[(long long)b * S + s] > 0.f);
  v[b] = ok ? 1 : 0;
}
__global__ void __launch_bounds__(256) onehot_kernel(float* __restrict__ out, int row0, int R, int n) {
  const long long i = ((long long)blockIdx.x * blockDim.x + threadIdx.x) * 4;
  if (i >= (long long)R * n) return;
  const int r = (int)(i / n), j = (int)(i % n);       // n % 4 == 0 is checked by the launcher (else the scalar path)
  const int hot = row0 + r;
  float4 v = make_float4(j == hot ? 1.f : 0.f, j + 1 == hot ? 1.f : 0.f, j + 2 == hot ? 1.f : 0.f, j + 3 == hot ? 1.f : 0.f);
  *reinterpret_cast<float4*>(out + i) = v;
}
__global__ void __launch_bounds__(256) onehot_scalar_kernel(float* __restrict__ out, int row0, int R, int n) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= (long long)R * n) return;
  out[i] = ((int)(i % n) == row0 + (int)(i / n)) ? 1.f : 0.f;
}
void launch_onehot(float* out, int row0, int R, int n, cudaStream_t s) {
  const long long cnt = (long long)R * n;
  if (cnt <= 0) return;
  if (n % 4 == 0 && (reinterpret_cast<uintptr_t>(out) & 15) == 0) onehot_kernel<<<ceil_div(cnt / 4, 256), 256, 0, s>>>(out, row0, R, n);
  else onehot_scalar_kernel<<<ceil_div(cnt, 256), 256, 0, s>>>(out, row0, R, n);
}

__global__ void bias_sum_kernel(const float* a, const float* b, float* out, int n) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) out[i] = (a ? a[i] : 0.f) + (b ? b[i] : 0.f);
}
void launch_bias_sum(const float* a, const float* b, float* out, int n, cudaStream_t s) {
  if (n <= 0) return;
  bias_sum_kernel<<<ceil_div(n, 128), 128, 0, s>>>(a, b, out, n);
}

void launch_verdict(const float* lb, uint8_t* verified, int B, int S, cudaStream_t s) {
  if (B <= 0) return;
  verdict_kernel<<<ceil_div(B, 128), 128, 0, s>>>(lb, verified, B, S);
}

__global__ void ibp_relu_kernel(const float* l, const float* u, float* lo, float* uo, long long count) {
  long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= count) return;
  lo[i] = fmaxf(l[i], 0.f);
  uo[i] = fmaxf(u[i], 0.f);
}
void launch_ibp_relu(const float* l, const float* u, float* lo, float* uo, long long count, cudaStream_t s) {
  if (count <= 0) return;
  ibp_relu_kernel<<<ceil_div(count, 256), 256, 0, s>>>(l, u, lo, uo, count);
}
__global__ void ibp_add_kernel(const float* l0, const float* u0, const float* l1, const float* u1,
                               float* lo, float* uo, long long count) {
  long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= count) return;
  lo[i] = l0[i] + l1[i];
  uo[i] = u0[i] + u1[i];
}
void launch_ibp_add(const float* l0, const float* u0, const float* l1, const float* u1, float* lo,
                    float* uo, long long count, cudaStream_t s) {
  if (count <= 0) return;
  ibp_add_kernel<<<ceil_div(count, 256), 256, 0, s>>>(l0, u0, l1, u1, lo, uo, count);
}

// X [rows, cols] -> hi/lo TF32 parts; transpose=1 writes [cols, rows] through a 32x33 smem tile.
__global__ void split_tf32_kernel(const float* __restrict__ X, int rows, int cols, int transpose,
                                  float* __restrict__ hi, float* __restrict__ lo) {
  __shared__ float tile[32][33];
  int bx = blockIdx.x * 32, by = blockIdx.y * 32;
  int tx = threadIdx.x, ty = threadIdx.y;  // 32 x 8
  if (!transpose) {
    for (int k = ty; k < 32; k += 8) {
      int r = by + k, c = bx + tx;
      if (r < rows && c < cols) {
        float h, l2;
        tf32_split(X[(long long)r * cols + c], h, l2);
        hi[(long long)r * cols + c] = h;
        lo[(long long)r * cols + c] = l2;
      }
    }
    return;
  }
  for (int k = ty; k < 32; k += 8) {
    int r = by + k, c = bx + tx;
    tile[k][tx] = (r < rows && c < cols) ? X[(long long)r * cols + c] : 0.f;
  }
  __syncthreads();
  for (int k = ty; k < 32; k += 8) {
    int c = bx + k, r = by + tx;  // output [c, r]
    if (r < rows && c < cols) {
      float h, l2;
      tf32_split(tile[tx][k], h, l2);
      hi[(long long)c * rows + r] = h;
      lo[(long long)c * rows + r] = l2;
    }
  }
}
void launch_split_tf32(const float* X, int rows, int cols, int transpose, float* hi, float* lo,
                       cudaStream_t s) {
  if (rows <= 0 || cols <= 0) return;
  dim3 grid(ceil_div(cols, 32), ceil_div(rows, 32)), block(32, 8);
  split_tf32_kernel<<<grid, block, 0, s>>>(X, rows, cols, transpose, hi, lo);
}

}  // namespace crownb200
