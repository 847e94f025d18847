// Host-side launchers of the crownb200 kernels.  One declaration per kernel; each says which step
// of SURVEY.md sec. 8(a) / which passage of PAPER.md it implements.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace crownb200 {

// A strided view of an A-matrix [2, B, R, n] (branch-major).  sBr / sB may be 0 when both branches /
// all properties still share the same rows (start of a pass: A = W_k rows or C.W_L).
struct AView {
  const float* p = nullptr;   // fp32 values (or TF32 "hi" part when lo != nullptr)
  const float* lo = nullptr;  // TF32 "lo" part, same addressing, or nullptr
  long long sBr = 0, sB = 0;  // element strides of the branch and property axes
  long long ld = 0;           // row stride (elements)
  int n = 0;                  // row length
};

// a3 -- relaxation coefficients of a ReLU from its pre-activation bounds.
// coef[b*n+j] = {dU, bU, dL_fixed, unstable?1:0}.  rule: 0 adaptive, 1 zero, 2 one.
// split (NEXT-2; reading G26), int8 [count] or nullptr: +1 clamps l to max(l, 0), -1 clamps u to min(u, 0)
// before the classification, so a split neuron gets the exact line of its fixed state.
void launch_relax_coeffs(const float* l, const float* u, float4* coef, long long count, int rule, cudaStream_t s,
                         const int8_t* split = nullptr);

// a4 -- fused relaxation of A through a ReLU, both branches, with the bias
// accumulation of the ReLU (bU through the sign-selected part of A) and of the linear layer below
// (d += Abar . b), and the TF32 hi/lo operand split for the contraction that follows.
struct RelaxArgs {
  AView A;                   // input view (fp32)
  const float4* coef;        // [B, n] or nullptr: no ReLU here (split / bias only)
  const float* alpha_lo;     // [B, R, n] or nullptr (fixed rule)
  const float* alpha_up;     // [B, R, n] or nullptr
  const float* bias;         // bias of the layer below, [n / bias_div], or nullptr
  int bias_div;              // 1 for Linear; H'*W' for a Conv2d bias per channel
  float* out;                // [2,B,R,n] contiguous: fp32 result, or TF32 hi part when out_lo given
  float* out_lo;             // TF32 lo part or nullptr
  float* d;                  // [2,B,R] in/out: d += ...
  int B, R, n;
  // NEXT-2 -- beta-CROWN split constraints (reading G27): after the relaxation,
  // lower: Abar -= max(beta_lo, 0) * s, upper: Abar += max(beta_up, 0) * s  (the bias term d += Abar . b sees the sum)
  const int8_t* split = nullptr;   // [B, n] in {-1, 0, +1} or nullptr
  const float* beta_lo = nullptr;  // [B, R, n] or nullptr (= 0)
  const float* beta_up = nullptr;
};
void launch_relax(const RelaxArgs& a, cudaStream_t s);

// a8 -- concretisation: lb = A.x_c - |A|.x_r + d (br 0), ub = A.x_c + |A|.x_r + d.
void launch_concretize(const AView& A, const float* d, const float* x_lo, const float* x_hi,
                       float* lb, float* ub, int out_stride, int B, int R, cudaStream_t s);

// a1 -- IBP through a Linear layer in centre/radius form:
// c' = W c + b, r' = |W| r; l' = c' - r', u' = c' + r'.  relu_in: clamp the input interval at 0 first.
// ldo: row pitch of l_out/u_out (= n_out, or the full layer width when W is a streamed row slab).
void launch_ibp_linear(const float* W, const float* bias, const float* l_in, const float* u_in,
                       int relu_in, float* l_out, float* u_out, int B, int n_out, int n_in, int ldo,
                       cudaStream_t s);

// IBP through ReLU / Add (elementwise).
void launch_ibp_relu(const float* l, const float* u, float* lo, float* uo, long long count, cudaStream_t s);
void launch_ibp_add(const float* l0, const float* u0, const float* l1, const float* u1,
                    float* lo, float* uo, long long count, cudaStream_t s);

// out[r, :] = e_{row0 + r} for r < R (row-major [R, n]): identity rows of a start node without a weight matrix (NEXT-3)
void launch_onehot(float* out, int row0, int R, int n, cudaStream_t s);
// d[br,b,r] = bias[row0 + r] (start of an identity pass: d = I . b_k), or 0 when bias == nullptr.
void launch_init_d(float* d, const float* bias, int row0, int B, int R, cudaStream_t s);
// d[br,b,r] += sum_j A[br,b,r,j] * bias[j / bias_div]   (unfused bias of a Linear / Conv2d layer)
void launch_rowdot_bias(const AView& A, const float* bias, int bias_div, float* d, int B, int R,
                        cudaStream_t s);
// out[c] = (a ? a[c] : 0) + (b ? b[c] : 0), c < n (summed conv biases of a residual Add's operands; crown_init)
void launch_bias_sum(const float* a, const float* b, float* out, int n, cudaStream_t s);
// out[2,B,R,n] contiguous = view a (+ view b)
void launch_view_add(const AView& a, const AView* b, float* out, int B, int R, cudaStream_t s);
// a9 -- verdict: verified[b] = min_s lb[b,s] > 0
void launch_verdict(const float* lb, uint8_t* verified, int B, int S, cudaStream_t s);

// X [rows, cols] -> TF32 hi/lo parts, optionally transposed to [cols, rows] (weight prepack).
void launch_split_tf32(const float* X, int rows, int cols, int transpose, float* hi, float* lo,
                       cudaStream_t s);

// a5 fallback -- fp32 FFMA contraction D[M,N] = A[M,K] . W[K,N] (arbitrary shapes, CUDA cores).
void launch_gemm_ffma(const float* A, long long lda, const float* W, long long ldw, float* D,
                      long long ldd, int M, int N, int K, cudaStream_t s);

// a5 -- 3xTF32 contraction on tcgen05 tensor cores (CTA-pair tiles, gemm_tc.cu):
// D[M,N] = (A_hi + A_lo)[M,K] . (Wt_hi + Wt_lo)[N,K]^T with the three products hi.hi + hi.lo + lo.hi accumulated in
// fp32 (TMEM), drained to an fp32 CUDA-core running sum every k_drain elements of K.  Two fused epilogues replace the
// store of D; both need K to be a single panel (gemm_tc_single_panel) and emit one partial sum per (row, 32-column
// piece of the FULL row), which a small kernel adds in index order -- the grouping does not depend on the tiling,
// so N-slabbed (streamed) and row-chunked runs give bitwise the same sums:
//   a8 fused (ConcArgs):     no D; part[(row*parts + piece)] = float2(sum A.x_c, sum |A|.x_r) against the row's box;
//                            launch_concretize_parts finishes lb/ub.  A_0 never reaches HBM.
//   a4 fused (RelaxEpiArgs): D receives the TF32 hi limb and out_lo the lo limb of Abar = relaxation of the product
//                            through the ReLU below (fixed-rule slopes); part[row*parts + piece] = that piece's
//                            contribution to d (A-/+ . bU and Abar . bias); launch_reduce_parts adds them into d.
struct ConcArgs {
  const float* x_lo = nullptr; const float* x_hi = nullptr;   // [B, ldx]
  float* part = nullptr;                                       // [M, parts] float2
  int B = 0, R = 0, parts = 0;
  int ldx = 0;        // row pitch of x_lo / x_hi (the full input width)
  int col_off = 0;    // first input column of this launch (N-slab of a streamed operand), multiple of 32
};
struct RelaxEpiArgs {
  const float4* coef = nullptr;   // [B, coef_ld] {dU, bU, dL, unstable} of the ReLU below
  long long coef_ld = 0;          // = width of the full row (neurons of the ReLU)
  const float* bias = nullptr;    // bias of the Linear below the ReLU [coef_ld] or nullptr
  float* out_lo = nullptr;        // lo limb output, same addressing as D
  float* part = nullptr;          // [M, parts] float
  int B = 0, R = 0, parts = 0;
  int col_off = 0;                // first column of this launch inside the full row, multiple of 32
};
int gemm_tc_parts(int N_total);                // 32-column pieces per row of an N_total-wide output
int gemm_tc_single_panel(int K);               // 1 if the contraction runs as one K panel (fused epilogues allowed)
int gemm_tc_num_panels(int K);                 // kernel launches of one contraction over K
void launch_concretize_parts(const float* part, int parts, const float* d, float* lb, float* ub, int out_stride,
                             int B, int R, cudaStream_t s);
// d[m] += part[m*parts + 0] + part[m*parts + 1] + ... (index order), m < rows
void launch_reduce_parts(const float* part, int parts, float* d, long long rows, cudaStream_t s);
int gemm_tc_supported(int M, int N, int K);
int launch_gemm_tc(const float* A_hi, const float* A_lo, const float* Wt_hi, const float* Wt_lo,
                   float* D, long long ldd, int M, int N, int K, int k_drain, int num_sms,
                   cudaStream_t s, const char** err, const ConcArgs* conc = nullptr,
                   const RelaxEpiArgs* rel = nullptr);

// a2 / a6 -- Conv2d IBP (centre/radius) and conv-transpose backward of A.
void launch_ibp_conv(const float* W, const float* bias, const float* l_in, const float* u_in,
                     int relu_in, float* l_out, float* u_out, int B, int c_in, int h, int w,
                     int c_out, int kh, int kw, int stride, int pad, int ho, int wo, cudaStream_t s);
// allow_tc: 3x3 / stride 1 / pad 1 layers on 16- or 32-wide maps with <= 32 channels run as a per-tap implicit GEMM on
// tcgen05 (conv_tc.cu, 3xTF32); everything else on the CUDA-core kernels of conv.cu.
void launch_conv_transpose(const AView& A, const float* W, const float* addend, float* out,
                           int B, int R, int c_in, int h, int w, int c_out, int kh, int kw,
                           int stride, int pad, int ho, int wo, cudaStream_t s, int allow_tc = 0, int num_sms = 148);
int conv_tc_supported(int c_in, int h, int w, int c_out, int kh, int kw, int stride, int pad, int ho, int wo);
// 3x3 / stride 2 / pad 1 layers with h = 2 ho take the specialised kernel of conv.cu, whose epilogue adds `addend` for free
int conv_s2_supported(int c_in, int h, int w, int c_out, int kh, int kw, int stride, int pad, int ho, int wo);
int launch_conv_transpose_tc(const AView& A, const float* W, const float* addend, float* out, int B, int R,
                             int c_in, int h, int w, int c_out, int num_sms, cudaStream_t s);

// NEXT-1 -- alpha optimisation: kernels of the forward sweep G = d bound / d A (alpha.cu).
void launch_alpha_corner(const float* A0, const float* x_lo, const float* x_hi, float* G, int B, int S, int n0,
                         cudaStream_t s, float* G_lo = nullptr);   // G_lo: write TF32 limbs (only when alpha_corner_limbs_ok)
bool alpha_corner_limbs_ok(const float* A0, const float* x_lo, const float* x_hi, const float* G, const float* G_lo, int n0);
void launch_alpha_linear(const float* G, const float* W, const float* bias, float* D, int M, int N, int K,
                         cudaStream_t s);
void launch_alpha_conv(const float* W, const float* bias, const float* in, float* out, long long M, int c_in, int h,
                       int w, int c_out, int kh, int kw, int stride, int pad, int ho, int wo, cudaStream_t s);
// 3x3 / stride 1 / pad 1 forward conv of M points on the strip kernel of conv.cu (Wk = flipped, role-swapped filters)
int conv3x3s1_points_supported(int c_in, int h, int w, int c_out);
int launch_conv3x3s1_points(const float* in, const float* Wk, float* out, long long M, int c_in, int h, int w, int c_out,
                            cudaStream_t s);
void launch_flip_conv_weights(const float* W, float* Wk, int c_out, int c_in, cudaStream_t s);
// D[i] += bias[(i / div) % N] (div = H*W: per-channel bias of a conv map; div = 1: per-column bias of a Linear output)
void launch_add_bias_div(float* D, const float* bias, long long cnt, int N, int div, cudaStream_t s);
void launch_alpha_add(const float* a, const float* b, float* o, long long cnt, cudaStream_t s);
// D[m, j] += bias[j] for m < M, j < N (bias of a Linear layer after its tensor-core product in the forward sweep)
void launch_add_bias_rows(float* D, const float* bias, long long M, int N, cudaStream_t s);
// split / beta_lo / beta_up / gb_lo / gb_up (NEXT-2, reading G28; all nullptr = alpha only): d lb / d beta_lo = -s * Gin,
// d ub / d beta_up = +s * Gin; step mode: beta <- max(max(beta, 0) +/- step[1] * dir, 0) in place.
void launch_alpha_relu(const float* A, const float* Gin, const float4* coef, float* alpha_lo, float* alpha_up,
                       float* Gout, float* g_lo, float* g_up, const float* step, int mode, int B, int S, int n,
                       cudaStream_t s, const int8_t* split = nullptr, float* beta_lo = nullptr, float* beta_up = nullptr,
                       float* gb_lo = nullptr, float* gb_up = nullptr,
                       const float* gin_bias = nullptr,   // [n]: added to Gin on the fly (the bias of the Linear that made Gin)
                       float* Gout_lo = nullptr);         // non-null: Gout / Gout_lo receive the TF32 limbs of the output
void launch_alpha_best(const float* lb, const float* ub, float* lb_best, float* ub_best, float* step, float decay,
                       int first, int count, cudaStream_t s);
void launch_alpha_set_step(float* step, float v, cudaStream_t s, float v_beta = 0.f);   // step[0] = alpha step, step[1] = beta step

// Per-device kernel attributes (opt-in dynamic shared memory sizes).  cudaFuncSetAttribute applies to the CURRENT
// device only, so crown_init calls this for the device of every new context (a process-wide "done" flag would
// leave a second device without them).  Returns 0 on success.
int gemm_tc_init_device();
int ibp_init_device();
int conv_init_device();
int conv_tc_init_device();
inline int kernels_init_device() { return gemm_tc_init_device() | ibp_init_device() | conv_init_device() | conv_tc_init_device(); }

}  // namespace crownb200
