/* crownb200.h -- C-ABI boundary of the B200-native bound-propagation hot path.
 *
 * What is computed (citations are /root/reference/PAPER.md line + section):
 *   IBP interval forward                          PAPER.md:58-62  (sec. 2.1)
 *   ReLU linear relaxation                        PAPER.md:64     (sec. 2.1)
 *   CROWN / alpha-CROWN backward pass (Eq. 1)     PAPER.md:64-70  (sec. 2.1), :128 (sec. 3.3.2)
 *   concretisation against the L_inf box          PAPER.md:27, :66 (reading G1 in DESIGN.md)
 *   intermediate bounds choose the slopes         PAPER.md:130    (sec. 3.3.2)
 *   verdict
 *
 * Conventions
 *   - Every pointer named *_dev is a DEVICE pointer owned by the CALLER (the Python binding
 *     allocates them as torch tensors).  Pointers named *_host are host pointers.
 *   - The library never calls cudaMalloc: the caller passes ONE device workspace at init;
 *     crown_workspace_bytes() says how large it must be.
 *   - All tensors are dense float32, row-major, no padding.
 *   - Work is issued asynchronously on the CUDA stream given to crown_init; results are valid
 *     after the caller synchronises that stream.  (Host-buffer entry points *_host synchronise
 *     before returning.)
 *   - Every call returns 0 (CROWN_OK) or a negative crown_status; no C++ exception crosses.
 *     crown_last_error() gives the text of the last failure on that context.
 *   - There is no CPU fallback: without a CUDA device every compute call returns CROWN_ECUDA.
 *
 * Row layout of A-matrices and bias vectors ("branch-major"):
 *   A_dev [2, B, R, n]   index ((br*B + b)*R + r)*n + j,  br = 0 lower branch, 1 upper branch
 *   d_dev [2, B, R]
 * Each (br, b, r) row is an independent linear bound  A x + d  (Eq. 1 is row-wise).
 */
#ifndef CROWNB200_H
#define CROWNB200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  CROWN_OK = 0,
  CROWN_EINVAL = -1,       /* bad shape / null pointer / non-topological node list / bad option   */
  CROWN_ENOMEM = -2,       /* workspace smaller than crown_workspace_bytes(), or cap too small    */
  CROWN_ECUDA = -3,        /* CUDA runtime / driver error (sticky); text via crown_last_error     */
  CROWN_EUNSUPPORTED = -4  /* op or graph shape outside Linear/Conv2d/ReLU/Add/Flatten            */
} crown_status;

typedef enum {
  CROWN_LINEAR = 1,  /* y = W x + b,  W [n_out, n_in] row-major                   */
  CROWN_CONV2D = 2,  /* y = conv(x, W) + b, W [c_out, c_in, kh, kw], zero padding, NCHW         */
  CROWN_RELU = 3,    /* y = max(x, 0)                                                            */
  CROWN_ADD = 4,     /* y = in0 + in1 (residual add)                                            */
  CROWN_FLATTEN = 5  /* row-major (C,H,W) -> (C*H*W)                                            */
} crown_op;

/* One node of a topologically ordered DAG.  Producers are node ids < own id; -1 = network input. */
typedef struct {
  int32_t op;                 /* crown_op                                                       */
  int32_t in0, in1;           /* in1 only for CROWN_ADD, else -1                                */
  int32_t n_out, n_in;        /* LINEAR: sizes.  Other ops: filled by the library (may be 0)    */
  int32_t c_out, c_in, kh, kw, stride, pad, h_in, w_in; /* CONV2D                               */
  const float* W_dev;         /* LINEAR [n_out,n_in]; CONV2D [c_out,c_in,kh,kw]; device memory.
                                 May be NULL for a LINEAR layer that is streamed (see W_host)     */
  const float* b_dev;         /* [n_out] / [c_out]; device memory                               */
  const float* W_host;        /* optional PINNED host copy of W (caller-owned, must outlive the context).
                                 With opts.stream_weights != 0 and n_in*n_out >= stream_min_elems
                                 the layer is STREAMED: nothing of it stays resident; IBP copies raw
                                 row slabs from here, the backward pass copies N-slabs of the
                                 prepacked operand the library keeps in its own pinned host memory */
} crown_node;

typedef struct {
  uint64_t mem_cap_bytes;   /* cap on workspace use; 0 = no cap.  Start-spec rows are chunked so
                               that prepacked weights + live A buffers stay below it
                               (single-GPU restatement of Eq. 2)               */
  int32_t stream_weights;   /* 1: LINEAR layers with >= stream_min_elems weights and a W_host are not
                               resident: their GEMM operand is prepacked into pinned host memory at
                               init and copied H2D on a side stream per use through two staging
                               buffers of <= 1 GiB in the workspace ("gather before / free after",
                               PAPER.md:146); results are bitwise those of the resident mode      */
  int32_t mma_scheme;       /* 0 = 3xTF32 on tcgen05 tensor cores (fp32-accurate, never plain
                               TF32); 2 = fp32 FFMA on CUDA cores (debug / odd shapes)           */
  int32_t slope_rule;       /* fixed lower slope for unstable neurons when no alpha is given:
                               0 adaptive (1 iff u > -l, reading G4), 1 all-zero, 2 all-one       */
  int32_t k_drain;          /* 3xTF32: accumulate at most this many K in TMEM before the fp32
                               CUDA-core running sum takes over (0 = library default)            */
  uint64_t stream_min_elems;/* see stream_weights (0 = library default 2^28 elements)            */
  uint64_t stream_stage_bytes; /* size cap of each of the two staging buffers (0 = default 1 GiB) */
  int32_t disable_epi_fusion; /* 0 (default): where a contraction has a single K panel and is followed by a ReLU over a
                               tensor-core Linear with fixed-rule slopes, its epilogue applies that relaxation, both
                               bias accumulations and the TF32 split (a4 fused into a5: A <- A.Lambda_i W_i is ONE
                               kernel).  1: always run the separate relaxation kernel               */
  int32_t disable_conc_fusion; /* 1: always materialise A_0 and run the concretise kernel (default 0: when the
                               last contraction of a pass has a single K panel, concretise in its epilogue) */
  int32_t disable_graph;    /* 0 (default): crown_run captures its launch sequence once per (B, S, pointer set) into
                               a CUDA graph and replays it (the sequence depends on shapes only); 1: plain launches */
  int32_t disable_conv_tc;  /* 0 (default): 3x3 stride-1 BoundConv backward steps on 16/32-wide maps with <= 32 channels run as a
                               per-tap implicit GEMM on the tensor cores (3xTF32); 1: CUDA-core kernel everywhere */
} crown_opts;

typedef struct crown_ctx crown_ctx;   /* opaque; owned by the library; freed by crown_destroy */

/* Bytes of device workspace crown_init needs for batches up to B_max properties and final
 * specs up to S_max rows, under opts (mem_cap_bytes bounds the answer or CROWN_ENOMEM).
 * in_c/in_h/in_w: input shape; for flat inputs pass (n0, 1, 1). */
int crown_workspace_bytes(const crown_node* nodes, int n_nodes, int in_c, int in_h, int in_w,
                          int B_max, int S_max, const crown_opts* opts, size_t* out_bytes);

/* Builds the plan, prepacks GEMM weight operands (transpose + TF32 hi/lo split, a device kernel)
 * into the workspace (or pinned host memory when streaming), creates TMA descriptors.
 * cuda_stream: a cudaStream_t (0 = default stream). */
int crown_init(crown_ctx** out, const crown_node* nodes, int n_nodes, int in_c, int in_h, int in_w,
               int B_max, int S_max, void* workspace_dev, size_t workspace_bytes,
               const crown_opts* opts, void* cuda_stream);

/* O1 -- IBP for B properties with boxes [x_lo, x_hi] ([B, n0] each).
 * l_dev[i], u_dev[i] (arrays of n_nodes device pointers, entries may be NULL = not wanted):
 * interval of node i's OUTPUT, [B, size_i].  If C_dev != NULL ([B,S,n_L]) also writes the IBP
 * bound of C.f(x) with C and the last Linear fused into one layer (reading G10) to
 * lb_dev/ub_dev [B,S]. */
int ibp_forward(crown_ctx* ctx, int B, const float* x_lo_dev, const float* x_hi_dev,
                float* const* l_dev, float* const* u_dev,
                const float* C_dev, int S, float* lb_dev, float* ub_dev);

/* O3 -- one CROWN backward pass (PAPER.md:64-68 Eq. 1, :128 A <- A.Lambda_i W_i) from node
 * `start` down to the input, for `rows` start-spec rows per property.
 *   C_dev == NULL : start matrix = rows [row0, row0+rows) of the identity on node `start`'s
 *                   output (intermediate bounds).  `start` is any non-ReLU node: for a Linear node
 *                   the rows of W are read in place; for a conv-shaped node (Conv2d / Add / Flatten output; full-CROWN
 *                   intermediate bounds of a conv net) the rows are materialised
 *                   one-hot and the sweep starts at the node itself.
 *   C_dev != NULL : [B, rows, size_start] start matrix (row0 ignored).
 *   l_dev/u_dev   : arrays of n_nodes pointers; for every ReLU node i below `start`, the
 *                   pre-activation bounds of its INPUT, [B, size_i].
 *   alpha_lo_dev / alpha_up_dev : arrays of n_nodes pointers or NULL; entry i, if non-NULL, is
 *                   the lower-relaxation slope [B, rows, size_i] of ReLU i used by the lower /
 *                   upper branch, clipped to [0,1]; NULL = opts.slope_rule.
 *                   The two may alias.
 *   A_dev [2,B,rows,n0], d_dev [2,B,rows] : outputs (branch-major, see top).  Either may be NULL
 *                   when lb_dev/ub_dev are given.
 *   x_lo_dev/x_hi_dev/lb_dev/ub_dev : if lb_dev != NULL the pass ends with the concretisation
 *                   (same arithmetic as concretize()) into lb_dev/ub_dev [B, rows]. */
int crown_backward(crown_ctx* ctx, int B, int start, int row0, int rows, const float* C_dev,
                   const float* const* l_dev, const float* const* u_dev,
                   const float* const* alpha_lo_dev, const float* const* alpha_up_dev,
                   float* A_dev, float* d_dev,
                   const float* x_lo_dev, const float* x_hi_dev, float* lb_dev, float* ub_dev);

/* Numbers from Eq. 1 over the box (Hoelder dual of the L_inf ball):
 *   lb = A_lo.x_c - |A_lo|.x_r + d_lo,  ub = A_up.x_c + |A_up|.x_r + d_up,
 *   x_c = (x_lo+x_hi)/2, x_r = (x_hi-x_lo)/2.   A_dev [2,B,rows,n0], d_dev [2,B,rows].
 * lb_dev/ub_dev: element (b, r) is written at lb_dev[b*out_stride + r]. */
int concretize(crown_ctx* ctx, int B, int rows, const float* A_dev, const float* d_dev,
               const float* x_lo_dev, const float* x_hi_dev,
               float* lb_dev, float* ub_dev, int out_stride);

/* a9 on its own -- verdict: verified_dev[b] = 1 iff every lb_dev[b, s] > 0 (a NaN bound fails
 * closed), lb_dev [B, S], verified_dev [B] uint8.  For callers that assemble the path from the calls above. */
int crown_verdict(crown_ctx* ctx, int B, int S, const float* lb_dev, uint8_t* verified_dev);

/* The whole hot path for a batch (O4 then O5 then the verdict):
 *   intermediate = 0: CROWN intermediate bounds for every ReLU in topological order (first
 *                     layer by IBP, which coincides), row-chunked under mem_cap; Linear AND
 *                     conv-shaped pre-activations (conv nets: dense A, chunks of crown_row_chunk rows);
 *   intermediate = 1: IBP for every pre-activation (cfg5, reading G22);
 *   then the final pass from the last node with C_dev [B,S,n_L] and alpha (array of n_nodes
 *   pointers, entry i = [B,S,size_i] for ReLU i, or NULL array/entries = slope rule).
 * Outputs: l_dev/u_dev (arrays of n_nodes pointers; entries for ReLU nodes must be non-NULL
 * [B,size_i] and receive that ReLU's pre-activation bounds), lb_dev/ub_dev [B,S],
 * verified_dev [B] uint8 (1 iff min_s lb > 0). */
int crown_run(crown_ctx* ctx, int B, const float* x_lo_dev, const float* x_hi_dev,
              const float* C_dev, int S, const float* const* alpha_dev, int intermediate,
              float* const* l_dev, float* const* u_dev,
              float* lb_dev, float* ub_dev, uint8_t* verified_dev);

/* Same as crown_run with HOST buffers: copies x_lo/x_hi/C/alpha H2D, runs, copies lb/ub/verified
 * D2H, synchronises.  Staging comes from the workspace.  alpha_host entries as in crown_run.
 * Returns CROWN_EINVAL if some x_lo > x_hi (checked here because the box is in host memory; the device-pointer
 * entry points do not check it: NaN/Inf and inverted boxes propagate). */
int crown_run_host(crown_ctx* ctx, int B, const float* x_lo_host, const float* x_hi_host,
                   const float* C_host, int S, const float* const* alpha_host, int intermediate,
                   float* lb_host, float* ub_host, uint8_t* verified_host);

/* NEXT-1 -- alpha optimisation (sec. 2.1: "alpha-CROWN promotes the fixed slopes to per-neuron optimisable
 * parameters alpha_i in [0,1]; gradient ascent over alpha tightens the lower bound (or lowers the upper bound)"; alpha
 * tensors are [B, S, size_i] per ReLU).  The intermediate bounds l_dev/u_dev stay fixed (reading G8);
 * only the final pass from the last node with C_dev [B,S,n_L] is differentiated / optimised.  The gradient is the
 * transpose of that pass: a forward sweep of the 2*B*S bound-attaining box corners through the
 * network with every ReLU replaced by the line the sign of the saved A selects; at A = 0 the one-sided derivative 0 is
 * taken (reading G23).  Every ReLU needs an alpha_lo and an alpha_up entry.  scratch_dev: caller-owned device memory of
 * at least crown_alpha_scratch_bytes(B, S) bytes, 256-byte aligned (saved A per ReLU, the sweep's vectors, TF32 limbs of the
 * weights the sweep multiplies on the tensor cores).
 * Streamed layers are CROWN_EUNSUPPORTED here. */
int crown_alpha_scratch_bytes(crown_ctx* ctx, int B, int S, size_t* out);

/* Bounds of the final pass at the given alpha (lb_dev / ub_dev [B,S], may be NULL) and their derivatives
 * g_lo_dev[i] = d lb[b,s] / d alpha_lo[i][b,s,:], g_up_dev[i] = d ub[b,s] / d alpha_up[i][b,s,:]  (arrays of n_nodes
 * pointers, [B,S,size_i] for ReLU i; NULL array or entry = not wanted).  Zero on stable neurons.  alpha may alias. */
int crown_alpha_grad(crown_ctx* ctx, int B, const float* C_dev, int S,
                     const float* const* l_dev, const float* const* u_dev,
                     const float* const* alpha_lo_dev, const float* const* alpha_up_dev,
                     const float* x_lo_dev, const float* x_hi_dev,
                     float* const* g_lo_dev, float* const* g_up_dev, float* lb_dev, float* ub_dev,
                     void* scratch_dev, size_t scratch_bytes);

/* `iters` projected gradient steps, in place: with a = clip(alpha, 0, 1),
 *   alpha_lo <- clip(a + step * dir(g_lo), 0, 1)   (ascent on lb),   alpha_up <- clip(a - step * dir(g_up), 0, 1),
 * dir = g (mode 0, plain) or sign(g) (mode 1) -- the step rule is reading G24; step = eta * decay^t at iteration t.
 * The bounds are evaluated at iters + 1 points (the start and after every step); every iterate is a valid alpha, so every
 * iterate is sound and the best per spec row is returned (reading G25):
 *   lb_best_dev = max_t lb_t, ub_best_dev = min_t ub_t  [B,S];  lb_last_dev / ub_last_dev [B,S] (may be NULL) = bounds
 *   at the final alpha;  verified_dev [B] (may be NULL) = verdict on lb_best.
 * alpha_lo_dev[i] and alpha_up_dev[i] must be DISTINCT tensors for every ReLU (CROWN_EINVAL otherwise). */
int crown_alpha_ascent(crown_ctx* ctx, int B, const float* C_dev, int S,
                       const float* const* l_dev, const float* const* u_dev,
                       float* const* alpha_lo_dev, float* const* alpha_up_dev,
                       const float* x_lo_dev, const float* x_hi_dev,
                       float eta, float decay, int iters, int mode,
                       float* lb_best_dev, float* ub_best_dev, float* lb_last_dev, float* ub_last_dev,
                       uint8_t* verified_dev, void* scratch_dev, size_t scratch_bytes);

/* NEXT-2 -- beta-CROWN bounds of batched branch-and-bound sub-domains (sec. 2.1.1: BaB fixes "a ReLU state
 * x >= 0 or x < 0" and bounds are recomputed per sub-region; sec. 2.2: the split constraints enter the
 * bound-propagation pass "via Lagrangian dual variables beta ... bounds for thousands of sub-problems are evaluated in
 * parallel on GPU as batched matrix multiplications, and alpha/beta parameters are jointly optimised by gradient
 * descent"; PAPER.md:96 batch BaB).  A sub-domain is one entry of the batch: its box, its (parent's) intermediate bounds
 * l_dev/u_dev and, per ReLU i, split_dev[i] (array of n_nodes pointers; entry = int8 [B, size_i], 4-byte aligned, or NULL):
 * +1 fixes the pre-activation z >= 0, -1 fixes z <= 0, 0 = not split.  Readings G26-G28:
 *   - the interval of a split neuron is clamped inside the library (l <- max(l,0) resp. u <- min(u,0)); l_dev/u_dev are
 *     not modified;
 *   - right after the relaxation of ReLU i (A w.r.t. its pre-activation):  lower branch A -= max(beta_lo_i, 0) * s_i,
 *     upper branch A += max(beta_up_i, 0) * s_i  with beta [B, rows, size_i]; sound for every beta >= 0 (weak duality);
 *     beta arrays / entries may be NULL (= 0); values on unsplit neurons are ignored.
 * crown_backward_split: crown_backward with these two additions (same outputs, same errors). */
int crown_backward_split(crown_ctx* ctx, int B, int start, int row0, int rows, const float* C_dev,
                         const float* const* l_dev, const float* const* u_dev, const int8_t* const* split_dev,
                         const float* const* alpha_lo_dev, const float* const* alpha_up_dev,
                         const float* const* beta_lo_dev, const float* const* beta_up_dev,
                         float* A_dev, float* d_dev,
                         const float* x_lo_dev, const float* x_hi_dev, float* lb_dev, float* ub_dev);

/* crown_alpha_grad for a batch of sub-domains: additionally gb_lo_dev[i] = d lb / d beta_lo[i] = -s_i * z_i(x*) and
 * gb_up_dev[i] = d ub / d beta_up[i] = +s_i * z_i(x*)  ([B,S,size_i]; z_i(x*) = the pre-activation at the bound-attaining
 * corner through the selected lines, i.e. the forward sweep of crown_alpha_grad); zero on unsplit neurons.  Written only
 * for ReLUs with a split entry.  Scratch as for crown_alpha_grad. */
int crown_beta_grad(crown_ctx* ctx, int B, const float* C_dev, int S,
                    const float* const* l_dev, const float* const* u_dev, const int8_t* const* split_dev,
                    const float* const* alpha_lo_dev, const float* const* alpha_up_dev,
                    const float* const* beta_lo_dev, const float* const* beta_up_dev,
                    const float* x_lo_dev, const float* x_hi_dev,
                    float* const* g_lo_dev, float* const* g_up_dev, float* const* gb_lo_dev, float* const* gb_up_dev,
                    float* lb_dev, float* ub_dev, void* scratch_dev, size_t scratch_bytes);

/* Joint projected ascent on (alpha, beta), in place (reading G28): alpha as in crown_alpha_ascent with step eta_alpha;
 *   beta_lo <- max(max(beta_lo,0) + eta_beta * dir(gb_lo), 0),  beta_up <- max(max(beta_up,0) - eta_beta * dir(gb_up), 0);
 * both steps decay by `decay` per iteration.  Every iterate is sound; outputs as crown_alpha_ascent (best over iterates).
 * Every ReLU with a split entry needs DISTINCT beta_lo / beta_up tensors (CROWN_EINVAL otherwise). */
int crown_beta_ascent(crown_ctx* ctx, int B, const float* C_dev, int S,
                      const float* const* l_dev, const float* const* u_dev, const int8_t* const* split_dev,
                      float* const* alpha_lo_dev, float* const* alpha_up_dev,
                      float* const* beta_lo_dev, float* const* beta_up_dev,
                      const float* x_lo_dev, const float* x_hi_dev,
                      float eta_alpha, float eta_beta, float decay, int iters, int mode,
                      float* lb_best_dev, float* ub_best_dev, float* lb_last_dev, float* ub_last_dev,
                      uint8_t* verified_dev, void* scratch_dev, size_t scratch_bytes);

/* D[M,N] = A[M,K] . W[K,N] (row-major fp32) through the same contraction kernel the backward
 * pass uses (scheme: 0 = 3xTF32 tcgen05 on prepared limbs, 2 = FFMA; 1 -- reserved in SURVEY.md for a split-bf16
 * scheme -- is intentionally absent); exposed for parity tests and roofline
 * measurement of kernel 1.  Wt_hi/Wt_lo [N,K] and A_hi/A_lo [M,K] are produced by
 * crown_split_tf32 (transpose=1 for W). */
int crown_gemm(crown_ctx* ctx, int scheme, int M, int N, int K,
               const float* A_hi_dev, const float* A_lo_dev,
               const float* Wt_hi_dev, const float* Wt_lo_dev, float* D_dev);
int crown_split_tf32(crown_ctx* ctx, const float* X_dev, int rows, int cols, int transpose,
                     float* hi_dev, float* lo_dev);

/* The same contraction for callers that cannot allocate device memory (code under CUDA-graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc): D[M,N] = A[M,K] . W[K,N], row-major fp32 DEVICE pointers, 3xTF32 on tcgen05
 * (PAPER.md:66-68 Eq. 1, :128).  The TF32 limbs that crown_gemm takes from the caller live here in one file-scope
 * device array inside the library (16 MiB, held by every GPU that loads the library until the process exits); the call
 * needs no crown_ctx and calls no cudaMalloc / cudaFree / allocating library routine.  Work is queued on `stream`
 * (a cudaStream_t of the CURRENT device, or NULL) and the call returns without synchronising.
 *   limits: N >= 128, K >= 32, N % 4 == 0, K % 4 == 0, D_dev 16-byte aligned, and
 *           round64(M*K) + round64(N*K) <= CROWN_GEMM_NOALLOC_MAX_ELEMS  (crown_gemm_noalloc_max_elems() returns it);
 *           anything beyond is CROWN_EINVAL with the sizes in crown_gemm_noalloc_error() (thread-local text).
 *   sharing: every call uses the same array, which keeps the previous call's contents; each call overwrites all it
 *           reads, so nothing needs clearing.  Calls whose kernels may overlap on the GPU (different streams without
 *           a dependency, or different host threads on different streams) RACE -- serialise them on one stream.
 *   result: bitwise equal to crown_split_tf32 x 2 + crown_gemm(scheme 0) of a context with default options. */
#define CROWN_GEMM_NOALLOC_MAX_ELEMS (1u << 21)
int crown_gemm_noalloc(int M, int N, int K, const float* A_dev, const float* W_dev, float* D_dev, void* stream);
int crown_gemm_noalloc_max_elems(void);
const char* crown_gemm_noalloc_error(void);

/* Introspection. */
int crown_peak_bytes(crown_ctx* ctx, size_t* out);         /* high-water mark of workspace use   */
int crown_row_chunk(crown_ctx* ctx, int* out);             /* rows per chunk of identity-start passes under mem_cap */
int crown_launch_count(crown_ctx* ctx, uint64_t* out);      /* kernels launched so far (graph replays count their kernels) */
int crown_graph_replays(crown_ctx* ctx, uint64_t* out);     /* crown_run calls served by a CUDA-graph replay */
int crown_gemm_flops(crown_ctx* ctx, double* out);          /* useful 2MNK flops of A.W so far    */
int crown_h2d_bytes(crown_ctx* ctx, double* out);           /* weight bytes streamed H2D so far   */
int crown_timing(crown_ctx* ctx, int enable);               /* 1: record CUDA events per kernel class */
int crown_timing_read(crown_ctx* ctx, int kernel_class, double* ms_total, uint64_t* launches,
                      double* bytes_total, double* flops_total);
const char* crown_last_error(crown_ctx* ctx);
int crown_destroy(crown_ctx* ctx);
const char* crown_version(void);

/* kernel classes for crown_timing_read */
enum {
  CROWN_K_IBP = 0, CROWN_K_COEFF = 1, CROWN_K_RELAX = 2, CROWN_K_GEMM_TC = 3, CROWN_K_GEMM_FFMA = 4,
  CROWN_K_CONCRETIZE = 5, CROWN_K_CONV = 6, CROWN_K_MISC = 7, CROWN_K_NUM = 8
};

#ifdef __cplusplus
}
#endif
#endif /* CROWNB200_H */
