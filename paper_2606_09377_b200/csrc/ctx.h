// Internal host-side state of the crownb200 library shared by api.cu and backward.cu (not installed).
#pragma once
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdio>
#include <cstring>
#include <map>
#include <string>
#include <vector>

#include "../../include/crownb200.h"
#include "kernels.h"

using namespace crownb200;

namespace {

struct NodeInfo {
  crown_node n;
  int size = 0;            // elements of the output
  int c = 0, h = 0, w = 0; // output shape for conv-shaped nodes (c*h*w == size), else (size,1,1)
  int n_consumers = 0;
  float* Wt_hi = nullptr;  // prepacked GEMM operand [n_in, n_out] (device)
  float* Wt_lo = nullptr;
  bool tc_ok = false;
  // a7: weight streaming ("gather before / free after").  A streamed layer has no resident copy:
  // raw W lives in the caller's pinned host buffer (n.W_host), the prepacked GEMM operand in pinned host memory
  // owned by the library; both are copied H2D slab by slab through two staging buffers on a side stream.
  bool streamed = false;
  float* hWt_hi = nullptr;  // pinned host [n_in, n_out]
  float* hWt_lo = nullptr;
};

struct Plan {
  size_t prepack_bytes = 0, coef_bytes = 0, ibp_bytes = 0, d_bytes = 0, io_bytes = 0;
  size_t buf_bytes = 0;
  size_t part_bytes = 0;  // per-(row, 32-column piece) partial sums of the fused epilogues (a4 / a8 fused)
  size_t stage_bytes = 0; // one of the two weight-streaming staging buffers (0: nothing is streamed)
  int nbuf = 0;
  int rc = 0;             // row chunk for identity passes
  int rows_cap = 0;       // max(rc, S_max)
  size_t total = 0;
};

struct TimingRec { cudaEvent_t a, b; int cls; double bytes, flops; };

// one captured step of crown_run: key = (B, S, intermediate, every pointer argument)
struct GraphEntry { std::vector<uintptr_t> key; cudaGraphExec_t exec = nullptr; uint64_t launches = 0; double flops = 0; };

}  // namespace

struct crown_ctx {
  std::vector<NodeInfo> nodes;
  int in_c = 0, in_h = 0, in_w = 0, n0 = 0;
  int input_consumers = 0;   // nodes that read the network input; the fused concretisation needs exactly one
  int B_max = 0, S_max = 0;
  crown_opts opts{};
  cudaStream_t stream = nullptr;
  int num_sms = 148;
  uint8_t* ws = nullptr;
  size_t ws_bytes = 0;
  Plan plan;
  // carved regions
  uint8_t* coef_base = nullptr; std::vector<size_t> coef_off;   // per node: ReLU coefficient records; Add: summed conv biases
  std::vector<char> add_bias_ok;                                // per node: the Add's operands' biases are in its vector
  uint8_t* ibp_base = nullptr;  std::vector<size_t> ibp_off;    // per node: l then u
  float* d_buf = nullptr;
  float* part_buf = nullptr;
  uint8_t* io_base = nullptr;
  uint8_t* hpack = nullptr;        // pinned mirror of the host-call staging region (small problems only, crown_run_host)
  uint8_t* pool_base = nullptr;
  std::vector<int> pool_ref;
  size_t peak = 0;
  bool has_add = false;
  std::string err;
  uint64_t launches = 0;
  double gemm_flops = 0;
  bool timing = false;
  std::vector<TimingRec> recs;
  std::vector<cudaEvent_t> free_events;
  // CUDA-graph replay of crown_run
  std::vector<GraphEntry> graphs;
  cudaStream_t gstream = nullptr;            // capture / replay stream when the caller's stream is the legacy default
  cudaEvent_t ev_gin = nullptr, ev_gout = nullptr;
  uint64_t graph_replays = 0;
  // weight streaming
  cudaStream_t copy_stream = nullptr;
  uint8_t* stage[2] = {nullptr, nullptr};
  cudaEvent_t ev_copied[2] = {nullptr, nullptr}, ev_free[2] = {nullptr, nullptr};
  uint64_t slab_seq = 0;      // slabs issued so far (parity = staging buffer)
  double h2d_bytes = 0;
};

namespace {

int fail(crown_ctx* ctx, int code, const std::string& msg) {
  if (ctx) ctx->err = msg;
  return code;
}

#define CK(ctx, expr)                                                                      \
  do {                                                                                     \
    cudaError_t e__ = (expr);                                                              \
    if (e__ != cudaSuccess)                                                                \
      return fail(ctx, CROWN_ECUDA, std::string(#expr) + ": " + cudaGetErrorString(e__)); \
  } while (0)

size_t align_up(size_t x, size_t a = 1024) { return (x + a - 1) / a * a; }

// ---- graph analysis ---------------------------------------------------------------------------
int analyse(const crown_node* nodes, int n_nodes, int in_c, int in_h, int in_w,
            std::vector<NodeInfo>& out, std::string& err, bool& has_add, int* input_consumers = nullptr) {
  if (!nodes || n_nodes <= 0 || in_c <= 0 || in_h <= 0 || in_w <= 0) { err = "bad network description"; return CROWN_EINVAL; }
  out.assign(n_nodes, NodeInfo());
  has_add = false;
  int in_cons = 0;     // consumers of the network input (node -1): a skip connection from x makes it > 1
  auto shape_of = [&](int idx, int& c, int& h, int& w) {
    if (idx < 0) { c = in_c; h = in_h; w = in_w; } else { c = out[idx].c; h = out[idx].h; w = out[idx].w; }
  };
  for (int i = 0; i < n_nodes; ++i) {
    NodeInfo& ni = out[i];
    ni.n = nodes[i];
    const crown_node& n = nodes[i];
    if (n.in0 >= i || n.in0 < -1) { err = "node list is not topologically ordered"; return CROWN_EINVAL; }
    int c, h, w; shape_of(n.in0, c, h, w);
    long long in_size = (long long)c * h * w;
    switch (n.op) {
      case CROWN_LINEAR:
        if (n.n_out <= 0 || n.n_in != in_size || (!n.W_dev && !n.W_host)) { err = "LINEAR: n_in does not match producer or W missing"; return CROWN_EINVAL; }
        ni.c = n.n_out; ni.h = 1; ni.w = 1;
        break;
      case CROWN_CONV2D: {
        if (n.c_in != c || n.h_in != h || n.w_in != w || n.c_out <= 0 || n.kh <= 0 || n.kw <= 0 || n.stride <= 0 || n.pad < 0 || !n.W_dev) {
          err = "CONV2D: shape does not match producer"; return CROWN_EINVAL; }
        int ho = (h + 2 * n.pad - n.kh) / n.stride + 1, wo = (w + 2 * n.pad - n.kw) / n.stride + 1;
        if (ho <= 0 || wo <= 0) { err = "CONV2D: empty output"; return CROWN_EINVAL; }
        ni.c = n.c_out; ni.h = ho; ni.w = wo;
        break; }
      case CROWN_RELU:
        ni.c = c; ni.h = h; ni.w = w;
        break;
      case CROWN_ADD: {
        if (n.in1 >= i || n.in1 < -1) { err = "ADD: bad in1"; return CROWN_EINVAL; }
        int c2, h2, w2; shape_of(n.in1, c2, h2, w2);
        if (c2 != c || h2 != h || w2 != w) { err = "ADD: operand shapes differ"; return CROWN_EINVAL; }
        ni.c = c; ni.h = h; ni.w = w; has_add = true;
        break; }
      case CROWN_FLATTEN:
        ni.c = (int)in_size; ni.h = 1; ni.w = 1;
        break;
      default:
        err = "unsupported op"; return CROWN_EUNSUPPORTED;
    }
    ni.size = ni.c * ni.h * ni.w;
    if (n.in0 >= 0) out[n.in0].n_consumers++; else ++in_cons;
    if (n.op == CROWN_ADD) { if (n.in1 >= 0) out[n.in1].n_consumers++; else ++in_cons; }
  }
  if (input_consumers) *input_consumers = in_cons;
  return CROWN_OK;
}

bool is_streamed(const crown_node& n, const crown_opts& o) {
  if (n.op != CROWN_LINEAR || !o.stream_weights || !n.W_host) return false;
  const uint64_t min_elems = o.stream_min_elems ? o.stream_min_elems : (1ull << 28);
  return (uint64_t)n.n_in * (uint64_t)n.n_out >= min_elems;
}

constexpr size_t kStageBytesMax = (size_t)1 << 30;   // 1 GiB per staging buffer

// rows of a [rows_total, row_elems] fp32 matrix (x limbs) that fit one staging buffer, multiple of 128
int slab_rows(size_t stage_bytes, int rows_total, int row_elems, int limbs) {
  size_t r = stage_bytes / ((size_t)limbs * row_elems * 4);
  if (r >= (size_t)rows_total) return rows_total;
  r = r / 128 * 128;
  return (int)(r < 128 ? 128 : r);
}

bool wants_prepack(const NodeInfo& ni, const crown_opts& o) {
  if (ni.n.op != CROWN_LINEAR || o.mma_scheme != 0) return false;
  // as GEMM operand: K = n_out, N = n_in; M is decided per pass
  return gemm_tc_supported(128, ni.n.n_in, ni.n.n_out) != 0;
}

int make_plan(const std::vector<NodeInfo>& nodes, int n0, int B, int S, const crown_opts& o, bool has_add,
              Plan& p, std::string& err) {
  p = Plan();
  int nmax = n0, max_start = 1;
  bool any_epi = false;
  for (const auto& ni : nodes) {
    if (ni.n.op == CROWN_LINEAR && o.mma_scheme == 0 && !o.disable_epi_fusion && gemm_tc_supported(128, ni.n.n_in, ni.n.n_out) &&
        gemm_tc_single_panel(ni.n.n_out)) any_epi = true;
    nmax = std::max(nmax, ni.size);
    if (ni.n.op == CROWN_LINEAR && ni.n.in0 >= 0) max_start = std::max(max_start, ni.size);
    // conv-shaped pre-activations (NEXT-3 identity passes) are chunked too; they ask for at most 512 rows per chunk so that
    // a conv net whose CROWN intermediate bounds are never requested (cfg5 benchmark: IBP ones) does not pay for them
    if (ni.n.op == CROWN_RELU && ni.n.in0 >= 0 && nodes[ni.n.in0].n.op != CROWN_LINEAR && nodes[ni.n.in0].n.in0 >= 0)
      max_start = std::max(max_start, std::min(nodes[ni.n.in0].size, 512));
    if (is_streamed(ni.n, o)) {
      // staging must hold 128 rows of the prepacked operand (2 limbs x n_out) and 128 raw rows (n_in)
      size_t need = std::max((size_t)2 * 128 * ni.n.n_out * 4, (size_t)128 * ni.n.n_in * 4);
      size_t full = (size_t)2 * ni.n.n_in * ni.n.n_out * 4;
      p.stage_bytes = std::max(p.stage_bytes, std::max(need, std::min(full, o.stream_stage_bytes ? (size_t)o.stream_stage_bytes : kStageBytesMax)));
    } else if (wants_prepack(ni, o)) p.prepack_bytes += 2 * align_up((size_t)ni.n.n_in * ni.n.n_out * 4);
    if (ni.n.op == CROWN_RELU) p.coef_bytes += align_up((size_t)B * ni.size * 16);   // float4 records {dU, bU, dL, unstable}
    if (ni.n.op == CROWN_ADD) p.coef_bytes += align_up((size_t)ni.c * 4);            // summed biases of its conv operands
    p.ibp_bytes += 2 * align_up((size_t)B * ni.size * 4);
    if (ni.n.op == CROWN_RELU) p.io_bytes += align_up((size_t)B * S * ni.size * 4) + 2 * align_up((size_t)B * ni.size * 4);
  }
  p.io_bytes += 2 * align_up((size_t)B * n0 * 4) + align_up((size_t)B * S * nodes.back().size * 4) +
                2 * align_up((size_t)B * S * 4) + align_up((size_t)B);
  // live A buffers of a chain: operand hi + lo and the product; when the product's epilogue also emits the next
  // operand's hi + lo limbs (a4 fused, single-K-panel layers) one more
  p.nbuf = has_add ? 8 : (any_epi ? 4 : 3);
  size_t per_row = (size_t)2 * B * nmax * 4;            // bytes of one start-spec row in one buffer
  const size_t per_row_part = (size_t)2 * B * ((nmax + 31) / 32) * 8;
  p.stage_bytes = align_up(p.stage_bytes);
  size_t fixed = p.prepack_bytes + p.coef_bytes + p.ibp_bytes + p.io_bytes + 2 * p.stage_bytes;
  int rc = max_start;
  if (o.mem_cap_bytes) {
    size_t d_est = align_up((size_t)2 * B * std::max(max_start, S) * 4);
    if (o.mem_cap_bytes <= fixed + d_est) { err = "mem_cap_bytes below the fixed footprint"; return CROWN_ENOMEM; }
    size_t avail = o.mem_cap_bytes - fixed - d_est;
    size_t fit = avail / ((size_t)p.nbuf * per_row + per_row_part);
    if (fit < (size_t)std::max(1, S)) { err = "mem_cap_bytes too small for one row chunk"; return CROWN_ENOMEM; }
    if (fit < (size_t)rc) rc = (int)fit;
    if (rc < max_start && rc > 64) rc = rc / 64 * 64;
    if (rc < max_start && rc >= 64) {
      // equal chunks: a short tail chunk runs the same number of K panels over a nearly empty grid
      // (cfg4, ncu: 4096 rows as 1984 + 1984 + 128 spent 6 % of the contraction time on 3 % of the rows)
      const int nchunks = (max_start + rc - 1) / rc;
      const int even = ((max_start + nchunks - 1) / nchunks + 63) / 64 * 64;
      if (even < rc) rc = even;
    }
  }
  p.rc = rc;
  p.rows_cap = std::max(rc, S);
  p.d_bytes = align_up((size_t)2 * B * p.rows_cap * 4);
  p.buf_bytes = align_up((size_t)p.rows_cap * per_row);
  p.part_bytes = align_up((size_t)p.rows_cap * per_row_part);
  p.total = fixed + p.d_bytes + p.part_bytes + (size_t)p.nbuf * p.buf_bytes;
  return CROWN_OK;
}

// ---- launch bookkeeping -----------------------------------------------------------------------
struct Scope {
  crown_ctx* ctx; int cls; double bytes, flops; cudaEvent_t a = nullptr, b = nullptr;
  Scope(crown_ctx* c, int cls_, double bytes_ = 0, double flops_ = 0) : ctx(c), cls(cls_), bytes(bytes_), flops(flops_) {
    ctx->launches++;
    if (ctx->timing) {
      auto get = [&]() { cudaEvent_t e; if (!ctx->free_events.empty()) { e = ctx->free_events.back(); ctx->free_events.pop_back(); } else cudaEventCreate(&e); return e; };
      a = get(); b = get();
      cudaEventRecord(a, ctx->stream);
    }
  }
  ~Scope() {
    if (ctx->timing) {
      cudaEventRecord(b, ctx->stream);
      ctx->recs.push_back({a, b, cls, bytes, flops});
    }
  }
};

// ---- a7: weight streaming through the two staging buffers ------------------------------------------
// copy(slab, dst, copy_stream) enqueues the H2D copies of one slab; use(slab, src) launches the kernels that
// read it on the main stream.  Slab s+1 is copied while slab s is consumed ("gather before / free after",
// PAPER.md:146); because every call is only an enqueue, the copy of the NEXT layer's first slab also starts
// as soon as a staging buffer is free, i.e. while the current layer still computes.
template <class Copy, class Use>
int stream_slabs(crown_ctx* ctx, int nslabs, Copy copy, Use use) {
  auto issue = [&](int s) -> int {
    const int buf = (int)((ctx->slab_seq + s) & 1);
    CK(ctx, cudaStreamWaitEvent(ctx->copy_stream, ctx->ev_free[buf], 0));
    CK(ctx, copy(s, ctx->stage[buf], ctx->copy_stream));
    CK(ctx, cudaEventRecord(ctx->ev_copied[buf], ctx->copy_stream));
    return CROWN_OK;
  };
  int rc = issue(0);
  if (rc) return rc;
  for (int s = 0; s < nslabs; ++s) {
    const int buf = (int)((ctx->slab_seq + s) & 1);
    if (s + 1 < nslabs && (rc = issue(s + 1))) return rc;
    CK(ctx, cudaStreamWaitEvent(ctx->stream, ctx->ev_copied[buf], 0));
    if ((rc = use(s, ctx->stage[buf]))) return rc;
    CK(ctx, cudaEventRecord(ctx->ev_free[buf], ctx->stream));
  }
  ctx->slab_seq += nslabs;
  return CROWN_OK;
}

// ---- A-buffer pool ----------------------------------------------------------------------------
int pool_get(crown_ctx* ctx) {
  for (int i = 0; i < (int)ctx->pool_ref.size(); ++i)
    if (ctx->pool_ref[i] == 0) {
      ctx->pool_ref[i] = 1;
      size_t used = (size_t)(ctx->pool_base - ctx->ws) + (size_t)(i + 1) * ctx->plan.buf_bytes;
      ctx->peak = std::max(ctx->peak, used);
      return i;
    }
  return -1;
}
float* pool_ptr(crown_ctx* ctx, int i) { return reinterpret_cast<float*>(ctx->pool_base + (size_t)i * ctx->plan.buf_bytes); }
void pool_release(crown_ctx* ctx, int i) { if (i >= 0 && ctx->pool_ref[i] > 0) ctx->pool_ref[i]--; }
void pool_retain(crown_ctx* ctx, int i) { if (i >= 0) ctx->pool_ref[i]++; }

struct Pending {
  AView v;
  int buf = -1, buf_lo = -1;   // pool ids backing v.p / v.lo (-1: caller memory or weights)
  int bias_done_for = -2;      // node id whose bias has already been added to d through this view
};
void release(crown_ctx* ctx, Pending& p) { pool_release(ctx, p.buf); pool_release(ctx, p.buf_lo); p.buf = p.buf_lo = -1; }

AView canon_view(const float* p, int B, int R, int n) {
  AView v; v.p = p; v.ld = n; v.n = n; v.sB = (long long)R * n; v.sBr = (long long)B * R * n; return v;
}

// number of distinct rows of a view and whether they are uniformly spaced (one GEMM can take them)
bool view_uniform(const AView& v, int B, int R, int& m_eff) {
  int nb = v.sB ? B : 1, nbr = v.sBr ? 2 : 1;
  if (v.sB && v.sB != (long long)R * v.ld) return false;
  if (v.sBr && v.sBr != (long long)nb * R * v.ld) return false;
  m_eff = nbr * nb * R;
  return true;
}

}  // namespace

// api.cu: interval of every node's OUTPUT (O1).  L/U receive the pointer used per node (caller's or scratch).
int ibp_internal(crown_ctx* ctx, int B, const float* x_lo, const float* x_hi, float* const* l_dev,
                 float* const* u_dev, std::vector<float*>& L, std::vector<float*>& U, bool only_first_layer);
