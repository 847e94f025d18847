// C-ABI boundary + host scheduler of the crownb200 hot path (include/crownb200.h).
// The scheduler walks the layer DAG in reverse topological order (A <- A.Lambda_i W_i),
// keeps at most a handful of A-matrix buffers alive in the caller's workspace, chunks start-spec rows
// under mem_cap (single-GPU restatement of Eq. 2) and launches the kernels of
// kernels.h.  No device memory is allocated here and there is no CPU fallback.
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
};

struct Plan {
  size_t prepack_bytes = 0, coef_bytes = 0, ibp_bytes = 0, d_bytes = 0, io_bytes = 0;
  size_t buf_bytes = 0;
  int nbuf = 0;
  int rc = 0;             // row chunk for identity passes
  int rows_cap = 0;       // max(rc, S_max)
  size_t total = 0;
};

struct TimingRec { cudaEvent_t a, b; int cls; double bytes, flops; };

}  // namespace

struct crown_ctx {
  std::vector<NodeInfo> nodes;
  int in_c = 0, in_h = 0, in_w = 0, n0 = 0;
  int B_max = 0, S_max = 0;
  crown_opts opts{};
  cudaStream_t stream = nullptr;
  int num_sms = 148;
  uint8_t* ws = nullptr;
  size_t ws_bytes = 0;
  Plan plan;
  // carved regions
  uint8_t* coef_base = nullptr; std::vector<size_t> coef_off;   // per node (ReLU only)
  uint8_t* ibp_base = nullptr;  std::vector<size_t> ibp_off;    // per node: l then u
  float* d_buf = nullptr;
  uint8_t* io_base = nullptr;
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
            std::vector<NodeInfo>& out, std::string& err, bool& has_add) {
  if (!nodes || n_nodes <= 0 || in_c <= 0 || in_h <= 0 || in_w <= 0) { err = "bad network description"; return CROWN_EINVAL; }
  out.assign(n_nodes, NodeInfo());
  has_add = false;
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
        if (n.n_out <= 0 || n.n_in != in_size || !n.W_dev) { err = "LINEAR: n_in does not match producer or W missing"; return CROWN_EINVAL; }
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
    if (n.in0 >= 0) out[n.in0].n_consumers++;
    if (n.op == CROWN_ADD && n.in1 >= 0) out[n.in1].n_consumers++;
  }
  return CROWN_OK;
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
  for (const auto& ni : nodes) {
    nmax = std::max(nmax, ni.size);
    if (ni.n.op == CROWN_LINEAR && ni.n.in0 >= 0) max_start = std::max(max_start, ni.size);
    if (wants_prepack(ni, o)) p.prepack_bytes += 2 * align_up((size_t)ni.n.n_in * ni.n.n_out * 4);
    if (ni.n.op == CROWN_RELU) p.coef_bytes += align_up((size_t)B * ni.size * 16);
    p.ibp_bytes += 2 * align_up((size_t)B * ni.size * 4);
    if (ni.n.op == CROWN_RELU) p.io_bytes += align_up((size_t)B * S * ni.size * 4) + 2 * align_up((size_t)B * ni.size * 4);
  }
  p.io_bytes += 2 * align_up((size_t)B * n0 * 4) + align_up((size_t)B * S * nodes.back().size * 4) +
                2 * align_up((size_t)B * S * 4) + align_up((size_t)B);
  p.nbuf = has_add ? 8 : 3;
  size_t per_row = (size_t)2 * B * nmax * 4;            // bytes of one start-spec row in one buffer
  size_t fixed = p.prepack_bytes + p.coef_bytes + p.ibp_bytes + p.io_bytes;
  int rc = max_start;
  if (o.mem_cap_bytes) {
    size_t d_est = align_up((size_t)2 * B * std::max(max_start, S) * 4);
    if (o.mem_cap_bytes <= fixed + d_est) { err = "mem_cap_bytes below the fixed footprint"; return CROWN_ENOMEM; }
    size_t avail = o.mem_cap_bytes - fixed - d_est;
    size_t fit = avail / ((size_t)p.nbuf * per_row);
    if (fit < (size_t)std::max(1, S)) { err = "mem_cap_bytes too small for one row chunk"; return CROWN_ENOMEM; }
    if (fit < (size_t)rc) rc = (int)fit;
    if (rc < max_start && rc > 64) rc = rc / 64 * 64;
  }
  p.rc = rc;
  p.rows_cap = std::max(rc, S);
  p.d_bytes = align_up((size_t)2 * B * p.rows_cap * 4);
  p.buf_bytes = align_up((size_t)p.rows_cap * per_row);
  p.total = fixed + p.d_bytes + (size_t)p.nbuf * p.buf_bytes;
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

// ================================================================================================
// init / destroy / introspection
// ================================================================================================
extern "C" int crown_workspace_bytes(const crown_node* nodes, int n_nodes, int in_c, int in_h, int in_w,
                                     int B_max, int S_max, const crown_opts* opts, size_t* out_bytes) {
  if (!out_bytes || !opts || B_max <= 0 || S_max < 0) return CROWN_EINVAL;
  std::vector<NodeInfo> ni; std::string err; bool has_add;
  int rc = analyse(nodes, n_nodes, in_c, in_h, in_w, ni, err, has_add);
  if (rc) return rc;
  Plan p;
  rc = make_plan(ni, in_c * in_h * in_w, B_max, std::max(S_max, 1), *opts, has_add, p, err);
  if (rc) return rc;
  *out_bytes = p.total + 4096;
  return CROWN_OK;
}

extern "C" int crown_init(crown_ctx** out, const crown_node* nodes, int n_nodes, int in_c, int in_h, int in_w,
                          int B_max, int S_max, void* workspace_dev, size_t workspace_bytes,
                          const crown_opts* opts, void* cuda_stream) {
  if (!out || !opts || !workspace_dev || B_max <= 0 || S_max < 0) return CROWN_EINVAL;
  *out = nullptr;
  crown_ctx* ctx = new crown_ctx();
  ctx->opts = *opts;
  if (ctx->opts.mma_scheme != 0 && ctx->opts.mma_scheme != 2) { delete ctx; return CROWN_EINVAL; }
  if (ctx->opts.slope_rule < 0 || ctx->opts.slope_rule > 2) { delete ctx; return CROWN_EINVAL; }
  int rc = analyse(nodes, n_nodes, in_c, in_h, in_w, ctx->nodes, ctx->err, ctx->has_add);
  if (rc) { delete ctx; return rc; }
  ctx->in_c = in_c; ctx->in_h = in_h; ctx->in_w = in_w; ctx->n0 = in_c * in_h * in_w;
  ctx->B_max = B_max; ctx->S_max = std::max(S_max, 1);
  ctx->stream = reinterpret_cast<cudaStream_t>(cuda_stream);
  rc = make_plan(ctx->nodes, ctx->n0, B_max, ctx->S_max, ctx->opts, ctx->has_add, ctx->plan, ctx->err);
  if (rc) { delete ctx; return rc; }
  if (workspace_bytes < ctx->plan.total) { delete ctx; return CROWN_ENOMEM; }
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess ||
      cudaDeviceGetAttribute(&ctx->num_sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
    delete ctx; return CROWN_ECUDA;
  }
  // carve the workspace
  ctx->ws = reinterpret_cast<uint8_t*>(workspace_dev);
  ctx->ws_bytes = workspace_bytes;
  uint8_t* cur = reinterpret_cast<uint8_t*>(align_up(reinterpret_cast<size_t>(ctx->ws)));
  for (auto& ni : ctx->nodes) {
    if (wants_prepack(ni, ctx->opts)) {
      size_t sz = align_up((size_t)ni.n.n_in * ni.n.n_out * 4);
      ni.Wt_hi = reinterpret_cast<float*>(cur); cur += sz;
      ni.Wt_lo = reinterpret_cast<float*>(cur); cur += sz;
      ni.tc_ok = true;
    }
  }
  ctx->coef_base = cur; ctx->coef_off.assign(n_nodes, 0);
  { size_t off = 0; for (int i = 0; i < n_nodes; ++i) if (ctx->nodes[i].n.op == CROWN_RELU) { ctx->coef_off[i] = off; off += align_up((size_t)B_max * ctx->nodes[i].size * 16); } cur += ctx->plan.coef_bytes; }
  ctx->ibp_base = cur; ctx->ibp_off.assign(n_nodes, 0);
  { size_t off = 0; for (int i = 0; i < n_nodes; ++i) { ctx->ibp_off[i] = off; off += 2 * align_up((size_t)B_max * ctx->nodes[i].size * 4); } cur += ctx->plan.ibp_bytes; }
  ctx->d_buf = reinterpret_cast<float*>(cur); cur += ctx->plan.d_bytes;
  ctx->io_base = cur; cur += ctx->plan.io_bytes;
  ctx->pool_base = cur;
  ctx->pool_ref.assign(ctx->plan.nbuf, 0);
  ctx->peak = (size_t)(ctx->pool_base - ctx->ws);
  // prepack: transpose + TF32 split of every GEMM weight operand (one pass over W)
  for (auto& ni : ctx->nodes) {
    if (!ni.tc_ok) continue;
    Scope sc(ctx, CROWN_K_MISC);
    launch_split_tf32(ni.n.W_dev, ni.n.n_out, ni.n.n_in, 1, ni.Wt_hi, ni.Wt_lo, ctx->stream);
  }
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) { std::string m = cudaGetErrorString(e); delete ctx; (void)m; return CROWN_ECUDA; }
  *out = ctx;
  return CROWN_OK;
}

extern "C" int crown_destroy(crown_ctx* ctx) {
  if (!ctx) return CROWN_EINVAL;
  for (auto& r : ctx->recs) { cudaEventDestroy(r.a); cudaEventDestroy(r.b); }
  for (auto e : ctx->free_events) cudaEventDestroy(e);
  delete ctx;
  return CROWN_OK;
}
extern "C" const char* crown_last_error(crown_ctx* ctx) { return ctx ? ctx->err.c_str() : "null context"; }
extern "C" const char* crown_version(void) { return "crownb200 0.1 (sm_100a)"; }
extern "C" int crown_peak_bytes(crown_ctx* ctx, size_t* out) { if (!ctx || !out) return CROWN_EINVAL; *out = ctx->peak; return CROWN_OK; }
extern "C" int crown_launch_count(crown_ctx* ctx, uint64_t* out) { if (!ctx || !out) return CROWN_EINVAL; *out = ctx->launches; return CROWN_OK; }
extern "C" int crown_gemm_flops(crown_ctx* ctx, double* out) { if (!ctx || !out) return CROWN_EINVAL; *out = ctx->gemm_flops; return CROWN_OK; }
extern "C" int crown_timing(crown_ctx* ctx, int enable) {
  if (!ctx) return CROWN_EINVAL;
  for (auto& r : ctx->recs) { ctx->free_events.push_back(r.a); ctx->free_events.push_back(r.b); }
  ctx->recs.clear();
  ctx->timing = enable != 0;
  return CROWN_OK;
}
extern "C" int crown_timing_read(crown_ctx* ctx, int cls, double* ms_total, uint64_t* launches,
                                 double* bytes_total, double* flops_total) {
  if (!ctx || cls < 0 || cls >= CROWN_K_NUM) return CROWN_EINVAL;
  CK(ctx, cudaStreamSynchronize(ctx->stream));
  double ms = 0, by = 0, fl = 0; uint64_t n = 0;
  for (auto& r : ctx->recs) {
    if (r.cls != cls) continue;
    float t = 0; CK(ctx, cudaEventElapsedTime(&t, r.a, r.b));
    ms += t; by += r.bytes; fl += r.flops; ++n;
  }
  if (ms_total) *ms_total = ms;
  if (launches) *launches = n;
  if (bytes_total) *bytes_total = by;
  if (flops_total) *flops_total = fl;
  return CROWN_OK;
}

// ================================================================================================
// O1 -- IBP forward
// ================================================================================================
namespace {

float* ibp_tmp_l(crown_ctx* ctx, int i) { return reinterpret_cast<float*>(ctx->ibp_base + ctx->ibp_off[i]); }
float* ibp_tmp_u(crown_ctx* ctx, int i) {
  return reinterpret_cast<float*>(ctx->ibp_base + ctx->ibp_off[i] + align_up((size_t)ctx->B_max * ctx->nodes[i].size * 4));
}

// Interval of every node's output.  L/U receive the pointer actually used per node (caller's or scratch).
// only_first_layer: stop after the Linear/Conv nodes fed directly by the network input.
int ibp_internal(crown_ctx* ctx, int B, const float* x_lo, const float* x_hi, float* const* l_dev,
                 float* const* u_dev, std::vector<float*>& L, std::vector<float*>& U, bool only_first_layer) {
  const int n = (int)ctx->nodes.size();
  cudaStream_t s = ctx->stream;
  L.assign(n, nullptr); U.assign(n, nullptr);
  std::vector<char> have(n, 0);
  for (int i = 0; i < n; ++i) {
    const NodeInfo& ni = ctx->nodes[i];
    const crown_node& nd = ni.n;
    if (only_first_layer && !((nd.op == CROWN_LINEAR || nd.op == CROWN_CONV2D) && nd.in0 < 0)) continue;
    float* lo = (l_dev && l_dev[i]) ? l_dev[i] : ibp_tmp_l(ctx, i);
    float* uo = (u_dev && u_dev[i]) ? u_dev[i] : ibp_tmp_u(ctx, i);
    // input interval; a ReLU producer is folded into the consumer (relu_in) when it was not materialised
    auto input_of = [&](int src, const float*& li, const float*& ui, int& relu_in) -> bool {
      relu_in = 0;
      if (src < 0) { li = x_lo; ui = x_hi; return true; }
      if (have[src]) { li = L[src]; ui = U[src]; return true; }
      if (ctx->nodes[src].n.op == CROWN_RELU) {
        int s2 = ctx->nodes[src].n.in0;
        if (s2 < 0) { li = x_lo; ui = x_hi; } else { if (!have[s2]) return false; li = L[s2]; ui = U[s2]; }
        relu_in = 1;
        return true;
      }
      return false;
    };
    const float *li = nullptr, *ui = nullptr; int relu_in = 0;
    switch (nd.op) {
      case CROWN_LINEAR: {
        if (!input_of(nd.in0, li, ui, relu_in)) return fail(ctx, CROWN_EINVAL, "ibp: producer interval missing");
        Scope sc(ctx, CROWN_K_IBP, 4.0 * nd.n_out * nd.n_in * ((B + 7) / 8), 4.0 * B * nd.n_out * (double)nd.n_in);
        launch_ibp_linear(nd.W_dev, nd.b_dev, li, ui, relu_in, lo, uo, B, nd.n_out, nd.n_in, s);
        break; }
      case CROWN_CONV2D: {
        if (!input_of(nd.in0, li, ui, relu_in)) return fail(ctx, CROWN_EINVAL, "ibp: producer interval missing");
        Scope sc(ctx, CROWN_K_CONV);
        launch_ibp_conv(nd.W_dev, nd.b_dev, li, ui, relu_in, lo, uo, B, nd.c_in, nd.h_in, nd.w_in, nd.c_out,
                        nd.kh, nd.kw, nd.stride, nd.pad, ni.h, ni.w, s);
        break; }
      case CROWN_RELU: {
        // materialise only when someone other than a Linear/Conv consumer needs it
        bool wanted = (l_dev && l_dev[i]) || (u_dev && u_dev[i]);
        bool needed = false;
        for (int j = i + 1; j < n; ++j) {
          const crown_node& c = ctx->nodes[j].n;
          if ((c.in0 == i && c.op != CROWN_LINEAR && c.op != CROWN_CONV2D) || (c.op == CROWN_ADD && c.in1 == i)) needed = true;
        }
        if (i == n - 1) needed = true;
        if (!wanted && !needed) continue;
        int r2;
        if (!input_of(nd.in0, li, ui, r2)) return fail(ctx, CROWN_EINVAL, "ibp: producer interval missing");
        Scope sc(ctx, CROWN_K_MISC);
        launch_ibp_relu(li, ui, lo, uo, (long long)B * ni.size, s);
        break; }
      case CROWN_ADD: {
        const float *l1 = nullptr, *u1 = nullptr; int r0, r1;
        if (!input_of(nd.in0, li, ui, r0) || !input_of(nd.in1, l1, u1, r1) || r0 || r1)
          return fail(ctx, CROWN_EINVAL, "ibp: ADD operand interval missing");
        Scope sc(ctx, CROWN_K_MISC);
        launch_ibp_add(li, ui, l1, u1, lo, uo, (long long)B * ni.size, s);
        break; }
      case CROWN_FLATTEN: {
        if (!input_of(nd.in0, li, ui, relu_in)) return fail(ctx, CROWN_EINVAL, "ibp: producer interval missing");
        if (relu_in) {
          Scope sc(ctx, CROWN_K_MISC);
          launch_ibp_relu(li, ui, lo, uo, (long long)B * ni.size, s);
        } else {
          // same memory order: alias instead of copying unless the caller wants its own copy
          if ((l_dev && l_dev[i]) || (u_dev && u_dev[i])) {
            CK(ctx, cudaMemcpyAsync(lo, li, (size_t)B * ni.size * 4, cudaMemcpyDeviceToDevice, s));
            CK(ctx, cudaMemcpyAsync(uo, ui, (size_t)B * ni.size * 4, cudaMemcpyDeviceToDevice, s));
          } else { lo = const_cast<float*>(li); uo = const_cast<float*>(ui); }
        }
        break; }
      default:
        return fail(ctx, CROWN_EUNSUPPORTED, "ibp: unsupported op");
    }
    L[i] = lo; U[i] = uo; have[i] = 1;
  }
  CK(ctx, cudaGetLastError());
  return CROWN_OK;
}

}  // namespace

extern "C" int ibp_forward(crown_ctx* ctx, int B, const float* x_lo_dev, const float* x_hi_dev,
                           float* const* l_dev, float* const* u_dev, const float* C_dev, int S,
                           float* lb_dev, float* ub_dev) {
  if (!ctx) return CROWN_EINVAL;
  if (B <= 0 || B > ctx->B_max || !x_lo_dev || !x_hi_dev) return fail(ctx, CROWN_EINVAL, "ibp_forward: bad arguments");
  std::vector<float*> L, U;
  int rc = ibp_internal(ctx, B, x_lo_dev, x_hi_dev, l_dev, u_dev, L, U, false);
  if (rc) return rc;
  if (!C_dev) return CROWN_OK;
  // spec: C and the last Linear fused into ONE linear layer (reading G10)
  const int last = (int)ctx->nodes.size() - 1;
  const NodeInfo& ln = ctx->nodes[last];
  if (ln.n.op != CROWN_LINEAR) return fail(ctx, CROWN_EUNSUPPORTED, "ibp_forward: spec needs a final Linear node");
  if (S <= 0 || S > ctx->plan.rows_cap || !lb_dev || !ub_dev) return fail(ctx, CROWN_EINVAL, "ibp_forward: bad spec arguments");
  cudaStream_t s = ctx->stream;
  std::fill(ctx->pool_ref.begin(), ctx->pool_ref.end(), 0);
  const float *li, *ui;
  int src = ln.n.in0;
  if (src < 0) { li = x_lo_dev; ui = x_hi_dev; }
  else if (L[src]) { li = L[src]; ui = U[src]; }
  else {  // un-materialised ReLU: clamp its input interval into the ReLU's scratch slot
    int s2 = ctx->nodes[src].n.in0;
    const float* pl = s2 < 0 ? x_lo_dev : L[s2];
    const float* pu = s2 < 0 ? x_hi_dev : U[s2];
    Scope sc(ctx, CROWN_K_MISC);
    launch_ibp_relu(pl, pu, ibp_tmp_l(ctx, src), ibp_tmp_u(ctx, src), (long long)B * ctx->nodes[src].size, s);
    li = ibp_tmp_l(ctx, src); ui = ibp_tmp_u(ctx, src);
  }
  int nb = pool_get(ctx);
  float* CW = pool_ptr(ctx, nb);
  { Scope sc(ctx, CROWN_K_GEMM_FFMA);
    launch_gemm_ffma(C_dev, ln.n.n_out, ln.n.W_dev, ln.n.n_in, CW, ln.n.n_in, B * S, ln.n.n_in, ln.n.n_out, s); }
  AView cv; cv.p = C_dev; cv.ld = ln.n.n_out; cv.n = ln.n.n_out; cv.sB = (long long)S * ln.n.n_out; cv.sBr = 0;
  { Scope sc(ctx, CROWN_K_MISC); launch_init_d(ctx->d_buf, nullptr, 0, B, S, s); }
  { Scope sc(ctx, CROWN_K_MISC); launch_rowdot_bias(cv, ln.n.b_dev, 1, ctx->d_buf, B, S, s); }
  AView av; av.p = CW; av.ld = ln.n.n_in; av.n = ln.n.n_in; av.sB = (long long)S * ln.n.n_in; av.sBr = 0;
  { Scope sc(ctx, CROWN_K_CONCRETIZE);
    launch_concretize(av, ctx->d_buf, li, ui, lb_dev, ub_dev, S, B, S, s); }
  pool_release(ctx, nb);
  CK(ctx, cudaGetLastError());
  return CROWN_OK;
}
