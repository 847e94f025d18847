// C-ABI boundary + host scheduler of the crownb200 hot path (include/crownb200.h).
// The scheduler walks the layer DAG in reverse topological order (A <- A.Lambda_i W_i),
// keeps at most a handful of A-matrix buffers alive in the caller's workspace, chunks start-spec rows
// under mem_cap (single-GPU restatement of Eq. 2) and launches the kernels of
// kernels.h.  No device memory is allocated here and there is no CPU fallback.
#include "ctx.h"

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
  // every failure below releases whatever was created so far through crown_destroy (streams, events, pinned buffers)
  auto bail = [&](int code) { crown_destroy(ctx); return code; };
  ctx->opts = *opts;
  if (ctx->opts.mma_scheme != 0 && ctx->opts.mma_scheme != 2) return bail(CROWN_EINVAL);
  if (ctx->opts.slope_rule < 0 || ctx->opts.slope_rule > 2) return bail(CROWN_EINVAL);
  int rc = analyse(nodes, n_nodes, in_c, in_h, in_w, ctx->nodes, ctx->err, ctx->has_add, &ctx->input_consumers);
  if (rc) return bail(rc);
  ctx->in_c = in_c; ctx->in_h = in_h; ctx->in_w = in_w; ctx->n0 = in_c * in_h * in_w;
  ctx->B_max = B_max; ctx->S_max = std::max(S_max, 1);
  ctx->stream = reinterpret_cast<cudaStream_t>(cuda_stream);
  rc = make_plan(ctx->nodes, ctx->n0, B_max, ctx->S_max, ctx->opts, ctx->has_add, ctx->plan, ctx->err);
  if (rc) return bail(rc);
  if (workspace_bytes < ctx->plan.total) return bail(CROWN_ENOMEM);
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess ||
      cudaDeviceGetAttribute(&ctx->num_sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
    return bail(CROWN_ECUDA);
  // kernel attributes (opt-in dynamic shared memory) are per device: set them for the device of this context
  if (kernels_init_device() != 0) return bail(CROWN_ECUDA);
  // carve the workspace
  ctx->ws = reinterpret_cast<uint8_t*>(workspace_dev);
  ctx->ws_bytes = workspace_bytes;
  uint8_t* cur = reinterpret_cast<uint8_t*>(align_up(reinterpret_cast<size_t>(ctx->ws)));
  for (auto& ni : ctx->nodes) {
    ni.streamed = is_streamed(ni.n, ctx->opts);
    if (ni.n.op == CROWN_LINEAR && !ni.streamed && !ni.n.W_dev) return bail(CROWN_EINVAL);   // no resident copy: must stream
    if (ni.streamed) {
      if (ctx->opts.mma_scheme != 0 || !gemm_tc_supported(128, ni.n.n_in, ni.n.n_out)) return bail(CROWN_EUNSUPPORTED);
      ni.tc_ok = true;
    } else if (wants_prepack(ni, ctx->opts)) {
      size_t sz = align_up((size_t)ni.n.n_in * ni.n.n_out * 4);
      ni.Wt_hi = reinterpret_cast<float*>(cur); cur += sz;
      ni.Wt_lo = reinterpret_cast<float*>(cur); cur += sz;
      ni.tc_ok = true;
    }
  }
  if (ctx->plan.stage_bytes) {
    ctx->stage[0] = cur; cur += ctx->plan.stage_bytes;
    ctx->stage[1] = cur; cur += ctx->plan.stage_bytes;
    if (cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking) != cudaSuccess) return bail(CROWN_ECUDA);
    for (int b = 0; b < 2; ++b)
      if (cudaEventCreateWithFlags(&ctx->ev_copied[b], cudaEventDisableTiming) != cudaSuccess ||
          cudaEventCreateWithFlags(&ctx->ev_free[b], cudaEventDisableTiming) != cudaSuccess) return bail(CROWN_ECUDA);
  }
  ctx->coef_base = cur; ctx->coef_off.assign(n_nodes, 0);
  { size_t off = 0;
    for (int i = 0; i < n_nodes; ++i) {
      if (ctx->nodes[i].n.op == CROWN_RELU) { ctx->coef_off[i] = off; off += align_up((size_t)B_max * ctx->nodes[i].size * 16); }
      if (ctx->nodes[i].n.op == CROWN_ADD) { ctx->coef_off[i] = off; off += align_up((size_t)ctx->nodes[i].c * 4); }
    }
    cur += ctx->plan.coef_bytes; }
  ctx->ibp_base = cur; ctx->ibp_off.assign(n_nodes, 0);
  { size_t off = 0; for (int i = 0; i < n_nodes; ++i) { ctx->ibp_off[i] = off; off += 2 * align_up((size_t)B_max * ctx->nodes[i].size * 4); } cur += ctx->plan.ibp_bytes; }
  ctx->d_buf = reinterpret_cast<float*>(cur); cur += ctx->plan.d_bytes;
  ctx->part_buf = reinterpret_cast<float*>(cur); cur += ctx->plan.part_bytes;
  ctx->io_base = cur; cur += ctx->plan.io_bytes;
  ctx->pool_base = cur;
  ctx->pool_ref.assign(ctx->plan.nbuf, 0);
  ctx->peak = (size_t)(ctx->pool_base - ctx->ws);
  // residual Add nodes fed by convolutions: the sum of the operands' biases per channel, so that the relaxation kernel of
  // the ReLU above the Add accumulates d += Abar . (b_in0 + b_in1) in the pass it makes anyway (a6: the Add fans the same A
  // out to both operands) instead of one extra pass over A per conv operand
  ctx->add_bias_ok.assign(n_nodes, 0);
  for (int i = 0; i < n_nodes; ++i) {
    const NodeInfo& ni = ctx->nodes[i];
    if (ni.n.op != CROWN_ADD || ni.h * ni.w <= 0) continue;
    const float* b0 = nullptr; const float* b1 = nullptr;
    bool any = false, ok = true;
    for (int k = 0; k < 2; ++k) {
      const int src = k == 0 ? ni.n.in0 : ni.n.in1;
      if (src < 0) continue;
      const NodeInfo& sn = ctx->nodes[src];
      if (sn.n.op == CROWN_CONV2D) { (k == 0 ? b0 : b1) = sn.n.b_dev; any = true; if (sn.c != ni.c || sn.h != ni.h || sn.w != ni.w) ok = false; }
      else if (sn.n.op == CROWN_LINEAR) ok = false;         // Linear operands keep their own bias pass
    }
    if (ni.n.in0 == ni.n.in1) ok = false;
    if (!any || !ok) continue;
    Scope sc(ctx, CROWN_K_MISC);
    launch_bias_sum(b0, b1, reinterpret_cast<float*>(ctx->coef_base + ctx->coef_off[i]), ni.c, ctx->stream);
    ctx->add_bias_ok[i] = 1;
  }
  // prepack: transpose + TF32 split of every GEMM weight operand (one pass over W)
  for (auto& ni : ctx->nodes) {
    if (!ni.tc_ok || ni.streamed) continue;
    Scope sc(ctx, CROWN_K_MISC);
    launch_split_tf32(ni.n.W_dev, ni.n.n_out, ni.n.n_in, 1, ni.Wt_hi, ni.Wt_lo, ctx->stream);
  }
  // streamed layers: the same prepack, N-slab by N-slab through the staging buffers, into pinned host memory
  for (auto& ni : ctx->nodes) {
    if (!ni.streamed) continue;
    const int K = ni.n.n_out, N = ni.n.n_in;
    const size_t bytes = (size_t)N * K * 4;
    if (cudaHostAlloc(reinterpret_cast<void**>(&ni.hWt_hi), bytes, cudaHostAllocDefault) != cudaSuccess ||
        cudaHostAlloc(reinterpret_cast<void**>(&ni.hWt_lo), bytes, cudaHostAllocDefault) != cudaSuccess) {
      return bail(CROWN_ENOMEM);
    }
    // stage[1] holds the raw column slab W[:, n0:n0+ns] as [K, ns]; stage[0] its transposed hi/lo parts [ns, K]
    const int ns_max = slab_rows(ctx->plan.stage_bytes, N, K, 2);
    for (int n0 = 0; n0 < N; n0 += ns_max) {
      const int ns = std::min(ns_max, N - n0);
      float* raw = reinterpret_cast<float*>(ctx->stage[1]);
      float* hi = reinterpret_cast<float*>(ctx->stage[0]);
      float* lo = hi + (size_t)ns * K;
      cudaError_t e1 = cudaMemcpy2DAsync(raw, (size_t)ns * 4, ni.n.W_host + n0, (size_t)N * 4, (size_t)ns * 4, K,
                                         cudaMemcpyHostToDevice, ctx->stream);
      { Scope sc(ctx, CROWN_K_MISC); launch_split_tf32(raw, K, ns, 1, hi, lo, ctx->stream); }
      cudaError_t e2 = cudaMemcpyAsync(ni.hWt_hi + (size_t)n0 * K, hi, (size_t)ns * K * 4, cudaMemcpyDeviceToHost, ctx->stream);
      cudaError_t e3 = cudaMemcpyAsync(ni.hWt_lo + (size_t)n0 * K, lo, (size_t)ns * K * 4, cudaMemcpyDeviceToHost, ctx->stream);
      cudaError_t e4 = cudaStreamSynchronize(ctx->stream);
      if (e1 != cudaSuccess || e2 != cudaSuccess || e3 != cudaSuccess || e4 != cudaSuccess) return bail(CROWN_ECUDA);
    }
  }
  if (cudaGetLastError() != cudaSuccess) return bail(CROWN_ECUDA);
  *out = ctx;
  return CROWN_OK;
}

extern "C" int crown_destroy(crown_ctx* ctx) {
  if (!ctx) return CROWN_EINVAL;
  for (auto& r : ctx->recs) { cudaEventDestroy(r.a); cudaEventDestroy(r.b); }
  for (auto e : ctx->free_events) cudaEventDestroy(e);
  for (auto& ni : ctx->nodes) { if (ni.hWt_hi) cudaFreeHost(ni.hWt_hi); if (ni.hWt_lo) cudaFreeHost(ni.hWt_lo); }
  for (int b = 0; b < 2; ++b) { if (ctx->ev_copied[b]) cudaEventDestroy(ctx->ev_copied[b]); if (ctx->ev_free[b]) cudaEventDestroy(ctx->ev_free[b]); }
  if (ctx->hpack) cudaFreeHost(ctx->hpack);
  if (ctx->copy_stream) cudaStreamDestroy(ctx->copy_stream);
  for (auto& g : ctx->graphs) if (g.exec) cudaGraphExecDestroy(g.exec);
  if (ctx->ev_gin) cudaEventDestroy(ctx->ev_gin);
  if (ctx->ev_gout) cudaEventDestroy(ctx->ev_gout);
  if (ctx->gstream) cudaStreamDestroy(ctx->gstream);
  delete ctx;
  return CROWN_OK;
}
extern "C" const char* crown_last_error(crown_ctx* ctx) { return ctx ? ctx->err.c_str() : "null context"; }
extern "C" const char* crown_version(void) { return "crownb200 0.1 (sm_100a)"; }
extern "C" int crown_peak_bytes(crown_ctx* ctx, size_t* out) { if (!ctx || !out) return CROWN_EINVAL; *out = ctx->peak; return CROWN_OK; }
extern "C" int crown_row_chunk(crown_ctx* ctx, int* out) { if (!ctx || !out) return CROWN_EINVAL; *out = ctx->plan.rc; return CROWN_OK; }
extern "C" int crown_launch_count(crown_ctx* ctx, uint64_t* out) { if (!ctx || !out) return CROWN_EINVAL; *out = ctx->launches; return CROWN_OK; }
extern "C" int crown_gemm_flops(crown_ctx* ctx, double* out) { if (!ctx || !out) return CROWN_EINVAL; *out = ctx->gemm_flops; return CROWN_OK; }
extern "C" int crown_h2d_bytes(crown_ctx* ctx, double* out) { if (!ctx || !out) return CROWN_EINVAL; *out = ctx->h2d_bytes; return CROWN_OK; }
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

}  // namespace

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
        if (ni.streamed) {
          // raw row slabs of W from pinned host memory, double-buffered on the side stream (a7)
          const int rs_max = slab_rows(ctx->plan.stage_bytes, nd.n_out, nd.n_in, 1);
          const int nslabs = (nd.n_out + rs_max - 1) / rs_max;
          int rc2 = stream_slabs(ctx, nslabs,
            [&](int sl, uint8_t* dst, cudaStream_t cs) {
              const int r0 = sl * rs_max, rs = std::min(rs_max, nd.n_out - r0);
              ctx->h2d_bytes += (double)rs * nd.n_in * 4;
              return cudaMemcpyAsync(dst, nd.W_host + (size_t)r0 * nd.n_in, (size_t)rs * nd.n_in * 4, cudaMemcpyHostToDevice, cs);
            },
            [&](int sl, uint8_t* src) {
              const int r0 = sl * rs_max, rs = std::min(rs_max, nd.n_out - r0);
              Scope sc(ctx, CROWN_K_IBP, 4.0 * rs * nd.n_in * ((B + 3) / 4), 4.0 * B * rs * (double)nd.n_in);
              launch_ibp_linear(reinterpret_cast<const float*>(src), nd.b_dev ? nd.b_dev + r0 : nullptr, li, ui, relu_in,
                                lo + r0, uo + r0, B, rs, nd.n_in, nd.n_out, s);
              return 0;
            });
          if (rc2) return rc2;
          break;
        }
        Scope sc(ctx, CROWN_K_IBP, 4.0 * nd.n_out * nd.n_in * ((B + 3) / 4), 4.0 * B * nd.n_out * (double)nd.n_in);
        launch_ibp_linear(nd.W_dev, nd.b_dev, li, ui, relu_in, lo, uo, B, nd.n_out, nd.n_in, nd.n_out, s);
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
  if (ln.streamed || !ln.n.W_dev) return fail(ctx, CROWN_EUNSUPPORTED, "ibp_forward: the spec bound needs a resident last Linear layer");
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
