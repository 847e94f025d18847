// O3 -- the CROWN backward pass (PAPER.md:64-68 Eq. 1, :128 A <- A.Lambda_i W_i), the concretisation
// and the whole-path drivers crown_run / crown_run_host (O4, O5, verdict).
// Host scheduling only: every arithmetic step is a kernel of kernels.h.
#include "ctx.h"

namespace {

// NEXT-2: split constraints of a BaB sub-domain and their Lagrange multipliers (arrays of n_nodes pointers, entries for
// ReLU nodes; nullptr arrays / entries = no split / beta = 0)
struct SplitSpec {
  const int8_t* const* split = nullptr;     // [B, size_i] in {-1, 0, +1}
  const float* const* beta_lo = nullptr;    // [B, R, size_i]
  const float* const* beta_up = nullptr;
};

struct Pass {
  crown_ctx* ctx;
  int B, R;
  std::map<int, Pending> pend;   // node id (-1 = network input) -> A w.r.t. that node's OUTPUT
};

// a fresh contiguous [2,B,R,n] buffer from the pool
int new_buf(Pass& ps, float*& ptr) {
  int id = pool_get(ps.ctx);
  if (id < 0) return -1;
  ptr = pool_ptr(ps.ctx, id);
  return id;
}

// d += A . bias of Linear/Conv node j, unless the view already carries it
void add_bias(Pass& ps, Pending& p, int j) {
  crown_ctx* ctx = ps.ctx;
  if (p.bias_done_for == j) return;
  const NodeInfo& nj = ctx->nodes[j];
  if (!nj.n.b_dev) return;
  int div = nj.n.op == CROWN_CONV2D ? nj.h * nj.w : 1;
  Scope sc(ctx, CROWN_K_MISC, 4.0 * 2 * ps.B * ps.R * p.v.n);
  launch_rowdot_bias(p.v, nj.n.b_dev, div, ctx->d_buf, ps.B, ps.R, ctx->stream);
}

// Add a contribution to node `idx`.  A node with several consumers (residual fork) receives the SUM of
// their contributions.
int contribute(Pass& ps, int idx, Pending p) {
  crown_ctx* ctx = ps.ctx;
  auto it = ps.pend.find(idx);
  if (it == ps.pend.end()) { ps.pend[idx] = p; return CROWN_OK; }
  Pending& q = it->second;
  float* out = nullptr;
  int nb = new_buf(ps, out);
  if (nb < 0) return fail(ctx, CROWN_ENOMEM, "backward: A-buffer pool exhausted at a fork");
  int done = -2;
  if (idx >= 0 && (ctx->nodes[idx].n.op == CROWN_LINEAR || ctx->nodes[idx].n.op == CROWN_CONV2D)) {
    add_bias(ps, q, idx); add_bias(ps, p, idx); done = idx;   // each part carries its own A.b before the sum
  }
  { Scope sc(ctx, CROWN_K_MISC, 12.0 * 2 * ps.B * ps.R * p.v.n);
    launch_view_add(q.v, &p.v, out, ps.B, ps.R, ctx->stream); }
  release(ctx, q); release(ctx, p);
  Pending m; m.v = canon_view(out, ps.B, ps.R, p.v.n); m.buf = nb; m.bias_done_for = done;
  it->second = m;
  return CROWN_OK;
}


float4* coef_ptr(crown_ctx* ctx, int i) { return reinterpret_cast<float4*>(ctx->coef_base + ctx->coef_off[i]); }

// One contraction A.W_i on the tensor cores, resident or streamed (N-slabs of the prepacked operand from pinned host
// memory, a7: slab s+1 -- or the next layer's first slab -- is copied on the side stream while slab s is multiplied).
// mode 0: D = product; 1: a8 fused (conc partials into part_buf); 2: a4 fused (D = hi limb, D_lo = lo limb of the
// relaxed product, d partials into part_buf).  The same rule picks the mode in both residency modes: bitwise equality.
int tc_contract(crown_ctx* ctx, const NodeInfo& ni, const float* hi, const float* lo, float* D, float* D_lo, int M_full,
                int mode, const ConcArgs* conc, const RelaxEpiArgs* rel) {
  const int K = ni.n.n_out, N = ni.n.n_in;
  cudaStream_t s = ctx->stream;
  const char* e = nullptr;
  const double out_bytes = mode == 1 ? 0.0 : (mode == 2 ? 8.0 : 4.0) * (double)M_full;
  if (!ni.streamed) {
    Scope sc(ctx, CROWN_K_GEMM_TC, 8.0 * (double)M_full * K + 8.0 * (double)K * N + out_bytes * N, 2.0 * M_full * (double)N * K);
    if (launch_gemm_tc(hi, lo, ni.Wt_hi, ni.Wt_lo, D, N, M_full, N, K, ctx->opts.k_drain, ctx->num_sms, s, &e, conc, rel))
      return fail(ctx, CROWN_ECUDA, std::string("gemm_tc: ") + (e ? e : "?"));
    ctx->launches += gemm_tc_num_panels(K) - 1;      // the Scope counted one kernel
    return CROWN_OK;
  }
  const int ns_max = slab_rows(ctx->plan.stage_bytes, N, K, 2);
  const int nslabs = (N + ns_max - 1) / ns_max;
  return stream_slabs(ctx, nslabs,
    [&](int sl, uint8_t* dst, cudaStream_t cs) {
      const int n0 = sl * ns_max, ns = std::min(ns_max, N - n0);
      float* dhi = reinterpret_cast<float*>(dst);
      ctx->h2d_bytes += 2.0 * ns * K * 4;
      cudaError_t e1 = cudaMemcpyAsync(dhi, ni.hWt_hi + (size_t)n0 * K, (size_t)ns * K * 4, cudaMemcpyHostToDevice, cs);
      if (e1 != cudaSuccess) return e1;
      return cudaMemcpyAsync(dhi + (size_t)ns * K, ni.hWt_lo + (size_t)n0 * K, (size_t)ns * K * 4, cudaMemcpyHostToDevice, cs);
    },
    [&](int sl, uint8_t* src) {
      const int n0 = sl * ns_max, ns = std::min(ns_max, N - n0);
      const float* whi = reinterpret_cast<const float*>(src);
      Scope sc(ctx, CROWN_K_GEMM_TC, 8.0 * (double)M_full * K + 8.0 * (double)K * ns + out_bytes * ns, 2.0 * M_full * (double)ns * K);
      ConcArgs ca; RelaxEpiArgs ra;
      if (conc) { ca = *conc; ca.col_off = n0; }
      if (rel) { ra = *rel; ra.col_off = n0; ra.out_lo = D_lo + n0; }
      if (launch_gemm_tc(hi, lo, whi, whi + (size_t)ns * K, D ? D + n0 : nullptr, N, M_full, ns, K, ctx->opts.k_drain,
                         ctx->num_sms, s, &e, conc ? &ca : nullptr, rel ? &ra : nullptr))
        return fail(ctx, CROWN_ECUDA, std::string("gemm_tc: ") + (e ? e : "?"));
      ctx->launches += gemm_tc_num_panels(K) - 1;
      return (int)CROWN_OK;
    });
}

// One backward pass.  coef_ready: per node, 1 if coef_ptr(i) already holds the coefficients of ReLU i for the
// bounds in l_dev/u_dev (crown_run computes each ReLU's coefficients once); may be nullptr.
int run_pass(crown_ctx* ctx, int B, int start, int row0, int R, const float* C_dev,
             const float* const* l_dev, const float* const* u_dev, const float* const* alpha_lo,
             const float* const* alpha_up, float* A_dev, float* d_dev, const float* x_lo, const float* x_hi,
             float* lb, float* ub, int out_stride, std::vector<char>* coef_ready, float* const* A_save = nullptr,
             const SplitSpec* sp = nullptr) {
  const int n = (int)ctx->nodes.size();
  cudaStream_t s = ctx->stream;
  if (B <= 0 || B > ctx->B_max || R <= 0 || R > ctx->plan.rows_cap || start < 0 || start >= n)
    return fail(ctx, CROWN_EINVAL, "crown_backward: bad B / rows / start");
  if (lb && (!ub || !x_lo || !x_hi)) return fail(ctx, CROWN_EINVAL, "crown_backward: concretisation needs ub, x_lo, x_hi");
  std::fill(ctx->pool_ref.begin(), ctx->pool_ref.end(), 0);
  Pass ps; ps.ctx = ctx; ps.B = B; ps.R = R;
  bool conc_done = false; int conc_parts = 0;
  const NodeInfo& sn = ctx->nodes[start];
  int first = start;   // first node to visit in the reverse sweep
  auto ensure_coef = [&](int i) -> int {
    if (!l_dev || !u_dev || !l_dev[i] || !u_dev[i]) return fail(ctx, CROWN_EINVAL, "crown_backward: bounds of a ReLU below start are missing");
    if (!coef_ready || !(*coef_ready)[i]) {
      Scope sc(ctx, CROWN_K_COEFF, 24.0 * B * ctx->nodes[i].size);
      launch_relax_coeffs(l_dev[i], u_dev[i], coef_ptr(ctx, i), (long long)B * ctx->nodes[i].size, ctx->opts.slope_rule, s,
                          (sp && sp->split) ? sp->split[i] : nullptr);
      if (coef_ready) (*coef_ready)[i] = 1;
    }
    return CROWN_OK;
  };
  if (C_dev) {
    { Scope sc(ctx, CROWN_K_MISC); launch_init_d(ctx->d_buf, nullptr, 0, B, R, s); }
    Pending p; p.v.p = C_dev; p.v.ld = sn.size; p.v.n = sn.size; p.v.sB = (long long)R * sn.size; p.v.sBr = 0;
    ps.pend[start] = p;
  } else if (sn.n.op != CROWN_LINEAR) {
    // NEXT-3: rows [row0, row0+R) of the identity on a conv-shaped node (Conv2d / Add / Flatten
    // output).  The start matrix is materialised once as R one-hot rows shared by all branches and properties
    // (zero-stride view) and the sweep begins AT the start node: its conv-transpose turns the rows into the 3x3xC_in
    // patches of the layer, the rest of the pass is the dense recursion, row-chunked like every identity pass.
    if (sn.n.op == CROWN_RELU) return fail(ctx, CROWN_EUNSUPPORTED, "crown_backward: identity start on a ReLU node");
    if (row0 < 0 || row0 + R > sn.size) return fail(ctx, CROWN_EINVAL, "crown_backward: row range outside the start node");
    { Scope sc(ctx, CROWN_K_MISC); launch_init_d(ctx->d_buf, nullptr, 0, B, R, s); }
    float* oh = nullptr;
    Pending p; p.buf = new_buf(ps, oh);
    if (p.buf < 0) return fail(ctx, CROWN_ENOMEM, "backward: A-buffer pool exhausted");
    { Scope sc(ctx, CROWN_K_MISC, 4.0 * R * sn.size); launch_onehot(oh, row0, R, sn.size, s); }
    p.v.p = oh; p.v.ld = sn.size; p.v.n = sn.size; p.v.sB = 0; p.v.sBr = 0;
    ps.pend[start] = p;
  } else {
    // rows [row0, row0+R) of the identity on a Linear node: I.W = those rows of W, I.b = those biases
    if (row0 < 0 || row0 + R > sn.size) return fail(ctx, CROWN_EINVAL, "crown_backward: row range outside the start node");
    { Scope sc(ctx, CROWN_K_MISC); launch_init_d(ctx->d_buf, sn.n.b_dev, row0, B, R, s); }
    Pending p; p.v.ld = sn.n.n_in; p.v.n = sn.n.n_in; p.v.sB = 0; p.v.sBr = 0;
    if (sn.streamed) {   // no resident copy: fetch the R rows from the caller's pinned host buffer into an A buffer
      float* rowsbuf = nullptr;
      p.buf = new_buf(ps, rowsbuf);
      if (p.buf < 0) return fail(ctx, CROWN_ENOMEM, "backward: A-buffer pool exhausted");
      CK(ctx, cudaMemcpyAsync(rowsbuf, sn.n.W_host + (size_t)row0 * sn.n.n_in, (size_t)R * sn.n.n_in * 4,
                              cudaMemcpyHostToDevice, s));
      ctx->h2d_bytes += (double)R * sn.n.n_in * 4;
      p.v.p = rowsbuf;
    } else {
      p.v.p = sn.n.W_dev + (long long)row0 * sn.n.n_in;
    }
    ps.pend[sn.n.in0] = p;
    first = start - 1;
  }
  for (int i = first; i >= 0; --i) {
    auto it = ps.pend.find(i);
    if (it == ps.pend.end()) continue;
    Pending cur = it->second;
    ps.pend.erase(it);
    const NodeInfo& ni = ctx->nodes[i];
    const crown_node& nd = ni.n;
    int rc = CROWN_OK;
    switch (nd.op) {
      case CROWN_RELU: {
        if ((rc = ensure_coef(i))) return rc;
        const int j = nd.in0;
        if (A_save && A_save[i] && cur.v.p != A_save[i]) {   // alpha optimisation: keep A as it arrives at this ReLU, contiguous
                                                              // [2,B,R,n] (unless the contraction above already wrote it there)
          Scope sc(ctx, CROWN_K_MISC, 8.0 * 2 * B * R * ni.size);
          launch_view_add(cur.v, nullptr, A_save[i], B, R, s);
        }
        const bool lin_below = j >= 0 && (ctx->nodes[j].n.op == CROWN_LINEAR || ctx->nodes[j].n.op == CROWN_CONV2D);
        // the product that follows runs on the tensor cores when the producer is a prepacked Linear
        const bool tc = lin_below && ctx->nodes[j].tc_ok && (ctx->nodes[j].streamed || gemm_tc_supported(2 * B * R, ctx->nodes[j].n.n_in, ctx->nodes[j].n.n_out));
        RelaxArgs ra;
        ra.A = cur.v; ra.coef = coef_ptr(ctx, i);
        ra.alpha_lo = alpha_lo ? alpha_lo[i] : nullptr;
        ra.alpha_up = alpha_up ? alpha_up[i] : nullptr;
        ra.bias = lin_below ? ctx->nodes[j].n.b_dev : nullptr;
        ra.bias_div = (lin_below && ctx->nodes[j].n.op == CROWN_CONV2D) ? ctx->nodes[j].h * ctx->nodes[j].w : 1;
        // ReLU over a residual Add of convolutions: the Add hands the same A to both operands, so their biases are
        // accumulated here as one summed vector (crown_init) and the operands' own bias passes are skipped
        const bool add_below = j >= 0 && ctx->nodes[j].n.op == CROWN_ADD && ctx->add_bias_ok[j] && ctx->nodes[j].n_consumers == 1 &&
                               ps.pend.find(j) == ps.pend.end();
        if (add_below) {
          ra.bias = reinterpret_cast<const float*>(ctx->coef_base + ctx->coef_off[j]);
          ra.bias_div = ctx->nodes[j].h * ctx->nodes[j].w;
        }
        ra.d = ctx->d_buf; ra.B = B; ra.R = R; ra.n = ni.size;
        if (sp && sp->split && sp->split[i]) {
          ra.split = sp->split[i];
          ra.beta_lo = sp->beta_lo ? sp->beta_lo[i] : nullptr;
          ra.beta_up = sp->beta_up ? sp->beta_up[i] : nullptr;
        }
        Pending out;
        out.buf = new_buf(ps, ra.out);
        if (out.buf < 0) return fail(ctx, CROWN_ENOMEM, "backward: A-buffer pool exhausted");
        ra.out_lo = nullptr;
        if (tc) { out.buf_lo = new_buf(ps, ra.out_lo); if (out.buf_lo < 0) return fail(ctx, CROWN_ENOMEM, "backward: A-buffer pool exhausted"); }
        // algorithmic bytes: every DISTINCT input row is read once (at the start of a pass all branches / properties
        // share the R rows of W_k), every output row is written once (+ the lo limb), alpha once per (row, neuron)
        const double in_rows = (double)(cur.v.sBr ? 2 : 1) * (cur.v.sB ? B : 1) * R;
        const double out_rows = 2.0 * B * R;
        { Scope sc(ctx, CROWN_K_RELAX, 4.0 * ni.size * (in_rows + out_rows * (tc ? 2.0 : 1.0)) +
                                       ((ra.alpha_lo || ra.alpha_up) ? 4.0 * B * R * ni.size : 0.0) +
                                       ((ra.beta_lo ? 4.0 : 0.0) + (ra.beta_up && ra.beta_up != ra.beta_lo ? 4.0 : 0.0)) * B * R * ni.size);
          launch_relax(ra, s); }
        out.v = canon_view(ra.out, B, R, ni.size); out.v.lo = ra.out_lo;
        out.bias_done_for = (lin_below || add_below) ? j : -2;
        release(ctx, cur);
        rc = contribute(ps, j, out);
        break; }
      case CROWN_LINEAR: {
        add_bias(ps, cur, i);
        const int M_full = 2 * B * R;
        Pending out;
        float* D = nullptr;
        if (ni.tc_ok && (ni.streamed || gemm_tc_supported(M_full, nd.n_in, nd.n_out))) {
          const float *hi = cur.v.p, *lo = cur.v.lo;
          Pending tmp;
          if (!lo) {   // operand not split yet (start matrix, fork sum): split pass, also makes it contiguous
            RelaxArgs ra; ra.A = cur.v; ra.coef = nullptr; ra.alpha_lo = ra.alpha_up = nullptr; ra.bias = nullptr; ra.bias_div = 1;
            ra.d = nullptr; ra.B = B; ra.R = R; ra.n = ni.size;
            tmp.buf = new_buf(ps, ra.out); tmp.buf_lo = new_buf(ps, ra.out_lo);
            if (tmp.buf < 0 || tmp.buf_lo < 0) return fail(ctx, CROWN_ENOMEM, "backward: A-buffer pool exhausted");
            const double in_rows = (double)(cur.v.sBr ? 2 : 1) * (cur.v.sB ? B : 1) * R;
            { Scope sc(ctx, CROWN_K_RELAX, 4.0 * ni.size * (in_rows + 2.0 * M_full)); launch_relax(ra, s); }
            hi = ra.out; lo = ra.out_lo;
            release(ctx, cur); cur = tmp;
          }
          const int K = nd.n_out, N = nd.n_in;
          const int parts = gemm_tc_parts(N);
          const bool single = gemm_tc_single_panel(K) != 0;
          // a8 fused: the last contraction of the pass concretises in its epilogue, A_0 never reaches HBM
          const bool fc = nd.in0 < 0 && lb && !A_dev && ctx->input_consumers == 1 && ps.pend.find(-1) == ps.pend.end() &&
                          !ctx->opts.disable_conc_fusion && single && (size_t)M_full * parts * 8 <= ctx->plan.part_bytes;
          // a4 fused: the product feeds a ReLU (only consumer: this layer) over a tensor-core Linear, fixed-rule slopes:
          // the epilogue applies that relaxation and emits the next operand's limbs (A <- A.Lambda W as one kernel)
          int r = nd.in0, j = -1;
          bool fr = false;
          if (!fc && r >= 0 && ctx->nodes[r].n.op == CROWN_RELU && ctx->nodes[r].n_consumers == 1 &&
              ps.pend.find(r) == ps.pend.end() && !ctx->opts.disable_epi_fusion && single && (R % 32) == 0 &&
              !(alpha_lo && alpha_lo[r]) && !(alpha_up && alpha_up[r]) && !(sp && sp->split && sp->split[r]) &&
              (size_t)M_full * parts * 4 <= ctx->plan.part_bytes) {
            j = ctx->nodes[r].n.in0;
            fr = j >= 0 && ctx->nodes[j].n.op == CROWN_LINEAR && ctx->nodes[j].tc_ok &&
                 (ctx->nodes[j].streamed || gemm_tc_supported(M_full, ctx->nodes[j].n.n_in, ctx->nodes[j].n.n_out));
          }
          if (fc) {
            ConcArgs ca;
            ca.x_lo = x_lo; ca.x_hi = x_hi; ca.part = ctx->part_buf; ca.B = B; ca.R = R; ca.parts = parts; ca.ldx = N;
            if ((rc = tc_contract(ctx, ni, hi, lo, nullptr, nullptr, M_full, 1, &ca, nullptr))) return rc;
            conc_done = true; conc_parts = parts;
            ctx->gemm_flops += 2.0 * M_full * (double)N * K;
            release(ctx, cur);
            break;                      // nothing is contributed to the input node: the bound is finished below
          }
          // alpha / beta optimisation: the product that arrives at a ReLU whose A is kept goes straight into that buffer
          // (one copy of A per ReLU and evaluation less)
          float* direct = (!fr && A_save && r >= 0 && ctx->nodes[r].n.op == CROWN_RELU && A_save[r] &&
                           ctx->nodes[r].n_consumers == 1 && ps.pend.find(r) == ps.pend.end() && !ni.streamed) ? A_save[r] : nullptr;
          if (direct) { D = direct; out.buf = -1; }
          else {
            out.buf = new_buf(ps, D);
            if (out.buf < 0) return fail(ctx, CROWN_ENOMEM, "backward: A-buffer pool exhausted");
          }
          if (fr) {
            if ((rc = ensure_coef(r))) return rc;
            float* D_lo = nullptr;
            out.buf_lo = new_buf(ps, D_lo);
            if (out.buf_lo < 0) return fail(ctx, CROWN_ENOMEM, "backward: A-buffer pool exhausted");
            RelaxEpiArgs re;
            re.coef = coef_ptr(ctx, r); re.coef_ld = N; re.bias = ctx->nodes[j].n.b_dev; re.out_lo = D_lo;
            re.part = ctx->part_buf; re.B = B; re.R = R; re.parts = parts;
            if ((rc = tc_contract(ctx, ni, hi, lo, D, D_lo, M_full, 2, nullptr, &re))) return rc;
            { Scope sc(ctx, CROWN_K_MISC, 4.0 * M_full * parts); launch_reduce_parts(ctx->part_buf, parts, ctx->d_buf, M_full, s); }
            ctx->gemm_flops += 2.0 * M_full * (double)N * K;
            out.v = canon_view(D, B, R, N); out.v.lo = D_lo;
            out.bias_done_for = j;
            release(ctx, cur);
            rc = contribute(ps, j, out);      // ReLU r is done: the relaxed product is A w.r.t. node j's output
            break;
          }
          if ((rc = tc_contract(ctx, ni, hi, lo, D, nullptr, M_full, 0, nullptr, nullptr))) return rc;
          ctx->gemm_flops += 2.0 * M_full * (double)N * K;
          out.v = canon_view(D, B, R, N);
        } else {
          // CUDA-core contraction; rows shared between branches / properties are multiplied once
          int m_eff = 0;
          if (ni.streamed) return fail(ctx, CROWN_EUNSUPPORTED, "backward: a streamed layer needs the tensor-core path");
          if (!view_uniform(cur.v, B, R, m_eff)) return fail(ctx, CROWN_EINVAL, "backward: non-uniform A view");
          if (cur.v.lo) return fail(ctx, CROWN_EINVAL, "backward: split operand on the CUDA-core path");
          out.buf = new_buf(ps, D);
          if (out.buf < 0) return fail(ctx, CROWN_ENOMEM, "backward: A-buffer pool exhausted");
          { Scope sc(ctx, CROWN_K_GEMM_FFMA, 4.0 * ((double)m_eff * nd.n_out + (double)nd.n_out * nd.n_in + (double)m_eff * nd.n_in),
                     2.0 * m_eff * (double)nd.n_in * nd.n_out);
            launch_gemm_ffma(cur.v.p, cur.v.ld, nd.W_dev, nd.n_in, D, nd.n_in, m_eff, nd.n_in, nd.n_out, s); }
          ctx->gemm_flops += 2.0 * m_eff * (double)nd.n_in * nd.n_out;
          out.v.p = D; out.v.ld = nd.n_in; out.v.n = nd.n_in;
          out.v.sB = cur.v.sB ? (long long)R * nd.n_in : 0;
          out.v.sBr = cur.v.sBr ? (long long)(cur.v.sB ? B : 1) * R * nd.n_in : 0;
        }
        release(ctx, cur);
        rc = contribute(ps, nd.in0, out);
        break; }
      case CROWN_CONV2D: {
        if (cur.v.lo) {   // the conv kernels take plain fp32: fold a TF32-split view back (hi + lo is exact)
          float* F = nullptr;
          Pending f; f.buf = new_buf(ps, F);
          if (f.buf < 0) return fail(ctx, CROWN_ENOMEM, "backward: A-buffer pool exhausted");
          { Scope sc(ctx, CROWN_K_MISC, 12.0 * 2 * B * R * cur.v.n); launch_view_add(cur.v, nullptr, F, B, R, s); }
          f.v = canon_view(F, B, R, cur.v.n); f.bias_done_for = cur.bias_done_for;
          release(ctx, cur); cur = f;
        }
        add_bias(ps, cur, i);
        Pending out;
        float* D = nullptr;
        out.buf = new_buf(ps, D);
        if (out.buf < 0) return fail(ctx, CROWN_ENOMEM, "backward: A-buffer pool exhausted");
        const int in_size = nd.c_in * nd.h_in * nd.w_in;
        // residual fork: when the node this conv feeds already holds the other consumer's contribution (a plain
        // contiguous buffer, no bias bookkeeping attached), the kernel adds it in its epilogue (no separate sum pass)
        const float* addend = nullptr;
        Pending other;
        {
          auto itp = ps.pend.find(nd.in0);
          const bool plain_node = nd.in0 < 0 || (ctx->nodes[nd.in0].n.op != CROWN_LINEAR && ctx->nodes[nd.in0].n.op != CROWN_CONV2D);
          // only the tensor-core kernel absorbs the addend for free (its loads hide behind the MMAs); on the CUDA-core
          // kernel it measured the same as the separate sum pass
          const bool tc_conv = ctx->opts.mma_scheme == 0 && !ctx->opts.disable_conv_tc && !cur.v.lo &&
                               conv_tc_supported(nd.c_in, nd.h_in, nd.w_in, nd.c_out, nd.kh, nd.kw, nd.stride, nd.pad, ni.h, ni.w);
          const bool s2_conv = !cur.v.lo && conv_s2_supported(nd.c_in, nd.h_in, nd.w_in, nd.c_out, nd.kh, nd.kw, nd.stride, nd.pad, ni.h, ni.w) &&
                               (2LL * B * R * in_size) % 2 == 0;
          if (itp != ps.pend.end() && plain_node && (tc_conv || s2_conv) && !itp->second.v.lo && itp->second.v.n == in_size && itp->second.v.ld == in_size &&
              itp->second.v.sB == (long long)R * in_size && itp->second.v.sBr == (long long)B * R * in_size) {
            other = itp->second; addend = other.v.p; ps.pend.erase(itp);
          }
        }
        // rows still shared by all branches and properties (the first hops of an identity pass on a conv map, NEXT-3) are
        // transposed ONCE: the R rows run as a B = 1 problem whose "upper branch" is the second half of the rows
        const bool shared_rows = cur.v.sB == 0 && cur.v.sBr == 0 && !cur.v.lo && !addend && (R % 2) == 0 && B * 2 > 1;
        if (shared_rows) {
          AView v2 = cur.v; v2.sBr = (long long)(R / 2) * cur.v.ld;
          { Scope sc(ctx, CROWN_K_CONV, 4.0 * R * ((double)ni.size + in_size), 2.0 * R * (double)ni.size * nd.c_in * nd.kh * nd.kw);
            launch_conv_transpose(v2, nd.W_dev, nullptr, D, 1, R / 2, nd.c_in, nd.h_in, nd.w_in, nd.c_out, nd.kh, nd.kw,
                                  nd.stride, nd.pad, ni.h, ni.w, s, ctx->opts.mma_scheme == 0 && !ctx->opts.disable_conv_tc, ctx->num_sms); }
          out.v.p = D; out.v.ld = in_size; out.v.n = in_size; out.v.sB = 0; out.v.sBr = 0;
          release(ctx, cur);
          rc = contribute(ps, nd.in0, out);
          break;
        }
        { Scope sc(ctx, CROWN_K_CONV, 4.0 * 2 * B * R * ((double)ni.size + in_size * (addend ? 2.0 : 1.0)),
                   2.0 * 2 * B * R * (double)ni.size * nd.c_in * nd.kh * nd.kw);
          launch_conv_transpose(cur.v, nd.W_dev, addend, D, B, R, nd.c_in, nd.h_in, nd.w_in, nd.c_out, nd.kh, nd.kw,
                                nd.stride, nd.pad, ni.h, ni.w, s, ctx->opts.mma_scheme == 0 && !ctx->opts.disable_conv_tc, ctx->num_sms); }
        out.v = canon_view(D, B, R, in_size);
        if (addend) release(ctx, other);
        release(ctx, cur);
        rc = contribute(ps, nd.in0, out);
        break; }
      case CROWN_ADD: {
        Pending second = cur;
        pool_retain(ctx, second.buf); pool_retain(ctx, second.buf_lo);
        {
          // the summed bias of the conv operands went into d with the relaxation above this Add (see CROWN_RELU)
          const bool done = cur.bias_done_for == i && ctx->add_bias_ok[i];
          auto mark = [&](int src) { return (done && src >= 0 && ctx->nodes[src].n.op == CROWN_CONV2D) ? src : -2; };
          cur.bias_done_for = mark(nd.in0);
          second.bias_done_for = mark(nd.in1);
        }
        rc = contribute(ps, nd.in0, cur);
        if (rc == CROWN_OK) rc = contribute(ps, nd.in1, second);
        break; }
      case CROWN_FLATTEN:
        rc = contribute(ps, nd.in0, cur);
        break;
      default:
        return fail(ctx, CROWN_EUNSUPPORTED, "crown_backward: unsupported op");
    }
    if (rc) return rc;
  }
  if (conc_done) {   // the bound was concretised inside the last contraction
    if (d_dev) CK(ctx, cudaMemcpyAsync(d_dev, ctx->d_buf, (size_t)2 * B * R * 4, cudaMemcpyDeviceToDevice, s));
    { Scope sc(ctx, CROWN_K_CONCRETIZE, 8.0 * 2 * B * R * conc_parts);
      launch_concretize_parts(ctx->part_buf, conc_parts, ctx->d_buf, lb, ub, out_stride, B, R, s); }
    CK(ctx, cudaGetLastError());
    return CROWN_OK;
  }
  // A w.r.t. the network input
  auto it = ps.pend.find(-1);
  if (it == ps.pend.end()) return fail(ctx, CROWN_EINVAL, "crown_backward: start node does not reach the input");
  Pending a0 = it->second;
  if (a0.v.n != ctx->n0) return fail(ctx, CROWN_EINVAL, "crown_backward: internal size mismatch at the input");
  if (A_dev) { Scope sc(ctx, CROWN_K_MISC, 8.0 * 2 * B * R * ctx->n0); launch_view_add(a0.v, nullptr, A_dev, B, R, s); }
  if (d_dev) CK(ctx, cudaMemcpyAsync(d_dev, ctx->d_buf, (size_t)2 * B * R * 4, cudaMemcpyDeviceToDevice, s));
  if (lb) { Scope sc(ctx, CROWN_K_CONCRETIZE, 4.0 * 2 * B * R * ctx->n0, 4.0 * 2 * B * R * ctx->n0);
            launch_concretize(a0.v, ctx->d_buf, x_lo, x_hi, lb, ub, out_stride, B, R, s); }
  release(ctx, a0);
  CK(ctx, cudaGetLastError());
  return CROWN_OK;
}

}  // namespace

extern "C" int crown_backward(crown_ctx* ctx, int B, int start, int row0, int rows, const float* C_dev,
                              const float* const* l_dev, const float* const* u_dev,
                              const float* const* alpha_lo_dev, const float* const* alpha_up_dev,
                              float* A_dev, float* d_dev, const float* x_lo_dev, const float* x_hi_dev,
                              float* lb_dev, float* ub_dev) {
  if (!ctx) return CROWN_EINVAL;
  if (!A_dev && !d_dev && !lb_dev) return fail(ctx, CROWN_EINVAL, "crown_backward: no output requested");
  return run_pass(ctx, B, start, row0, rows, C_dev, l_dev, u_dev, alpha_lo_dev, alpha_up_dev, A_dev, d_dev,
                  x_lo_dev, x_hi_dev, lb_dev, ub_dev, rows, nullptr);
}

extern "C" int concretize(crown_ctx* ctx, int B, int rows, const float* A_dev, const float* d_dev,
                          const float* x_lo_dev, const float* x_hi_dev, float* lb_dev, float* ub_dev,
                          int out_stride) {
  if (!ctx) return CROWN_EINVAL;
  if (B <= 0 || rows <= 0 || !A_dev || !x_lo_dev || !x_hi_dev || !lb_dev || !ub_dev || out_stride < rows)
    return fail(ctx, CROWN_EINVAL, "concretize: bad arguments");
  AView v = canon_view(A_dev, B, rows, ctx->n0);
  { Scope sc(ctx, CROWN_K_CONCRETIZE, 4.0 * 2 * B * rows * ctx->n0, 4.0 * 2 * B * rows * ctx->n0);
    launch_concretize(v, d_dev, x_lo_dev, x_hi_dev, lb_dev, ub_dev, out_stride, B, rows, ctx->stream); }
  CK(ctx, cudaGetLastError());
  return CROWN_OK;
}

extern "C" int crown_verdict(crown_ctx* ctx, int B, int S, const float* lb_dev, uint8_t* verified_dev) {
  if (!ctx) return CROWN_EINVAL;
  if (B <= 0 || S <= 0 || !lb_dev || !verified_dev) return fail(ctx, CROWN_EINVAL, "crown_verdict: bad arguments");
  { Scope sc(ctx, CROWN_K_MISC); launch_verdict(lb_dev, verified_dev, B, S, ctx->stream); }
  CK(ctx, cudaGetLastError());
  return CROWN_OK;
}

// ================================================================================================
// O4 + O5 + verdict: the whole hot path for one batch
// ================================================================================================
static int crown_run_enqueue(crown_ctx* ctx, int B, const float* x_lo_dev, const float* x_hi_dev,
                             const float* C_dev, int S, const float* const* alpha_dev, int intermediate,
                             float* const* l_dev, float* const* u_dev, float* lb_dev, float* ub_dev,
                             uint8_t* verified_dev) {
  if (!ctx) return CROWN_EINVAL;
  const int n = (int)ctx->nodes.size();
  if (B <= 0 || B > ctx->B_max || S <= 0 || S > ctx->S_max || !x_lo_dev || !x_hi_dev || !C_dev || !l_dev ||
      !u_dev || !lb_dev || !ub_dev || (intermediate != 0 && intermediate != 1))
    return fail(ctx, CROWN_EINVAL, "crown_run: bad arguments");
  std::vector<int> relus;
  for (int i = 0; i < n; ++i)
    if (ctx->nodes[i].n.op == CROWN_RELU) {
      if (!l_dev[i] || !u_dev[i]) return fail(ctx, CROWN_EINVAL, "crown_run: l_dev/u_dev entry of a ReLU node is NULL");
      if (ctx->nodes[i].n.in0 < 0) return fail(ctx, CROWN_EUNSUPPORTED, "crown_run: ReLU directly on the input");
      relus.push_back(i);
    }
  // IBP writes the OUTPUT interval of node in0(relu) straight into the caller's pre-activation buffers
  std::vector<float*> lmap(n, nullptr), umap(n, nullptr), L, U;
  std::vector<const float*> lc(n, nullptr), uc(n, nullptr);
  for (int i : relus) {
    const int src = ctx->nodes[i].n.in0;
    if (lmap[src]) return fail(ctx, CROWN_EUNSUPPORTED, "crown_run: two ReLUs on one node");
    lmap[src] = l_dev[i]; umap[src] = u_dev[i];
    lc[i] = l_dev[i]; uc[i] = u_dev[i];
  }
  std::vector<char> coef_ready(n, 0);
  int rc;
  if (intermediate == 1) {
    rc = ibp_internal(ctx, B, x_lo_dev, x_hi_dev, lmap.data(), umap.data(), L, U, false);
    if (rc) return rc;
  } else {
    rc = ibp_internal(ctx, B, x_lo_dev, x_hi_dev, lmap.data(), umap.data(), L, U, true);
    if (rc) return rc;
    for (int i : relus) {
      const int src = ctx->nodes[i].n.in0;
      const crown_node& sn = ctx->nodes[src].n;
      if ((sn.op == CROWN_LINEAR || sn.op == CROWN_CONV2D) && sn.in0 < 0) continue;   // first layer: O1 (exact)
      const int size = ctx->nodes[src].size;
      for (int row0 = 0; row0 < size; row0 += ctx->plan.rc) {
        const int rows = std::min(ctx->plan.rc, size - row0);
        rc = run_pass(ctx, B, src, row0, rows, nullptr, lc.data(), uc.data(), nullptr, nullptr, nullptr, nullptr,
                      x_lo_dev, x_hi_dev, l_dev[i] + row0, u_dev[i] + row0, size, &coef_ready);
        if (rc) return rc;
      }
    }
  }
  rc = run_pass(ctx, B, n - 1, 0, S, C_dev, lc.data(), uc.data(), alpha_dev, alpha_dev, nullptr, nullptr,
                x_lo_dev, x_hi_dev, lb_dev, ub_dev, S, &coef_ready);
  if (rc) return rc;
  if (verified_dev) { Scope sc(ctx, CROWN_K_MISC); launch_verdict(lb_dev, verified_dev, B, S, ctx->stream); }
  CK(ctx, cudaGetLastError());
  return CROWN_OK;
}


// ---- CUDA-graph replay of crown_run ------------------------------------------------------------------------------
// The launch sequence of a step depends only on shapes and pointers, never on data, so a step is captured once per
// (B, S, intermediate, pointer set) into a CUDA graph and replayed: one cudaGraphLaunch instead of 12-70 kernel
// launches.  For the latency-bound configs (cfg1: ~0.2 GFLOP behind a dozen dependent launches) the host launch
// path is the step time.  Capture needs a capturable stream: when the caller gave the legacy default stream, the
// graph runs on a side stream joined to it by events.  Streamed layers (side-stream copies) and timing mode bypass it.
static bool graph_eligible(crown_ctx* ctx) {
  if (ctx->opts.disable_graph || ctx->timing) return false;
  for (const auto& ni : ctx->nodes) if (ni.streamed) return false;
  return true;
}

extern "C" int crown_run(crown_ctx* ctx, int B, const float* x_lo_dev, const float* x_hi_dev,
                         const float* C_dev, int S, const float* const* alpha_dev, int intermediate,
                         float* const* l_dev, float* const* u_dev, float* lb_dev, float* ub_dev,
                         uint8_t* verified_dev) {
  if (!ctx) return CROWN_EINVAL;
  if (!graph_eligible(ctx) || !l_dev || !u_dev)
    return crown_run_enqueue(ctx, B, x_lo_dev, x_hi_dev, C_dev, S, alpha_dev, intermediate, l_dev, u_dev, lb_dev, ub_dev, verified_dev);
  const int n = (int)ctx->nodes.size();
  std::vector<uintptr_t> key;
  key.reserve(8 + 3 * n);
  key.push_back((uintptr_t)B); key.push_back((uintptr_t)S); key.push_back((uintptr_t)intermediate);
  for (const void* q : {(const void*)x_lo_dev, (const void*)x_hi_dev, (const void*)C_dev, (const void*)lb_dev,
                        (const void*)ub_dev, (const void*)verified_dev}) key.push_back((uintptr_t)q);
  for (int i = 0; i < n; ++i) {
    key.push_back((uintptr_t)l_dev[i]); key.push_back((uintptr_t)u_dev[i]);
    key.push_back(alpha_dev ? (uintptr_t)alpha_dev[i] : 0);
  }
  const bool legacy = ctx->stream == nullptr || ctx->stream == cudaStreamLegacy;
  cudaStream_t user = ctx->stream;
  if (legacy && !ctx->gstream) {
    CK(ctx, cudaStreamCreateWithFlags(&ctx->gstream, cudaStreamNonBlocking));
    CK(ctx, cudaEventCreateWithFlags(&ctx->ev_gin, cudaEventDisableTiming));
    CK(ctx, cudaEventCreateWithFlags(&ctx->ev_gout, cudaEventDisableTiming));
  }
  cudaStream_t gs = legacy ? ctx->gstream : user;
  GraphEntry* ge = nullptr;
  for (auto& e : ctx->graphs) if (e.key == key) { ge = &e; break; }
  if (!ge) {
    // capture: the normal enqueue path runs with the capture stream as the context's stream; nothing executes yet
    GraphEntry e; e.key = key;
    const uint64_t l0 = ctx->launches; const double f0 = ctx->gemm_flops;
    ctx->stream = gs;
    cudaError_t ce = cudaStreamBeginCapture(gs, cudaStreamCaptureModeThreadLocal);
    int rc = CROWN_OK;
    if (ce == cudaSuccess) {
      rc = crown_run_enqueue(ctx, B, x_lo_dev, x_hi_dev, C_dev, S, alpha_dev, intermediate, l_dev, u_dev, lb_dev, ub_dev, verified_dev);
      cudaGraph_t g = nullptr;
      ce = cudaStreamEndCapture(gs, &g);
      if (rc == CROWN_OK && ce == cudaSuccess && g) ce = cudaGraphInstantiate(&e.exec, g, 0);
      if (g) cudaGraphDestroy(g);
    }
    ctx->stream = user;
    e.launches = ctx->launches - l0; e.flops = ctx->gemm_flops - f0;
    ctx->launches = l0; ctx->gemm_flops = f0;
    if (rc != CROWN_OK) { (void)cudaGetLastError(); return rc; }
    if (ce != cudaSuccess || !e.exec) {
      // capture not possible here (e.g. an uncapturable stream): run the plain path from now on
      (void)cudaGetLastError();
      ctx->opts.disable_graph = 1;
      return crown_run_enqueue(ctx, B, x_lo_dev, x_hi_dev, C_dev, S, alpha_dev, intermediate, l_dev, u_dev, lb_dev, ub_dev, verified_dev);
    }
    if (ctx->graphs.size() >= 8) { cudaGraphExecDestroy(ctx->graphs.front().exec); ctx->graphs.erase(ctx->graphs.begin()); }
    ctx->graphs.push_back(e);
    ge = &ctx->graphs.back();
  }
  if (legacy) { CK(ctx, cudaEventRecord(ctx->ev_gin, user)); CK(ctx, cudaStreamWaitEvent(gs, ctx->ev_gin, 0)); }
  CK(ctx, cudaGraphLaunch(ge->exec, gs));
  if (legacy) { CK(ctx, cudaEventRecord(ctx->ev_gout, gs)); CK(ctx, cudaStreamWaitEvent(user, ctx->ev_gout, 0)); }
  ctx->launches += ge->launches; ctx->gemm_flops += ge->flops;
  ctx->graph_replays++;
  return CROWN_OK;
}

extern "C" int crown_graph_replays(crown_ctx* ctx, uint64_t* out) { if (!ctx || !out) return CROWN_EINVAL; *out = ctx->graph_replays; return CROWN_OK; }

extern "C" int crown_run_host(crown_ctx* ctx, int B, const float* x_lo_host, const float* x_hi_host,
                              const float* C_host, int S, const float* const* alpha_host, int intermediate,
                              float* lb_host, float* ub_host, uint8_t* verified_host) {
  if (!ctx) return CROWN_EINVAL;
  const int n = (int)ctx->nodes.size();
  if (B <= 0 || B > ctx->B_max || S <= 0 || S > ctx->S_max || !x_lo_host || !x_hi_host || !C_host || !lb_host || !ub_host)
    return fail(ctx, CROWN_EINVAL, "crown_run_host: bad arguments");
  // the box is in host memory here, so x_lo <= x_hi is checked (CROWN_EINVAL); the device-pointer
  // entry points do not check it (it would need a device->host sync) and propagate whatever they are given
  for (size_t k = 0; k < (size_t)B * ctx->n0; ++k)
    if (x_lo_host[k] > x_hi_host[k]) return fail(ctx, CROWN_EINVAL, "crown_run_host: x_lo > x_hi");
  cudaStream_t s = ctx->stream;
  // staging layout inside the workspace: [inputs: alpha per ReLU, x_lo, x_hi, C] [l, u per ReLU] [outputs: lb, ub, verified]
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t o = off; off += align_up(bytes); return o; };
  std::vector<size_t> a_off(n, 0), l_off(n, 0), u_off(n, 0);
  for (int i = 0; i < n; ++i)
    if (ctx->nodes[i].n.op == CROWN_RELU) a_off[i] = take((size_t)ctx->B_max * ctx->S_max * ctx->nodes[i].size * 4);
  const size_t nL = ctx->nodes.back().size;
  const size_t xl_off = take((size_t)ctx->B_max * ctx->n0 * 4), xh_off = take((size_t)ctx->B_max * ctx->n0 * 4);
  const size_t C_off = take((size_t)ctx->B_max * ctx->S_max * nL * 4);
  const size_t in_bytes = off;
  for (int i = 0; i < n; ++i)
    if (ctx->nodes[i].n.op == CROWN_RELU) {
      l_off[i] = take((size_t)ctx->B_max * ctx->nodes[i].size * 4);
      u_off[i] = take((size_t)ctx->B_max * ctx->nodes[i].size * 4);
    }
  const size_t out0 = off;
  const size_t lb_off = take((size_t)ctx->B_max * ctx->S_max * 4), ub_off = take((size_t)ctx->B_max * ctx->S_max * 4);
  const size_t ver_off = take((size_t)ctx->B_max);
  const size_t out_bytes = off - out0;
  if (off > ctx->plan.io_bytes) return fail(ctx, CROWN_ENOMEM, "crown_run_host: staging region too small");
  uint8_t* io = ctx->io_base;
  // Small problems (cfg1: 25 KB in, 73 B out) are latency-bound on the NUMBER of copies: everything is packed into one
  // pinned mirror of the staging region (allocated once) and moved by ONE copy per direction instead of 4 + 2 per ReLU.
  constexpr size_t kPackMax = (size_t)1 << 20;
  const bool pack = in_bytes + out_bytes <= kPackMax;
  if (pack && !ctx->hpack) {
    if (cudaHostAlloc(reinterpret_cast<void**>(&ctx->hpack), in_bytes + out_bytes, cudaHostAllocDefault) != cudaSuccess) {
      (void)cudaGetLastError();
      ctx->hpack = nullptr;
    }
  }
  const bool packed = pack && ctx->hpack != nullptr;
  std::vector<float*> l(n, nullptr), u(n, nullptr);
  std::vector<const float*> al(n, nullptr);
  bool any_alpha = false;
  for (int i = 0; i < n; ++i) {
    if (ctx->nodes[i].n.op != CROWN_RELU) continue;
    const size_t sz = ctx->nodes[i].size;
    l[i] = reinterpret_cast<float*>(io + l_off[i]);
    u[i] = reinterpret_cast<float*>(io + u_off[i]);
    if (alpha_host && alpha_host[i]) {
      if (packed) std::memcpy(ctx->hpack + a_off[i], alpha_host[i], (size_t)B * S * sz * 4);
      else CK(ctx, cudaMemcpyAsync(io + a_off[i], alpha_host[i], (size_t)B * S * sz * 4, cudaMemcpyHostToDevice, s));
      al[i] = reinterpret_cast<const float*>(io + a_off[i]); any_alpha = true;
    }
  }
  float* xl = reinterpret_cast<float*>(io + xl_off);
  float* xh = reinterpret_cast<float*>(io + xh_off);
  float* C = reinterpret_cast<float*>(io + C_off);
  float* lb = reinterpret_cast<float*>(io + lb_off);
  float* ub = reinterpret_cast<float*>(io + ub_off);
  uint8_t* ver = io + ver_off;
  if (packed) {
    std::memcpy(ctx->hpack + xl_off, x_lo_host, (size_t)B * ctx->n0 * 4);
    std::memcpy(ctx->hpack + xh_off, x_hi_host, (size_t)B * ctx->n0 * 4);
    std::memcpy(ctx->hpack + C_off, C_host, (size_t)B * S * nL * 4);
    CK(ctx, cudaMemcpyAsync(io, ctx->hpack, in_bytes, cudaMemcpyHostToDevice, s));
  } else {
    CK(ctx, cudaMemcpyAsync(xl, x_lo_host, (size_t)B * ctx->n0 * 4, cudaMemcpyHostToDevice, s));
    CK(ctx, cudaMemcpyAsync(xh, x_hi_host, (size_t)B * ctx->n0 * 4, cudaMemcpyHostToDevice, s));
    CK(ctx, cudaMemcpyAsync(C, C_host, (size_t)B * S * nL * 4, cudaMemcpyHostToDevice, s));
  }
  int rc = crown_run(ctx, B, xl, xh, C, S, any_alpha ? al.data() : nullptr, intermediate, l.data(), u.data(), lb, ub, ver);
  if (rc) return rc;
  if (packed) {
    uint8_t* ho = ctx->hpack + in_bytes;          // mirror of [out0, out0 + out_bytes)
    CK(ctx, cudaMemcpyAsync(ho, io + out0, out_bytes, cudaMemcpyDeviceToHost, s));
    CK(ctx, cudaStreamSynchronize(s));
    std::memcpy(lb_host, ho + (lb_off - out0), (size_t)B * S * 4);
    std::memcpy(ub_host, ho + (ub_off - out0), (size_t)B * S * 4);
    if (verified_host) std::memcpy(verified_host, ho + (ver_off - out0), (size_t)B);
    return CROWN_OK;
  }
  CK(ctx, cudaMemcpyAsync(lb_host, lb, (size_t)B * S * 4, cudaMemcpyDeviceToHost, s));
  CK(ctx, cudaMemcpyAsync(ub_host, ub, (size_t)B * S * 4, cudaMemcpyDeviceToHost, s));
  if (verified_host) CK(ctx, cudaMemcpyAsync(verified_host, ver, (size_t)B, cudaMemcpyDeviceToHost, s));
  CK(ctx, cudaStreamSynchronize(s));
  return CROWN_OK;
}

// ================================================================================================
// NEXT-1 -- alpha optimisation of the final bound
// ================================================================================================
namespace {

struct AlphaScratch {
  float* A0 = nullptr;             // [2,B,S,n0]   A w.r.t. the input, as the final pass leaves it
  float* Gin = nullptr;            // [2,B,S,n0]   the corner of the box that attains each bound
  std::vector<float*> Asave;       // per ReLU node [2,B,S,size]: A as it arrived at that ReLU
  std::vector<float*> G;           // per node [2,B,S,size]: d bound / d A_i (Flatten aliases its producer)
  float* lb = nullptr; float* ub = nullptr;   // [B,S] bounds of the current iterate
  float* step = nullptr;           // current step size (device scalar: the iteration is data-independent on the host)
  // forward sweep through Linear layers on the tensor cores: the layer's weight split into TF32 limbs (not transposed:
  // G_i = G_in . W_i^T wants W_i [n_out, n_in] as the K-major B operand) and the split of G_in
  std::vector<float*> Wf_hi, Wf_lo;   // per Linear node (nullptr: CUDA-core kernel)
  std::vector<float*> Wk;             // per Conv2d node: flipped, role-swapped filters for the strip kernel (nullptr: gather kernel)
  float* Gs_hi = nullptr; float* Gs_lo = nullptr;
  int last_relu = -1;
  size_t bytes = 0;
};

void alpha_layout(crown_ctx* ctx, int B, int S, uint8_t* base, AlphaScratch& sc) {
  const int n = (int)ctx->nodes.size();
  size_t off = 0;
  auto take = [&](size_t elems) { float* p = reinterpret_cast<float*>(base + off); off += align_up(elems * 4, 256); return p; };
  const size_t rows = (size_t)2 * B * S;
  sc.A0 = take(rows * ctx->n0);
  sc.Gin = take(rows * ctx->n0);
  sc.Asave.assign(n, nullptr); sc.G.assign(n, nullptr);
  sc.last_relu = -1;
  for (int i = 0; i < n; ++i) if (ctx->nodes[i].n.op == CROWN_RELU) sc.last_relu = i;
  for (int i = 0; i <= sc.last_relu; ++i) {
    const NodeInfo& ni = ctx->nodes[i];
    if (ni.n.op == CROWN_RELU) sc.Asave[i] = take(rows * ni.size);
    if (ni.n.op == CROWN_FLATTEN) sc.G[i] = ni.n.in0 < 0 ? sc.Gin : sc.G[ni.n.in0];
    else sc.G[i] = take(rows * ni.size);
  }
  sc.lb = take((size_t)B * S); sc.ub = take((size_t)B * S);
  sc.step = take(2);                 // {alpha step, beta step}
  sc.Wf_hi.assign(n, nullptr); sc.Wf_lo.assign(n, nullptr);
  size_t kmax = 0;
  if (ctx->opts.mma_scheme == 0)
    for (int i = 0; i <= sc.last_relu; ++i) {
      const NodeInfo& ni = ctx->nodes[i];
      if (ni.n.op != CROWN_LINEAR || !gemm_tc_supported((int)rows, ni.n.n_out, ni.n.n_in)) continue;
      sc.Wf_hi[i] = take((size_t)ni.n.n_out * ni.n.n_in);
      sc.Wf_lo[i] = take((size_t)ni.n.n_out * ni.n.n_in);
      kmax = std::max(kmax, (size_t)ni.n.n_in);
    }
  if (kmax) { sc.Gs_hi = take(rows * kmax); sc.Gs_lo = take(rows * kmax); }
  sc.Wk.assign(n, nullptr);
  for (int i = 0; i <= sc.last_relu; ++i) {
    const NodeInfo& ni = ctx->nodes[i];
    const crown_node& nd = ni.n;
    if (nd.op == CROWN_CONV2D && nd.kh == 3 && nd.kw == 3 && nd.stride == 1 && nd.pad == 1 && (rows % 2) == 0 &&
        conv3x3s1_points_supported(nd.c_in, nd.h_in, nd.w_in, nd.c_out))
      sc.Wk[i] = take((size_t)nd.c_out * nd.c_in * 9);
  }
  sc.bytes = off;
}

// TF32 limbs of the weights the forward sweep multiplies on the tensor cores (once per call: one pass over those W)
void alpha_prepare(crown_ctx* ctx, const AlphaScratch& sc) {
  for (size_t i = 0; i < ctx->nodes.size(); ++i) {
    if (!sc.Wf_hi[i]) continue;
    const crown_node& nd = ctx->nodes[i].n;
    Scope scp(ctx, CROWN_K_MISC, 12.0 * nd.n_out * nd.n_in);
    launch_split_tf32(nd.W_dev, nd.n_out, nd.n_in, 0, sc.Wf_hi[i], sc.Wf_lo[i], ctx->stream);
  }
  for (size_t i = 0; i < ctx->nodes.size(); ++i) {
    if (!sc.Wk[i]) continue;
    const crown_node& nd = ctx->nodes[i].n;
    Scope scp(ctx, CROWN_K_MISC, 8.0 * nd.c_out * nd.c_in * 9);
    launch_flip_conv_weights(nd.W_dev, sc.Wk[i], nd.c_out, nd.c_in, ctx->stream);
  }
}

int alpha_check(crown_ctx* ctx, int B, int S, const float* C_dev, const float* const* l_dev, const float* const* u_dev,
                const float* const* alpha_lo, const float* const* alpha_up, const float* x_lo, const float* x_hi,
                const void* scratch, size_t scratch_bytes, bool distinct, AlphaScratch& sc) {
  if (B <= 0 || B > ctx->B_max || S <= 0 || S > ctx->S_max || !C_dev || !l_dev || !u_dev || !alpha_lo || !alpha_up ||
      !x_lo || !x_hi || !scratch)
    return fail(ctx, CROWN_EINVAL, "crown_alpha: bad arguments");
  if (reinterpret_cast<uintptr_t>(scratch) & 255) return fail(ctx, CROWN_EINVAL, "crown_alpha: scratch must be 256-byte aligned");
  for (size_t i = 0; i < ctx->nodes.size(); ++i) {
    const NodeInfo& ni = ctx->nodes[i];
    if (ni.n.op == CROWN_RELU && (!alpha_lo[i] || !alpha_up[i] || !l_dev[i] || !u_dev[i]))
      return fail(ctx, CROWN_EINVAL, "crown_alpha: every ReLU needs alpha_lo, alpha_up and its pre-activation bounds");
    if (ni.n.op == CROWN_RELU && distinct && alpha_lo[i] == alpha_up[i])
      return fail(ctx, CROWN_EINVAL, "crown_alpha_ascent: alpha_lo and alpha_up must be distinct tensors (they are optimised separately)");
    if (ni.n.op == CROWN_LINEAR && !ni.n.W_dev) return fail(ctx, CROWN_EUNSUPPORTED, "crown_alpha: streamed layers are not supported");
  }
  alpha_layout(ctx, B, S, reinterpret_cast<uint8_t*>(const_cast<void*>(scratch)), sc);
  if (scratch_bytes < sc.bytes) return fail(ctx, CROWN_ENOMEM, "crown_alpha: scratch smaller than crown_alpha_scratch_bytes");
  return CROWN_OK;
}

// final pass at the current alpha (keeping A at every ReLU and at the input), bounds into sc.lb / sc.ub
int alpha_backward(crown_ctx* ctx, int B, int S, const float* C_dev, const float* const* l_dev, const float* const* u_dev,
                   const float* const* alpha_lo, const float* const* alpha_up, const float* x_lo, const float* x_hi,
                   const AlphaScratch& sc, std::vector<char>* coef_ready, const SplitSpec* sp = nullptr) {
  return run_pass(ctx, B, (int)ctx->nodes.size() - 1, 0, S, C_dev, l_dev, u_dev, alpha_lo, alpha_up, sc.A0, nullptr, x_lo, x_hi,
                  sc.lb, sc.ub, S, coef_ready, sc.Asave.data(), sp);
}

// what the forward sweep does with beta (NEXT-2): gradients out, or the projected step in place (with `step`)
struct BetaSweep {
  const int8_t* const* split = nullptr;
  float* const* beta_lo = nullptr; float* const* beta_up = nullptr;
  float* const* gb_lo = nullptr; float* const* gb_up = nullptr;
};

// forward sweep of G; step == nullptr: gradients into g_lo / g_up, else the projected step on alpha in place
int alpha_forward(crown_ctx* ctx, int B, int S, const AlphaScratch& sc, const float* x_lo, const float* x_hi,
                  float* const* alpha_lo, float* const* alpha_up, float* const* g_lo, float* const* g_up,
                  const float* step, int mode, const BetaSweep* bs = nullptr) {
  cudaStream_t s = ctx->stream;
  const long long M = 2LL * B * S;
  // the corner of the box per row; when the input feeds exactly one tensor-core Linear (node 0), its limbs are written
  // straight into that contraction's operand scratch
  const bool corner_limbs = ctx->input_consumers == 1 && sc.last_relu >= 0 && ctx->nodes[0].n.op == CROWN_LINEAR &&
                            ctx->nodes[0].n.in0 < 0 && sc.Wf_hi[0] && sc.Gs_hi &&
                            alpha_corner_limbs_ok(sc.A0, x_lo, x_hi, sc.Gs_hi, sc.Gs_lo, ctx->n0);
  { Scope scp(ctx, CROWN_K_MISC, 4.0 * M * ctx->n0 * (corner_limbs ? 3 : 2));
    launch_alpha_corner(sc.A0, x_lo, x_hi, corner_limbs ? sc.Gs_hi : sc.Gin, B, S, ctx->n0, s, corner_limbs ? sc.Gs_lo : nullptr); }
  // Two passes over G are folded into the ReLU kernel where the graph is a plain chain: the bias of a tensor-core Linear
  // whose only consumer is a ReLU is added when that ReLU reads G (deferred_bias), and a ReLU whose only consumer is a
  // tensor-core Linear writes that contraction's TF32 limbs itself (presplit).
  const int nn = (int)ctx->nodes.size();
  std::vector<const float*> deferred_bias(nn, nullptr);
  std::vector<char> presplit(nn, 0);
  auto sole_consumer = [&](int i) -> int {      // the one node that reads node i, or -1
    if (ctx->nodes[i].n_consumers != 1) return -1;
    for (int k = i + 1; k < nn; ++k)
      if (ctx->nodes[k].n.in0 == i || (ctx->nodes[k].n.op == CROWN_ADD && ctx->nodes[k].n.in1 == i)) return k;
    return -1;
  };
  for (int i = 0; i <= sc.last_relu; ++i) {
    const NodeInfo& ni = ctx->nodes[i];
    const crown_node& nd = ni.n;
    const float* gin = nd.in0 < 0 ? sc.Gin : sc.G[nd.in0];
    switch (nd.op) {
      case CROWN_LINEAR: {
        if (sc.Wf_hi[i]) {
          // tensor cores (3xTF32): split G_in, contract with the limbs of W_i made by alpha_prepare, add the bias
          if (!(nd.in0 >= 0 ? presplit[nd.in0] != 0 : (corner_limbs && i == 0)))
          { Scope scp(ctx, CROWN_K_MISC, 12.0 * M * nd.n_in); launch_split_tf32(gin, (int)M, nd.n_in, 0, sc.Gs_hi, sc.Gs_lo, s); }
          const char* e = nullptr;
          { Scope scp(ctx, CROWN_K_GEMM_TC, 8.0 * M * nd.n_in + 8.0 * nd.n_in * nd.n_out + 4.0 * M * nd.n_out, 2.0 * M * (double)nd.n_in * nd.n_out);
            if (launch_gemm_tc(sc.Gs_hi, sc.Gs_lo, sc.Wf_hi[i], sc.Wf_lo[i], sc.G[i], nd.n_out, (int)M, nd.n_out, nd.n_in,
                               ctx->opts.k_drain, ctx->num_sms, s, &e))
              return fail(ctx, CROWN_ECUDA, std::string("alpha forward gemm_tc: ") + (e ? e : "?"));
            ctx->launches += gemm_tc_num_panels(nd.n_in) - 1; }
          if (nd.b_dev) {
            const int k = sole_consumer(i);
            if (k >= 0 && k <= sc.last_relu && ctx->nodes[k].n.op == CROWN_RELU) deferred_bias[i] = nd.b_dev;
            else { Scope scp(ctx, CROWN_K_MISC, 8.0 * M * nd.n_out); launch_add_bias_rows(sc.G[i], nd.b_dev, M, nd.n_out, s); }
          }
          break;
        }
        Scope scp(ctx, CROWN_K_GEMM_FFMA, 4.0 * ((double)M * nd.n_in + (double)nd.n_in * nd.n_out + (double)M * nd.n_out),
                  2.0 * M * (double)nd.n_in * nd.n_out);
        launch_alpha_linear(gin, nd.W_dev, nd.b_dev, sc.G[i], (int)M, nd.n_out, nd.n_in, s);
        break; }
      case CROWN_CONV2D: {
        Scope scp(ctx, CROWN_K_CONV, 4.0 * M * ((double)ni.size + (double)nd.c_in * nd.h_in * nd.w_in),
                  2.0 * M * (double)ni.size * nd.c_in * nd.kh * nd.kw);
        if (sc.Wk[i] && launch_conv3x3s1_points(gin, sc.Wk[i], sc.G[i], M, nd.c_in, nd.h_in, nd.w_in, nd.c_out, s) == 0) {
          if (nd.b_dev) launch_add_bias_div(sc.G[i], nd.b_dev, M * ni.size, nd.c_out, ni.h * ni.w, s);
          break;
        }
        launch_alpha_conv(nd.W_dev, nd.b_dev, gin, sc.G[i], M, nd.c_in, nd.h_in, nd.w_in, nd.c_out, nd.kh, nd.kw, nd.stride,
                          nd.pad, ni.h, ni.w, s);
        break; }
      case CROWN_ADD: {
        const float* gb = nd.in1 < 0 ? sc.Gin : sc.G[nd.in1];
        Scope scp(ctx, CROWN_K_MISC, 12.0 * M * ni.size);
        launch_alpha_add(gin, gb, sc.G[i], M * ni.size, s);
        break; }
      case CROWN_FLATTEN:
        break;                                  // aliases its producer
      case CROWN_RELU: {
        const bool sp = bs && bs->split && bs->split[i];
        const int k = sole_consumer(i);
        // k == i + 1: nothing between the two may reuse the limb scratch
        const bool limbs = k == i + 1 && k <= sc.last_relu && ctx->nodes[k].n.op == CROWN_LINEAR && ctx->nodes[k].n.in0 == i && sc.Wf_hi[k];
        presplit[i] = limbs ? 1 : 0;
        Scope scp(ctx, CROWN_K_RELAX, 4.0 * ni.size * ((limbs ? 4.0 : 3.0) * M + 2.0 * B * S + (sp ? 2.0 * B * S : 0.0)));
        launch_alpha_relu(sc.Asave[i], gin, coef_ptr(ctx, i), alpha_lo[i], alpha_up[i], limbs ? sc.Gs_hi : sc.G[i],
                          g_lo ? g_lo[i] : nullptr, g_up ? g_up[i] : nullptr, step, mode, B, S, ni.size, s,
                          sp ? bs->split[i] : nullptr, sp && bs->beta_lo ? bs->beta_lo[i] : nullptr,
                          sp && bs->beta_up ? bs->beta_up[i] : nullptr, sp && bs->gb_lo ? bs->gb_lo[i] : nullptr,
                          sp && bs->gb_up ? bs->gb_up[i] : nullptr, nd.in0 >= 0 ? deferred_bias[nd.in0] : nullptr,
                          limbs ? sc.Gs_lo : nullptr);
        break; }
      default:
        return fail(ctx, CROWN_EUNSUPPORTED, "crown_alpha: unsupported op");
    }
  }
  CK(ctx, cudaGetLastError());
  return CROWN_OK;
}

}  // namespace

extern "C" int crown_alpha_scratch_bytes(crown_ctx* ctx, int B, int S, size_t* out) {
  if (!ctx || !out || B <= 0 || S <= 0) return CROWN_EINVAL;
  AlphaScratch sc;
  alpha_layout(ctx, B, S, nullptr, sc);
  *out = sc.bytes;
  return CROWN_OK;
}

static int beta_grad_impl(crown_ctx* ctx, int B, const float* C_dev, int S, const float* const* l_dev,
                          const float* const* u_dev, const int8_t* const* split_dev, const float* const* alpha_lo_dev,
                          const float* const* alpha_up_dev, const float* const* beta_lo_dev, const float* const* beta_up_dev,
                          const float* x_lo_dev, const float* x_hi_dev, float* const* g_lo_dev, float* const* g_up_dev,
                          float* const* gb_lo_dev, float* const* gb_up_dev, float* lb_dev, float* ub_dev,
                          void* scratch_dev, size_t scratch_bytes) {
  AlphaScratch sc;
  int rc = alpha_check(ctx, B, S, C_dev, l_dev, u_dev, alpha_lo_dev, alpha_up_dev, x_lo_dev, x_hi_dev, scratch_dev,
                       scratch_bytes, false, sc);
  if (rc) return rc;
  CK(ctx, cudaMemsetAsync(scratch_dev, 0, sc.bytes, ctx->stream));
  alpha_prepare(ctx, sc);
  SplitSpec sp; sp.split = split_dev; sp.beta_lo = beta_lo_dev; sp.beta_up = beta_up_dev;
  rc = alpha_backward(ctx, B, S, C_dev, l_dev, u_dev, alpha_lo_dev, alpha_up_dev, x_lo_dev, x_hi_dev, sc, nullptr,
                      split_dev ? &sp : nullptr);
  if (rc) return rc;
  if (lb_dev) CK(ctx, cudaMemcpyAsync(lb_dev, sc.lb, (size_t)B * S * 4, cudaMemcpyDeviceToDevice, ctx->stream));
  if (ub_dev) CK(ctx, cudaMemcpyAsync(ub_dev, sc.ub, (size_t)B * S * 4, cudaMemcpyDeviceToDevice, ctx->stream));
  BetaSweep bs; bs.split = split_dev; bs.gb_lo = gb_lo_dev; bs.gb_up = gb_up_dev;
  return alpha_forward(ctx, B, S, sc, x_lo_dev, x_hi_dev, const_cast<float* const*>(reinterpret_cast<const float* const*>(alpha_lo_dev)),
                       const_cast<float* const*>(reinterpret_cast<const float* const*>(alpha_up_dev)), g_lo_dev, g_up_dev, nullptr, 0,
                       split_dev ? &bs : nullptr);
}

static int beta_ascent_impl(crown_ctx* ctx, int B, const float* C_dev, int S, const float* const* l_dev,
                            const float* const* u_dev, const int8_t* const* split_dev, float* const* alpha_lo_dev,
                            float* const* alpha_up_dev, float* const* beta_lo_dev, float* const* beta_up_dev,
                            const float* x_lo_dev, const float* x_hi_dev, float eta_alpha, float eta_beta, float decay,
                            int iters, int mode, float* lb_best_dev, float* ub_best_dev, float* lb_last_dev,
                            float* ub_last_dev, uint8_t* verified_dev, void* scratch_dev, size_t scratch_bytes,
                            const char* who) {
  if (iters < 0 || (mode != 0 && mode != 1) || !(eta_alpha >= 0.f) || !(eta_beta >= 0.f) || !(decay > 0.f) || !lb_best_dev || !ub_best_dev)
    return fail(ctx, CROWN_EINVAL, std::string(who) + ": bad arguments");
  AlphaScratch sc;
  const float* const* al = reinterpret_cast<const float* const*>(alpha_lo_dev);
  const float* const* au = reinterpret_cast<const float* const*>(alpha_up_dev);
  int rc = alpha_check(ctx, B, S, C_dev, l_dev, u_dev, al, au, x_lo_dev, x_hi_dev, scratch_dev, scratch_bytes, true, sc);
  if (rc) return rc;
  if (split_dev)
    for (size_t i = 0; i < ctx->nodes.size(); ++i)
      if (split_dev[i] && (!beta_lo_dev || !beta_up_dev || !beta_lo_dev[i] || !beta_up_dev[i] || beta_lo_dev[i] == beta_up_dev[i]))
        return fail(ctx, CROWN_EINVAL, std::string(who) + ": every split ReLU needs distinct beta_lo and beta_up tensors");
  cudaStream_t s = ctx->stream;
  CK(ctx, cudaMemsetAsync(scratch_dev, 0, sc.bytes, s));
  alpha_prepare(ctx, sc);
  { Scope scp(ctx, CROWN_K_MISC); launch_alpha_set_step(sc.step, eta_alpha, s, eta_beta); }
  SplitSpec sp; sp.split = split_dev;
  sp.beta_lo = reinterpret_cast<const float* const*>(beta_lo_dev); sp.beta_up = reinterpret_cast<const float* const*>(beta_up_dev);
  BetaSweep bs; bs.split = split_dev; bs.beta_lo = beta_lo_dev; bs.beta_up = beta_up_dev;
  std::vector<char> coef_ready(ctx->nodes.size(), 0);      // the intermediate bounds and the split are fixed: coefficients once
  for (int t = 0; t <= iters; ++t) {
    rc = alpha_backward(ctx, B, S, C_dev, l_dev, u_dev, al, au, x_lo_dev, x_hi_dev, sc, &coef_ready, split_dev ? &sp : nullptr);
    if (rc) return rc;
    { Scope scp(ctx, CROWN_K_MISC); launch_alpha_best(sc.lb, sc.ub, lb_best_dev, ub_best_dev, sc.step, decay, t == 0, B * S, s); }
    if (t == iters) break;
    rc = alpha_forward(ctx, B, S, sc, x_lo_dev, x_hi_dev, alpha_lo_dev, alpha_up_dev, nullptr, nullptr, sc.step, mode,
                       split_dev ? &bs : nullptr);
    if (rc) return rc;
  }
  if (lb_last_dev) CK(ctx, cudaMemcpyAsync(lb_last_dev, sc.lb, (size_t)B * S * 4, cudaMemcpyDeviceToDevice, s));
  if (ub_last_dev) CK(ctx, cudaMemcpyAsync(ub_last_dev, sc.ub, (size_t)B * S * 4, cudaMemcpyDeviceToDevice, s));
  if (verified_dev) { Scope scp(ctx, CROWN_K_MISC); launch_verdict(lb_best_dev, verified_dev, B, S, s); }
  CK(ctx, cudaGetLastError());
  return CROWN_OK;
}

extern "C" int crown_alpha_grad(crown_ctx* ctx, int B, const float* C_dev, int S, const float* const* l_dev,
                                const float* const* u_dev, const float* const* alpha_lo_dev,
                                const float* const* alpha_up_dev, const float* x_lo_dev, const float* x_hi_dev,
                                float* const* g_lo_dev, float* const* g_up_dev, float* lb_dev, float* ub_dev,
                                void* scratch_dev, size_t scratch_bytes) {
  if (!ctx) return CROWN_EINVAL;
  return beta_grad_impl(ctx, B, C_dev, S, l_dev, u_dev, nullptr, alpha_lo_dev, alpha_up_dev, nullptr, nullptr, x_lo_dev,
                        x_hi_dev, g_lo_dev, g_up_dev, nullptr, nullptr, lb_dev, ub_dev, scratch_dev, scratch_bytes);
}

extern "C" int crown_alpha_ascent(crown_ctx* ctx, int B, const float* C_dev, int S, const float* const* l_dev,
                                  const float* const* u_dev, float* const* alpha_lo_dev, float* const* alpha_up_dev,
                                  const float* x_lo_dev, const float* x_hi_dev, float eta, float decay, int iters,
                                  int mode, float* lb_best_dev, float* ub_best_dev, float* lb_last_dev,
                                  float* ub_last_dev, uint8_t* verified_dev, void* scratch_dev, size_t scratch_bytes) {
  if (!ctx) return CROWN_EINVAL;
  return beta_ascent_impl(ctx, B, C_dev, S, l_dev, u_dev, nullptr, alpha_lo_dev, alpha_up_dev, nullptr, nullptr, x_lo_dev,
                          x_hi_dev, eta, 0.f, decay, iters, mode, lb_best_dev, ub_best_dev, lb_last_dev, ub_last_dev,
                          verified_dev, scratch_dev, scratch_bytes, "crown_alpha_ascent");
}

// ================================================================================================
// NEXT-2 -- beta-CROWN bounds of batched BaB sub-domains
// ================================================================================================
extern "C" int crown_backward_split(crown_ctx* ctx, int B, int start, int row0, int rows, const float* C_dev,
                                    const float* const* l_dev, const float* const* u_dev,
                                    const int8_t* const* split_dev, const float* const* alpha_lo_dev,
                                    const float* const* alpha_up_dev, const float* const* beta_lo_dev,
                                    const float* const* beta_up_dev, float* A_dev, float* d_dev,
                                    const float* x_lo_dev, const float* x_hi_dev, float* lb_dev, float* ub_dev) {
  if (!ctx) return CROWN_EINVAL;
  if (!A_dev && !d_dev && !lb_dev) return fail(ctx, CROWN_EINVAL, "crown_backward_split: no output requested");
  SplitSpec sp; sp.split = split_dev; sp.beta_lo = beta_lo_dev; sp.beta_up = beta_up_dev;
  return run_pass(ctx, B, start, row0, rows, C_dev, l_dev, u_dev, alpha_lo_dev, alpha_up_dev, A_dev, d_dev,
                  x_lo_dev, x_hi_dev, lb_dev, ub_dev, rows, nullptr, nullptr, split_dev ? &sp : nullptr);
}

extern "C" int crown_beta_grad(crown_ctx* ctx, int B, const float* C_dev, int S, const float* const* l_dev,
                               const float* const* u_dev, const int8_t* const* split_dev,
                               const float* const* alpha_lo_dev, const float* const* alpha_up_dev,
                               const float* const* beta_lo_dev, const float* const* beta_up_dev,
                               const float* x_lo_dev, const float* x_hi_dev, float* const* g_lo_dev,
                               float* const* g_up_dev, float* const* gb_lo_dev, float* const* gb_up_dev,
                               float* lb_dev, float* ub_dev, void* scratch_dev, size_t scratch_bytes) {
  if (!ctx) return CROWN_EINVAL;
  return beta_grad_impl(ctx, B, C_dev, S, l_dev, u_dev, split_dev, alpha_lo_dev, alpha_up_dev, beta_lo_dev, beta_up_dev,
                        x_lo_dev, x_hi_dev, g_lo_dev, g_up_dev, gb_lo_dev, gb_up_dev, lb_dev, ub_dev, scratch_dev, scratch_bytes);
}

extern "C" int crown_beta_ascent(crown_ctx* ctx, int B, const float* C_dev, int S, const float* const* l_dev,
                                 const float* const* u_dev, const int8_t* const* split_dev,
                                 float* const* alpha_lo_dev, float* const* alpha_up_dev, float* const* beta_lo_dev,
                                 float* const* beta_up_dev, const float* x_lo_dev, const float* x_hi_dev,
                                 float eta_alpha, float eta_beta, float decay, int iters, int mode,
                                 float* lb_best_dev, float* ub_best_dev, float* lb_last_dev, float* ub_last_dev,
                                 uint8_t* verified_dev, void* scratch_dev, size_t scratch_bytes) {
  if (!ctx) return CROWN_EINVAL;
  return beta_ascent_impl(ctx, B, C_dev, S, l_dev, u_dev, split_dev, alpha_lo_dev, alpha_up_dev, beta_lo_dev, beta_up_dev,
                          x_lo_dev, x_hi_dev, eta_alpha, eta_beta, decay, iters, mode, lb_best_dev, ub_best_dev,
                          lb_last_dev, ub_last_dev, verified_dev, scratch_dev, scratch_bytes, "crown_beta_ascent");
}

// ================================================================================================
// kernel 1 exposed on its own (parity tests, roofline measurement)
// ================================================================================================
extern "C" int crown_split_tf32(crown_ctx* ctx, const float* X_dev, int rows, int cols, int transpose,
                                float* hi_dev, float* lo_dev) {
  if (!ctx) return CROWN_EINVAL;
  if (!X_dev || !hi_dev || !lo_dev || rows <= 0 || cols <= 0) return fail(ctx, CROWN_EINVAL, "crown_split_tf32: bad arguments");
  { Scope sc(ctx, CROWN_K_MISC); launch_split_tf32(X_dev, rows, cols, transpose, hi_dev, lo_dev, ctx->stream); }
  CK(ctx, cudaGetLastError());
  return CROWN_OK;
}

extern "C" int crown_gemm(crown_ctx* ctx, int scheme, int M, int N, int K, const float* A_hi_dev,
                          const float* A_lo_dev, const float* Wt_hi_dev, const float* Wt_lo_dev, float* D_dev) {
  if (!ctx) return CROWN_EINVAL;
  if (M <= 0 || N <= 0 || K <= 0 || !A_hi_dev || !Wt_hi_dev || !D_dev) return fail(ctx, CROWN_EINVAL, "crown_gemm: bad arguments");
  if (scheme == 0) {
    if (!A_lo_dev || !Wt_lo_dev) return fail(ctx, CROWN_EINVAL, "crown_gemm: 3xTF32 needs the lo parts");
    const char* e = nullptr;
    Scope sc(ctx, CROWN_K_GEMM_TC, 4.0 * ((double)M * K + (double)K * N + (double)M * N), 2.0 * M * (double)N * K);
    if (launch_gemm_tc(A_hi_dev, A_lo_dev, Wt_hi_dev, Wt_lo_dev, D_dev, N, M, N, K, ctx->opts.k_drain, ctx->num_sms, ctx->stream, &e))
      return fail(ctx, CROWN_EINVAL, std::string("crown_gemm: ") + (e ? e : "?"));
    ctx->launches += gemm_tc_num_panels(K) - 1;
  } else if (scheme == 2) {
    // FFMA path takes W [K,N] row-major in Wt_hi_dev (NOT transposed) and fp32 A in A_hi_dev
    Scope sc(ctx, CROWN_K_GEMM_FFMA, 4.0 * ((double)M * K + (double)K * N + (double)M * N), 2.0 * M * (double)N * K);
    launch_gemm_ffma(A_hi_dev, K, Wt_hi_dev, N, D_dev, N, M, N, K, ctx->stream);
  } else {
    return fail(ctx, CROWN_EINVAL, "crown_gemm: unknown scheme");
  }
  CK(ctx, cudaGetLastError());
  return CROWN_OK;
}
