"""float64 CPU oracle for IBP / CROWN / alpha-CROWN bound propagation.

TEST INFRASTRUCTURE ONLY.  Only `tests/`, `__graft_entry__.smoke()` and
`bench.py`'s `cpu_baseline` / `--impl reference` legs may import this module.
It shares no code with the CUDA path (`paper_2606_09377_b200/`): the only
common module is the seeded input generator `workloads.py`, which holds none
of the method's arithmetic.  NumPy only, float64 throughout, operating on the
same float32-rounded inputs upcast to float64, one property at a time, no
blocking / fusion / reordering beyond what the cited passages state.

What it follows (citations are /root/reference/PAPER.md line + section):
  O1  ibp()              PAPER.md:58-62 (§2.1), literally the W+/W- form
  O2  relax_coeffs()     PAPER.md:64    (§2.1) ReLU linear relaxation
  O3  backward()         PAPER.md:64-68 (§2.1, Eq. 1), :128 (§3.3.2) A <- A.Lambda_i W_i
      concretize()       PAPER.md:27 (eps-ball), :66 (Eq. 1)   [reading G1: Hoelder dual]
  O4  crown_bounds()     PAPER.md:130 (§3.3.2) intermediate bounds choose the slopes
  O5  final_bounds()     PAPER.md:70 (§2.1) alpha-CROWN with given alpha; :25, :74 verdict
  O6  sample_check()     PAPER.md:74 (§2.1.1) definition of soundness
  (O7 brute force lives in oracle/brute_force.py)

Readings of points where the paper is silent (listed in
DESIGN.md): stable neurons are classified active (l >= 0) -> inactive (u <= 0)
-> unstable in that order (G3); the fixed lower slope is the adaptive rule of
the CROWN paper the text cites: lambda = 1 iff u > -l (strict), else 0 (G4);
lower-relaxation intercept is 0; no intersection of CROWN and IBP bounds (G9);
the box is not clipped (G11).

Pins (tests/test_oracle_*.py, `-m "not gpu"`): the paper's worked example
(PAPER.md:134), closed forms (single linear layer; all-active / all-inactive
nets), hand-worked relaxations E2/E3 (tests/golden/), W+/W- == centre/radius,
conv == dense Toeplitz matrix, conv-transpose adjoint identity, containment of
10^4 samples incl. adversarial corners, lb <= exact min <= sampled min from
brute-force activation-pattern enumeration + LP, eps-monotonicity, sign
symmetry, row independence.  Absolute bound VALUES on cfg1-cfg5 have no
published reference: for those "parity unpinned" beyond the pins above.
"""
from __future__ import annotations

from typing import Dict, List, Optional, Sequence, Tuple

import numpy as np

LINEAR, CONV, RELU, ADD, FLATTEN = "linear", "conv", "relu", "add", "flatten"

F64 = np.float64


# ------------------------------------------------------------------------------------------
# linear operators of the network, written out from their definitions
# ------------------------------------------------------------------------------------------
def conv2d(x: np.ndarray, W: np.ndarray, stride: int, pad: int) -> np.ndarray:
    """Cross-correlation y[o,p,q] = sum_{c,i,j} W[o,c,i,j] * x[c, p*s+i-pad, q*s+j-pad]; no bias.
    x: [..., C_in, H, W] -> [..., C_out, H', W'].  Zero padding."""
    W = W.astype(F64)
    c_out, c_in, kh, kw = W.shape
    lead = x.shape[:-3]
    xp = np.zeros(lead + (c_in, x.shape[-2] + 2 * pad, x.shape[-1] + 2 * pad), dtype=F64)
    xp[..., pad:pad + x.shape[-2], pad:pad + x.shape[-1]] = x
    ho = (xp.shape[-2] - kh) // stride + 1
    wo = (xp.shape[-1] - kw) // stride + 1
    y = np.zeros(lead + (c_out, ho, wo), dtype=F64)
    for i in range(kh):
        for j in range(kw):
            patch = xp[..., :, i:i + stride * ho:stride, j:j + stride * wo:stride]
            y += np.einsum("oc,...chw->...ohw", W[:, :, i, j], patch)
    return y


def conv2d_transpose(A: np.ndarray, W: np.ndarray, stride: int, pad: int,
                     in_hw: Tuple[int, int]) -> np.ndarray:
    """Adjoint of conv2d w.r.t. x: A_x[c, p*s+i-pad, q*s+j-pad] += W[o,c,i,j] * A[o,p,q].
    A: [..., C_out, H', W'] -> [..., C_in, H, W] with (H, W) = in_hw (PAPER.md:144, :289:
    a conv layer is linear, so the backward recursion uses its transpose)."""
    W = W.astype(F64)
    c_out, c_in, kh, kw = W.shape
    lead = A.shape[:-3]
    ho, wo = A.shape[-2], A.shape[-1]
    H, Wd = in_hw
    xp = np.zeros(lead + (c_in, H + 2 * pad, Wd + 2 * pad), dtype=F64)
    for i in range(kh):
        for j in range(kw):
            xp[..., :, i:i + stride * ho:stride, j:j + stride * wo:stride] += \
                np.einsum("oc,...ohw->...chw", W[:, :, i, j], A)
    return xp[..., pad:pad + H, pad:pad + Wd]


def _in_shape(net, idx):
    return net.in_shape if idx < 0 else net.nodes[idx].shape


def forward(net, x: np.ndarray) -> List[np.ndarray]:
    """Exact network evaluation in float64 for ONE input; returns every node's output."""
    x = np.asarray(x, dtype=F64).reshape(net.in_shape)
    vals: List[np.ndarray] = []
    for n in net.nodes:
        a = x if n.in0 < 0 else vals[n.in0]
        if n.op == LINEAR:
            v = n.W.astype(F64) @ a.reshape(-1) + n.b.astype(F64)
        elif n.op == CONV:
            v = conv2d(a, n.W, n.stride, n.pad) + n.b.astype(F64)[:, None, None]
        elif n.op == RELU:
            v = np.maximum(a, 0.0)
        elif n.op == ADD:
            v = a + (x if n.in1 < 0 else vals[n.in1])
        elif n.op == FLATTEN:
            v = a.reshape(-1)
        else:
            raise ValueError(n.op)
        vals.append(v)
    return vals


def forward_batch(net, X: np.ndarray) -> np.ndarray:
    """f(x) for many inputs X [n, n0] (float64), vectorised over the leading axis."""
    X = np.asarray(X, dtype=F64).reshape((X.shape[0],) + tuple(net.in_shape))
    vals: List[np.ndarray] = []
    for n in net.nodes:
        a = X if n.in0 < 0 else vals[n.in0]
        if n.op == LINEAR:
            v = a.reshape(a.shape[0], -1) @ n.W.astype(F64).T + n.b.astype(F64)
        elif n.op == CONV:
            v = conv2d(a, n.W, n.stride, n.pad) + n.b.astype(F64)[:, None, None]
        elif n.op == RELU:
            v = np.maximum(a, 0.0)
        elif n.op == ADD:
            v = a + (X if n.in1 < 0 else vals[n.in1])
        elif n.op == FLATTEN:
            v = a.reshape(a.shape[0], -1)
        else:
            raise ValueError(n.op)
        vals.append(v)
    return vals[-1]


# ------------------------------------------------------------------------------------------
# O1 -- IBP
# ------------------------------------------------------------------------------------------
def ibp(net, x_lo: np.ndarray, x_hi: np.ndarray) -> List[Tuple[np.ndarray, np.ndarray]]:
    """Interval bounds (l, u) of every node's output for ONE property with box [x_lo, x_hi].

    Linear / conv:  l_y = W+ l_x + W- u_x + b,  u_y = W+ u_x + W- l_x + b
    with W+ = max(W,0), W- = min(W,0) elementwise.
    ReLU: l' = max(l,0), u' = max(u,0).  Add: intervals add.  Flatten: row-major reshape.
    """
    lo = np.asarray(x_lo, dtype=F64).reshape(net.in_shape)
    hi = np.asarray(x_hi, dtype=F64).reshape(net.in_shape)
    out: List[Tuple[np.ndarray, np.ndarray]] = []
    for n in net.nodes:
        l, u = (lo, hi) if n.in0 < 0 else out[n.in0]
        if n.op == LINEAR:
            W = n.W.astype(F64)
            Wp, Wm = np.maximum(W, 0.0), np.minimum(W, 0.0)
            b = n.b.astype(F64)
            l, u = l.reshape(-1), u.reshape(-1)
            r = (Wp @ l + Wm @ u + b, Wp @ u + Wm @ l + b)
        elif n.op == CONV:
            W = n.W.astype(F64)
            Wp, Wm = np.maximum(W, 0.0), np.minimum(W, 0.0)
            b = n.b.astype(F64)[:, None, None]
            r = (conv2d(l, Wp, n.stride, n.pad) + conv2d(u, Wm, n.stride, n.pad) + b,
                 conv2d(u, Wp, n.stride, n.pad) + conv2d(l, Wm, n.stride, n.pad) + b)
        elif n.op == RELU:
            r = (np.maximum(l, 0.0), np.maximum(u, 0.0))
        elif n.op == ADD:
            l2, u2 = (lo, hi) if n.in1 < 0 else out[n.in1]
            r = (l + l2, u + u2)
        elif n.op == FLATTEN:
            r = (l.reshape(-1), u.reshape(-1))
        else:
            raise ValueError(n.op)
        out.append(r)
    return out


def ibp_spec(net, x_lo, x_hi, C: np.ndarray) -> Tuple[np.ndarray, np.ndarray]:
    """IBP bound of C.f(x): the last linear layer and C are ONE linear layer with weight C.W_L and
    bias C.b_L (reading G10; PAPER.md:134 shows that un-fused stacking loses tightness)."""
    last = net.nodes[-1]
    assert last.op == LINEAR
    bounds = ibp(net, x_lo, x_hi)
    l, u = (np.asarray(x_lo, F64), np.asarray(x_hi, F64)) if last.in0 < 0 else bounds[last.in0]
    l, u = l.reshape(-1), u.reshape(-1)
    CW = C.astype(F64) @ last.W.astype(F64)
    Cb = C.astype(F64) @ last.b.astype(F64)
    Wp, Wm = np.maximum(CW, 0.0), np.minimum(CW, 0.0)
    return Wp @ l + Wm @ u + Cb, Wp @ u + Wm @ l + Cb


# ------------------------------------------------------------------------------------------
# O2 -- ReLU relaxation coefficients
# ------------------------------------------------------------------------------------------
def relax_coeffs(l: np.ndarray, u: np.ndarray, alpha: Optional[np.ndarray] = None,
                 rule: str = "adaptive"):
    """Per-neuron (dU, bU, dL) for pre-activation bounds [l, u] (flat arrays [n]).

    Unstable l < 0 < u:  lambda_l x <= ReLU(x) <= u/(u-l) (x - l)
        dU = u/(u-l),  bU = -l u/(u-l),  dL = alpha clipped to [0,1] (alpha-mode)
        or the fixed rule: 'adaptive' lambda=1 iff u > -l (G4), 'zero', 'one'.
    Active  l >= 0: dU = dL = 1, bU = 0.   Inactive u <= 0: dU = dL = 0, bU = 0   (G3, this order).
    alpha may be [n] or [R, n]; dL takes alpha's shape.  Lower intercept is always 0.
    """
    l = np.asarray(l, F64).reshape(-1)
    u = np.asarray(u, F64).reshape(-1)
    active = l >= 0.0
    inactive = (~active) & (u <= 0.0)
    unstable = ~(active | inactive)
    den = np.where(unstable, u - l, 1.0)
    dU = np.where(unstable, u / den, np.where(active, 1.0, 0.0))
    bU = np.where(unstable, -l * u / den, 0.0)
    if alpha is not None:
        slope = np.clip(np.asarray(alpha, F64), 0.0, 1.0)
    elif rule == "adaptive":
        slope = (u > -l).astype(F64)
    elif rule == "zero":
        slope = np.zeros_like(l)
    elif rule == "one":
        slope = np.ones_like(l)
    else:
        raise ValueError(rule)
    dL = np.where(unstable, slope, np.where(active, 1.0, 0.0))
    return dU, bU, dL


# ------------------------------------------------------------------------------------------
# O3 -- CROWN backward pass (PAPER.md:64-68 Eq. 1, :128)
# ------------------------------------------------------------------------------------------
def backward(net, start: int, C0: np.ndarray,
             pre: Dict[int, Tuple[np.ndarray, np.ndarray]],
             alpha_lo: Optional[Dict[int, np.ndarray]] = None,
             alpha_up: Optional[Dict[int, np.ndarray]] = None,
             rule: str = "adaptive", trace: Optional[Dict[int, Tuple[np.ndarray, np.ndarray]]] = None):
    """Linear bounds  A_lo x + d_lo <= C0 . v_start(x) <= A_up x + d_up  for ONE property.

    start : node whose OUTPUT the start matrix C0 [R, n_start] multiplies.
    pre   : {relu node id: (l, u) of that ReLU's INPUT} for every ReLU below `start`.
    alpha_lo / alpha_up : {relu node id: [R, n_k]} lower-relaxation slopes used by the lower /
            upper branch ("different slope choices are used for the lower- and upper-bound
            branches"); None => fixed `rule`.
    Nodes are visited in reverse topological order; a node's A is the SUM of the contributions
    of all its consumers (residual fork).  Per branch, with A the coefficients w.r.t. the node's
    output y and d the accumulated bias (b^(L), b^(U) of Eq. 1, reading G2):
      Linear y = W x + b : d += A b ;  A_x += A W
      Conv               : d += sum_o b_o sum_pq A[o,p,q] ;  A_x += conv^T(A, W)
      Add  y = a + b     : A_a += A ;  A_b += A
      Flatten            : A_x += A (row-major reshape)
      ReLU y = ReLU(x)   : lower: A_x = A+ * dL + A- * dU ; d += A- . bU
                           upper: A_x = A+ * dU + A- * dL ; d += A+ . bU
    trace : if a dict is given, it receives {relu node id: (A_lo, A_up)}: the coefficients w.r.t. each
            ReLU's OUTPUT as they arrive at that ReLU (what oracle/alpha_oracle.py differentiates through).
    Returns (A_lo [R,n0], A_up [R,n0], d_lo [R], d_up [R]).
    """
    C0 = np.asarray(C0, F64)
    R = C0.shape[0]
    n0 = int(np.prod(net.in_shape))
    pend: Dict[int, List[np.ndarray]] = {start: [C0.reshape(R, -1).copy(), C0.reshape(R, -1).copy()]}
    d = [np.zeros(R), np.zeros(R)]

    def contribute(idx: int, parts: Sequence[np.ndarray]):
        parts = [p.reshape(R, -1) for p in parts]
        if idx in pend:
            pend[idx][0] = pend[idx][0] + parts[0]
            pend[idx][1] = pend[idx][1] + parts[1]
        else:
            pend[idx] = [parts[0].copy(), parts[1].copy()]

    for i in range(start, -1, -1):
        if i not in pend:
            continue
        A = pend.pop(i)
        n = net.nodes[i]
        if n.op == LINEAR:
            W = n.W.astype(F64)
            b = n.b.astype(F64)
            for br in (0, 1):
                d[br] = d[br] + A[br] @ b
            contribute(n.in0, [A[0] @ W, A[1] @ W])
        elif n.op == CONV:
            b = n.b.astype(F64)
            c_out, ho, wo = n.shape
            in_shape = _in_shape(net, n.in0)
            outs = []
            for br in (0, 1):
                Ab = A[br].reshape(R, c_out, ho, wo)
                d[br] = d[br] + np.einsum("rohw,o->r", Ab, b)
                outs.append(conv2d_transpose(Ab, n.W, n.stride, n.pad, (in_shape[1], in_shape[2])))
            contribute(n.in0, outs)
        elif n.op == ADD:
            contribute(n.in0, A)
            contribute(n.in1, A)
        elif n.op == FLATTEN:
            contribute(n.in0, A)
        elif n.op == RELU:
            l, u = pre[i]
            if trace is not None:
                trace[i] = (A[0].copy(), A[1].copy())
            a_lo = None if alpha_lo is None or alpha_lo.get(i) is None else alpha_lo[i]
            a_up = None if alpha_up is None or alpha_up.get(i) is None else alpha_up[i]
            dU, bU, dL_lo = relax_coeffs(l, u, a_lo, rule)
            _, _, dL_up = relax_coeffs(l, u, a_up, rule)
            Ap, Am = np.maximum(A[0], 0.0), np.minimum(A[0], 0.0)
            new_lo = Ap * dL_lo + Am * dU
            d[0] = d[0] + Am @ bU
            Ap, Am = np.maximum(A[1], 0.0), np.minimum(A[1], 0.0)
            new_up = Ap * dU + Am * dL_up
            d[1] = d[1] + Ap @ bU
            contribute(n.in0, [new_lo, new_up])
        else:
            raise ValueError(n.op)
    if -1 in pend:
        A_lo, A_up = pend[-1]
    else:
        A_lo, A_up = np.zeros((R, n0)), np.zeros((R, n0))
    return A_lo, A_up, d[0], d[1]


def concretize(A_lo, A_up, d_lo, d_up, x_lo, x_hi):
    """Numbers from Eq. 1 over the box [x_lo, x_hi] (reading G1 -- Hoelder dual of
    the L_inf ball):  min_{x in box} a.x = a.x_c - |a|.x_r,  max = a.x_c + |a|.x_r,
    x_c = (x_lo+x_hi)/2, x_r = (x_hi-x_lo)/2;  for x0 +- eps this is a.x0 -+ eps ||a||_1."""
    x_lo = np.asarray(x_lo, F64).reshape(-1)
    x_hi = np.asarray(x_hi, F64).reshape(-1)
    xc = 0.5 * (x_lo + x_hi)
    xr = 0.5 * (x_hi - x_lo)
    lb = A_lo @ xc - np.abs(A_lo) @ xr + d_lo
    ub = A_up @ xc + np.abs(A_up) @ xr + d_up
    return lb, ub


# ------------------------------------------------------------------------------------------
# O4 -- intermediate (pre-activation) bounds for every ReLU
# ------------------------------------------------------------------------------------------
def _reaches_only_input_linearly(net, idx: int) -> bool:
    """True if node idx is a Linear/Conv fed directly by the network input (first layer):
    its CROWN bound coincides with IBP (single linear layer is exact) and O1 is used."""
    n = net.nodes[idx]
    return n.op in (LINEAR, CONV) and n.in0 < 0


def crown_bounds(net, x_lo, x_hi, intermediate: str = "crown", rule: str = "adaptive",
                 forced: Optional[Dict[int, Tuple[np.ndarray, np.ndarray]]] = None,
                 rows: Optional[Dict[int, np.ndarray]] = None
                 ) -> Dict[int, Tuple[np.ndarray, np.ndarray]]:
    """Pre-activation bounds {relu id: (l, u)} for ONE property.

    intermediate='ibp'  : O1 for every ReLU input (cfg5, reading G22).
    intermediate='crown': for each ReLU in topological order, O3 started at its input node with
        C0 = I and fixed-rule slopes, using the bounds already computed for earlier ReLUs; for a
        first-layer node O1 is used (same value in exact arithmetic).
    forced : if given, {relu id: (l, u)} to use for EARLIER ReLUs instead of the oracle's own
        (forced-bounds layer-wise parity).
    rows   : if given, {relu id: index array}: only these rows of I are propagated for that ReLU
        (row-sampled parity; rows are independent linear bounds); entries not
        computed are NaN.
    """
    ib = ibp(net, x_lo, x_hi)
    lo = np.asarray(x_lo, F64).reshape(-1)
    hi = np.asarray(x_hi, F64).reshape(-1)
    pre: Dict[int, Tuple[np.ndarray, np.ndarray]] = {}
    for i in net.relu_ids():
        src = net.nodes[i].in0
        n_src = net.nodes[src].size
        if intermediate == "ibp" or _reaches_only_input_linearly(net, src):
            l, u = ib[src]
            pre[i] = (l.reshape(-1).copy(), u.reshape(-1).copy())
            continue
        use = pre if forced is None else {k: forced[k] for k in forced if k < i}
        if rows is not None and rows.get(i) is not None:
            idx = np.asarray(rows[i])
            C0 = np.zeros((idx.size, n_src))
            C0[np.arange(idx.size), idx] = 1.0
            A_lo, A_up, d_lo, d_up = backward(net, src, C0, use, rule=rule)
            lb, ub = concretize(A_lo, A_up, d_lo, d_up, lo, hi)
            l = np.full(n_src, np.nan)
            u = np.full(n_src, np.nan)
            l[idx], u[idx] = lb, ub
        else:
            A_lo, A_up, d_lo, d_up = backward(net, src, np.eye(n_src), use, rule=rule)
            l, u = concretize(A_lo, A_up, d_lo, d_up, lo, hi)
        pre[i] = (l, u)
    return pre


# ------------------------------------------------------------------------------------------
# O5 -- final bound and verdict
# ------------------------------------------------------------------------------------------
def final_bounds(net, x_lo, x_hi, C: np.ndarray, pre, alpha_lo=None, alpha_up=None,
                 rule: str = "adaptive"):
    """lb, ub [S] of C.f(x) over the box: O3 from the output node with C0 = C; alpha-mode where alpha
    is supplied ({relu id: [S, n_k]}), else the fixed rule.  Also returns (A_lo, A_up, d_lo, d_up)."""
    A_lo, A_up, d_lo, d_up = backward(net, len(net.nodes) - 1, C, pre, alpha_lo, alpha_up, rule)
    lb, ub = concretize(A_lo, A_up, d_lo, d_up, x_lo, x_hi)
    return lb, ub, (A_lo, A_up, d_lo, d_up)


def verified(lb: np.ndarray) -> bool:
    """A property is verified iff every margin row has a positive lower bound."""
    return bool(np.min(lb) > 0.0)


def run_property(net, x_lo, x_hi, C, alpha: Optional[Sequence[np.ndarray]] = None,
                 intermediate: str = "crown", rule: str = "adaptive"):
    """Whole hot path for ONE property: O4 then O5.  alpha: per ReLU (topological order) [S, n_k],
    used for both branches (reading G7: benchmarks alias alpha_lo and alpha_up)."""
    pre = crown_bounds(net, x_lo, x_hi, intermediate, rule)
    a = None
    if alpha is not None:
        a = {i: alpha[j] for j, i in enumerate(net.relu_ids())}
    lb, ub, lin = final_bounds(net, x_lo, x_hi, C, pre, a, a, rule)
    return {"pre": pre, "lb": lb, "ub": ub, "lin": lin, "verified": verified(lb)}


def run_workload(wl, eps: Optional[float] = None, props: Optional[Sequence[int]] = None):
    """Whole hot path for a workloads.Workload (batch = loop over properties)."""
    lo, hi = wl.box() if eps is None else _box(wl.x0, eps)
    out = []
    for p in (range(wl.B) if props is None else props):
        al = None if wl.alpha is None else [a[p] for a in wl.alpha]
        out.append(run_property(wl.net, lo[p], hi[p], wl.C[p], al, wl.intermediate))
    return out


def _box(x0, eps):
    e = np.float32(eps).astype(F64)
    return ((x0.astype(F64) - e).astype(np.float32), (x0.astype(F64) + e).astype(np.float32))


# ------------------------------------------------------------------------------------------
# O6 -- sample containment ("lower bounds never exceed true minima; upper bounds
#       never fall below true maxima")
# ------------------------------------------------------------------------------------------
def adversarial_corners(A_lo, A_up, x_lo, x_hi) -> np.ndarray:
    """Per spec row the two box corners that minimise A_lo.x and maximise A_up.x: the tightest
    probes of a linear bound."""
    x_lo = np.asarray(x_lo, F64).reshape(-1)
    x_hi = np.asarray(x_hi, F64).reshape(-1)
    mins = np.where(A_lo >= 0.0, x_lo[None, :], x_hi[None, :])
    maxs = np.where(A_up >= 0.0, x_hi[None, :], x_lo[None, :])
    return np.concatenate([mins, maxs], axis=0)


def sample_check(net, C, X: np.ndarray, lb: np.ndarray, ub: np.ndarray, slack_rel: float = 1e-9,
                 slack_abs: float = 0.0):
    """C.f(x) in float64 for all probe points X [n, n0]; returns (ok, worst_lb_violation,
    worst_ub_violation, vmin [S], vmax [S]); violation > 0 means the bound was crossed by more than
    slack = slack_abs + slack_rel * (1 + |v|)."""
    Y = forward_batch(net, X) @ np.asarray(C, F64).T            # [n, S]
    vmin, vmax = Y.min(axis=0), Y.max(axis=0)
    sl_lo = slack_abs + slack_rel * (1.0 + np.abs(vmin))
    sl_hi = slack_abs + slack_rel * (1.0 + np.abs(vmax))
    v_lo = float(np.max(np.asarray(lb, F64) - vmin - sl_lo))
    v_hi = float(np.max(vmax - np.asarray(ub, F64) - sl_hi))
    return (v_lo <= 0.0 and v_hi <= 0.0), v_lo, v_hi, vmin, vmax
