"""float64 CPU oracle for the alpha optimisation of alpha-CROWN.

TEST INFRASTRUCTURE ONLY (same rules as oracle/crown_oracle.py: only `tests/`, `__graft_entry__.smoke()`
and `bench.py`'s `cpu_baseline` / `--impl reference` legs may import it; no code shared with the CUDA path).

What it follows (/root/reference/PAPER.md line + section):
  PAPER.md:70 (§2.1)  "alpha-CROWN promotes the fixed slopes lambda_i to per-neuron optimisable parameters
                       alpha_i in [0,1].  Gradient ascent over alpha tightens the lower bound (or lowers the
                       upper bound) without any branching."
  PAPER.md:266, :304  alpha tensors have shape (layers) x (specs) x (batch) x (neurons).

The paper gives no formula for the gradient; it is the derivative of O3 + concretisation
(oracle/crown_oracle.py `backward`, `concretize`) with respect to the lower-relaxation slopes, written out:

  O3 (lower branch, per spec row; A_i = coefficients w.r.t. the OUTPUT of node i):
      ReLU   i: A_in += A_i^+ * dL_i + A_i^- * dU_i ;   d += A_i^- . bU_i          (dL_i = alpha_i on unstable neurons)
      Linear i: A_in += A_i W_i ;                        d += A_i . b_i
      Conv   i: A_in += conv^T(A_i, W_i) ;               d += sum_o b_o sum_pq A_i[o,p,q]
      Add    i: A_in0 += A_i ; A_in1 += A_i              Flatten: A_in += A_i
      input   : lb = A_0 . x_c - |A_0| . x_r + d
  Chain rule with G_i := d lb / d A_i (one vector per spec row, shape of node i's output), taken in
  topological order (the transpose of every step above):
      input   : G_in = x_c - sign(A_0) * x_r            (the corner of the box that attains the minimum)
      Linear i: G_i = G_in W_i^T + b_i                   Conv i: G_i = conv(G_in, W_i) + b_i
      Add    i: G_i = G_in0 + G_in1                      Flatten: G_i = G_in
      ReLU   i: G_i = [A_i > 0] * dL_i * G_in + [A_i < 0] * (dU_i * G_in + bU_i)
                d lb / d alpha_i = A_i^+ * G_in  on unstable neurons, 0 on stable ones      (*)
  i.e. G is the network evaluated at the minimising corner with every ReLU replaced by the line the sign of A_i
  selects.  Upper branch: lb -> ub, the corner is x_c + sign(A_0) * x_r, ReLU: G_i = [A_i > 0] * (dU_i * G_in + bU_i)
  + [A_i < 0] * dL_i * G_in, and d ub / d alpha_i = A_i^- * G_in.
  At A = 0 (a kink of |.| and of the sign split) the one-sided derivative 0 is taken (reading G23 in DESIGN.md).

  Projected gradient ascent (step rule is a reading, G24): with a = clip(alpha, 0, 1),
      'plain': alpha <- clip(a + eta * g, 0, 1)        'sign': alpha <- clip(a + eta * sign(g), 0, 1)
  for the lower branch (ascent on lb) and with -g for the upper branch (descent on ub).  Every iterate is a valid
  alpha, so every iterate's bound is sound; the reported bound is the best over the iterates per spec row (G25).
  Intermediate bounds stay fixed (reading G8: alpha only on the final pass).

Pins (tests/test_oracle_alpha_pins.py, `-m "not gpu"`): central finite differences of `final_bounds` in alpha
(away from kinks); the hand-worked example E3 (tests/golden/e3_alpha_gradient.json: lb = -(|a1+a2| + |a1-a2|));
Euler's identity lb_s = C_s . G_last,s (lb is positively homogeneous of degree 1 in the spec row); zero gradient
on stable neurons; best-so-far bound never decreases and alpha stays in [0,1]; every iterate's bound is below the
exact minimum from brute-force activation-pattern enumeration.
"""
from __future__ import annotations

from typing import Dict, Optional, Tuple

import numpy as np

from . import crown_oracle as O
from .crown_oracle import ADD, CONV, FLATTEN, LINEAR, RELU

F64 = np.float64


def _unstable(l, u):
    l = np.asarray(l, F64).reshape(-1)
    u = np.asarray(u, F64).reshape(-1)
    return (l < 0.0) & (u > 0.0)          # not active (l >= 0), not inactive (u <= 0): reading G3


def bound_and_gradient(net, x_lo, x_hi, C, pre, alpha_lo: Dict[int, np.ndarray], alpha_up: Dict[int, np.ndarray],
                       rule: str = "adaptive"):
    """lb, ub [S] of O5 at the given alpha, and their derivatives with respect to the slopes:
    returns (lb, ub, g_lo, g_up, G_last) with g_lo[i] = d lb_s / d alpha_lo[i][s, :] and g_up[i] =
    d ub_s / d alpha_up[i][s, :]  ({relu id: [S, n_i]}), G_last = (G_lo, G_up) [S, n_out] at the output node.
    alpha_lo / alpha_up must hold an entry [S, n_i] for every ReLU (alpha-mode on every layer)."""
    C = np.asarray(C, F64)
    S = C.shape[0]
    trace: Dict[int, Tuple[np.ndarray, np.ndarray]] = {}
    A_lo, A_up, d_lo, d_up = O.backward(net, len(net.nodes) - 1, C, pre, alpha_lo, alpha_up, rule, trace=trace)
    lb, ub = O.concretize(A_lo, A_up, d_lo, d_up, x_lo, x_hi)
    x_lo = np.asarray(x_lo, F64).reshape(-1)
    x_hi = np.asarray(x_hi, F64).reshape(-1)
    xc, xr = 0.5 * (x_lo + x_hi), 0.5 * (x_hi - x_lo)
    # G[br][i]: d bound / d A_i, [S, size_i]; node -1 = network input
    G = [{-1: xc[None, :] - np.sign(A_lo) * xr[None, :]}, {-1: xc[None, :] + np.sign(A_up) * xr[None, :]}]
    g = [dict(), dict()]
    for i, n in enumerate(net.nodes):
        for br in (0, 1):
            Gb = G[br]
            if n.in0 not in Gb or (n.op == ADD and n.in1 not in Gb):
                continue
            if n.op == LINEAR:
                Gb[i] = Gb[n.in0].reshape(S, -1) @ n.W.astype(F64).T + n.b.astype(F64)[None, :]
            elif n.op == CONV:
                shp = O._in_shape(net, n.in0)
                x = Gb[n.in0].reshape((S,) + tuple(shp))
                y = np.stack([O.conv2d(x[s], n.W, n.stride, n.pad) for s in range(S)])
                Gb[i] = (y + n.b.astype(F64)[None, :, None, None]).reshape(S, -1)
            elif n.op == ADD:
                Gb[i] = Gb[n.in0].reshape(S, -1) + Gb[n.in1].reshape(S, -1)
            elif n.op == FLATTEN:
                Gb[i] = Gb[n.in0].reshape(S, -1)
            elif n.op == RELU:
                l, u = pre[i]
                a = (alpha_lo, alpha_up)[br][i]
                dU, bU, dL = O.relax_coeffs(l, u, a, rule)          # dL [S, n] = clip(alpha) on unstable neurons
                A = trace[i][br] if i in trace else np.zeros((S, n.size))
                Gin = Gb[n.in0].reshape(S, -1)
                pos, neg = (A > 0.0), (A < 0.0)
                if br == 0:
                    Gb[i] = pos * (dL * Gin) + neg * (dU[None, :] * Gin + bU[None, :])
                    g[0][i] = np.maximum(A, 0.0) * Gin * _unstable(l, u)[None, :]
                else:
                    Gb[i] = pos * (dU[None, :] * Gin + bU[None, :]) + neg * (dL * Gin)
                    g[1][i] = np.minimum(A, 0.0) * Gin * _unstable(l, u)[None, :]
            else:
                raise ValueError(n.op)
    last = len(net.nodes) - 1
    return lb, ub, g[0], g[1], (G[0][last], G[1][last])


def ascent_step(alpha: np.ndarray, grad: np.ndarray, eta: float, mode: str, ascend: bool) -> np.ndarray:
    """One projected step (reading G24): a = clip(alpha); a + eta * dir, clipped to [0,1]; dir = g or sign(g),
    negated for descent (upper branch)."""
    a = np.clip(np.asarray(alpha, F64), 0.0, 1.0)
    step = grad if mode == "plain" else np.sign(grad)
    if not ascend:
        step = -step
    return np.clip(a + eta * step, 0.0, 1.0)


def alpha_ascent(net, x_lo, x_hi, C, pre, alpha_lo: Dict[int, np.ndarray], alpha_up: Dict[int, np.ndarray],
                 eta: float, iters: int, mode: str = "sign", decay: float = 1.0, rule: str = "adaptive"):
    """`iters` projected gradient steps on alpha_lo (ascent on lb) and alpha_up (descent on ub), bounds evaluated
    at iters + 1 points (the start and after every step); step t uses eta * decay^t.  Returns a dict with the final
    alpha, the bounds at every evaluation (`lb_hist`, `ub_hist` [iters+1, S]) and the best per spec row
    (`lb_best` = max_t lb_t, `ub_best` = min_t ub_t): all iterates are sound, so the best is (G25)."""
    al = {i: np.clip(np.asarray(a, F64), 0.0, 1.0) for i, a in alpha_lo.items()}
    au = {i: np.clip(np.asarray(a, F64), 0.0, 1.0) for i, a in alpha_up.items()}
    lb_hist, ub_hist = [], []
    step = float(eta)
    for t in range(iters + 1):
        lb, ub, g_lo, g_up, _ = bound_and_gradient(net, x_lo, x_hi, C, pre, al, au, rule)
        lb_hist.append(lb)
        ub_hist.append(ub)
        if t == iters:
            break
        al = {i: ascent_step(al[i], g_lo[i], step, mode, True) for i in al}
        au = {i: ascent_step(au[i], g_up[i], step, mode, False) for i in au}
        step *= decay
    lb_hist, ub_hist = np.stack(lb_hist), np.stack(ub_hist)
    return {"alpha_lo": al, "alpha_up": au, "lb_hist": lb_hist, "ub_hist": ub_hist,
            "lb_best": lb_hist.max(axis=0), "ub_best": ub_hist.min(axis=0)}
