"""float64 CPU oracle for beta-CROWN bounds of branch-and-bound sub-domains.

TEST INFRASTRUCTURE ONLY (same rules as oracle/crown_oracle.py: only `tests/`, `__graft_entry__.smoke()`
and `bench.py`'s `cpu_baseline` / `--impl reference` legs may import it; no code shared with the CUDA path).

What it follows (/root/reference/PAPER.md line + section):
  PAPER.md:76 (§2.1.1) "Branch-and-Bound (BaB): when bounds are insufficient, the input space is split into
                        sub-regions (e.g. by fixing a ReLU state x >= 0 or x < 0), and bounds are recomputed for
                        each sub-region."
  PAPER.md:80 (§2.2)   "The key innovation of beta-CROWN is encoding ReLU-split constraints directly into the
                        bound-propagation pass via Lagrangian dual variables beta ... bounds for thousands of
                        sub-problems are evaluated in parallel on GPU as batched matrix multiplications, and
                        alpha/beta parameters are jointly optimised by gradient descent."
  PAPER.md:96 (§2.4)   batch BaB: sub-problems are batched and bounded in a single pass.
  PAPER.md:180 (§3.4.4) "Branching-constraint variables beta are managed identically to single-GPU mode."

The paper names the mechanism and gives no formula; it is weak Lagrangian duality written into O3
(oracle/crown_oracle.py `backward`), restated here step by step (readings G26-G28 in DESIGN.md):

  A sub-domain = the box [x_lo, x_hi] plus, per ReLU i, a sign vector s_i in {-1, 0, +1}^{n_i} on its
  PRE-activation z_i:  s_ij = +1 fixes z_ij >= 0 (active),  -1 fixes z_ij <= 0 (inactive),  0 = not split.
  (G26) A split neuron's pre-activation interval is clamped: l_ij <- max(l_ij, 0) if s_ij = +1,
        u_ij <- min(u_ij, 0) if s_ij = -1; its relaxation is then the exact line of that state (O2: active / inactive).
  (G27) For any beta_i >= 0 (one value per spec row and neuron, shape [R, n_i]; used only where s_ij != 0):
            min_{x in box, s_i * z_i(x) >= 0}  c.f(x)   >=   min_{x in box}  c.f(x) - sum_i (beta_i * s_i) . z_i(x)
        because the subtracted term is >= 0 on the sub-domain.  In the backward recursion this adds, right after
        the relaxation of ReLU i (where A is the coefficient matrix w.r.t. z_i):
            lower branch:  A_z <- A_z - beta_lo_i * s_i          upper branch:  A_z <- A_z + beta_up_i * s_i
        (upper bound of c.f = minus the lower bound of -c.f).  Everything else is O3 unchanged; beta = 0 gives
        plain CROWN on the clamped intervals.
  (G28) Joint projected gradient ascent on (alpha, beta): alpha as in oracle/alpha_oracle.py; with
        G_z := d bound / d A_z (the forward sweep of alpha_oracle: z_i evaluated at the bound-attaining corner
        through the selected lines),   d lb / d beta_lo_i = -s_i * G_z,   d ub / d beta_up_i = +s_i * G_z;
        beta <- max(beta +- eta_beta * dir, 0), dir = g or sign(g).  Every iterate is sound (G27 holds for every
        beta >= 0 and every alpha in [0,1]); the best bound per spec row over the iterates is reported (G25).

Pins (tests/test_oracle_beta_pins.py, `-m "not gpu"`): a hand-worked example (tests/golden/e4_beta_split.json:
lb(alpha, beta) = -|1 + alpha - beta|, exact sub-domain minimum 0 reached at beta = 1 + alpha); beta = 0 equals
crown_oracle.backward on the clamped intervals; weak duality against the exact sub-domain minimum from brute-force
activation-pattern enumeration restricted to the split (oracle/brute_force.py); central finite differences of the
bound in beta; best-so-far monotone, beta >= 0; containment of sampled points that satisfy the split constraints.
"""
from __future__ import annotations

from typing import Dict, Optional, Tuple

import numpy as np

from . import crown_oracle as O
from .crown_oracle import ADD, CONV, FLATTEN, LINEAR, RELU

F64 = np.float64


def clamp_split(pre: Dict[int, Tuple[np.ndarray, np.ndarray]], split: Optional[Dict[int, np.ndarray]]):
    """(G26) pre-activation intervals of a sub-domain: l <- max(l, 0) where s = +1, u <- min(u, 0) where s = -1."""
    out = {}
    for i, (l, u) in pre.items():
        l = np.asarray(l, F64).reshape(-1).copy()
        u = np.asarray(u, F64).reshape(-1).copy()
        s = None if split is None else split.get(i)
        if s is not None:
            s = np.asarray(s).reshape(-1)
            l = np.where(s > 0, np.maximum(l, 0.0), l)
            u = np.where(s < 0, np.minimum(u, 0.0), u)
        out[i] = (l, u)
    return out


def _beta_term(beta, s, R, n):
    """max(beta, 0) * s broadcast to [R, n]; zero where the neuron is not split or no beta is given."""
    if beta is None or s is None:
        return np.zeros((R, n))
    b = np.maximum(np.asarray(beta, F64), 0.0)
    return np.broadcast_to(b, (R, n)) * np.asarray(s, F64).reshape(1, n)


def backward(net, start: int, C0: np.ndarray, pre, split=None, beta_lo=None, beta_up=None,
             alpha_lo=None, alpha_up=None, rule: str = "adaptive", trace=None):
    """O3 with split constraints (G26, G27) for ONE sub-domain.  `pre` are the UNCLAMPED intervals (clamped here);
    split: {relu id: s [n_i] in {-1,0,+1}};  beta_lo / beta_up: {relu id: [R, n_i]} (None / missing = 0).
    Returns (A_lo, A_up, d_lo, d_up) as crown_oracle.backward; trace receives A w.r.t. each ReLU's OUTPUT."""
    C0 = np.asarray(C0, F64)
    R = C0.shape[0]
    n0 = int(np.prod(net.in_shape))
    prec = clamp_split(pre, split)
    pend = {start: [C0.reshape(R, -1).copy(), C0.reshape(R, -1).copy()]}
    d = [np.zeros(R), np.zeros(R)]

    def contribute(idx, parts):
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
            W, b = n.W.astype(F64), n.b.astype(F64)
            for br in (0, 1):
                d[br] = d[br] + A[br] @ b
            contribute(n.in0, [A[0] @ W, A[1] @ W])
        elif n.op == CONV:
            b = n.b.astype(F64)
            c_out, ho, wo = n.shape
            ish = O._in_shape(net, n.in0)
            outs = []
            for br in (0, 1):
                Ab = A[br].reshape(R, c_out, ho, wo)
                d[br] = d[br] + np.einsum("rohw,o->r", Ab, b)
                outs.append(O.conv2d_transpose(Ab, n.W, n.stride, n.pad, (ish[1], ish[2])))
            contribute(n.in0, outs)
        elif n.op == ADD:
            contribute(n.in0, A)
            contribute(n.in1, A)
        elif n.op == FLATTEN:
            contribute(n.in0, A)
        elif n.op == RELU:
            l, u = prec[i]
            if trace is not None:
                trace[i] = (A[0].copy(), A[1].copy())
            a_lo = None if alpha_lo is None else alpha_lo.get(i)
            a_up = None if alpha_up is None else alpha_up.get(i)
            dU, bU, dL_lo = O.relax_coeffs(l, u, a_lo, rule)
            _, _, dL_up = O.relax_coeffs(l, u, a_up, rule)
            s = None if split is None else split.get(i)
            nn = A[0].shape[1]
            Ap, Am = np.maximum(A[0], 0.0), np.minimum(A[0], 0.0)
            new_lo = Ap * dL_lo + Am * dU - _beta_term(None if beta_lo is None else beta_lo.get(i), s, R, nn)
            d[0] = d[0] + Am @ bU
            Ap, Am = np.maximum(A[1], 0.0), np.minimum(A[1], 0.0)
            new_up = Ap * dU + Am * dL_up + _beta_term(None if beta_up is None else beta_up.get(i), s, R, nn)
            d[1] = d[1] + Ap @ bU
            contribute(n.in0, [new_lo, new_up])
        else:
            raise ValueError(n.op)
    if -1 in pend:
        A_lo, A_up = pend[-1]
    else:
        A_lo, A_up = np.zeros((R, n0)), np.zeros((R, n0))
    return A_lo, A_up, d[0], d[1]


def final_bounds(net, x_lo, x_hi, C, pre, split=None, beta_lo=None, beta_up=None, alpha_lo=None, alpha_up=None,
                 rule: str = "adaptive"):
    """lb, ub [S] of C.f over the sub-domain (box + split), for the given alpha / beta."""
    A_lo, A_up, d_lo, d_up = backward(net, len(net.nodes) - 1, C, pre, split, beta_lo, beta_up, alpha_lo, alpha_up, rule)
    return O.concretize(A_lo, A_up, d_lo, d_up, x_lo, x_hi)


def bound_and_gradient(net, x_lo, x_hi, C, pre, split, beta_lo, beta_up, alpha_lo, alpha_up, rule: str = "adaptive"):
    """Bounds and their derivatives w.r.t. alpha and beta (G28).  alpha_* / beta_* hold an entry [S, n_i] for every
    ReLU.  Returns (lb, ub, ga_lo, ga_up, gb_lo, gb_up): {relu id: [S, n_i]} each; gb is zero off the split set,
    ga is zero on stable (incl. split) neurons."""
    C = np.asarray(C, F64)
    S = C.shape[0]
    trace = {}
    A_lo, A_up, d_lo, d_up = backward(net, len(net.nodes) - 1, C, pre, split, beta_lo, beta_up, alpha_lo, alpha_up, rule, trace)
    lb, ub = O.concretize(A_lo, A_up, d_lo, d_up, x_lo, x_hi)
    prec = clamp_split(pre, split)
    x_lo = np.asarray(x_lo, F64).reshape(-1)
    x_hi = np.asarray(x_hi, F64).reshape(-1)
    xc, xr = 0.5 * (x_lo + x_hi), 0.5 * (x_hi - x_lo)
    G = [{-1: xc[None, :] - np.sign(A_lo) * xr[None, :]}, {-1: xc[None, :] + np.sign(A_up) * xr[None, :]}]
    ga, gb = [dict(), dict()], [dict(), dict()]
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
                l, u = prec[i]
                a = (alpha_lo, alpha_up)[br][i]
                dU, bU, dL = O.relax_coeffs(l, u, a, rule)
                unstable = ((l < 0.0) & (u > 0.0))[None, :]
                A = trace[i][br] if i in trace else np.zeros((S, n.size))
                Gin = Gb[n.in0].reshape(S, -1)                       # z_i at the bound-attaining corner
                pos, neg = (A > 0.0), (A < 0.0)
                s = np.zeros(n.size) if split is None or split.get(i) is None else np.asarray(split[i], F64).reshape(-1)
                if br == 0:
                    Gb[i] = pos * (dL * Gin) + neg * (dU[None, :] * Gin + bU[None, :])
                    ga[0][i] = np.maximum(A, 0.0) * Gin * unstable
                    gb[0][i] = -s[None, :] * Gin
                else:
                    Gb[i] = pos * (dU[None, :] * Gin + bU[None, :]) + neg * (dL * Gin)
                    ga[1][i] = np.minimum(A, 0.0) * Gin * unstable
                    gb[1][i] = s[None, :] * Gin
            else:
                raise ValueError(n.op)
    return lb, ub, ga[0], ga[1], gb[0], gb[1]


def _dir(g, mode):
    return g if mode == "plain" else np.sign(g)


def joint_ascent(net, x_lo, x_hi, C, pre, split, beta_lo, beta_up, alpha_lo, alpha_up, eta_alpha: float,
                 eta_beta: float, iters: int, mode: str = "sign", decay: float = 1.0, rule: str = "adaptive"):
    """`iters` joint projected steps (G28); bounds at iters + 1 points; step t uses eta * decay^t.
    Lower branch ascends lb in (alpha_lo, beta_lo); upper branch descends ub in (alpha_up, beta_up)."""
    al = {i: np.clip(np.asarray(a, F64), 0.0, 1.0) for i, a in alpha_lo.items()}
    au = {i: np.clip(np.asarray(a, F64), 0.0, 1.0) for i, a in alpha_up.items()}
    bl = {i: np.maximum(np.asarray(b, F64), 0.0) for i, b in beta_lo.items()}
    bu = {i: np.maximum(np.asarray(b, F64), 0.0) for i, b in beta_up.items()}
    lb_hist, ub_hist = [], []
    ea, eb = float(eta_alpha), float(eta_beta)
    for t in range(iters + 1):
        lb, ub, ga_lo, ga_up, gb_lo, gb_up = bound_and_gradient(net, x_lo, x_hi, C, pre, split, bl, bu, al, au, rule)
        lb_hist.append(lb)
        ub_hist.append(ub)
        if t == iters:
            break
        al = {i: np.clip(al[i] + ea * _dir(ga_lo[i], mode), 0.0, 1.0) for i in al}
        au = {i: np.clip(au[i] - ea * _dir(ga_up[i], mode), 0.0, 1.0) for i in au}
        bl = {i: np.maximum(bl[i] + eb * _dir(gb_lo[i], mode), 0.0) for i in bl}
        bu = {i: np.maximum(bu[i] - eb * _dir(gb_up[i], mode), 0.0) for i in bu}
        ea *= decay
        eb *= decay
    lb_hist, ub_hist = np.stack(lb_hist), np.stack(ub_hist)
    return {"alpha_lo": al, "alpha_up": au, "beta_lo": bl, "beta_up": bu, "lb_hist": lb_hist, "ub_hist": ub_hist,
            "lb_best": lb_hist.max(axis=0), "ub_best": ub_hist.min(axis=0)}
