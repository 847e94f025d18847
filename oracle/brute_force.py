"""O7 -- exact output range of a tiny ReLU MLP by activation-pattern enumeration + LP.

TEST INFRASTRUCTURE ONLY (see oracle/crown_oracle.py header).  Independent of the bound
propagation code: it never forms a relaxation.  For a fixed activation pattern s in {0,1}^n the
network is affine on the polytope {x in box : pattern constraints}; the exact minimum / maximum of
c.f(x) is the min / max over all feasible patterns of an LP optimum (BaB fixes ReLU
states x >= 0 or x < 0 -- full enumeration is BaB run to exhaustion; PAPER.md:74 defines what the
bounds must enclose).  Feasible only for <= ~12 ReLU neurons and small n0 (2^n LPs).
"""
from __future__ import annotations

import itertools
from typing import Tuple

import numpy as np
from scipy.optimize import linprog

LINEAR, RELU = "linear", "relu"


def exact_range(net, x_lo, x_hi, C: np.ndarray, split=None) -> Tuple[np.ndarray, np.ndarray]:
    """Exact (min, max) [S] of C.f(x) over the box for a plain MLP (linear/relu chain).
    split (optional): {relu node id: s in {-1,0,+1}^n}: the BaB sub-domain that fixes pre-activation j of that ReLU to
    >= 0 (s = +1) or <= 0 (s = -1); only activation patterns that agree with it are enumerated.
    Returns (+inf, -inf) for an empty sub-domain."""
    x_lo = np.asarray(x_lo, np.float64).reshape(-1)
    x_hi = np.asarray(x_hi, np.float64).reshape(-1)
    C = np.asarray(C, np.float64)
    n0 = x_lo.size
    layers = []
    for i, n in enumerate(net.nodes):
        if n.op == LINEAR:
            assert n.in0 == i - 1, "chain MLP expected"
            layers.append((n.W.astype(np.float64), n.b.astype(np.float64)))
        else:
            assert n.op == RELU and n.in0 == i - 1, "chain MLP expected"
    hidden = [W.shape[0] for W, _ in layers[:-1]]
    n_relu = int(sum(hidden))
    assert n_relu <= 14, "too many neurons to enumerate"
    S = C.shape[0]
    best_min = np.full(S, np.inf)
    best_max = np.full(S, -np.inf)
    bounds = list(zip(x_lo, x_hi))
    fixed = np.zeros(n_relu, dtype=int)          # per enumerated neuron: 0 free, +1 must be active, -1 must be inactive
    if split is not None:
        off, k = 0, 0
        for i, n in enumerate(net.nodes):
            if n.op == RELU:
                if split.get(i) is not None:
                    fixed[off:off + hidden[k]] = np.sign(np.asarray(split[i]).reshape(-1)).astype(int)
                off += hidden[k]
                k += 1
    for pattern in itertools.product((0, 1), repeat=n_relu):
        pat = np.array(pattern)
        if np.any((fixed > 0) & (pat == 0)) or np.any((fixed < 0) & (pat == 1)):
            continue
        # affine map of the current layer's post-activation: z = M x + v
        M = np.eye(n0)
        v = np.zeros(n0)
        A_ub, b_ub = [], []
        off = 0
        for (W, b), h in zip(layers[:-1], hidden):
            Mz = W @ M
            vz = W @ v + b
            s = np.array(pattern[off:off + h], dtype=np.float64)
            off += h
            for j in range(h):
                if s[j] > 0:      # active: Mz_j x + vz_j >= 0
                    A_ub.append(-Mz[j]); b_ub.append(vz[j])
                else:             # inactive: Mz_j x + vz_j <= 0
                    A_ub.append(Mz[j]); b_ub.append(-vz[j])
            M = s[:, None] * Mz
            v = s * vz
        W, b = layers[-1]
        Mo = C @ (W @ M)
        vo = C @ (W @ v + b)
        A_ub_a = np.array(A_ub) if A_ub else None
        b_ub_a = np.array(b_ub) if b_ub else None
        # feasibility once per pattern
        feas = linprog(np.zeros(n0), A_ub=A_ub_a, b_ub=b_ub_a, bounds=bounds, method="highs")
        if feas.status != 0:
            continue
        for r in range(S):
            lo = linprog(Mo[r], A_ub=A_ub_a, b_ub=b_ub_a, bounds=bounds, method="highs")
            hi = linprog(-Mo[r], A_ub=A_ub_a, b_ub=b_ub_a, bounds=bounds, method="highs")
            if lo.status == 0:
                best_min[r] = min(best_min[r], lo.fun + vo[r])
            if hi.status == 0:
                best_max[r] = max(best_max[r], -hi.fun + vo[r])
    return best_min, best_max
