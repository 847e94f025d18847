"""Pins of oracle/alpha_oracle.py (alpha optimisation of alpha-CROWN) against
things other than itself: a hand-worked example, finite differences of the (separately pinned) bound, Euler's
identity, brute-force exact minima.  CPU only."""
import json
import os

import numpy as np
import pytest

import workloads as wl_mod
from oracle import alpha_oracle as AO
from oracle import brute_force as BF
from oracle import crown_oracle as O
from workloads import Net, Node

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _load(name):
    with open(os.path.join(GOLD, name)) as f:
        return json.load(f)


def _e3_net():
    g = _load("e3_alpha_rows.json")
    W1 = np.array(g["W1"], np.float32); b1 = np.array(g["b1"], np.float32)
    W2 = np.array(g["W2"], np.float32); b2 = np.array(g["b2"], np.float32)
    net = Net(in_shape=(2,))
    net.nodes.append(Node("linear", -1, W=W1, b=b1, shape=(2,)))
    net.nodes.append(Node("relu", 0, shape=(2,)))
    net.nodes.append(Node("linear", 1, W=W2, b=b2, shape=(1,)))
    return net, np.array(g["x_lo"]), np.array(g["x_hi"])


def test_e3_gradient_closed_form_and_sign_ascent():
    """tests/golden/e3_alpha_gradient.json: lb(a) = -(|a1+a2| + |a1-a2|) and its derivative, the upper bound's
    independence of alpha_up, and a three-step sign ascent that reaches the true minimum 0."""
    g = _load("e3_alpha_gradient.json")
    net, lo, hi = _e3_net()
    pre = O.crown_bounds(net, lo, hi)
    al = np.array([c["alpha"] for c in g["gradient_cases"]])
    C = np.ones((al.shape[0], 1))
    lb, ub, g_lo, g_up, _ = AO.bound_and_gradient(net, lo, hi, C, pre, {1: al}, {1: al})
    np.testing.assert_allclose(lb, [c["lb"] for c in g["gradient_cases"]], atol=1e-15)
    np.testing.assert_allclose(g_lo[1], [c["g_lo"] for c in g["gradient_cases"]], atol=1e-15)
    np.testing.assert_allclose(g_up[1], np.broadcast_to(g["g_up"], al.shape), atol=1e-15)
    a = g["ascent"]
    a0 = np.array([a["alpha0"]])
    r = AO.alpha_ascent(net, lo, hi, np.ones((1, 1)), pre, {1: a0}, {1: a0}, a["eta"], a["iters"], a["mode"])
    np.testing.assert_allclose(r["lb_hist"][:, 0], a["lb_hist"], atol=1e-15)
    np.testing.assert_allclose(r["alpha_lo"][1][0], a["alpha_final"], atol=1e-15)
    assert r["lb_best"][0] == 0.0
    mn, _ = BF.exact_range(net, lo, hi, np.ones((1, 1)))
    assert abs(mn[0] - r["lb_best"][0]) < 1e-9            # the optimum of alpha-CROWN is the exact minimum here


def _fd_check(net, lo, hi, C, pre, al, au, rng, n_probe=40, h=1e-6):
    """central differences of O.final_bounds in single alpha entries vs the analytic gradient"""
    lb, ub, g_lo, g_up, _ = AO.bound_and_gradient(net, lo, hi, C, pre, al, au)
    lb_ref, ub_ref, _ = O.final_bounds(net, lo, hi, C, pre, al, au)
    np.testing.assert_allclose(lb, lb_ref, atol=0, rtol=0)
    np.testing.assert_allclose(ub, ub_ref, atol=0, rtol=0)
    S = C.shape[0]
    checked = 0
    for _ in range(n_probe):
        i = int(rng.choice(list(al.keys())))
        s = int(rng.integers(S)); j = int(rng.integers(al[i].shape[1]))
        for br, alpha, grad in ((0, al, g_lo), (1, au, g_up)):
            if not (h < alpha[i][s, j] < 1 - h):
                continue
            ap = {k: v.copy() for k, v in alpha.items()}; am = {k: v.copy() for k, v in alpha.items()}
            ap[i][s, j] += h; am[i][s, j] -= h
            if br == 0:
                fp = O.final_bounds(net, lo, hi, C, pre, ap, au)[0]; fm = O.final_bounds(net, lo, hi, C, pre, am, au)[0]
            else:
                fp = O.final_bounds(net, lo, hi, C, pre, al, ap)[1]; fm = O.final_bounds(net, lo, hi, C, pre, al, am)[1]
            fd = (fp - fm) / (2 * h)
            # alpha[i][s, j] only enters row s
            other = np.delete(fd, s)
            assert np.all(np.abs(other) < 1e-7), "alpha of one spec row changed another row's bound"
            an = grad[i][s, j]
            assert abs(fd[s] - an) <= 1e-5 * (1 + abs(an)), (i, s, j, br, fd[s], an)
            checked += 1
    return checked


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_gradient_matches_finite_differences_mlp(seed):
    w = wl_mod.small_mlp([5, 8, 7, 6, 4], seed=10 + seed, B=1, eps=0.3, S=3)
    lo, hi = w.box()
    rng = np.random.default_rng(seed)
    for inter in ("crown", "ibp"):
        pre = O.crown_bounds(w.net, lo[0], hi[0], inter)
        al = {i: rng.uniform(0.05, 0.95, w.alpha[j][0].shape) for j, i in enumerate(w.net.relu_ids())}
        au = {i: rng.uniform(0.05, 0.95, w.alpha[j][0].shape) for j, i in enumerate(w.net.relu_ids())}
        assert _fd_check(w.net, lo[0], hi[0], w.C[0].astype(np.float64), pre, al, au, rng) >= 40
        # stable neurons have zero gradient, unstable ones (generically) not all zero
        _, _, g_lo, g_up, _ = AO.bound_and_gradient(w.net, lo[0], hi[0], w.C[0], pre, al, au)
        n_unstable = 0
        for i in w.net.relu_ids():
            l, u = pre[i]
            st = ~((l < 0) & (u > 0))
            assert np.all(g_lo[i][:, st] == 0) and np.all(g_up[i][:, st] == 0)
            n_unstable += int((~st).sum())
        assert n_unstable > 0
        assert any(np.any(g_lo[i] != 0) for i in g_lo)


def test_gradient_matches_finite_differences_residual_conv_net():
    """the DAG case: conv, residual add (fork sum in O3 = both parents in the forward sweep), flatten, linear"""
    rng = np.random.Generator(np.random.PCG64(77))
    net = wl_mod.resnet(rng, in_shape=(2, 6, 6), stem=3, blocks=((3, 1), (4, 2)), fc=6, n_classes=4)
    x0 = rng.random(net.n_in).astype(np.float32)
    lo, hi = (x0 - 0.05).astype(np.float32), (x0 + 0.05).astype(np.float32)
    C = rng.standard_normal((2, net.n_out))
    pre = O.crown_bounds(net, lo, hi, "ibp")
    al = {i: rng.uniform(0.05, 0.95, (2, net.nodes[i].size)) for i in net.relu_ids()}
    au = {i: rng.uniform(0.05, 0.95, (2, net.nodes[i].size)) for i in net.relu_ids()}
    assert _fd_check(net, lo, hi, C, pre, al, au, rng, n_probe=30) >= 30


def test_euler_identity_bound_equals_spec_dot_G():
    """lb_s (ub_s) is positively homogeneous of degree 1 in spec row s (O3 and the concretisation are), hence
    lb_s = <C_s, d lb_s / d C_s> = C_s . G_last[s]: pins the whole forward sweep G without finite differences."""
    w = wl_mod.small_mlp([6, 9, 7, 5], seed=5, B=1, eps=0.25, S=4)
    lo, hi = w.box()
    pre = O.crown_bounds(w.net, lo[0], hi[0])
    al = {i: w.alpha[j][0].astype(np.float64) for j, i in enumerate(w.net.relu_ids())}
    lb, ub, _, _, (G_lo, G_up) = AO.bound_and_gradient(w.net, lo[0], hi[0], w.C[0], pre, al, al)
    C = w.C[0].astype(np.float64)
    np.testing.assert_allclose(np.sum(C * G_lo, axis=1), lb, rtol=1e-12, atol=1e-12)
    np.testing.assert_allclose(np.sum(C * G_up, axis=1), ub, rtol=1e-12, atol=1e-12)
    # and G_last is d lb / d C by finite differences in C
    h = 1e-6
    for s, j in ((0, 1), (2, 0), (3, 4)):
        Cp, Cm = C.copy(), C.copy()
        Cp[s, j] += h; Cm[s, j] -= h
        fd = (O.final_bounds(w.net, lo[0], hi[0], Cp, pre, al, al)[0][s] -
              O.final_bounds(w.net, lo[0], hi[0], Cm, pre, al, al)[0][s]) / (2 * h)
        assert abs(fd - G_lo[s, j]) < 1e-6 * (1 + abs(fd))


@pytest.mark.parametrize("mode,eta", [("sign", 0.05), ("plain", 0.02)])
def test_ascent_best_is_monotone_sound_and_projected(mode, eta):
    w = wl_mod.small_mlp([2, 4, 4, 3], seed=1, B=1, eps=0.8, S=3)
    lo, hi = w.box()
    pre = O.crown_bounds(w.net, lo[0], hi[0])
    al = {i: w.alpha[j][0].astype(np.float64) * 1.6 - 0.3 for j, i in enumerate(w.net.relu_ids())}   # partly outside [0,1]
    r = AO.alpha_ascent(w.net, lo[0], hi[0], w.C[0], pre, al, al, eta, 25, mode, decay=0.97)
    for a in list(r["alpha_lo"].values()) + list(r["alpha_up"].values()):
        assert a.min() >= 0.0 and a.max() <= 1.0
    # best-so-far never decreases; the optimised bound is at least the starting one and strictly better somewhere
    best = np.maximum.accumulate(r["lb_hist"], axis=0)
    assert np.all(best[-1] == r["lb_best"]) and np.all(r["lb_best"] >= r["lb_hist"][0])
    assert np.all(r["ub_best"] <= r["ub_hist"][0])
    assert np.any(r["lb_best"] > r["lb_hist"][0] + 1e-6) and np.any(r["ub_best"] < r["ub_hist"][0] - 1e-6)
    # every iterate is sound: below the exact minimum / above the exact maximum (brute force, O7)
    mn, mx = BF.exact_range(w.net, lo[0], hi[0], w.C[0])
    assert np.all(r["lb_hist"] <= mn[None, :] + 1e-9) and np.all(r["ub_hist"] >= mx[None, :] - 1e-9)
    # the bound at the final alpha is what O5 returns for it
    lb, ub, _ = O.final_bounds(w.net, lo[0], hi[0], w.C[0], pre, r["alpha_lo"], r["alpha_up"])
    np.testing.assert_allclose(lb, r["lb_hist"][-1], atol=0, rtol=0)
    np.testing.assert_allclose(ub, r["ub_hist"][-1], atol=0, rtol=0)


def test_ascent_step_rule():
    a = np.array([[-0.2, 0.5, 0.98, 0.3]])
    g = np.array([[1.0, -3.0, 2.0, 0.0]])
    np.testing.assert_allclose(AO.ascent_step(a, g, 0.1, "sign", True), [[0.1, 0.4, 1.0, 0.3]])
    np.testing.assert_allclose(AO.ascent_step(a, g, 0.1, "sign", False), [[0.0, 0.6, 0.88, 0.3]])
    np.testing.assert_allclose(AO.ascent_step(a, g, 0.1, "plain", True), [[0.1, 0.2, 1.0, 0.3]])
