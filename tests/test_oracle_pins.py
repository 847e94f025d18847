"""Pins for the float64 oracle (`-m "not gpu"`): each test checks the oracle against something
OTHER than itself -- values the paper prints, hand-worked closed forms, invariants, library
routines (dense matmul for conv), brute force.  A dropped term, wrong sign/index or transposed
operand anywhere in oracle/crown_oracle.py must fail at least one of these."""
import json
import os

import numpy as np
import pytest

import workloads as wl_mod
from workloads import Net, Node
from oracle import crown_oracle as O
from oracle import brute_force as BF

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _load(name):
    with open(os.path.join(GOLD, name)) as f:
        return json.load(f)


def _net_from(g, relu_between=True):
    W1 = np.array(g["W1"], np.float32); b1 = np.array(g["b1"], np.float32)
    W2 = np.array(g["W2"], np.float32); b2 = np.array(g["b2"], np.float32)
    net = Net(in_shape=(W1.shape[1],))
    net.nodes.append(Node("linear", -1, W=W1, b=b1, shape=(W1.shape[0],)))
    src = 0
    if relu_between:
        net.nodes.append(Node("relu", 0, shape=(W1.shape[0],)))
        src = 1
    net.nodes.append(Node("linear", src, W=W2, b=b2, shape=(W2.shape[0],)))
    return net


# ---------------------------------------------------------------- paper's worked example
def test_paper_example_ibp_unfused_and_crown_exact():
    g = _load("paper_example_wrapping.json")
    net = _net_from(g, relu_between=False)        # two stacked linear layers, no ReLU
    lo, hi = np.array(g["x_lo"]), np.array(g["x_hi"])
    ib = O.ibp(net, lo, hi)
    np.testing.assert_allclose(ib[0][0], g["ibp_y"][0], atol=0)
    np.testing.assert_allclose(ib[0][1], g["ibp_y"][1], atol=0)
    assert ib[1][0][0] == g["ibp_z1"][0] and ib[1][1][0] == g["ibp_z1"][1]
    A_lo, A_up, d_lo, d_up = O.backward(net, 1, np.eye(1), {})
    np.testing.assert_allclose(A_lo[0], g["crown_A"], atol=0)
    np.testing.assert_allclose(A_up[0], g["crown_A"], atol=0)
    lb, ub = O.concretize(A_lo, A_up, d_lo, d_up, lo, hi)
    assert lb[0] == g["crown_z1"][0] and ub[0] == g["crown_z1"][1]


# ---------------------------------------------------------------- hand-worked relaxations
def test_e2_relaxation_sign_split_and_bias():
    g = _load("e2_relaxation.json")
    net = _net_from(g)
    lo, hi = np.array(g["x_lo"]), np.array(g["x_hi"])
    pre = O.crown_bounds(net, lo, hi)
    np.testing.assert_allclose(pre[1][0], g["pre_l"], atol=1e-15)
    np.testing.assert_allclose(pre[1][1], g["pre_u"], atol=1e-15)
    dU, bU, _ = O.relax_coeffs(*pre[1])
    np.testing.assert_allclose(dU, g["dU"], atol=1e-15)
    np.testing.assert_allclose(bU, g["bU"], atol=1e-15)
    C = np.eye(1)
    for case in g["cases"]:
        a = {1: np.array([case["alpha"]])}
        lb, ub, (A_lo, A_up, d_lo, d_up) = O.final_bounds(net, lo, hi, C, pre, a, a)
        assert abs(A_lo[0, 0] - case["A_lo"]) < 1e-15
        assert abs(d_lo[0] - case["d_lo"]) < 1e-15
        assert abs(lb[0] - case["lb"]) < 1e-15
        assert abs(A_up[0, 0] - g["A_up"]) < 1e-15
        assert abs(d_up[0] - g["d_up"]) < 1e-15
        assert abs(ub[0] - g["ub"]) < 1e-15
    l_ibp, u_ibp = O.ibp_spec(net, lo, hi, C)
    assert abs(l_ibp[0] - g["ibp"][0]) < 1e-15 and abs(u_ibp[0] - g["ibp"][1]) < 1e-15
    # exact range from an independent routine
    mn, mx = BF.exact_range(net, lo, hi, C)
    assert abs(mn[0] - g["true_min"]) < 1e-9 and abs(mx[0] - g["true_max"]) < 1e-9


def test_e3_alpha_per_row_and_l1_concretisation():
    g = _load("e3_alpha_rows.json")
    net = _net_from(g)
    lo, hi = np.array(g["x_lo"]), np.array(g["x_hi"])
    pre = O.crown_bounds(net, lo, hi)
    # all alpha cases at once as three spec rows sharing C = [1]: alpha is per (row, neuron)
    al = np.array([c["alpha"] for c in g["alpha_cases"]])
    C = np.ones((al.shape[0], 1))
    lb, ub, (A_lo, A_up, d_lo, d_up) = O.final_bounds(net, lo, hi, C, pre, {1: al}, {1: al})
    np.testing.assert_allclose(lb, [c["lb"] for c in g["alpha_cases"]], atol=1e-15)
    np.testing.assert_allclose(ub, g["ub"], atol=1e-15)
    np.testing.assert_allclose(A_up[0], g["A_up"], atol=1e-15)
    np.testing.assert_allclose(d_up, g["d_up"], atol=1e-15)
    lb_ad, _, _ = O.final_bounds(net, lo, hi, np.ones((1, 1)), pre)
    assert abs(lb_ad[0] - g["adaptive_lb"]) < 1e-15
    mn, mx = BF.exact_range(net, lo, hi, np.ones((1, 1)))
    assert abs(mn[0] - g["true_min"]) < 1e-9 and abs(mx[0] - g["true_max"]) < 1e-9


# ---------------------------------------------------------------- closed forms
def test_single_linear_layer_closed_form():
    """One linear layer: bounds are exact, c.W.x0 + c.b -+ eps*||c.W||_1 (north_star; G1)."""
    rng = np.random.default_rng(1)
    W = rng.standard_normal((7, 13)).astype(np.float32)
    b = rng.standard_normal(7).astype(np.float32)
    net = Net(in_shape=(13,), nodes=[Node("linear", -1, W=W, b=b, shape=(7,))])
    x0 = rng.standard_normal(13)
    eps = 0.3
    C = rng.standard_normal((5, 7))
    lb, ub, _ = O.final_bounds(net, x0 - eps, x0 + eps, C, {})
    CW = C @ W.astype(np.float64)
    mid = CW @ x0 + C @ b.astype(np.float64)
    rad = eps * np.abs(CW).sum(axis=1)
    np.testing.assert_allclose(lb, mid - rad, rtol=1e-13, atol=1e-13)
    np.testing.assert_allclose(ub, mid + rad, rtol=1e-13, atol=1e-13)
    l2, u2 = O.ibp_spec(net, x0 - eps, x0 + eps, C)
    np.testing.assert_allclose(l2, mid - rad, rtol=1e-13, atol=1e-13)
    np.testing.assert_allclose(u2, mid + rad, rtol=1e-13, atol=1e-13)
    # the extreme corners attain the bounds
    Xc = O.adversarial_corners(CW, CW, x0 - eps, x0 + eps)
    Y = O.forward_batch(net, Xc) @ C.T
    np.testing.assert_allclose(np.diag(Y[:5]), lb, rtol=1e-12, atol=1e-12)
    np.testing.assert_allclose(np.diag(Y[5:]), ub, rtol=1e-12, atol=1e-12)


@pytest.mark.parametrize("shift,kind", [(1.0, "active"), (-1.0, "inactive")])
def test_all_stable_nets_are_exact(shift, kind):
    """All-active nets are affine => CROWN bounds are the exact affine range, independent of alpha;
    all-inactive nets are constant (north_star closed form)."""
    w = wl_mod.small_mlp([6, 9, 8, 4], seed=3, B=2, eps=0.2, bias_shift=shift, weight_scale=0.05)
    lo, hi = w.box()
    for p in range(w.B):
        res = O.run_property(w.net, lo[p], hi[p], w.C[p], [a[p] for a in w.alpha])
        for l, u in res["pre"].values():        # the premise: every neuron is stable
            assert np.all(l > 0) if kind == "active" else np.all(u < 0)
        Ws = [n.W.astype(np.float64) for n in w.net.nodes if n.op == "linear"]
        bs = [n.b.astype(np.float64) for n in w.net.nodes if n.op == "linear"]
        C = w.C[p].astype(np.float64)
        if kind == "active":
            M = Ws[2] @ Ws[1] @ Ws[0]
            v = Ws[2] @ (Ws[1] @ bs[0] + bs[1]) + bs[2]
        else:
            M = np.zeros((4, 6))
            v = Ws[2] @ np.zeros(8) + bs[2]
            # hidden layer 2 pre-activation is b2 (+shift) < 0 -> inactive too
        CM, Cv = C @ M, C @ v
        xc = 0.5 * (lo[p].astype(np.float64) + hi[p].astype(np.float64))
        xr = 0.5 * (hi[p].astype(np.float64) - lo[p].astype(np.float64))
        np.testing.assert_allclose(res["lb"], CM @ xc - np.abs(CM) @ xr + Cv, rtol=1e-11, atol=1e-11)
        np.testing.assert_allclose(res["ub"], CM @ xc + np.abs(CM) @ xr + Cv, rtol=1e-11, atol=1e-11)
        res2 = O.run_property(w.net, lo[p], hi[p], w.C[p], None)
        np.testing.assert_allclose(res2["lb"], res["lb"], rtol=1e-13, atol=1e-13)


def test_ibp_wplus_wminus_equals_centre_radius():
    """W+ l + W- u == W c - |W| r: the GPU kernel uses the right-hand form."""
    rng = np.random.default_rng(5)
    W = rng.standard_normal((11, 17)).astype(np.float32)
    b = rng.standard_normal(11).astype(np.float32)
    net = Net(in_shape=(17,), nodes=[Node("linear", -1, W=W, b=b, shape=(11,))])
    lo = rng.standard_normal(17)
    hi = lo + rng.random(17)
    l, u = O.ibp(net, lo, hi)[0]
    W64 = W.astype(np.float64)
    c, r = 0.5 * (lo + hi), 0.5 * (hi - lo)
    np.testing.assert_allclose(l, W64 @ c - np.abs(W64) @ r + b, rtol=1e-13, atol=1e-13)
    np.testing.assert_allclose(u, W64 @ c + np.abs(W64) @ r + b, rtol=1e-13, atol=1e-13)


def test_relax_coeffs_classes_and_geometry():
    l = np.array([-1.0, 0.0, 0.5, -2.0, -3.0, -1.0, 0.0])
    u = np.array([2.0, 1.0, 0.7, -0.5, 0.0, 1.0, 0.0])
    dU, bU, dL = O.relax_coeffs(l, u)
    # stable classes (G3): l>=0 active (incl. l=u=0), u<=0 inactive
    assert list(dU[[1, 2, 6]]) == [1, 1, 1] and list(dL[[1, 2, 6]]) == [1, 1, 1]
    assert list(dU[[3, 4]]) == [0, 0] and list(dL[[3, 4]]) == [0, 0]
    assert np.all(bU[[1, 2, 3, 4, 6]] == 0)
    # unstable: the upper line passes through (l,0) and (u,u) (u/(u-l) (x-l))
    for j in (0, 5):
        assert abs(dU[j] * l[j] + bU[j]) < 1e-15
        assert abs(dU[j] * u[j] + bU[j] - u[j]) < 1e-15
    # adaptive rule (G4): 1 iff u > -l strictly
    assert dL[0] == 1.0 and dL[5] == 0.0
    # alpha-mode: clipped to [0,1], only on unstable neurons
    _, _, dLa = O.relax_coeffs(l, u, alpha=np.array([1.7, 0.3, 0.3, 0.3, 0.3, -0.2, 0.4]))
    assert list(dLa) == [1.0, 1.0, 1.0, 0.0, 0.0, 0.0, 1.0]
    # relaxation really sandwiches ReLU on [l,u]
    xs = np.linspace(-1, 2, 301)
    assert np.all(dL[0] * xs <= np.maximum(xs, 0) + 1e-15)
    assert np.all(np.maximum(xs, 0) <= dU[0] * xs + bU[0] + 1e-15)


# ---------------------------------------------------------------- conv pins
def _dense_of_conv(W, stride, pad, in_shape):
    c_in, H, Wd = in_shape
    n_in = c_in * H * Wd
    cols = []
    for k in range(n_in):
        e = np.zeros(n_in); e[k] = 1.0
        cols.append(O.conv2d(e.reshape(in_shape), W, stride, pad).reshape(-1))
    return np.stack(cols, axis=1)       # [n_out, n_in]


def _dense_conv_by_definition(W, stride, pad, in_shape):
    """Toeplitz matrix written straight from the index definition (independent of O.conv2d)."""
    c_out, c_in, kh, kw = W.shape
    _, H, Wd = in_shape
    ho = (H + 2 * pad - kh) // stride + 1
    wo = (Wd + 2 * pad - kw) // stride + 1
    M = np.zeros((c_out * ho * wo, c_in * H * Wd))
    for o in range(c_out):
        for p in range(ho):
            for q in range(wo):
                for c in range(c_in):
                    for i in range(kh):
                        for j in range(kw):
                            y, x = p * stride + i - pad, q * stride + j - pad
                            if 0 <= y < H and 0 <= x < Wd:
                                M[(o * ho + p) * wo + q, (c * H + y) * Wd + x] += W[o, c, i, j]
    return M


@pytest.mark.parametrize("stride,pad,k", [(1, 1, 3), (2, 1, 3), (2, 0, 1)])
def test_conv_matches_dense_toeplitz_and_adjoint(stride, pad, k):
    rng = np.random.default_rng(7)
    in_shape = (3, 6, 5)
    W = rng.standard_normal((4, 3, k, k)).astype(np.float32)
    M = _dense_conv_by_definition(W.astype(np.float64), stride, pad, in_shape)
    x = rng.standard_normal(in_shape)
    y = O.conv2d(x, W, stride, pad)
    np.testing.assert_allclose(y.reshape(-1), M @ x.reshape(-1), rtol=1e-12, atol=1e-12)
    A = rng.standard_normal((5,) + y.shape)
    At = O.conv2d_transpose(A, W, stride, pad, in_shape[1:])
    np.testing.assert_allclose(At.reshape(5, -1), A.reshape(5, -1) @ M, rtol=1e-12, atol=1e-12)
    # adjoint identity <A, conv(x)> = <conv^T(A), x>
    np.testing.assert_allclose(np.sum(A[0] * y), np.sum(At[0] * x), rtol=1e-12)


def test_conv_net_equals_dense_net_bounds():
    """A small conv+residual net and its dense (Toeplitz) twin get identical IBP and CROWN bounds."""
    rng = np.random.Generator(np.random.PCG64(11))
    net = wl_mod.resnet(rng, in_shape=(2, 6, 6), stem=3, blocks=((3, 1), (4, 2)), fc=6, n_classes=4)
    # dense twin: every conv -> linear with its Toeplitz matrix, shapes flattened
    dn = Net(in_shape=(net.n_in,))
    for n in net.nodes:
        if n.op == "conv":
            ishape = net.shape_of(n.in0)
            M = _dense_conv_by_definition(n.W.astype(np.float64), n.stride, n.pad, ishape)
            hw = n.shape[1] * n.shape[2]
            dn.nodes.append(Node("linear", n.in0, W=M, b=np.repeat(n.b.astype(np.float64), hw),
                                 shape=(n.size,)))
        elif n.op == "linear":
            dn.nodes.append(Node("linear", n.in0, W=n.W, b=n.b, shape=n.shape))
        else:
            dn.nodes.append(Node(n.op, n.in0, n.in1, shape=(n.size,)))
    x0 = rng.random(net.n_in)
    lo, hi = x0 - 0.05, x0 + 0.05
    C = rng.standard_normal((3, 4))
    for inter in ("ibp", "crown"):
        pa = O.crown_bounds(net, lo, hi, inter)
        pb = O.crown_bounds(dn, lo, hi, inter)
        for i in net.relu_ids():
            np.testing.assert_allclose(pa[i][0], pb[i][0], rtol=1e-10, atol=1e-10)
            np.testing.assert_allclose(pa[i][1], pb[i][1], rtol=1e-10, atol=1e-10)
        al = {i: rng.random((3, net.nodes[i].size)) for i in net.relu_ids()}
        la, ua, _ = O.final_bounds(net, lo, hi, C, pa, al, al)
        lb, ub, _ = O.final_bounds(dn, lo, hi, C, pb, al, al)
        np.testing.assert_allclose(la, lb, rtol=1e-10, atol=1e-10)
        np.testing.assert_allclose(ua, ub, rtol=1e-10, atol=1e-10)
        # forward agrees too (the sample check relies on it), and with workloads.label_forward
        np.testing.assert_allclose(O.forward(net, x0)[-1], O.forward(dn, x0)[-1], rtol=1e-11, atol=1e-11)
        np.testing.assert_allclose(O.forward(net, x0)[-1], wl_mod.label_forward(net, x0), rtol=1e-12, atol=1e-12)


# ---------------------------------------------------------------- soundness / exact range
@pytest.mark.parametrize("seed", [0, 1, 2])
def test_bruteforce_sandwich_small_mlp(seed):
    """lb_CROWN <= exact_min <= sampled_min and symmetric for ub, on nets with <= 10 neurons (O7)."""
    w = wl_mod.small_mlp([2, 4, 4, 3], seed=seed, B=1, eps=0.8, S=3)
    lo, hi = w.box()
    for inter in ("crown", "ibp"):
        pre = O.crown_bounds(w.net, lo[0], hi[0], inter)
        al = {i: w.alpha[j][0] for j, i in enumerate(w.net.relu_ids())}
        for a in (None, al):
            lb, ub, _ = O.final_bounds(w.net, lo[0], hi[0], w.C[0], pre, a, a)
            mn, mx = BF.exact_range(w.net, lo[0], hi[0], w.C[0])
            X = wl_mod.sample_points(0, lo[0], hi[0], 2000, 500)
            Y = O.forward_batch(w.net, X) @ w.C[0].astype(np.float64).T
            assert np.all(lb <= mn + 1e-9), (lb, mn)
            assert np.all(mn <= Y.min(axis=0) + 1e-9)
            assert np.all(ub >= mx - 1e-9), (ub, mx)
            assert np.all(mx >= Y.max(axis=0) - 1e-9)
    # intermediate CROWN bounds enclose the exact pre-activation range of layer 2
    sub = Net(in_shape=w.net.in_shape, nodes=w.net.nodes[:3])
    mn, mx = BF.exact_range(sub, lo[0], hi[0], np.eye(4))
    pre = O.crown_bounds(w.net, lo[0], hi[0], "crown")
    assert np.all(pre[3][0] <= mn + 1e-9) and np.all(pre[3][1] >= mx - 1e-9)


@pytest.mark.parametrize("cfg,scale", [(1, 1), (2, 4), (5, 4)])
def test_sample_containment_10k(cfg, scale):
    """lower <= C.f(x) <= upper for 10^4 seeded samples incl. corners and adversarial corners (O6)."""
    w = wl_mod.make(cfg, scale=scale, B=2 if cfg != 1 else None)
    lo, hi = w.box()
    res = O.run_workload(w)
    for p, r in enumerate(res):
        assert np.all(r["lb"] <= r["ub"])
        for i, (l, u) in r["pre"].items():
            assert np.all(l <= u)
        X = wl_mod.sample_points(cfg, lo[p], hi[p], 8192, 1792)
        A_lo, A_up, _, _ = r["lin"]
        X = np.concatenate([X, O.adversarial_corners(A_lo, A_up, lo[p], hi[p])], axis=0)
        ok, v_lo, v_hi, vmin, vmax = O.sample_check(w.net, w.C[p], X, r["lb"], r["ub"])
        assert ok, (v_lo, v_hi)
        # pre-activation bounds contain the sampled pre-activations too
        Xs = X[:512]
        for x in Xs[:32]:
            vals = O.forward(w.net, x)
            for i, (l, u) in r["pre"].items():
                z = vals[w.net.nodes[i].in0].reshape(-1)
                assert np.all(z >= l - 1e-9 * (1 + np.abs(z))) and np.all(z <= u + 1e-9 * (1 + np.abs(z)))


# ---------------------------------------------------------------- invariants
def test_eps_monotonicity_ibp_and_forced_crown():
    w = wl_mod.small_mlp([8, 16, 16, 5], seed=9, B=1, eps=0.05)
    x0 = w.x0[0].astype(np.float64)
    prev = None
    pre_fix = O.crown_bounds(w.net, x0 - 0.2, x0 + 0.2)          # forced (l,u), valid for all eps<=0.2
    al = {i: w.alpha[j][0] for j, i in enumerate(w.net.relu_ids())}
    for eps in (0.01, 0.05, 0.1, 0.2):
        l, u = O.ibp_spec(w.net, x0 - eps, x0 + eps, w.C[0])
        lb, ub, _ = O.final_bounds(w.net, x0 - eps, x0 + eps, w.C[0], pre_fix, al, al)
        if prev is not None:
            assert np.all(l <= prev[0] + 1e-12) and np.all(u >= prev[1] - 1e-12)
            assert np.all(lb <= prev[2] + 1e-12) and np.all(ub >= prev[3] - 1e-12)
        prev = (l, u, lb, ub)


def test_sign_symmetry_and_row_independence():
    w = wl_mod.small_mlp([8, 16, 16, 5], seed=4, B=1, eps=0.1, S=6)
    lo, hi = w.box()
    pre = O.crown_bounds(w.net, lo[0], hi[0])
    rng = np.random.default_rng(0)
    ids = w.net.relu_ids()
    a1 = {i: rng.random((6, w.net.nodes[i].size)) for i in ids}
    a2 = {i: rng.random((6, w.net.nodes[i].size)) for i in ids}
    C = w.C[0].astype(np.float64)
    lb, ub, _ = O.final_bounds(w.net, lo[0], hi[0], C, pre, a1, a2)
    lbn, ubn, _ = O.final_bounds(w.net, lo[0], hi[0], -C, pre, a2, a1)
    np.testing.assert_allclose(lbn, -ub, rtol=0, atol=1e-13)
    np.testing.assert_allclose(ubn, -lb, rtol=0, atol=1e-13)
    # a row's result does not depend on which other rows are in the chunk
    sel = [4, 1]
    lbs, ubs, _ = O.final_bounds(w.net, lo[0], hi[0], C[sel], pre,
                                 {i: a1[i][sel] for i in ids}, {i: a2[i][sel] for i in ids})
    np.testing.assert_allclose(lbs, lb[sel], rtol=0, atol=1e-13)
    np.testing.assert_allclose(ubs, ub[sel], rtol=0, atol=1e-13)
    # row-sampled intermediate bounds == full
    full = O.crown_bounds(w.net, lo[0], hi[0])
    part = O.crown_bounds(w.net, lo[0], hi[0], rows={3: np.array([2, 7, 11])})
    np.testing.assert_allclose(part[3][0][[2, 7, 11]], full[3][0][[2, 7, 11]], rtol=0, atol=1e-13)
    assert np.isnan(part[3][0][0])


def test_crown_tighter_than_ibp_on_relu_free_chain_and_first_layer_equal():
    w = wl_mod.small_mlp([5, 7, 6, 3], seed=12, B=1, eps=0.3)
    lo, hi = w.box()
    ib = O.ibp(w.net, lo[0], hi[0])
    pre = O.crown_bounds(w.net, lo[0], hi[0])
    # first layer: CROWN == IBP (single linear layer exact)
    A_lo, A_up, d_lo, d_up = O.backward(w.net, 0, np.eye(7), {})
    l1, u1 = O.concretize(A_lo, A_up, d_lo, d_up, lo[0], hi[0])
    np.testing.assert_allclose(l1, ib[0][0], rtol=1e-13, atol=1e-13)
    np.testing.assert_allclose(u1, ib[0][1], rtol=1e-13, atol=1e-13)
    np.testing.assert_allclose(pre[1][0], ib[0][0], rtol=0, atol=0)


def test_margin_spec_and_workload_recipe():
    C = wl_mod.margin_spec(5, 2)
    assert C.shape == (4, 5) and np.all(C[:, 2] == 1) and list(np.argmin(C, axis=1)) == [0, 1, 3, 4]
    w = wl_mod.make(1)
    assert w.net.nodes[0].W.shape == (256, 784) and w.C.shape == (1, 9, 10) and w.alpha[0].shape == (1, 9, 256)
    assert abs(float(w.net.nodes[0].W.std()) - np.sqrt(2 / 784)) < 2e-3          # He-normal
    assert abs(float(np.concatenate([n.b for n in w.net.nodes if n.b is not None]).std()) - 0.1) < 0.02
    y = int(np.argmax(O.forward(w.net, w.x0[0])[-1]))
    assert y == w.labels[0]
    w2 = wl_mod.make(1)
    assert np.array_equal(w.net.nodes[2].W, w2.net.nodes[2].W) and np.array_equal(w.x0, w2.x0)
    w5 = wl_mod.make(5, scale=4, B=1)
    assert len(w5.net.relu_ids()) == 10


def test_residual_dag_affine_exactness():
    """Residual fork pin: on a conv/add/flatten/linear DAG whose ReLUs are all stably active the net
    is affine, so CROWN must return the exact affine range.  The affine map is recovered
    independently by probing `forward` at basis points (forward itself is pinned against the dense
    twin and workloads.label_forward above)."""
    rng = np.random.Generator(np.random.PCG64(21))
    net = wl_mod.resnet(rng, in_shape=(2, 4, 4), stem=3, blocks=((3, 1), (4, 2)), fc=5, n_classes=3)
    for n in net.nodes:                       # small weights, bias +1 => every pre-activation > 0
        if n.W is not None:
            n.W = (n.W * 0.05).astype(np.float32)
            n.b = (n.b + (1.0 if n is not net.nodes[-1] else 0.0)).astype(np.float32)
    n0 = net.n_in
    x0 = rng.random(n0)
    lo, hi = x0 - 0.1, x0 + 0.1
    f0 = O.forward(net, x0)[-1]
    M = np.stack([O.forward(net, x0 + np.eye(n0)[k] * 0.05)[-1] - f0 for k in range(n0)], axis=1) / 0.05
    v = f0 - M @ x0
    C = rng.standard_normal((4, 3))
    for inter in ("crown", "ibp"):
        pre = O.crown_bounds(net, lo, hi, inter)
        for l, u in pre.values():
            assert np.all(l > 0)
        lb, ub, (A_lo, A_up, d_lo, d_up) = O.final_bounds(net, lo, hi, C, pre)
        CM = C @ M
        np.testing.assert_allclose(A_lo, CM, rtol=1e-9, atol=1e-10)
        np.testing.assert_allclose(A_up, CM, rtol=1e-9, atol=1e-10)
        np.testing.assert_allclose(d_lo, C @ v, rtol=1e-9, atol=1e-10)
        np.testing.assert_allclose(lb, CM @ x0 - 0.1 * np.abs(CM).sum(1) + C @ v, rtol=1e-9, atol=1e-10)
        np.testing.assert_allclose(ub, CM @ x0 + 0.1 * np.abs(CM).sum(1) + C @ v, rtol=1e-9, atol=1e-10)
    # interval arithmetic through the fork: IBP of the Add node is the sum of its operands' intervals
    ib = O.ibp(net, lo, hi)
    for i, n in enumerate(net.nodes):
        if n.op == "add":
            np.testing.assert_allclose(ib[i][0], ib[n.in0][0] + ib[n.in1][0], rtol=0, atol=0)
            X = wl_mod.sample_points(0, lo, hi, 64, 64)
            for x in X:
                z = O.forward(net, x)[i]
                assert np.all(z >= ib[i][0] - 1e-12) and np.all(z <= ib[i][1] + 1e-12)


# ------------------------------------------------------------------------------------------ verdict and box helpers
def test_verified_is_strict_and_fails_closed():
    """a property is proved iff EVERY margin row is strictly positive; an undefined (NaN) bound
    proves nothing."""
    assert O.verified(np.array([0.5, 1e-30, 3.0])) is True
    assert O.verified(np.array([0.5, 0.0, 3.0])) is False          # strict: lb = 0 is not a proof
    assert O.verified(np.array([0.5, -1e-30, 3.0])) is False
    assert O.verified(np.array([np.nan, 1.0])) is False
    assert O.verified(np.array([np.inf])) is True


def test_box_is_x0_plus_minus_the_float32_radius():
    """_box(x0, eps): corners are float32(x0 -+ float32(eps)) with the subtraction done in float64, the same
    rounding as workloads.Workload.box (hand values: 0.5 -+ 0.25 exactly; 0.1 is not a float32 number)."""
    x0 = np.array([[0.5, -1.0]], dtype=np.float32)
    lo, hi = O._box(x0, 0.25)
    assert lo.dtype == np.float32 and hi.dtype == np.float32
    assert lo.tolist() == [[0.25, -1.25]] and hi.tolist() == [[0.75, -0.75]]
    lo, hi = O._box(x0, 0.1)
    e32 = 0.100000001490116119384765625                              # float32(0.1), written out
    assert lo[0, 0] == np.float32(0.5 - e32) and hi[0, 1] == np.float32(-1.0 + e32)
    wl = wl_mod.small_mlp([4, 4, 2], 0, eps=0.1)
    l2, h2 = O._box(wl.x0, 0.1)
    assert np.array_equal(l2, wl.box()[0]) and np.array_equal(h2, wl.box()[1])
