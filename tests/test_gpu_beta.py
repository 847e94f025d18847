"""GPU parity of the beta-CROWN bounds of batched BaB sub-domains (NEXT-2) through the C-ABI
(crown_backward_split / crown_beta_grad / crown_beta_ascent) against oracle/beta_oracle.py on the same seeded inputs.

A batch entry is a sub-domain: a property's box, its parent's intermediate bounds and a split vector per ReLU.
Protocol as in tests/test_gpu_alpha.py: forced bounds (the oracle starts from the GPU's (l, u) upcast to float64), element-
wise tolerance 1e-5 + 1e-4 |ref| for A, d, lb, ub; gradients compared on rows without a near-zero A entry (flagged rows
are counted and bounded); the ascent by the forced protocol (oracle bound at the GPU's final (alpha, beta) == the GPU's
last iterate) plus soundness on sampled points of the sub-domain."""
import json
import os

import numpy as np
import pytest

import workloads as W
from oracle import beta_oracle as BO
from oracle import crown_oracle as O
from workloads import Net, Node

pytestmark = pytest.mark.gpu

ATOL, RTOL = 1e-5, 1e-4
GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _ctx(net, B, S, **kw):
    from paper_2606_09377_b200 import CrownContext
    return CrownContext(net, B, S, **kw)


def _np(t):
    return t.detach().cpu().numpy()


def _close(gpu, ref, what, atol=ATOL, rtol=RTOL):
    gpu = np.asarray(gpu, np.float64); ref = np.asarray(ref, np.float64)
    err = np.abs(gpu - ref) - (atol + rtol * np.abs(ref))
    assert np.all(err <= 0), f"{what}: worst excess {err.max():.3e} at {np.unravel_index(err.argmax(), err.shape)}"


def _subdomains(wl, ctx, reps, n_split, seed, beta_scale=1.0, balanced=False):
    """reps sub-domains per property of wl: same box and (GPU-computed) intermediate bounds, random splits on
    n_split unstable neurons each.  Returns the stacked batch (numpy) and the per-entry oracle inputs."""
    lo, hi = wl.box()
    res = ctx.run(lo, hi, wl.C, None, wl.intermediate)
    rng = np.random.default_rng(seed)
    relus = wl.net.relu_ids()
    idx = np.repeat(np.arange(wl.B), reps)
    Bs = len(idx)
    pre = {i: (_np(res["pre"][i][0])[idx], _np(res["pre"][i][1])[idx]) for i in relus}
    split = {i: np.zeros((Bs, wl.net.nodes[i].size), np.int8) for i in relus}
    for e in range(Bs):
        cand = [(i, j) for i in relus for j in np.nonzero((pre[i][0][e] < 0) & (pre[i][1][e] > 0))[0]]
        if balanced:      # neurons whose sign really varies over the box (so that the sub-domain can be sampled)
            X = lo[idx[e]][None, :] + rng.random((400, lo.shape[1])) * (hi[idx[e]] - lo[idx[e]])[None, :]
            Z = {i: np.stack([O.forward(wl.net, x)[wl.net.nodes[i].in0].reshape(-1) for x in X]) for i in relus}
            cand = [(i, j) for (i, j) in cand if 0.2 < np.mean(Z[i][:, j] > 0) < 0.8]
        for k in rng.permutation(len(cand))[:n_split]:
            i, j = cand[k]
            split[i][e, j] = 1 if rng.random() < 0.5 else -1
    S = wl.S
    mk = lambda a, b: {i: rng.uniform(a, b, (Bs, S, wl.net.nodes[i].size)).astype(np.float32) for i in relus}
    al, au = mk(0.02, 0.98), mk(0.02, 0.98)
    bl, bu = mk(-0.2 * beta_scale, beta_scale), mk(-0.2 * beta_scale, beta_scale)     # some below 0: clipped inside
    return dict(idx=idx, B=Bs, lo=lo[idx], hi=hi[idx], C=wl.C[idx], pre=pre, split=split, al=al, au=au, bl=bl, bu=bu)


def _entry(sd, e):
    f64 = lambda d: {i: v[e].astype(np.float64) for i, v in d.items()}
    pre = {i: (l[e].astype(np.float64), u[e].astype(np.float64)) for i, (l, u) in sd["pre"].items()}
    return pre, {i: v[e] for i, v in sd["split"].items()}, f64(sd["al"]), f64(sd["au"]), f64(sd["bl"]), f64(sd["bu"])


def _torch_pre(ctx, sd):
    return {i: (ctx._dev(l), ctx._dev(u)) for i, (l, u) in sd["pre"].items()}


def test_e4_hand_worked_example_on_the_gpu():
    with open(os.path.join(GOLD, "e4_beta_split.json")) as f:
        g = json.load(f)
    net = Net(in_shape=(1,))
    net.nodes.append(Node("linear", -1, W=np.array(g["W1"], np.float32), b=np.array(g["b1"], np.float32), shape=(2,)))
    net.nodes.append(Node("relu", 0, shape=(2,)))
    net.nodes.append(Node("linear", 1, W=np.array(g["W2"], np.float32), b=np.array(g["b2"], np.float32), shape=(1,)))
    cases = g["lower_cases"]
    B = len(cases)
    ctx = _ctx(net, B, 1)
    lo = np.tile(np.array(g["x_lo"], np.float32), (B, 1)); hi = np.tile(np.array(g["x_hi"], np.float32), (B, 1))
    C = np.ones((B, 1, 1), np.float32)
    pre = {1: (np.tile(np.float32([-1, -1]), (B, 1)), np.tile(np.float32([1, 1]), (B, 1)))}
    split = {1: np.tile(np.int8(g["split"]), (B, 1))}
    beta = {1: np.float32([[[c["beta"], 7.0]] for c in cases])}
    alpha = {1: np.float32([[[c["alpha"], c["alpha"]]] for c in cases])}
    out = ctx.beta_grad(pre, split, C, alpha, alpha, beta, beta, (lo, hi))
    np.testing.assert_allclose(_np(out["lb"])[:, 0], [c["lb"] for c in cases], atol=1e-6)
    np.testing.assert_allclose(_np(out["gb_lo"][1])[:, 0, 0], [c["g_beta"] for c in cases], atol=1e-6)
    assert np.all(_np(out["gb_lo"][1])[:, 0, 1] == 0)
    a = g["ascent"]
    z = {1: np.zeros((1, 1, 2), np.float32)}
    r = ctx.beta_ascent({1: (pre[1][0][:1], pre[1][1][:1])}, {1: split[1][:1]}, C[:1], z, {1: z[1].copy()}, z, {1: z[1].copy()},
                        (lo[:1], hi[:1]), a["eta_alpha"], a["eta_beta"], a["iters"], a["mode"])
    assert float(_np(r["lb_best"])[0, 0]) == pytest.approx(a["lb_hist"][-1], abs=1e-6)
    assert float(_np(r["beta_lo"][1])[0, 0, 0]) == pytest.approx(a["beta_final"], abs=1e-6)
    ctx.close()


@pytest.mark.parametrize("scheme", [0, 2])
def test_backward_split_matches_oracle(scheme):
    """A, d, lb, ub of a batch of sub-domains vs oracle/beta_oracle.py, tensor-core and CUDA-core contraction"""
    wl = W.small_mlp([16, 160, 144, 5], seed=11, B=2, eps=0.05, S=4)
    ctx = _ctx(wl.net, 8, wl.S, mma_scheme=scheme)
    sd = _subdomains(wl, ctx, reps=4, n_split=10, seed=1)
    last = len(wl.net.nodes) - 1
    out = ctx.backward_split(sd["B"], last, _torch_pre(ctx, sd), sd["split"], sd["C"], alpha_lo=sd["al"], alpha_up=sd["au"],
                             beta_lo=sd["bl"], beta_up=sd["bu"], box=(sd["lo"], sd["hi"]))
    nob = ctx.backward_split(sd["B"], last, _torch_pre(ctx, sd), sd["split"], sd["C"], alpha_lo=sd["al"], alpha_up=sd["au"],
                             box=(sd["lo"], sd["hi"]))
    A, d, lb, ub = _np(out["A"]), _np(out["d"]), _np(out["lb"]), _np(out["ub"])
    moved = 0
    for e in range(sd["B"]):
        pre, sp, al, au, bl, bu = _entry(sd, e)
        assert sum(int(np.count_nonzero(v)) for v in sp.values()) >= 5
        A_lo, A_up, d_lo, d_up = BO.backward(wl.net, last, sd["C"][e], pre, sp, bl, bu, al, au)
        olb, oub = O.concretize(A_lo, A_up, d_lo, d_up, sd["lo"][e], sd["hi"][e])
        _close(A[0, e], A_lo, f"entry {e} A_lo")          # element by element, 1e-5 + 1e-4 |ref|
        _close(A[1, e], A_up, f"entry {e} A_up")
        _close(d[0, e], d_lo, f"entry {e} d_lo"); _close(d[1, e], d_up, f"entry {e} d_up")
        _close(lb[e], olb, f"entry {e} lb"); _close(ub[e], oub, f"entry {e} ub")
        # beta = NULL is beta = 0
        l0, u0 = BO.final_bounds(wl.net, sd["lo"][e], sd["hi"][e], sd["C"][e], pre, sp, None, None, al, au)
        _close(_np(nob["lb"])[e], l0, f"entry {e} lb at beta 0"); _close(_np(nob["ub"])[e], u0, f"entry {e} ub at beta 0")
        moved += int(np.any(np.abs(l0 - olb) > 1e-3 * (1 + np.abs(l0))))
    assert moved >= sd["B"] // 2, "beta did not change the bounds: the test does not exercise the split term"
    ctx.close()


def test_split_without_beta_equals_clamped_intervals():
    """crown_backward_split with beta = NULL == crown_backward on intervals clamped by the caller (bitwise: same kernels)"""
    import torch
    wl = W.make(2, B=3)
    ctx = _ctx(wl.net, 6, wl.S)
    sd = _subdomains(wl, ctx, reps=2, n_split=40, seed=2)
    last = len(wl.net.nodes) - 1
    a = ctx.backward_split(sd["B"], last, _torch_pre(ctx, sd), sd["split"], sd["C"], alpha_lo=sd["al"], alpha_up=sd["au"],
                           box=(sd["lo"], sd["hi"]))
    cl = {}
    for i, (l, u) in sd["pre"].items():
        s = sd["split"][i]
        cl[i] = (np.where(s > 0, np.maximum(l, 0), l).astype(np.float32), np.where(s < 0, np.minimum(u, 0), u).astype(np.float32))
    b = ctx.crown_backward(sd["B"], last, cl, sd["C"], alpha_lo=sd["al"], alpha_up=sd["au"], box=(sd["lo"], sd["hi"]))
    ctx.stream.synchronize()
    for k in ("A", "d", "lb", "ub"):
        assert torch.equal(a[k], b[k]), k
    ctx.close()


def _risky_rows(net, C, pre, sp, bl, bu, al, au):
    trace = {}
    A_lo, A_up, _, _ = BO.backward(net, len(net.nodes) - 1, C, pre, sp, bl, bu, al, au, trace=trace)
    risky = np.zeros((2, C.shape[0]), bool)
    for pair in [(A_lo, A_up)] + [trace[i] for i in trace]:
        for br in (0, 1):
            A = np.abs(pair[br])
            scale = A.max(axis=1, keepdims=True) + 1e-300
            risky[br] |= np.any((A < 1e-5 * scale) & (A > 0), axis=1)
    return risky


@pytest.mark.parametrize("which", ["small", "cfg2"])
def test_beta_gradient_matches_oracle(which):
    if which == "small":
        wl = W.small_mlp([16, 160, 144, 5], seed=12, B=2, eps=0.05, S=4)
        reps, n_split, bs = 3, 8, 1.0
    else:
        wl = W.make(2, B=2)
        reps, n_split, bs = 2, 30, 5.0
    ctx = _ctx(wl.net, wl.B * reps, wl.S)
    sd = _subdomains(wl, ctx, reps=reps, n_split=n_split, seed=3, beta_scale=bs)
    out = ctx.beta_grad(_torch_pre(ctx, sd), sd["split"], sd["C"], sd["al"], sd["au"], sd["bl"], sd["bu"], (sd["lo"], sd["hi"]))
    flagged = total = 0
    for e in range(sd["B"]):
        pre, sp, al, au, bl, bu = _entry(sd, e)
        C = sd["C"][e].astype(np.float64)
        lb, ub, ga_lo, ga_up, gb_lo, gb_up = BO.bound_and_gradient(wl.net, sd["lo"][e], sd["hi"][e], C, pre, sp, bl, bu, al, au)
        _close(_np(out["lb"])[e], lb, f"entry {e} lb"); _close(_np(out["ub"])[e], ub, f"entry {e} ub")
        risky = _risky_rows(wl.net, C, pre, sp, bl, bu, al, au)
        for br, pairs in enumerate((((out["g_lo"], ga_lo), (out["gb_lo"], gb_lo)), ((out["g_up"], ga_up), (out["gb_up"], gb_up)))):
            for gg, go in pairs:
                for i in wl.net.relu_ids():
                    G = _np(gg[i])[e]
                    sc = np.abs(go[i]).max(axis=1, keepdims=True) + 1e-30
                    for s in range(wl.S):
                        total += 1
                        if risky[br, s]:
                            flagged += 1
                            continue
                        err = np.abs(G[s] - go[i][s]) - (ATOL * max(1.0, sc[s, 0]) + RTOL * np.abs(go[i][s]))
                        assert np.all(err <= 0), f"entry {e} relu {i} branch {br} row {s}: worst excess {err.max():.3e}"
        for i in wl.net.relu_ids():      # beta gradient lives on the split set only
            assert np.all(_np(out["gb_lo"][i])[e][:, sp[i] == 0] == 0) and np.all(_np(out["gb_up"][i])[e][:, sp[i] == 0] == 0)
            assert np.any(_np(out["gb_lo"][i])[e][:, sp[i] != 0] != 0) or not np.any(sp[i] != 0)
    assert flagged <= 0.5 * total, f"{flagged} of {total} checks skipped as risky"
    ctx.close()


@pytest.mark.parametrize("mode,ea,eb", [("sign", 0.05, 0.05), ("plain", 0.02, 0.02)])
def test_beta_ascent_forced_parity_and_soundness(mode, ea, eb):
    wl = W.small_mlp([8, 160, 136, 4], seed=13, B=2, eps=0.3, S=3)
    reps = 3
    ctx = _ctx(wl.net, wl.B * reps, wl.S)
    sd = _subdomains(wl, ctx, reps=reps, n_split=3, seed=4, balanced=True)
    iters = 15
    zero = {i: np.zeros_like(v) for i, v in sd["bl"].items()}
    out = ctx.beta_ascent(_torch_pre(ctx, sd), sd["split"], sd["C"], sd["al"], sd["au"], zero, {i: v.copy() for i, v in zero.items()},
                          (sd["lo"], sd["hi"]), ea, eb, iters, mode, 0.97)
    start = ctx.beta_grad(_torch_pre(ctx, sd), sd["split"], sd["C"], sd["al"], sd["au"], zero, zero, (sd["lo"], sd["hi"]))
    lb0, ub0 = _np(start["lb"]), _np(start["ub"])
    lbb, ubb, lbl, ubl = (_np(out[k]) for k in ("lb_best", "ub_best", "lb_last", "ub_last"))
    assert np.all(lbb >= lb0) and np.all(ubb <= ub0) and np.all(lbb >= lbl) and np.all(ubb <= ubl)
    assert np.mean(lbb > lb0 + 1e-4 * np.abs(lb0)) > 0.5, "ascent did not tighten most lower bounds"
    moved = 0
    checked = 0
    for e in range(sd["B"]):
        pre, sp, _, _, _, _ = _entry(sd, e)
        g = lambda d: {i: _np(v)[e].astype(np.float64) for i, v in d.items()}
        al, au, bl, bu = g(out["alpha_lo"]), g(out["alpha_up"]), g(out["beta_lo"]), g(out["beta_up"])
        for i in bl:
            assert bl[i].min() >= 0 and bu[i].min() >= 0 and al[i].min() >= 0 and al[i].max() <= 1
            assert np.all(bl[i][:, sp[i] == 0] == 0) and np.all(bu[i][:, sp[i] == 0] == 0)
            moved += int(np.any(bl[i][:, sp[i] != 0] > 0))
        olb, oub = BO.final_bounds(wl.net, sd["lo"][e], sd["hi"][e], sd["C"][e], pre, sp, bl, bu, al, au)
        _close(lbl[e], olb, f"entry {e} lb at the optimised (alpha, beta)")
        _close(ubl[e], oub, f"entry {e} ub at the optimised (alpha, beta)")
        assert bool(_np(out["verified"])[e]) == O.verified(lbb[e].astype(np.float64))
        # free-running float64 ascent from the same start: trajectories may part at a kink, most rows must agree
        r = BO.joint_ascent(wl.net, sd["lo"][e], sd["hi"][e], sd["C"][e], pre, sp, {i: v[e] for i, v in zero.items()},
                            {i: v[e] for i, v in zero.items()}, {i: v[e] for i, v in sd["al"].items()},
                            {i: v[e] for i, v in sd["au"].items()}, ea, eb, iters, mode, 0.97)
        close = np.abs(lbb[e] - r["lb_best"]) <= 1e-3 * (1 + np.abs(r["lb_best"]))
        assert close.mean() >= 0.6, (lbb[e], r["lb_best"])
        # soundness on sampled points of the sub-domain (rejection sampling on the split constraints)
        rng = np.random.default_rng(100 + e)
        X = sd["lo"][e][None, :] + rng.random((6000, sd["lo"].shape[1])) * (sd["hi"][e] - sd["lo"][e])[None, :]
        keep = np.ones(len(X), bool)
        for i in sp:
            if not np.any(sp[i]):
                continue
            Z = np.stack([O.forward(wl.net, x)[wl.net.nodes[i].in0].reshape(-1) for x in X])
            keep &= ~np.any((sp[i][None, :] > 0) & (Z < 0), axis=1) & ~np.any((sp[i][None, :] < 0) & (Z > 0), axis=1)
        Xs = X[keep]
        if len(Xs) >= 10:
            checked += 1
            Y = O.forward_batch(wl.net, Xs) @ sd["C"][e].astype(np.float64).T
            tol = ATOL + RTOL * np.abs(Y)
            assert np.all(Y >= lbb[e][None, :] - tol) and np.all(Y <= ubb[e][None, :] + tol), f"entry {e}: sample outside"
    assert moved >= 1 and checked >= sd["B"] // 2
    ctx.close()


def test_beta_errors():
    import torch
    from paper_2606_09377_b200.binding import CrownError
    wl = W.small_mlp([8, 40, 4], seed=14, B=2, eps=0.2, S=2)
    ctx = _ctx(wl.net, 2, wl.S)
    sd = _subdomains(wl, ctx, reps=1, n_split=2, seed=5)
    t = lambda d: {i: ctx._dev(v) for i, v in d.items()}
    o = {k: torch.empty(2, wl.S, device=ctx.device) for k in ("lb_best", "ub_best", "lb_last", "ub_last")}
    o["verified"] = torch.empty(2, dtype=torch.uint8, device=ctx.device)
    pre = _torch_pre(ctx, sd)
    l = {i: v[0] for i, v in pre.items()}; u = {i: v[1] for i, v in pre.items()}
    bl = t(sd["bl"])
    with pytest.raises(CrownError):       # aliased beta tensors are refused by the ascent
        ctx.beta_ascent_device(l, u, ctx._split_dev(sd["split"]), ctx._dev(sd["C"]), t(sd["al"]), t(sd["au"]), bl, bl,
                               ctx._dev(sd["lo"]), ctx._dev(sd["hi"]), 0.1, 0.1, 1.0, 2, 1, o)
    ctx.close()


def test_branch_and_bound_loop_with_gpu_bounds_against_brute_force():
    """The batched sub-domain bounding inside an actual BaB loop (split, re-bound, repeat).  The loop itself
    (which neuron to split, the domain list) is host logic of the TEST; every bound comes from crown_beta_ascent on the
    whole frontier as ONE batch.  On nets small enough for brute force: every leaf's bound is sound against the exact minimum
    over that leaf, the global lower bound (min over the leaves, which cover the box) is sound at every depth, and a leaf is
    only ever declared verified when the exact minimum over it is positive.  (Tightness is not asserted: with a finite number
    of ascent steps from beta = 0 a child can start below its parent; weak duality is what must always hold.)"""
    from oracle import brute_force as BF
    n_leaves = []
    for seed in (51, 52, 53):
        wl = W.small_mlp([2, 6, 5, 2], seed=seed, B=1, eps=0.7, S=2)
        lo, hi = wl.box()
        net, C = wl.net, wl.C[0]
        exact_min, _ = BF.exact_range(net, lo[0], hi[0], C)
        relus = net.relu_ids()
        Bmax = 64
        ctx = _ctx(net, Bmax, wl.S)
        root = ctx.run(lo, hi, wl.C, None, wl.intermediate)
        pre0 = {i: (_np(root["pre"][i][0])[0], _np(root["pre"][i][1])[0]) for i in relus}
        frontier = [{i: np.zeros(net.nodes[i].size, np.int8) for i in relus}]      # split vectors of the open leaves
        glb_hist = []
        for depth in range(5):
            nb = len(frontier)
            assert nb <= Bmax
            rep = lambda v: np.repeat(v[None], nb, axis=0)
            pre = {i: (rep(pre0[i][0]), rep(pre0[i][1])) for i in relus}
            split = {i: np.stack([f[i] for f in frontier]) for i in relus}
            mk = lambda v: {i: np.full((nb, wl.S, net.nodes[i].size), v, np.float32) for i in relus}
            out = ctx.beta_ascent(pre, split, rep(C), mk(0.5), mk(0.5), mk(0.0), mk(0.0), (rep(lo[0]), rep(hi[0])),
                                  0.05, 0.1, 40, "sign", 0.97)
            lbb = _np(out["lb_best"]).astype(np.float64)
            ver = _np(out["verified"]).astype(bool)
            # soundness of every leaf bound against the exact minimum over that leaf (skip empty leaves)
            for e, f in enumerate(frontier):
                mn, _ = BF.exact_range(net, lo[0], hi[0], C, split=f)
                if np.all(np.isfinite(mn)):
                    assert np.all(lbb[e] <= mn + 1e-5 + 1e-4 * np.abs(mn)), (seed, depth, e, lbb[e], mn)
                    if ver[e]:
                        assert np.all(mn > 0)
            glb = lbb.min(axis=0)                      # a valid lower bound of the whole box: the leaves cover it
            assert np.all(glb <= exact_min + 1e-5 + 1e-4 * np.abs(exact_min))
            glb_hist.append(glb)
            # branch: every open leaf splits its unstable, unsplit neuron with the widest relaxation gap (-l u / (u - l))
            nxt = []
            for e, f in enumerate(frontier):
                best, score = None, 0.0
                for i in relus:
                    l, u = pre0[i]
                    gap = np.where((l < 0) & (u > 0) & (f[i] == 0), -l * u / np.maximum(u - l, 1e-30), 0.0)
                    j = int(np.argmax(gap))
                    if gap[j] > score:
                        best, score = (i, j), float(gap[j])
                if best is None or ver[e]:
                    nxt.append(f)                      # fully split or verified: stays a leaf
                    continue
                for sg in (1, -1):
                    c = {i: v.copy() for i, v in f.items()}
                    c[best[0]][best[1]] = sg
                    nxt.append(c)
            frontier = nxt
        n_leaves.append(len(frontier))
        ctx.close()
    assert max(n_leaves) >= 16            # the frontier really grew into a batch of sub-domains
