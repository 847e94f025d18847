"""GPU parity of the alpha optimisation (NEXT-1) through the C-ABI (crown_alpha_grad / crown_alpha_ascent)
against oracle/alpha_oracle.py on the same seeded inputs.

Protocol (extends reading G18): the gradient of a piecewise-linear bound is DISCONTINUOUS where an entry of A (at a
ReLU or at the input) changes sign; a (property, spec row) whose float64 run has such an entry within fp32 error of 0
is flagged and skipped (counted, bounded), every other row is compared element by element.  The ascent is compared by
the forced protocol: the oracle evaluates O5 at the GPU's final alpha (its bound must equal the GPU's last iterate),
best-so-far is monotone, alpha stays in [0,1], every sample stays inside the optimised bounds."""
import numpy as np
import pytest

import workloads as W
from oracle import alpha_oracle as AO
from oracle import crown_oracle as O

pytestmark = pytest.mark.gpu

ATOL, RTOL = 1e-5, 1e-4


def _ctx(net, B, S, **kw):
    from paper_2606_09377_b200 import CrownContext
    return CrownContext(net, B, S, **kw)


def _np(t):
    return t.detach().cpu().numpy()


def _close(gpu, ref, what, atol=ATOL, rtol=RTOL):
    gpu = np.asarray(gpu, np.float64); ref = np.asarray(ref, np.float64)
    err = np.abs(gpu - ref) - (atol + rtol * np.abs(ref))
    assert np.all(err <= 0), f"{what}: worst excess {err.max():.3e} at {np.unravel_index(err.argmax(), err.shape)}"


def _alphas(wl, seed):
    rng = np.random.default_rng(seed)
    al = {i: rng.uniform(0.02, 0.98, (wl.B, wl.S, wl.net.nodes[i].size)).astype(np.float32) for i in wl.net.relu_ids()}
    au = {i: rng.uniform(0.02, 0.98, (wl.B, wl.S, wl.net.nodes[i].size)).astype(np.float32) for i in wl.net.relu_ids()}
    return al, au


def _risky_rows(net, lo, hi, C, pre, al, au):
    """spec rows of one property whose A (at a ReLU or at the input) has an entry within fp32 error of a sign change"""
    trace = {}
    A_lo, A_up, _, _ = O.backward(net, len(net.nodes) - 1, C, pre, al, au, trace=trace)
    S = C.shape[0]
    risky = np.zeros((2, S), bool)
    mats = [(A_lo, A_up)] + [trace[i] for i in trace]
    for pair in mats:
        for br in (0, 1):
            A = np.abs(pair[br])
            scale = A.max(axis=1, keepdims=True) + 1e-300
            risky[br] |= np.any((A < 1e-5 * scale) & (A > 0), axis=1)
    return risky


def _check_gradient(wl, seed=0, max_flag_frac=0.5, **kw):
    lo, hi = wl.box()
    ctx = _ctx(wl.net, wl.B, wl.S, **kw)
    res = ctx.run(lo, hi, wl.C, None, wl.intermediate)
    al, au = _alphas(wl, seed)
    out = ctx.alpha_grad(res["pre"], wl.C, al, au, (lo, hi))
    flagged = total = 0
    for p in range(wl.B):
        forced = {i: (_np(l)[p].astype(np.float64), _np(u)[p].astype(np.float64)) for i, (l, u) in res["pre"].items()}
        alp = {i: a[p].astype(np.float64) for i, a in al.items()}
        aup = {i: a[p].astype(np.float64) for i, a in au.items()}
        lb, ub, g_lo, g_up, _ = AO.bound_and_gradient(wl.net, lo[p], hi[p], wl.C[p], forced, alp, aup)
        _close(_np(out["lb"])[p], lb, f"prop {p} lb")
        _close(_np(out["ub"])[p], ub, f"prop {p} ub")
        risky = _risky_rows(wl.net, lo[p], hi[p], wl.C[p].astype(np.float64), forced, alp, aup)
        for br, (gg, go) in enumerate(((out["g_lo"], g_lo), (out["g_up"], g_up))):
            for i in wl.net.relu_ids():
                G = _np(gg[i])[p]
                # the tolerance's absolute part is scaled to the row: a gradient entry is A^+ * G_in, a product of two
                # cancelling sums whose fp32 error is relative to the summands
                sc = np.abs(go[i]).max(axis=1, keepdims=True) + 1e-30
                for s in range(wl.S):
                    total += 1
                    if risky[br, s]:
                        flagged += 1
                        continue
                    err = np.abs(G[s] - go[i][s]) - (ATOL * max(1.0, sc[s, 0]) + RTOL * np.abs(go[i][s]))
                    assert np.all(err <= 0), f"prop {p} relu {i} branch {br} row {s}: worst excess {err.max():.3e}"
                # stable neurons: exactly zero
                l, u = forced[i]
                st = ~((l < 0) & (u > 0))
                assert np.all(G[:, st] == 0)
    assert flagged <= max_flag_frac * total, f"{flagged} of {total} (relu, row) checks skipped as risky"
    return ctx


def test_alpha_gradient_small_mlp():
    _check_gradient(W.small_mlp([6, 9, 7, 5, 3], seed=3, B=3, eps=0.2), mma_scheme=2)
    _check_gradient(W.small_mlp([6, 9, 7, 5, 3], seed=4, B=3, eps=0.2))


def test_alpha_gradient_cfg1_and_cfg2_subset():
    _check_gradient(W.make(1))
    _check_gradient(W.make(2, B=6), seed=1)


def test_alpha_gradient_residual_conv_net():
    _check_gradient(W.make(5, scale=4, B=2), seed=2)


def test_alpha_gradient_aliased_alpha():
    """alpha_lo and alpha_up may be the same tensor for the gradient call"""
    wl = W.make(2, B=3)
    lo, hi = wl.box()
    ctx = _ctx(wl.net, wl.B, wl.S)
    res = ctx.run(lo, hi, wl.C, None, wl.intermediate)
    al, _ = _alphas(wl, 5)
    o1 = ctx.alpha_grad(res["pre"], wl.C, al, al, (lo, hi))
    o2 = ctx.alpha_grad(res["pre"], wl.C, al, {i: a.copy() for i, a in al.items()}, (lo, hi))
    import torch
    for i in wl.net.relu_ids():
        assert torch.equal(o1["g_lo"][i], o2["g_lo"][i]) and torch.equal(o1["g_up"][i], o2["g_up"][i])


@pytest.mark.parametrize("mode,eta,decay", [("sign", 0.05, 0.98), ("plain", 0.02, 1.0)])
def test_alpha_ascent_forced_parity_and_soundness(mode, eta, decay):
    wl = W.make(2, B=4)
    lo, hi = wl.box()
    ctx = _ctx(wl.net, wl.B, wl.S)
    res = ctx.run(lo, hi, wl.C, None, wl.intermediate)
    al, au = _alphas(wl, 7)
    # partly outside [0,1]: the projection must bring them back
    al = {i: (a * 1.4 - 0.2).astype(np.float32) for i, a in al.items()}
    iters = 12
    out = ctx.alpha_ascent(res["pre"], wl.C, al, au, (lo, hi), eta, iters, mode, decay)
    start = ctx.alpha_grad(res["pre"], wl.C, al, au, (lo, hi))
    lb0, ub0 = _np(start["lb"]), _np(start["ub"])
    lbb, ubb, lbl, ubl = (_np(out[k]) for k in ("lb_best", "ub_best", "lb_last", "ub_last"))
    assert np.all(lbb >= lb0) and np.all(ubb <= ub0) and np.all(lbb >= lbl) and np.all(ubb <= ubl)
    assert np.mean(lbb > lb0 + 1e-4 * np.abs(lb0)) > 0.5, "ascent did not tighten most lower bounds"
    for a in list(out["alpha_lo"].values()) + list(out["alpha_up"].values()):
        assert float(a.min()) >= 0.0 and float(a.max()) <= 1.0
    for p in range(wl.B):
        forced = {i: (_np(l)[p].astype(np.float64), _np(u)[p].astype(np.float64)) for i, (l, u) in res["pre"].items()}
        alp = {i: _np(a)[p].astype(np.float64) for i, a in out["alpha_lo"].items()}
        aup = {i: _np(a)[p].astype(np.float64) for i, a in out["alpha_up"].items()}
        # forced protocol: O5 at the GPU's final alpha == the GPU's last iterate
        olb, oub, (A_lo, A_up, _, _) = O.final_bounds(wl.net, lo[p], hi[p], wl.C[p], forced, alp, aup)
        _close(lbl[p], olb, f"prop {p} lb at the optimised alpha")
        _close(ubl[p], oub, f"prop {p} ub at the optimised alpha")
        assert bool(_np(out["verified"])[p]) == O.verified(lbb[p].astype(np.float64))
        # free-running oracle ascent from the same start: same step rule, float64.  Trajectories may part at a kink;
        # the optimised bounds must still agree closely for most rows, and the GPU's must not be looser overall
        r = AO.alpha_ascent(wl.net, lo[p], hi[p], wl.C[p], forced, {i: a[p] for i, a in al.items()},
                            {i: a[p] for i, a in au.items()}, eta, iters, mode, decay)
        close = np.abs(lbb[p] - r["lb_best"]) <= 1e-3 * (1 + np.abs(r["lb_best"]))
        assert close.mean() >= 0.75, (lbb[p], r["lb_best"])
        # soundness of the optimised bounds on samples incl. the adversarial corners of the final linear bound
        X = np.concatenate([W.sample_points(2, lo[p], hi[p], 2048, 512), O.adversarial_corners(A_lo, A_up, lo[p], hi[p])])
        ok, vlo, vhi, _, _ = O.sample_check(wl.net, wl.C[p], X, lbb[p], ubb[p], slack_rel=RTOL, slack_abs=ATOL)
        assert ok, (vlo, vhi)


def test_alpha_ascent_zero_iterations_is_the_plain_bound_and_errors():
    from paper_2606_09377_b200.binding import CrownError
    wl = W.make(1)
    lo, hi = wl.box()
    ctx = _ctx(wl.net, wl.B, wl.S)
    res = ctx.run(lo, hi, wl.C, None, wl.intermediate)
    al, au = _alphas(wl, 9)
    out = ctx.alpha_ascent(res["pre"], wl.C, al, au, (lo, hi), 0.1, 0, "sign")
    ref = ctx.alpha_grad(res["pre"], wl.C, al, au, (lo, hi))
    import torch
    assert torch.equal(out["lb_best"], ref["lb"]) and torch.equal(out["ub_best"], ref["ub"])
    for i in wl.net.relu_ids():
        assert torch.equal(out["alpha_lo"][i].cpu(), torch.from_numpy(al[i]))
    # aliased alpha tensors are refused by the ascent (they are optimised separately)
    t = {i: ctx._dev(a) for i, a in al.items()}
    o = {k: torch.empty(wl.B, wl.S, device=ctx.device) for k in ("lb_best", "ub_best", "lb_last", "ub_last")}
    o["verified"] = torch.empty(wl.B, dtype=torch.uint8, device=ctx.device)
    l = {i: v[0] for i, v in res["pre"].items()}; u = {i: v[1] for i, v in res["pre"].items()}
    with pytest.raises(CrownError):
        ctx.alpha_ascent_device(l, u, ctx._dev(wl.C), t, t, ctx._dev(lo), ctx._dev(hi), 0.1, 1.0, 2, 1, o)
