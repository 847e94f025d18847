"""GPU parity (`-m gpu`) of every option and degenerate case of the boundary that the five BASELINE configs do not
reach: slope_rule 1 / 2, alpha_lo != alpha_up, alpha outside [0,1] (device clip), per-dimension boxes, all-stable
nets (closed form), neurons exactly on the relaxation discontinuities l = 0, u = 0, u = -l, verdicts (verified = 1,
NaN fails closed), skip connections from the network input and forks on a Linear output.
Tolerance |gpu - oracle| <= 1e-5 + 1e-4 |oracle| element by element (BASELINE.json north_star, reading G18)."""
import numpy as np
import pytest

import workloads as W
from oracle import crown_oracle as O

pytestmark = pytest.mark.gpu

ATOL, RTOL = 1e-5, 1e-4
RULES = {0: "adaptive", 1: "zero", 2: "one"}


def _ctx(net, B, S, **kw):
    from paper_2606_09377_b200 import CrownContext
    return CrownContext(net, B, S, **kw)


def _np64(t):
    return t.detach().cpu().numpy().astype(np.float64)


def _close(gpu, ref, what):
    gpu = np.asarray(gpu, np.float64)
    ref = np.asarray(ref, np.float64)
    err = np.abs(gpu - ref) - (ATOL + RTOL * np.abs(ref))
    assert np.all(err <= 0), f"{what}: worst excess {err.max():.3e} at {np.unravel_index(err.argmax(), err.shape)}"


def _forced(res, p):
    return {i: (_np64(l[p]), _np64(u[p])) for i, (l, u) in res["pre"].items()}


def _check_run(wl, lo, hi, alpha, rule_id=0, **kw):
    """crown_run vs the oracle with the GPU's earlier (l,u) forced (G18), every element of every layer."""
    ctx = _ctx(wl.net, wl.B, wl.S, slope_rule=rule_id, **kw)
    res = ctx.run(lo, hi, wl.C, alpha, wl.intermediate)
    rule = RULES[rule_id]
    for p in range(wl.B):
        forced = _forced(res, p)
        pre = O.crown_bounds(wl.net, lo[p], hi[p], wl.intermediate, rule=rule, forced=forced)
        for i in wl.net.relu_ids():
            _close(forced[i][0], pre[i][0], f"prop {p} relu {i} l")
            _close(forced[i][1], pre[i][1], f"prop {p} relu {i} u")
        al = None if alpha is None else {i: a[p] for i, a in zip(wl.net.relu_ids(), alpha)}
        olb, oub, _ = O.final_bounds(wl.net, lo[p], hi[p], wl.C[p], forced, al, al, rule=rule)
        _close(_np64(res["lb"][p]), olb, f"prop {p} lb")
        _close(_np64(res["ub"][p]), oub, f"prop {p} ub")
        assert bool(res["verified"][p].item()) == O.verified(_np64(res["lb"][p]))
    return ctx, res


# ------------------------------------------------------------------------------------------ slope rules
@pytest.mark.parametrize("rule_id", [1, 2])
@pytest.mark.parametrize("which", ["small", "cfg2"])
def test_fixed_slope_rules(rule_id, which):
    """slope_rule 1 (all-zero) and 2 (all-one) for the intermediate passes AND the final pass (no alpha)."""
    wl = W.small_mlp([6, 9, 7, 5, 3], seed=11, B=3, eps=0.2) if which == "small" else W.make(2, B=4)
    lo, hi = wl.box()
    _check_run(wl, lo, hi, None, rule_id)


# ------------------------------------------------------------------------------------------ alpha variants
def _final_pass_vs_oracle(wl, lo, hi, pre_dev, al_lo, al_up, ctx, rule="adaptive"):
    n_last = len(wl.net.nodes) - 1
    out = ctx.crown_backward(wl.B, n_last, pre_dev, Cmat=wl.C, alpha_lo=al_lo, alpha_up=al_up, box=(lo, hi), want_A=True)
    for p in range(wl.B):
        forced = {i: (_np64(l[p]), _np64(u[p])) for i, (l, u) in pre_dev.items()}
        a_lo = None if al_lo is None else {i: np.asarray(a[p]) for i, a in al_lo.items()}
        a_up = None if al_up is None else {i: np.asarray(a[p]) for i, a in al_up.items()}
        olb, oub, (A_lo, A_up, d_lo, d_up) = O.final_bounds(wl.net, lo[p], hi[p], wl.C[p], forced, a_lo, a_up, rule=rule)
        _close(_np64(out["lb"][p]), olb, f"prop {p} lb")
        _close(_np64(out["ub"][p]), oub, f"prop {p} ub")
        _close(_np64(out["A"][0, p]), A_lo, f"prop {p} A_lo")
        _close(_np64(out["A"][1, p]), A_up, f"prop {p} A_up")
        _close(_np64(out["d"][0, p]), d_lo, f"prop {p} d_lo")
        _close(_np64(out["d"][1, p]), d_up, f"prop {p} d_up")
    return out


@pytest.mark.parametrize("which", ["small", "cfg2"])
def test_alpha_lo_differs_from_alpha_up(which):
    """Separate slopes for the two branches: the `alU != alL` path of the relaxation kernel."""
    wl = W.small_mlp([6, 9, 7, 5, 3], seed=5, B=2, eps=0.15) if which == "small" else W.make(2, B=4)
    lo, hi = wl.box()
    ctx = _ctx(wl.net, wl.B, wl.S)
    res = ctx.run(lo, hi, wl.C, wl.alpha, wl.intermediate)
    rng = np.random.default_rng(77)
    al_lo = {i: a for i, a in zip(wl.net.relu_ids(), wl.alpha)}
    al_up = {i: rng.random(a.shape).astype(np.float32) for i, a in al_lo.items()}
    _final_pass_vs_oracle(wl, lo, hi, res["pre"], al_lo, al_up, ctx)


def test_alpha_outside_unit_interval_is_clipped():
    """alpha ~ U[-0.5, 1.5]: both sides clip to [0,1] (PAPER.md:70 lambda in [0,1])."""
    wl = W.make(2, B=4)
    lo, hi = wl.box()
    rng = np.random.default_rng(78)
    alpha = [(rng.random(a.shape) * 2.0 - 0.5).astype(np.float32) for a in wl.alpha]
    assert min(a.min() for a in alpha) < -0.4 and max(a.max() for a in alpha) > 1.4
    _check_run(wl, lo, hi, alpha)


# ------------------------------------------------------------------------------------------ boxes
@pytest.mark.parametrize("which", ["small", "cfg2"])
def test_per_dimension_box(which):
    """x_lo / x_hi that are not x0 +- eps: per-dimension radii incl. zero-width dimensions (general box, reading G1)."""
    wl = W.small_mlp([6, 9, 7, 5, 3], seed=9, B=3, eps=0.2) if which == "small" else W.make(2, B=4)
    rng = np.random.default_rng(79)
    rad = (rng.random(wl.x0.shape) * 0.05).astype(np.float32)
    rad[:, ::7] = 0.0                                           # some dimensions are fixed
    skew = (rng.random(wl.x0.shape) * 0.02).astype(np.float32)  # the box is not centred on x0
    lo = (wl.x0 - rad).astype(np.float32)
    hi = (wl.x0 + rad + skew).astype(np.float32)
    _check_run(wl, lo, hi, wl.alpha)


# ------------------------------------------------------------------------------------------ all-stable nets
@pytest.mark.parametrize("shift", [1.0, -1.0])
@pytest.mark.parametrize("widths", [[6, 9, 7, 3], [160, 192, 160, 12]])
def test_all_stable_nets_match_the_closed_form(shift, widths):
    """bias_shift = +1 with small weights: every neuron active, the net is affine and CROWN is exact
    (c.W_eff.x0 + c.b_eff -+ eps ||c.W_eff||_1); bias_shift = -1: every neuron inactive, f = b_L. Independent of alpha."""
    wl = W.small_mlp(widths, seed=21, B=2, eps=0.1, bias_shift=shift, weight_scale=0.05)
    lo, hi = wl.box()
    _, res = _check_run(wl, lo, hi, wl.alpha)
    lin = [n for n in wl.net.nodes if n.op == "linear"]
    for p in range(wl.B):
        xc, xr = 0.5 * (lo[p].astype(np.float64) + hi[p]), 0.5 * (hi[p].astype(np.float64) - lo[p])
        if shift > 0:
            Weff, beff = np.eye(wl.net.n_in), np.zeros(wl.net.n_in)
            for n in lin:
                Weff, beff = n.W.astype(np.float64) @ Weff, n.W.astype(np.float64) @ beff + n.b
        else:
            Weff, beff = np.zeros((wl.net.n_out, wl.net.n_in)), lin[-1].b.astype(np.float64)
        CW, Cb = wl.C[p].astype(np.float64) @ Weff, wl.C[p].astype(np.float64) @ beff
        for i, (l, u) in res["pre"].items():
            assert bool((l[p] >= 0).all()) if shift > 0 else bool((u[p] <= 0).all())
        _close(_np64(res["lb"][p]), CW @ xc - np.abs(CW) @ xr + Cb, "closed-form lb")
        _close(_np64(res["ub"][p]), CW @ xc + np.abs(CW) @ xr + Cb, "closed-form ub")


# ------------------------------------------------------------------------------------------ discontinuities
@pytest.mark.parametrize("with_alpha", [False, True])
@pytest.mark.parametrize("widths", [[6, 9, 7, 3], [160, 256, 192, 12]])
def test_planted_neurons_on_the_relaxation_discontinuities(with_alpha, widths):
    """Pre-activation bounds given by the caller with neurons EXACTLY at l = 0, u = 0, l = u = 0, u = -l (adaptive-rule
    tie, strict '>') and clearly stable ones: both sides must take the same branch (G3 order, G4 strictness)."""
    import torch
    wl = W.small_mlp(widths, seed=31, B=2, eps=0.1)
    lo, hi = wl.box()
    rng = np.random.default_rng(80)
    pre = {}
    for i in wl.net.relu_ids():
        n = wl.net.nodes[i].size
        l = (-rng.random((wl.B, n)) * 2.0).astype(np.float32)
        u = (rng.random((wl.B, n)) * 2.0).astype(np.float32)
        l[:, 0::8] = 0.0                                   # l = 0 < u          -> active
        u[:, 1::8] = 0.0                                   # l < 0 = u          -> inactive
        l[:, 2::8] = 0.0; u[:, 2::8] = 0.0                 # l = u = 0          -> active (G3 order)
        u[:, 3::8] = -l[:, 3::8]                           # u = -l exactly     -> adaptive lambda = 0 (strict >)
        l[:, 4::8] = np.abs(l[:, 4::8]) * 0.5              # 0 < l <= u         -> active
        u[:, 4::8] = l[:, 4::8] + 1.0
        u[:, 5::8] = -np.abs(u[:, 5::8]) * 0.5 - 0.1       # l <= u < 0         -> inactive
        l[:, 5::8] = u[:, 5::8] - 1.0
        pre[i] = (torch.from_numpy(l).cuda(), torch.from_numpy(u).cuda())
    ctx = _ctx(wl.net, wl.B, wl.S)
    al = {i: a for i, a in zip(wl.net.relu_ids(), wl.alpha)} if with_alpha else None
    _final_pass_vs_oracle(wl, lo, hi, pre, al, al, ctx)


# ------------------------------------------------------------------------------------------ verdict
def test_verified_properties_match_the_oracle():
    """A batch whose radii span 1e-5 .. 0.05: the small ones verify (margins at x0 are positive by construction of the
    label), the large ones do not; verified is compared with O.verified on the oracle's own lower bounds."""
    wl = W.make(2, B=8)
    wl.eps[:] = np.array([1e-5, 1e-4, 5e-4, 2e-3, 0.01, 0.026, 0.05, 1e-5], dtype=np.float32)
    lo, hi = wl.box()
    _, res = _check_run(wl, lo, hi, wl.alpha)
    ver = res["verified"].cpu().numpy().astype(bool)
    ref = []
    for p in range(wl.B):
        r = O.run_property(wl.net, lo[p], hi[p], wl.C[p], [a[p] for a in wl.alpha], wl.intermediate)
        assert np.min(np.abs(r["lb"])) > 1e-3, "margin too close to 0 for a robust verdict comparison"
        ref.append(r["verified"])
    assert ver.tolist() == ref
    assert any(ref) and not all(ref), ref            # both branches of the verdict are exercised


def test_verdict_fails_closed_on_nan():
    """A NaN lower bound must not verify (np.min(lb) > 0 is False in the oracle; fminf would have dropped the NaN)."""
    wl2 = W.small_mlp([6, 9, 7, 3], seed=41, B=3, eps=1e-4)
    lo, hi = wl2.box()
    hi = hi.copy(); hi[1, 2] = np.nan
    ctx = _ctx(wl2.net, wl2.B, wl2.S)
    res = ctx.run(lo, hi, wl2.C, wl2.alpha, wl2.intermediate)
    lb = _np64(res["lb"])
    assert np.isnan(lb[1]).any()
    assert res["verified"].cpu().numpy().tolist() == [int(O.verified(lb[p])) for p in range(3)]
    assert res["verified"][1].item() == 0


def test_host_entry_rejects_an_inverted_box():
    from paper_2606_09377_b200 import CrownError
    wl = W.small_mlp([6, 9, 7, 3], seed=42, B=2, eps=0.1)
    lo, hi = wl.box()
    ctx = _ctx(wl.net, wl.B, wl.S)
    lb = np.empty((wl.B, wl.S), np.float32); ub = np.empty_like(lb); ver = np.empty(wl.B, np.uint8)
    ctx.run_host(lo, hi, wl.C, wl.alpha, wl.intermediate, lb, ub, ver)          # fine
    bad = lo.copy(); bad[0, 0] = hi[0, 0] + 1.0
    with pytest.raises(CrownError):
        ctx.run_host(bad, hi, wl.C, wl.alpha, wl.intermediate, lb, ub, ver)


@pytest.mark.parametrize("which", ["cfg1", "cfg2", "small_B1of3", "cfg5"])
def test_host_entry_equals_device_entry_bitwise(which):
    """crown_run_host (H2D / D2H inside; one packed copy per direction for small problems, direct copies above 1 MiB)
    returns exactly what crown_run returns on resident tensors, also for B below B_max and on repeated calls"""
    if which == "cfg1":
        wl = W.make(1); Bmax = wl.B                      # 25 KB of inputs: packed path
    elif which == "cfg2":
        wl = W.make(2, B=24); Bmax = wl.B                # 1.4 MB of alpha: direct copies
    elif which == "cfg5":
        wl = W.make(5, B=2); Bmax = wl.B                 # 72 MB of alpha through the conv / residual graph
    else:
        wl = W.small_mlp([6, 9, 7, 3], seed=43, B=1, eps=0.1); Bmax = 3
    lo, hi = wl.box()
    ctx = _ctx(wl.net, Bmax, wl.S)
    ref = ctx.run(lo, hi, wl.C, wl.alpha, wl.intermediate)
    for rep in range(2):
        lb = np.full((wl.B, wl.S), np.nan, np.float32); ub = np.full_like(lb, np.nan); ver = np.full(wl.B, 7, np.uint8)
        ctx.run_host(lo, hi, wl.C, wl.alpha, wl.intermediate, lb, ub, ver)
        assert np.array_equal(lb, ref["lb"].cpu().numpy()) and np.array_equal(ub, ref["ub"].cpu().numpy())
        assert np.array_equal(ver, ref["verified"].cpu().numpy())
    ctx.close()


# ------------------------------------------------------------------------------------------ graph shapes
def _graph_workload(net, seed, B=2, eps=0.05, S=5):
    rng = np.random.Generator(np.random.PCG64(W.SEED_BASE + 5000 + seed))
    x0 = (rng.random((B, net.n_in)) * 2.0 - 1.0).astype(np.float32)
    C = rng.standard_normal((B, S, net.n_out)).astype(np.float32)
    al = [rng.random((B, S, net.nodes[i].size)).astype(np.float32) for i in net.relu_ids()]
    return W.Workload(cfg=0, name="graph", net=net, x0=x0, eps=np.full((B,), eps, np.float32), C=C,
                      labels=np.zeros(B, int), alpha=al, intermediate="ibp", eps_set=(eps,))


def _lin(rng, n_out, n_in):
    return (rng.standard_normal((n_out, n_in)) * np.sqrt(2.0 / n_in)).astype(np.float32), \
           (rng.standard_normal(n_out) * 0.1).astype(np.float32)


@pytest.mark.parametrize("n0,h", [(6, 9), (160, 192)])
def test_skip_connection_from_the_network_input(n0, h):
    """x -> Linear -> ReLU -> Linear(h -> n0) ; Add(., x) -> ReLU -> Linear: the input has TWO consumers, so the
    concretisation must not be fused into either contraction (both A.x terms are needed)."""
    rng = np.random.default_rng(90 + n0)
    N = W.Node
    W0, b0 = _lin(rng, h, n0); W2, b2 = _lin(rng, n0, h); W5, b5 = _lin(rng, 7, n0)
    net = W.Net(in_shape=(n0,), nodes=[
        N("linear", -1, W=W0, b=b0, shape=(h,)), N("relu", 0, shape=(h,)), N("linear", 1, W=W2, b=b2, shape=(n0,)),
        N("add", 2, -1, shape=(n0,)), N("relu", 3, shape=(n0,)), N("linear", 4, W=W5, b=b5, shape=(7,))])
    wl = _graph_workload(net, n0)
    lo, hi = wl.box()
    _check_run(wl, lo, hi, wl.alpha)
    _check_run(wl, lo, hi, None)


@pytest.mark.parametrize("n0,h", [(6, 9), (160, 192)])
def test_two_linear_branches_read_the_input(n0, h):
    rng = np.random.default_rng(190 + n0)
    N = W.Node
    W0, b0 = _lin(rng, h, n0); W2, b2 = _lin(rng, h, n0); W5, b5 = _lin(rng, 7, h)
    net = W.Net(in_shape=(n0,), nodes=[
        N("linear", -1, W=W0, b=b0, shape=(h,)), N("relu", 0, shape=(h,)), N("linear", -1, W=W2, b=b2, shape=(h,)),
        N("add", 1, 2, shape=(h,)), N("relu", 3, shape=(h,)), N("linear", 4, W=W5, b=b5, shape=(7,))])
    wl = _graph_workload(net, 100 + n0)
    lo, hi = wl.box()
    _check_run(wl, lo, hi, wl.alpha)
    _check_run(wl, lo, hi, None)


@pytest.mark.parametrize("n0,h", [(6, 9), (160, 192)])
def test_residual_fork_on_a_linear_output(n0, h):
    """The output of Linear 2 feeds ReLU 3 AND the Add 5: the TF32-split contribution arriving through the ReLU is
    merged with the fp32 one arriving through the skip (hi + lo must both be added)."""
    rng = np.random.default_rng(290 + n0)
    N = W.Node
    W0, b0 = _lin(rng, h, n0); W2, b2 = _lin(rng, h, h); W4, b4 = _lin(rng, h, h); W7, b7 = _lin(rng, 7, h)
    net = W.Net(in_shape=(n0,), nodes=[
        N("linear", -1, W=W0, b=b0, shape=(h,)), N("relu", 0, shape=(h,)), N("linear", 1, W=W2, b=b2, shape=(h,)),
        N("relu", 2, shape=(h,)), N("linear", 3, W=W4, b=b4, shape=(h,)), N("add", 4, 2, shape=(h,)),
        N("relu", 5, shape=(h,)), N("linear", 6, W=W7, b=b7, shape=(7,))])
    wl = _graph_workload(net, 200 + n0)
    lo, hi = wl.box()
    _check_run(wl, lo, hi, wl.alpha)
    _check_run(wl, lo, hi, None)
    _check_run(wl, lo, hi, None, disable_epi_fusion=1)


# ------------------------------------------------------------------------------------------ CUDA-graph replay
@pytest.mark.parametrize("cfg,kw", [(1, dict()), (2, dict(B=4)), (5, dict(scale=4, B=2))])
def test_graph_replay_is_bitwise_the_plain_launch_sequence(cfg, kw):
    """crown_run replays a captured CUDA graph from the second call with the same pointer set; the graph holds exactly
    the kernels of the plain path, so results are bitwise equal and fresh inputs written into the same buffers are
    picked up by the replay."""
    import torch
    wl = W.make(cfg, **kw)
    lo, hi = wl.box()
    inter = 1 if wl.intermediate == "ibp" else 0
    outs = {}
    for graph_off in (1, 0):
        ctx = _ctx(wl.net, wl.B, wl.S, disable_graph=graph_off)
        dev = ctx.device
        xlo, xhi = torch.from_numpy(lo).to(dev), torch.from_numpy(hi).to(dev)
        Cd = torch.from_numpy(wl.C).to(dev)
        al = {i: torch.from_numpy(a).to(dev) for i, a in zip(ctx.relu_ids, wl.alpha)}
        io = ctx.alloc_io(wl.B, wl.S)
        res = []
        for it in range(3):
            if it == 2:                      # new box in the SAME buffers: the replay must see it
                xlo.copy_(torch.from_numpy((lo - 0.001).astype(np.float32)))
                xhi.copy_(torch.from_numpy((hi + 0.001).astype(np.float32)))
            ctx.run_device(xlo, xhi, Cd, al, inter, io)
            torch.cuda.synchronize()
            res.append((io["lb"].clone(), io["ub"].clone(), io["verified"].clone()))
        assert ctx.graph_replays() == (0 if graph_off else 3)
        assert ctx.launch_count() > 0
        outs[graph_off] = res
    for a, b in zip(outs[0], outs[1]):
        for x, y in zip(a, b):
            assert torch.equal(x, y)
    assert not torch.equal(outs[0][1][0], outs[0][2][0])         # the third call really used the new box
