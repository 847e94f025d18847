"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (`-m gpu`).

Where the oracle cannot recompute everything in seconds (cfg3: 4.2e14 flops, cfg4: 7e13) parity is checked on
SAMPLED outputs the oracle can compute one by one: rows of a start spec are independent linear bounds
(PAPER.md:66), so the oracle propagates 128 identity rows per layer from the GPU's own earlier (l, u)
(forced-bounds protocol, reading G18) -- rows chosen to hit the first and last tile of the contraction, both sides
of every row-chunk boundary and the tail chunk, the rest seeded at random -- plus the final spec rows, on two
properties.  Tolerance |gpu - oracle| <= 1e-5 + 1e-4 |oracle| (BASELINE.json north_star).

Soundness (north_star: "must contain every sample"): for two properties of every config,
C.f(x) in float64 at 8192 uniform points + 1792 random corners + the centre + the two ADVERSARIAL corners of every
spec row (x0 -+ eps.sign(A0), the minimiser / maximiser of the linear bound, from the GPU's own A0) must lie inside
[lb, ub] with the parity tolerance as slack (reading G17)."""
import numpy as np
import pytest

import workloads as W
from oracle import crown_oracle as O

pytestmark = pytest.mark.gpu

ATOL, RTOL = 1e-5, 1e-4
N_UNIFORM, N_CORNER = 8192, 1792


def _np64(t):
    return t.detach().cpu().numpy().astype(np.float64)


def _excess(gpu, ref):
    return float(np.max(np.abs(gpu - ref) - (ATOL + RTOL * np.abs(ref))))


def _run(wl, **kw):
    from paper_2606_09377_b200 import CrownContext
    ctx = CrownContext(wl.net, wl.B, wl.S, **kw)
    lo, hi = wl.box()
    res = ctx.run(lo, hi, wl.C, wl.alpha, wl.intermediate)
    return ctx, res, lo, hi


def _targeted_rows(n, rc, count, rng):
    """`count` row indices of an n-row identity start: first / last 8 rows (first and last tile), 4 rows on each
    side of every chunk boundary k*rc, 8 rows of the tail chunk, rest random."""
    want = set(range(min(8, n))) | set(range(max(0, n - 8), n))
    for b in range(rc, n, rc):
        want |= set(range(max(0, b - 4), min(n, b + 4)))
    tail0 = (n - 1) // rc * rc
    want |= set(range(tail0, min(n, tail0 + 8)))
    want = sorted(want)[:count]
    rest = np.setdiff1d(np.arange(n), np.array(want, dtype=int))
    extra = rng.choice(rest, size=max(0, min(count, n) - len(want)), replace=False)
    return np.sort(np.concatenate([np.array(want, dtype=int), extra]))


def _check_props(wl, ctx, res, lo, hi, props, rows_per_layer=None, seed=0):
    """Forced-bounds parity of the pre-activation bounds (all rows, or a targeted sample) and of the final bound."""
    rng = np.random.default_rng(seed)
    lb, ub = _np64(res["lb"]), _np64(res["ub"])
    ver = res["verified"].cpu().numpy()
    rc = ctx.row_chunk()
    for p in props:
        forced = {i: (_np64(l[p]), _np64(u[p])) for i, (l, u) in res["pre"].items()}
        rows = None
        if rows_per_layer:
            rows = {i: _targeted_rows(wl.net.nodes[i].size, rc, rows_per_layer, rng) for i in wl.net.relu_ids()}
        pre = O.crown_bounds(wl.net, lo[p], hi[p], wl.intermediate, forced=forced, rows=rows)
        for i in wl.net.relu_ids():
            for k, nm in ((0, "l"), (1, "u")):
                ref = pre[i][k]
                m = ~np.isnan(ref)
                assert m.any()
                ex = _excess(forced[i][k][m], ref[m])
                assert ex <= 0, f"prop {p} relu {i} {nm}: excess {ex:.3e}"
        al = None if wl.alpha is None else {i: a[p] for i, a in zip(wl.net.relu_ids(), wl.alpha)}
        olb, oub, _ = O.final_bounds(wl.net, lo[p], hi[p], wl.C[p], forced, al, al)
        assert _excess(lb[p], olb) <= 0, f"prop {p} lb excess {_excess(lb[p], olb):.3e}"
        assert _excess(ub[p], oub) <= 0, f"prop {p} ub excess {_excess(ub[p], oub):.3e}"
        assert np.all(lb[p] <= ub[p] + ATOL + RTOL * np.abs(ub[p]))
        assert bool(ver[p]) == O.verified(lb[p])


def _check_containment(wl, ctx, res, lo, hi, props, chunk=2560):
    """O6 on the GPU's bounds: 8192 uniform + 1792 corners + centre + adversarial corners from the GPU's A0."""
    al = None if wl.alpha is None else {i: a for i, a in zip(wl.net.relu_ids(), wl.alpha)}
    out = ctx.crown_backward(wl.B, len(wl.net.nodes) - 1, res["pre"], Cmat=wl.C, alpha_lo=al, alpha_up=al,
                             box=(lo, hi), want_A=True)
    A = out["A"]
    lb, ub = _np64(res["lb"]), _np64(res["ub"])
    for p in props:
        X = W.sample_points(max(wl.cfg, 1), lo[p], hi[p], N_UNIFORM, N_CORNER)
        adv = O.adversarial_corners(_np64(A[0, p]), _np64(A[1, p]), lo[p], hi[p])
        X = np.concatenate([X, adv], axis=0)
        assert X.shape[0] == N_UNIFORM + N_CORNER + 1 + 2 * wl.S
        for s in range(0, X.shape[0], chunk):
            ok, vlo, vhi, _, _ = O.sample_check(wl.net, wl.C[p], X[s:s + chunk], lb[p], ub[p], slack_rel=RTOL, slack_abs=ATOL)
            assert ok, f"cfg{wl.cfg} prop {p}: a sample escapes the bounds (lb by {vlo:.3e}, ub by {vhi:.3e})"
        # the materialised-A pass and the fused-concretisation pass agree
        assert _excess(_np64(out["lb"][p]), lb[p]) <= 0 and _excess(_np64(out["ub"][p]), ub[p]) <= 0


def test_cfg1_full():
    wl = W.make(1)
    ctx, res, lo, hi = _run(wl)
    _check_props(wl, ctx, res, lo, hi, [0])
    _check_containment(wl, ctx, res, lo, hi, [0])            # B = 1: the one property


def test_cfg2_full_all_eps():
    wl = W.stack_eps(W.make(2))                      # 784-(256x6)-10, 64 points x 3 eps = ONE batch of 192, alpha
    assert wl.B == 192
    ctx, res, lo, hi = _run(wl)
    _check_props(wl, ctx, res, lo, hi, list(range(64, 128)) + [0, 21, 42, 63, 128, 149, 170, 191])
    _check_containment(wl, ctx, res, lo, hi, [0, 100, 191])   # one property of each eps


def test_cfg5_full():
    wl = W.make(5)                                   # ResNet, B = 8, S = 99, IBP intermediates + alpha backward
    ctx, res, lo, hi = _run(wl)
    _check_props(wl, ctx, res, lo, hi, [0, 7])
    _check_containment(wl, ctx, res, lo, hi, [0, 7])


def test_cfg3_full_sampled_rows():
    wl = W.make(3)                                   # 4096-16384x3-10, B = 16, chunked under a 64 GiB cap as in bench.py
    ctx, res, lo, hi = _run(wl, mem_cap_bytes=64 << 30)
    assert ctx.peak_bytes() <= 64 << 30
    assert ctx.row_chunk() < 16384                   # the cap really chunks the identity passes
    _check_props(wl, ctx, res, lo, hi, [5, 15], rows_per_layer=128, seed=3)
    # properties that hold at any size: lb <= ub everywhere, bounds finite
    for i, (l, u) in res["pre"].items():
        assert bool((l <= u).all()) and bool(l.isfinite().all()) and bool(u.isfinite().all())
    _check_containment(wl, ctx, res, lo, hi, [0, 15])


def test_cfg4_full_sampled_rows():
    wl = W.make(4)                                   # 4096-262144-4096-10, B = 4
    ctx, res, lo, hi = _run(wl, mem_cap_bytes=64 << 30)
    assert ctx.row_chunk() < 4096
    _check_props(wl, ctx, res, lo, hi, [0, 3], rows_per_layer=128, seed=4)
    for i, (l, u) in res["pre"].items():
        assert bool((l <= u).all()) and bool(l.isfinite().all()) and bool(u.isfinite().all())
    _check_containment(wl, ctx, res, lo, hi, [1, 2])
