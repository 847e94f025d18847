"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (`-m gpu`).

Where the oracle cannot recompute everything in seconds (cfg3: 4.2e14 flops, cfg4: 7e13) parity is checked on
SAMPLED outputs the oracle can compute one by one: rows of a start spec are independent linear bounds
(PAPER.md:66), so the oracle propagates a seeded sample of identity rows per layer from the GPU's own earlier
(l, u) (forced-bounds protocol, reading G18) plus the final spec rows of sampled properties.  Tolerance
|gpu - oracle| <= 1e-5 + 1e-4 |oracle| (BASELINE.json north_star)."""
import numpy as np
import pytest

import workloads as W
from oracle import crown_oracle as O

pytestmark = pytest.mark.gpu

ATOL, RTOL = 1e-5, 1e-4


def _np64(t):
    return t.detach().cpu().numpy().astype(np.float64)


def _excess(gpu, ref):
    return float(np.max(np.abs(gpu - ref) - (ATOL + RTOL * np.abs(ref))))


def _run(wl, eps=None, **kw):
    from paper_2606_09377_b200 import CrownContext
    ctx = CrownContext(wl.net, wl.B, wl.S, **kw)
    if eps is None:
        lo, hi = wl.box()
    else:
        e = np.float32(eps).astype(np.float64)
        lo = (wl.x0.astype(np.float64) - e).astype(np.float32)
        hi = (wl.x0.astype(np.float64) + e).astype(np.float32)
    res = ctx.run(lo, hi, wl.C, wl.alpha, wl.intermediate)
    return ctx, res, lo, hi


def _check_props(wl, res, lo, hi, props, rows_per_layer=None, seed=0):
    """Forced-bounds parity of the pre-activation bounds (all rows, or a seeded sample) and of the final bound."""
    rng = np.random.default_rng(seed)
    lb, ub = _np64(res["lb"]), _np64(res["ub"])
    ver = res["verified"].cpu().numpy()
    for p in props:
        forced = {i: (_np64(l[p]), _np64(u[p])) for i, (l, u) in res["pre"].items()}
        rows = None
        if rows_per_layer:
            rows = {i: np.sort(rng.choice(wl.net.nodes[i].size, size=min(rows_per_layer, wl.net.nodes[i].size),
                                          replace=False)) for i in wl.net.relu_ids()}
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
        assert bool(ver[p]) == bool(np.min(lb[p]) > 0)


def test_cfg2_full_all_eps():
    wl = W.stack_eps(W.make(2))                      # 784-(256x6)-10, 64 points x 3 eps = ONE batch of 192, alpha
    assert wl.B == 192
    _, res, lo, hi = _run(wl)
    _check_props(wl, res, lo, hi, list(range(64, 128)) + [0, 21, 42, 63, 128, 149, 170, 191])
    # soundness on samples for a property of each eps (O6; slack = parity tolerance, reading G17)
    lb, ub = _np64(res["lb"]), _np64(res["ub"])
    for p in (0, 100, 191):
        X = W.sample_points(2, lo[p], hi[p], 2048, 512)
        ok, vlo, vhi, _, _ = O.sample_check(wl.net, wl.C[p], X, lb[p], ub[p], slack_rel=RTOL, slack_abs=ATOL)
        assert ok, (vlo, vhi)


def test_cfg5_full():
    wl = W.make(5)                                   # ResNet, B = 8, S = 99, IBP intermediates + alpha backward
    _, res, lo, hi = _run(wl)
    _check_props(wl, res, lo, hi, [0, 7])


def test_cfg1_full():
    wl = W.make(1)
    _, res, lo, hi = _run(wl)
    _check_props(wl, res, lo, hi, [0])


def test_cfg3_full_sampled_rows():
    wl = W.make(3)                                   # 4096-16384x3-10, B = 16, chunked under a 64 GB cap as in bench.py
    ctx, res, lo, hi = _run(wl, mem_cap_bytes=64 << 30)
    assert ctx.peak_bytes() <= 64 << 30
    _check_props(wl, res, lo, hi, [5], rows_per_layer=24, seed=3)
    # properties that hold at any size: lb <= ub everywhere, bounds finite
    for i, (l, u) in res["pre"].items():
        assert bool((l <= u).all()) and bool(l.isfinite().all()) and bool(u.isfinite().all())


def test_cfg4_full_sampled_rows():
    wl = W.make(4)                                   # 4096-262144-4096-10, B = 4
    ctx, res, lo, hi = _run(wl, mem_cap_bytes=64 << 30)
    _check_props(wl, res, lo, hi, [2], rows_per_layer=16, seed=4)
    for i, (l, u) in res["pre"].items():
        assert bool((l <= u).all()) and bool(l.isfinite().all()) and bool(u.isfinite().all())
