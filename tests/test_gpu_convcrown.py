"""NEXT-3: full-CROWN intermediate bounds THROUGH conv layers on the GPU --
identity-start passes on conv-shaped nodes (Conv2d outputs, residual Add outputs), row-chunked, dense A -- against the
float64 oracle (O4 with `intermediate='crown'`, which handles any DAG and is pinned by the dense-Toeplitz twin in
tests/test_oracle_pins.py).  Same protocol and tolerance as the other parity tests (forced bounds layer-wise, free-running
where no neuron sits on a relaxation discontinuity, 1e-5 + 1e-4 |ref|)."""
import dataclasses
import importlib

import numpy as np
import pytest

import workloads as W
from oracle import crown_oracle as O

pytestmark = pytest.mark.gpu

P = importlib.import_module("test_gpu_parity")
F = importlib.import_module("test_gpu_fullsize")


def _crown(wl):
    return dataclasses.replace(wl, intermediate="crown")


@pytest.mark.parametrize("scale,kw", [(4, dict()), (4, dict(mma_scheme=2)), (2, dict(disable_graph=1))])
def test_conv_crown_scaled_resnet_matches_oracle(scale, kw):
    """every pre-activation bound of the residual conv net (stem by IBP, all others by identity-start CROWN passes
    through conv / add / flatten / linear) and the alpha-CROWN final bound, all elements, both properties"""
    wl = _crown(W.make(5, scale=scale, B=2))
    ctx, res = P._check_workload(wl, free_running=(scale == 4), **kw)
    # the point of NEXT-3: tighter than IBP intermediate bounds (reading G22), never looser
    lo, hi = wl.box()
    ibp = ctx.run(lo, hi, wl.C, wl.alpha, "ibp")
    w_crown = (res["ub"] - res["lb"]).cpu().numpy()
    w_ibp = (ibp["ub"] - ibp["lb"]).cpu().numpy()
    assert np.all(w_crown <= w_ibp * (1 + 1e-4) + 1e-5), "CROWN intermediate bounds gave a wider final interval than IBP ones"
    assert np.median(w_crown / w_ibp) < 0.9
    ctx.close()


def test_conv_crown_identity_start_one_by_one():
    """crown_backward with C = NULL on a Conv2d node and on an Add node: A, d and the concretised rows vs the oracle,
    for a row range that is not aligned to anything"""
    wl = _crown(W.make(5, scale=4, B=2))
    lo, hi = wl.box()
    from paper_2606_09377_b200 import CrownContext
    ctx = CrownContext(wl.net, wl.B, wl.S)
    res = ctx.run(lo, hi, wl.C, wl.alpha, "crown")
    net = wl.net
    conv_start = next(i for i in net.relu_ids() if net.nodes[net.nodes[i].in0].op == "conv" and net.nodes[net.nodes[i].in0].in0 >= 0)
    add_start = next(i for i in net.relu_ids() if net.nodes[net.nodes[i].in0].op == "add")
    for relu in (conv_start, add_start):
        src = net.nodes[relu].in0
        n = net.nodes[src].size
        row0, rows = 5, min(37, n - 5)
        out = ctx.crown_backward(wl.B, src, res["pre"], None, row0=row0, rows=rows, box=(lo, hi), want_A=True)
        ctx.stream.synchronize()
        for p in range(wl.B):
            forced = {i: (l[p].cpu().numpy().astype(np.float64), u[p].cpu().numpy().astype(np.float64)) for i, (l, u) in res["pre"].items()}
            C0 = np.zeros((rows, n)); C0[np.arange(rows), row0 + np.arange(rows)] = 1.0
            A_lo, A_up, d_lo, d_up = O.backward(net, src, C0, forced)
            olb, oub = O.concretize(A_lo, A_up, d_lo, d_up, lo[p], hi[p])
            P._close(out["A"][0, p].cpu().numpy(), A_lo, f"relu {relu} A_lo"); P._close(out["A"][1, p].cpu().numpy(), A_up, f"relu {relu} A_up")
            P._close(out["d"][0, p].cpu().numpy(), d_lo, "d_lo"); P._close(out["d"][1, p].cpu().numpy(), d_up, "d_up")
            P._close(out["lb"][p].cpu().numpy(), olb, "lb"); P._close(out["ub"][p].cpu().numpy(), oub, "ub")
            # and they are the rows crown_run produced
            P._close(out["lb"][p].cpu().numpy(), res["pre"][relu][0][p, row0:row0 + rows].cpu().numpy(), "rows of crown_run l")
    ctx.close()


def test_conv_crown_full_size_sampled_rows():
    """BASELINE cfg5 at full size (3x32x32, 16/32/32/64 channels), one property, CROWN intermediate bounds for all
    90 624 ReLU neurons: 24 targeted rows per ReLU + the final bound vs the oracle (forced bounds), sample containment
    incl. adversarial corners"""
    wl = _crown(W.make(5, B=1))
    ctx, res, lo, hi = F._run(wl)
    F._check_props(wl, ctx, res, lo, hi, props=[0], rows_per_layer=24, seed=5)
    F._check_containment(wl, ctx, res, lo, hi, props=[0])
    for i, (l, u) in res["pre"].items():
        assert bool((l <= u).all()) and bool(l.isfinite().all()) and bool(u.isfinite().all())
    ctx.close()
