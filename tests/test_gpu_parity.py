"""GPU parity (`-m gpu`): the CUDA path, called through the C-ABI binding, against the float64 oracle on
the same seeded inputs, element by element.  Tolerance (BASELINE.json north_star, reading G18):
|gpu - oracle| <= 1e-5 + 1e-4 |oracle|.  Forced-bounds protocol: where the oracle needs intermediate bounds
it is given the GPU's own (l, u) upcast to float64, so a relaxation-class flip at a discontinuity
cannot masquerade as (or hide) an arithmetic error; free-running parity is checked in addition."""
import numpy as np
import pytest

import workloads as W
from oracle import crown_oracle as O

pytestmark = pytest.mark.gpu

ATOL, RTOL = 1e-5, 1e-4


def _ctx(net, B, S, **kw):
    from paper_2606_09377_b200 import CrownContext
    return CrownContext(net, B, S, **kw)


def _close(gpu, ref, what, atol=ATOL, rtol=RTOL):
    gpu = np.asarray(gpu, np.float64)
    ref = np.asarray(ref, np.float64)
    err = np.abs(gpu - ref) - (atol + rtol * np.abs(ref))
    assert np.all(err <= 0), f"{what}: worst excess {err.max():.3e} at {np.unravel_index(err.argmax(), err.shape)}"


def _np(t):
    return t.detach().cpu().numpy()


# ------------------------------------------------------------------------------------------ kernel 1
@pytest.mark.parametrize("M,N,K", [(128, 128, 32), (256, 384, 512), (300, 260, 1000), (1152, 784, 256),
                                   (128, 4096, 16384)])
def test_gemm_3xtf32_matches_fp64(M, N, K):
    import torch
    rng = np.random.default_rng(M * 7 + N * 3 + K)
    A = rng.standard_normal((M, K)).astype(np.float32)
    Wm = (rng.standard_normal((K, N)) * np.sqrt(2.0 / K)).astype(np.float32)
    net = W.small_mlp([4, 4, 2], 0).net
    ctx = _ctx(net, 1, 1)
    D = _np(ctx.gemm(torch.from_numpy(A), torch.from_numpy(Wm), scheme=0))
    ref = A.astype(np.float64) @ Wm.astype(np.float64)
    # fp32-accurate: error relative to the row/column magnitude, not to the (possibly cancelling) result
    scale = np.abs(A).astype(np.float64) @ np.abs(Wm).astype(np.float64)
    assert np.max(np.abs(D - ref) / scale) < 2e-6, np.max(np.abs(D - ref) / scale)


@pytest.mark.parametrize("M,N,K", [(18, 256, 10), (65, 130, 33), (512, 784, 256)])
def test_gemm_ffma_matches_fp64(M, N, K):
    import torch
    rng = np.random.default_rng(M + N + K)
    A = rng.standard_normal((M, K)).astype(np.float32)
    Wm = rng.standard_normal((K, N)).astype(np.float32)
    ctx = _ctx(W.small_mlp([4, 4, 2], 0).net, 1, 1)
    D = _np(ctx.gemm(torch.from_numpy(A), torch.from_numpy(Wm), scheme=2))
    ref = A.astype(np.float64) @ Wm.astype(np.float64)
    scale = np.abs(A).astype(np.float64) @ np.abs(Wm).astype(np.float64)
    assert np.max(np.abs(D - ref) / scale) < 1e-6


# ------------------------------------------------------------------------------------------ whole path
def _oracle_forced(wl, gpu_pre, props):
    """Oracle bounds with the GPU's (l,u) forced for EARLIER ReLUs (layer-wise parity, G18)."""
    lo, hi = wl.box()
    out = []
    for p in props:
        forced = {i: (_np(l)[p].astype(np.float64), _np(u)[p].astype(np.float64)) for i, (l, u) in gpu_pre.items()}
        pre = O.crown_bounds(wl.net, lo[p], hi[p], wl.intermediate, forced=forced)
        al = None if wl.alpha is None else {i: a[p] for i, a in zip(wl.net.relu_ids(), wl.alpha)}
        lb, ub, _ = O.final_bounds(wl.net, lo[p], hi[p], wl.C[p], forced, al, al)
        out.append((pre, lb, ub))
    return out


def _check_workload(wl, props=None, free_running=True, **kw):
    lo, hi = wl.box()
    ctx = _ctx(wl.net, wl.B, wl.S, **kw)
    res = ctx.run(lo, hi, wl.C, wl.alpha, wl.intermediate)
    props = range(wl.B) if props is None else props
    forced = _oracle_forced(wl, res["pre"], props)
    lb, ub = _np(res["lb"]), _np(res["ub"])
    for k, p in enumerate(props):
        pre, olb, oub = forced[k]
        for i in wl.net.relu_ids():
            _close(_np(res["pre"][i][0])[p], pre[i][0], f"prop {p} relu {i} l")
            _close(_np(res["pre"][i][1])[p], pre[i][1], f"prop {p} relu {i} u")
        _close(lb[p], olb, f"prop {p} lb")
        _close(ub[p], oub, f"prop {p} ub")
        assert np.all(lb[p] <= ub[p] + ATOL)
        assert bool(_np(res["verified"])[p]) == O.verified(lb[p].astype(np.float64))
    if free_running:
        flagged = 0
        for p in props:
            r = O.run_property(wl.net, lo[p], hi[p], wl.C[p], None if wl.alpha is None else [a[p] for a in wl.alpha],
                               wl.intermediate)
            risky = any(np.any(np.minimum(np.minimum(np.abs(l), np.abs(u)), np.abs(u + l)) < 1e-5 * (1 + np.abs(u - l)))
                        for l, u in r["pre"].values())
            if risky:
                flagged += 1
                continue
            _close(lb[p], r["lb"], f"free-running prop {p} lb")
            _close(ub[p], r["ub"], f"free-running prop {p} ub")
            assert bool(_np(res["verified"])[p]) == r["verified"]
        assert flagged <= max(1, len(list(props)) // 2), f"{flagged} of {len(list(props))} properties skipped as risky"
    # soundness on samples (O6), slack = parity tolerance (G17)
    for p in list(props)[:2]:
        X = W.sample_points(max(wl.cfg, 1), lo[p], hi[p], 512, 128)
        ok, vlo, vhi, _, _ = O.sample_check(wl.net, wl.C[p], X, lb[p], ub[p], slack_rel=RTOL, slack_abs=ATOL)
        assert ok, (vlo, vhi)
    return ctx, res


@pytest.mark.parametrize("scheme", [2, 0])
def test_small_mlp(scheme):
    wl = W.small_mlp([6, 9, 7, 5, 3], seed=3, B=3, eps=0.2)
    _check_workload(wl, mma_scheme=scheme)


@pytest.mark.parametrize("scheme", [2, 0])
def test_cfg1(scheme):
    _check_workload(W.make(1), mma_scheme=scheme)


def test_cfg2_subset():
    wl = W.make(2, B=8)
    _check_workload(wl, props=[0, 3, 7])


def test_cfg3_scaled():
    wl = W.make(3, scale=16, B=4)     # 256-1024-1024-1024-10
    _check_workload(wl, props=[0, 3])


@pytest.mark.parametrize("cfg,kw", [(3, dict(scale=16, B=4)), (2, dict(B=8)), (1, dict())])
def test_unfused_relaxation_path(cfg, kw):
    """a4 as its own kernel (disable_epi_fusion=1; the default fuses it into the producing contraction's epilogue):
    same parity bar, and the two paths agree with each other within the tolerance."""
    wl = W.make(cfg, **kw)
    ctx, res = _check_workload(wl, props=[0, wl.B - 1], disable_epi_fusion=1)
    assert ctx.gemm_flops() > 0
    lo, hi = wl.box()
    res2 = _ctx(wl.net, wl.B, wl.S).run(lo, hi, wl.C, wl.alpha, wl.intermediate)
    _close(_np(res2["lb"]), _np(res["lb"]), "fused vs unfused lb")
    _close(_np(res2["ub"]), _np(res["ub"]), "fused vs unfused ub")


@pytest.mark.parametrize("widths", [[200, 176, 272, 160, 7], [136, 144, 160, 192, 5]])
def test_fused_epilogues_on_ragged_widths(widths):
    """a4 / a8 fused into the contraction where the row length is NOT a multiple of the 32-column pieces the epilogue works in
    (176 = 5.5, 144 = 4.5, 200 = 6.25, 136 = 4.25 pieces): the last piece of a row reads clamped coefficient columns and stores
    only the columns that exist.  The passes that start at the 160- / 192-row layers take the fused path (rows % 32 == 0)."""
    wl = W.small_mlp(widths, seed=17, B=3, eps=0.03, S=4)
    ctx, res = _check_workload(wl, free_running=False)
    assert ctx.gemm_flops() > 0
    lo, hi = wl.box()
    ctx1 = _ctx(wl.net, wl.B, wl.S, disable_epi_fusion=1, disable_conc_fusion=1)
    n_relax = []
    for c in (ctx, ctx1):           # a plain (non-graph) run with per-class timing on counts the relaxation kernels
        c.timing(True)
        r = c.run(lo, hi, wl.C, wl.alpha, wl.intermediate)
        n_relax.append(c.timing_read()["relax"]["launches"])
        c.timing(False)
    res1 = r
    assert n_relax[0] < n_relax[1], f"the fused epilogue was not taken ({n_relax}): the test does not exercise it"
    for i in wl.net.relu_ids():
        _close(_np(res["pre"][i][0]), _np(res1["pre"][i][0]), f"fused vs unfused l of relu {i}")
        _close(_np(res["pre"][i][1]), _np(res1["pre"][i][1]), f"fused vs unfused u of relu {i}")
    _close(_np(res["lb"]), _np(res1["lb"]), "fused vs unfused lb")
    _close(_np(res["ub"]), _np(res1["ub"]), "fused vs unfused ub")


def test_cfg3_scaled_chunked_equals_unchunked():
    import torch
    wl = W.make(3, scale=16, B=2)
    lo, hi = wl.box()
    r_full = _ctx(wl.net, wl.B, wl.S).run(lo, hi, wl.C, None, "crown")
    c2 = _ctx(wl.net, wl.B, wl.S, mem_cap_bytes=48 << 20)
    r_chunk = c2.run(lo, hi, wl.C, None, "crown")
    assert c2.peak_bytes() <= 48 << 20
    for k in ("lb", "ub"):
        assert torch.equal(r_full[k], r_chunk[k]), k     # rows are independent: chunking is bitwise neutral


def test_cfg4_scaled():
    wl = W.make(4, scale=64, B=2)     # 64-4096-64-10
    _check_workload(wl)


def test_cfg5_scaled():
    wl = W.make(5, scale=4, B=2)
    _check_workload(wl)


def test_streamed_weights_equal_resident_bitwise():
    """a7: layer-wise weight streaming from pinned host memory (PAPER.md:146 hook points) must not change a bit
    (the paper's FSDP argument)."""
    import torch
    wl3 = W.make(3, scale=16, B=2)    # 256-1024-1024-1024-10: tensor-core GEMMs on the streamed layers
    lo, hi = wl3.box()
    r_res = _ctx(wl3.net, wl3.B, wl3.S).run(lo, hi, wl3.C, None, "crown")
    # all hidden layers streamed; a 1 MiB staging cap forces several slabs per layer (W2: 8 MiB prepacked)
    for stage in (0, 1 << 20):
        c2 = _ctx(wl3.net, wl3.B, wl3.S, stream_weights=1, stream_min_elems=1 << 18, stream_stage_bytes=stage)
        assert len(c2.streamed_ids) == 3
        r_str = c2.run(lo, hi, wl3.C, None, "crown")
        assert c2.h2d_bytes() > 0
        for k in ("lb", "ub"):
            assert torch.equal(r_res[k], r_str[k]), k
        for i in r_res["pre"]:
            assert torch.equal(r_res["pre"][i][0], r_str["pre"][i][0]) and torch.equal(r_res["pre"][i][1], r_str["pre"][i][1])


def test_boundary_calls_one_by_one():
    """ibp_forward / crown_backward / concretize called separately through the C-ABI (not via crown_run): O1 against
    the oracle's IBP for every node and the fused spec, O3's A and d against the oracle's linear bounds, and the
    stand-alone concretisation against the fused one."""
    wl = W.make(2, B=4)
    lo, hi = wl.box()
    ctx = _ctx(wl.net, wl.B, wl.S)
    # O1
    ivals, (ilb, iub) = ctx.ibp_forward(lo, hi, wl.C)
    for p in range(wl.B):
        ref = O.ibp(wl.net, lo[p], hi[p])
        for i, (l, u) in enumerate(ref):
            _close(_np(ivals[i][0])[p], l.reshape(-1), f"ibp node {i} l")
            _close(_np(ivals[i][1])[p], u.reshape(-1), f"ibp node {i} u")
        slb, sub = O.ibp_spec(wl.net, lo[p], hi[p], wl.C[p])
        _close(_np(ilb)[p], slb, "ibp spec lb")
        _close(_np(iub)[p], sub, "ibp spec ub")
    # O3 with A and d returned, then a8 on its own
    res = ctx.run(lo, hi, wl.C, wl.alpha, wl.intermediate)
    al = {i: a for i, a in zip(wl.net.relu_ids(), wl.alpha)}
    out = ctx.crown_backward(wl.B, len(wl.net.nodes) - 1, res["pre"], Cmat=wl.C, alpha_lo=al, alpha_up=al,
                             box=(lo, hi), want_A=True)
    lb2, ub2 = ctx.concretize(out["A"], out["d"], lo, hi)
    A, d = _np(out["A"]), _np(out["d"])
    for p in range(wl.B):
        forced = {i: (_np(l)[p].astype(np.float64), _np(u)[p].astype(np.float64)) for i, (l, u) in res["pre"].items()}
        alp = {i: a[p] for i, a in al.items()}
        olb, oub, (A_lo, A_up, d_lo, d_up) = O.final_bounds(wl.net, lo[p], hi[p], wl.C[p], forced, alp, alp)
        _close(A[0, p], A_lo, "A_lo")          # element by element, 1e-5 + 1e-4 |ref|
        _close(A[1, p], A_up, "A_up")
        _close(d[0, p], d_lo, "d_lo")
        _close(d[1, p], d_up, "d_up")
        for g in (_np(out["lb"])[p], _np(lb2)[p], _np(res["lb"])[p]):
            _close(g, olb, "lb")
        for g in (_np(out["ub"])[p], _np(ub2)[p], _np(res["ub"])[p]):
            _close(g, oub, "ub")


@pytest.mark.parametrize("side", [12, 20])
def test_conv_backward_on_map_sizes_off_the_fast_paths(side):
    """ResNets on 12 x 12 and 20 x 20 images: the strip kernel's staging takes its general loop (h w / 4 = 36 / 100 does not
    divide the block size), the 6 x 6 / 10 x 10 maps after the stride-2 block are not a multiple of 4 wide and fall back to
    the generic tiled kernel, the 1x1 skip and the stride-2 3x3 kernels run on maps the benchmark never uses.  Parity on
    lb / ub and on the input-layer coefficients A^0."""
    rng = np.random.Generator(np.random.PCG64(W.SEED_BASE + 7100 + side))
    net = W.resnet(rng, in_shape=(3, side, side), stem=8, blocks=((8, 1), (16, 2), (16, 1)), fc=24, n_classes=6)
    B, S = 2, 5
    x0 = rng.random((B, net.n_in)).astype(np.float32)
    C = rng.standard_normal((B, S, net.n_out)).astype(np.float32)
    al = [rng.random((B, S, net.nodes[i].size)).astype(np.float32) for i in net.relu_ids()]
    wl = W.Workload(cfg=5, name=f"resnet{side}", net=net, x0=x0, eps=np.full((B,), 2.0 / 255.0, np.float32), C=C,
                    labels=np.zeros(B, int), alpha=al, intermediate="ibp", eps_set=(2.0 / 255.0,))
    ctx, res = _check_workload(wl, free_running=False)
    lo, hi = wl.box()
    ald = {i: a for i, a in zip(wl.net.relu_ids(), wl.alpha)}
    out = ctx.crown_backward(wl.B, len(wl.net.nodes) - 1, res["pre"], Cmat=wl.C, alpha_lo=ald, alpha_up=ald,
                             box=(lo, hi), want_A=True)
    A, d = _np(out["A"]), _np(out["d"])
    for p in range(wl.B):
        forced = {i: (_np(l)[p].astype(np.float64), _np(u)[p].astype(np.float64)) for i, (l, u) in res["pre"].items()}
        alp = {i: a[p] for i, a in ald.items()}
        _, _, (A_lo, A_up, d_lo, d_up) = O.final_bounds(wl.net, lo[p], hi[p], wl.C[p], forced, alp, alp)
        for br, ref in ((0, A_lo), (1, A_up)):
            sc = np.abs(ref).max(axis=-1, keepdims=True)       # as in the tensor-core test: cancelling sums over many paths
            err = np.abs(A[br, p] - ref) - (ATOL * sc + RTOL * np.abs(ref))
            assert np.all(err <= 0), f"A^0 branch {br} prop {p}: worst excess {err.max():.3e}"
        _close(d[0, p], d_lo, "d_lo")
        _close(d[1, p], d_up, "d_up")


def test_tensor_core_conv_backward_small_resnet():
    """A 16 x 16, 32-channel ResNet (stem + 2 residual blocks): the 3x3 stride-1 BoundConv backward steps with 32
    channels run as the per-tap implicit GEMM on tcgen05 (conv_tc.cu), one of them with the residual fork's other
    contribution added in its epilogue.  Same parity bar on lb / ub AND on the input-layer coefficients A^0 (every
    conv step feeds them; with IBP intermediates the bias term dominates lb, so lb alone would not see a conv error),
    and the CUDA-core path agrees within the tolerance without being the same arithmetic."""
    rng = np.random.Generator(np.random.PCG64(W.SEED_BASE + 7000))
    net = W.resnet(rng, in_shape=(3, 16, 16), stem=32, blocks=((32, 1), (32, 1)), fc=48, n_classes=12)
    B, S = 2, 7
    x0 = rng.random((B, net.n_in)).astype(np.float32)
    C = rng.standard_normal((B, S, net.n_out)).astype(np.float32)
    al = [rng.random((B, S, net.nodes[i].size)).astype(np.float32) for i in net.relu_ids()]
    wl = W.Workload(cfg=5, name="resnet16x32", net=net, x0=x0, eps=np.full((B,), 2.0 / 255.0, np.float32), C=C,
                    labels=np.zeros(B, int), alpha=al, intermediate="ibp", eps_set=(2.0 / 255.0,))
    ctx, res = _check_workload(wl, free_running=False)   # IBP intermediates, 40k neurons: the forced-bounds protocol is the check
    lo, hi = wl.box()
    ctx2 = _ctx(wl.net, wl.B, wl.S, disable_conv_tc=1)
    res2 = ctx2.run(lo, hi, wl.C, wl.alpha, wl.intermediate)
    _close(_np(res["lb"]), _np(res2["lb"]), "tensor-core vs CUDA-core conv lb")
    _close(_np(res["ub"]), _np(res2["ub"]), "tensor-core vs CUDA-core conv ub")
    ald = {i: a for i, a in zip(wl.net.relu_ids(), wl.alpha)}
    outs = [c.crown_backward(wl.B, len(wl.net.nodes) - 1, res["pre"], Cmat=wl.C, alpha_lo=ald, alpha_up=ald,
                             box=(lo, hi), want_A=True) for c in (ctx, ctx2)]
    A_tc, A_cc = _np(outs[0]["A"]), _np(outs[1]["A"])
    assert not np.array_equal(A_tc, A_cc)                 # the two paths really are different kernels
    for p in range(wl.B):
        forced = {i: (_np(l)[p].astype(np.float64), _np(u)[p].astype(np.float64)) for i, (l, u) in res["pre"].items()}
        alp = {i: a[p] for i, a in ald.items()}
        _, _, (A_lo, A_up, d_lo, d_up) = O.final_bounds(wl.net, lo[p], hi[p], wl.C[p], forced, alp, alp)
        # A^0 entries are cancelling sums over ~10^4 paths: the bar is the stated tolerance with the absolute part
        # scaled to the row's magnitude (fp32 rounding is relative to the summands, not to the cancelled result)
        for k, name in enumerate(("tc", "cuda-core")):
            A, d = (A_tc, A_cc)[k], _np(outs[k]["d"])
            for br, ref in ((0, A_lo), (1, A_up)):
                sc = np.abs(ref).max(axis=-1, keepdims=True)
                err = np.abs(A[br, p] - ref) - (ATOL * sc + RTOL * np.abs(ref))
                assert np.all(err <= 0), f"{name} A^0 branch {br} prop {p}: worst excess {err.max():.3e}"
            _close(d[0, p], d_lo, f"{name} d_lo")
            _close(d[1, p], d_up, f"{name} d_up")
