"""Seeded synthetic workloads for the five BASELINE.json configs.

This module is the ONLY code shared by the CPU oracle (`oracle/`) and the CUDA
path (`paper_2606_09377_b200/`).  It holds network descriptions and random
inputs and NONE of the method's arithmetic (no IBP, no relaxation, no
backward propagation, no concretisation).  The one numerical routine here,
`label_forward`, is a plain float64 evaluation of the network at x0, used only
to pick the label y = argmax f(x0) that defines the margin specification
(SURVEY.md §8(c) G12); it is network evaluation, not bound propagation.

The inputs stand in for the paper's workloads, which are not available
offline: VNN-COMP MNIST-FC 256xN MLPs, the wide
4096->262144 MLP of Experiment 1, the h x d MLPs of
Experiment 5 and the CIFAR-100 ResNets of Experiment 8
(PAPER.md:291).  Only shapes, eps values and input ranges are taken from the
paper; weights are He-normal random, no benchmark item is reproduced.

Recipe (restated in DESIGN.md):
  weights  ~ N(0, 2/fan_in)           (He-normal; fan_in = n_in or C_in*kh*kw)
  biases   ~ N(0, 0.01)  (variance => std 0.1)
  alpha    ~ U[0,1] per (property, spec row, neuron)
  x0       ~ U[0,1]^n0 (cfg 1,2,5) or N(0,1)^n0 (cfg 3,4)
  generator: numpy Generator(PCG64(seed)), seed = 26060937700 + 10*cfg + stream
  stream: 0 weights, 1 inputs, 2 alpha, 3 samples
  every value is drawn in float64 and rounded ONCE to float32.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Optional, Tuple

import numpy as np

SEED_BASE = 26060937700

LINEAR, CONV, RELU, ADD, FLATTEN = "linear", "conv", "relu", "add", "flatten"


@dataclass
class Node:
    """One node of a topologically ordered DAG. in0/in1 = producer ids, -1 = network input."""
    op: str
    in0: int
    in1: int = -1
    W: Optional[np.ndarray] = None      # linear: [n_out, n_in]; conv: [C_out, C_in, kh, kw]; float32
    b: Optional[np.ndarray] = None      # [n_out] / [C_out]; float32
    stride: int = 1
    pad: int = 0
    shape: Tuple[int, ...] = ()         # output shape: (n,) or (C, H, W)

    @property
    def size(self) -> int:
        return int(np.prod(self.shape))


@dataclass
class Net:
    in_shape: Tuple[int, ...]
    nodes: List[Node] = field(default_factory=list)

    @property
    def n_in(self) -> int:
        return int(np.prod(self.in_shape))

    @property
    def n_out(self) -> int:
        return self.nodes[-1].size

    def shape_of(self, idx: int) -> Tuple[int, ...]:
        return self.in_shape if idx < 0 else self.nodes[idx].shape

    def relu_ids(self) -> List[int]:
        return [i for i, n in enumerate(self.nodes) if n.op == RELU]


def rng_for(cfg: int, stream: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(SEED_BASE + 10 * cfg + stream))


def _normal32(rng: np.random.Generator, shape, std: float) -> np.ndarray:
    """N(0, std^2) drawn in float64, rounded once to float32; chunked so huge layers fit in RAM."""
    n = int(np.prod(shape))
    out = np.empty(n, dtype=np.float32)
    step = 1 << 24
    for s in range(0, n, step):
        e = min(n, s + step)
        out[s:e] = (rng.standard_normal(e - s) * std).astype(np.float32)
    return out.reshape(shape)


def _add_linear(net: Net, rng, src: int, n_out: int) -> int:
    n_in = int(np.prod(net.shape_of(src)))
    W = _normal32(rng, (n_out, n_in), np.sqrt(2.0 / n_in))
    b = _normal32(rng, (n_out,), 0.1)
    net.nodes.append(Node(LINEAR, src, W=W, b=b, shape=(n_out,)))
    return len(net.nodes) - 1


def _add_conv(net: Net, rng, src: int, c_out: int, k: int, stride: int, pad: int) -> int:
    c_in, h, w = net.shape_of(src)
    W = _normal32(rng, (c_out, c_in, k, k), np.sqrt(2.0 / (c_in * k * k)))
    b = _normal32(rng, (c_out,), 0.1)
    ho = (h + 2 * pad - k) // stride + 1
    wo = (w + 2 * pad - k) // stride + 1
    net.nodes.append(Node(CONV, src, W=W, b=b, stride=stride, pad=pad, shape=(c_out, ho, wo)))
    return len(net.nodes) - 1


def _add_relu(net: Net, src: int) -> int:
    net.nodes.append(Node(RELU, src, shape=net.shape_of(src)))
    return len(net.nodes) - 1


def _add_add(net: Net, a: int, b: int) -> int:
    assert net.shape_of(a) == net.shape_of(b)
    net.nodes.append(Node(ADD, a, b, shape=net.shape_of(a)))
    return len(net.nodes) - 1


def _add_flatten(net: Net, src: int) -> int:
    net.nodes.append(Node(FLATTEN, src, shape=(int(np.prod(net.shape_of(src))),)))
    return len(net.nodes) - 1


def mlp(widths, rng) -> Net:
    """ReLU MLP widths[0] -> ... -> widths[-1]; ReLU after every layer but the last."""
    net = Net(in_shape=(int(widths[0]),))
    cur = -1
    for k, n_out in enumerate(widths[1:], start=1):
        cur = _add_linear(net, rng, cur, int(n_out))
        if k < len(widths) - 1:
            cur = _add_relu(net, cur)
    return net


def resnet(rng, in_shape=(3, 32, 32), stem=16, blocks=((16, 1), (32, 2), (32, 1), (64, 2)),
           fc=512, n_classes=100) -> Net:
    """CIFAR-100-shaped ResNet of BASELINE.json cfg5.

    stem conv3x3(s1,p1)+ReLU; block: ReLU(conv2(ReLU(conv1(x))) + skip(x)), conv1 carries the
    stride; skip = identity when the shape is kept, else conv1x1 with the block's stride and a
    bias; flatten; FC fc + ReLU; FC n_classes.
    """
    net = Net(in_shape=tuple(in_shape))
    cur = _add_conv(net, rng, -1, stem, 3, 1, 1)
    cur = _add_relu(net, cur)
    for c_out, stride in blocks:
        x = cur
        c_in = net.shape_of(x)[0]
        h = _add_conv(net, rng, x, c_out, 3, stride, 1)
        h = _add_relu(net, h)
        h = _add_conv(net, rng, h, c_out, 3, 1, 1)
        if stride != 1 or c_in != c_out:
            s = _add_conv(net, rng, x, c_out, 1, stride, 0)
        else:
            s = x
        cur = _add_add(net, h, s)
        cur = _add_relu(net, cur)
    cur = _add_flatten(net, cur)
    cur = _add_linear(net, rng, cur, fc)
    cur = _add_relu(net, cur)
    _add_linear(net, rng, cur, n_classes)
    return net


# ----------------------------------------------------------------------------------------
# label + margin specification (network evaluation only; NOT part of the verified method)
# ----------------------------------------------------------------------------------------
def _conv_eval(x: np.ndarray, W: np.ndarray, b: np.ndarray, stride: int, pad: int) -> np.ndarray:
    c_out, c_in, kh, kw = W.shape
    xp = np.pad(x, ((0, 0), (pad, pad), (pad, pad)))
    ho = (xp.shape[1] - kh) // stride + 1
    wo = (xp.shape[2] - kw) // stride + 1
    y = np.zeros((c_out, ho, wo))
    for i in range(kh):
        for j in range(kw):
            patch = xp[:, i:i + stride * ho:stride, j:j + stride * wo:stride]
            y += np.einsum("oc,chw->ohw", W[:, :, i, j].astype(np.float64), patch)
    return y + b.astype(np.float64)[:, None, None]


def label_forward(net: Net, x: np.ndarray) -> np.ndarray:
    """f(x) in float64 for ONE input x (shape net.in_shape or flat). Used only to pick labels."""
    vals = []
    x = np.asarray(x, dtype=np.float64).reshape(net.in_shape)
    for n in net.nodes:
        a = x if n.in0 < 0 else vals[n.in0]
        if n.op == LINEAR:
            v = n.W.astype(np.float64) @ a.reshape(-1) + n.b.astype(np.float64)
        elif n.op == CONV:
            v = _conv_eval(a, n.W, n.b, n.stride, n.pad)
        elif n.op == RELU:
            v = np.maximum(a, 0.0)
        elif n.op == ADD:
            v = a + (x if n.in1 < 0 else vals[n.in1])
        elif n.op == FLATTEN:
            v = a.reshape(-1)
        else:
            raise ValueError(n.op)
        vals.append(v)
    return vals[-1]


def margin_spec(n_classes: int, y: int) -> np.ndarray:
    """Rows e_y - e_j for j != y ascending. float32 [n_classes-1, n_classes]."""
    C = np.zeros((n_classes - 1, n_classes), dtype=np.float32)
    r = 0
    for j in range(n_classes):
        if j == y:
            continue
        C[r, y] = 1.0
        C[r, j] = -1.0
        r += 1
    return C


@dataclass
class Workload:
    cfg: int
    name: str
    net: Net
    x0: np.ndarray            # [B, n0] float32
    eps: np.ndarray           # [B] float32
    C: np.ndarray             # [B, S, n_out] float32
    labels: np.ndarray        # [B] int
    alpha: Optional[List[np.ndarray]]   # per ReLU node (topological order): [B, S, n_k] float32, or None
    intermediate: str         # "crown" (full CROWN intermediate bounds) or "ibp" (cfg5, G22)
    eps_set: Tuple[float, ...] = ()      # cfg2: the three eps values, each run as its own batch (G13)

    @property
    def B(self) -> int:
        return self.x0.shape[0]

    @property
    def S(self) -> int:
        return self.C.shape[1]

    def box(self):
        lo = (self.x0.astype(np.float64) - self.eps.astype(np.float64)[:, None]).astype(np.float32)
        hi = (self.x0.astype(np.float64) + self.eps.astype(np.float64)[:, None]).astype(np.float32)
        return lo, hi


def _specs(net: Net, x0: np.ndarray):
    labels = np.array([int(np.argmax(label_forward(net, x))) for x in x0])
    C = np.stack([margin_spec(net.n_out, int(y)) for y in labels])
    return labels, C


def _alpha(cfg: int, net: Net, B: int, S: int):
    rng = rng_for(cfg, 2)
    return [rng.random((B, S, net.nodes[i].size)).astype(np.float32) for i in net.relu_ids()]


def make(cfg: int, scale: int = 1, B: Optional[int] = None, eps: Optional[float] = None) -> Workload:
    """Build BASELINE.json config `cfg` (1..5).

    scale > 1 divides every layer width except the output (cfg 1-4) to give the width-scaled
    copies used for full free-running parity (SURVEY.md §8(c) "Oracle cost"); for cfg5 it
    shrinks the image side and channel counts.  B / eps override the batch size and radius.
    """
    wrng = rng_for(cfg, 0)
    irng = rng_for(cfg, 1)
    s = int(scale)
    if cfg == 1:
        net = mlp([784 // s, 256 // s, 256 // s, 10], wrng)
        B_, eps_, dist, alpha, inter, name = 1, 0.02, "u", True, "crown", "mlp_784_256x2_10"
    elif cfg == 2:
        net = mlp([784 // s] + [256 // s] * 6 + [10], wrng)
        B_, eps_, dist, alpha, inter, name = 64, 0.026, "u", True, "crown", "mnistfc_784_256x6_10"
    elif cfg == 3:
        net = mlp([4096 // s] + [16384 // s] * 3 + [10], wrng)
        B_, eps_, dist, alpha, inter, name = 16, 0.01, "n", False, "crown", "wide_4096_16384x3_10"
    elif cfg == 4:
        net = mlp([4096 // s, 262144 // s, 4096 // s, 10], wrng)
        B_, eps_, dist, alpha, inter, name = 4, 0.005, "n", False, "crown", "vwide_4096_262144_4096_10"
    elif cfg == 5:
        if s == 1:
            net = resnet(wrng)
        else:
            side = max(8, 32 // s)
            ch = lambda c: max(2, c // s)
            net = resnet(wrng, in_shape=(3, side, side), stem=ch(16),
                         blocks=((ch(16), 1), (ch(32), 2), (ch(32), 1), (ch(64), 2)),
                         fc=max(8, 512 // s), n_classes=max(4, 100 // s))
        B_, eps_, dist, alpha, inter, name = 8, 2.0 / 255.0, "u", True, "ibp", "resnet_cifar100"
    else:
        raise ValueError(f"cfg must be 1..5, got {cfg}")
    B_ = B_ if B is None else int(B)
    eps_ = eps_ if eps is None else float(eps)
    n0 = net.n_in
    if dist == "u":
        x0 = irng.random((B_, n0)).astype(np.float32)
    else:
        x0 = irng.standard_normal((B_, n0)).astype(np.float32)
    labels, C = _specs(net, x0)
    al = _alpha(cfg, net, B_, C.shape[1]) if alpha else None
    return Workload(cfg=cfg, name=name + (f"_div{s}" if s > 1 else ""), net=net, x0=x0,
                    eps=np.full((B_,), eps_, dtype=np.float32), C=C, labels=labels, alpha=al,
                    intermediate=inter, eps_set=(0.015, 0.026, 0.05) if cfg == 2 else (eps_,))


def stack_eps(wl: Workload) -> Workload:
    """All eps values of a workload as ONE batch: property p of the result is point p % B with radius
    eps_set[p // B] (eps is a per-property input of the boundary, so the three batches of cfg2 are one
    call of 3*B properties, reading G13).  C, labels and alpha repeat per eps."""
    k = len(wl.eps_set)
    if k <= 1:
        return wl
    eps = np.concatenate([np.full((wl.B,), e, dtype=np.float32) for e in wl.eps_set])
    al = None if wl.alpha is None else [np.concatenate([a] * k, axis=0) for a in wl.alpha]
    return Workload(cfg=wl.cfg, name=wl.name + f"_x{k}eps", net=wl.net, x0=np.concatenate([wl.x0] * k, axis=0),
                    eps=eps, C=np.concatenate([wl.C] * k, axis=0), labels=np.concatenate([wl.labels] * k),
                    alpha=al, intermediate=wl.intermediate, eps_set=(float("nan"),))


def small_mlp(widths, seed: int, B: int = 2, eps: float = 0.1, S: Optional[int] = None,
              with_alpha: bool = True, bias_shift: float = 0.0, weight_scale: float = 1.0) -> Workload:
    """Tiny seeded MLP workload for unit tests / brute force. bias_shift is added to the hidden
    biases and weight_scale multiplies every weight (small weights + positive shift => all-active,
    negative shift => all-inactive nets)."""
    rng = np.random.Generator(np.random.PCG64(SEED_BASE + 1000 + seed))
    net = mlp(list(widths), rng)
    for n in net.nodes:
        if n.op == LINEAR:
            if weight_scale != 1.0:
                n.W = (n.W.astype(np.float64) * weight_scale).astype(np.float32)
            if bias_shift != 0.0 and n is not net.nodes[-1]:
                n.b = (n.b.astype(np.float64) + bias_shift).astype(np.float32)
    x0 = (rng.random((B, net.n_in)) * 2.0 - 1.0).astype(np.float32)
    if S is None:
        labels, C = _specs(net, x0)
    else:
        labels = np.zeros(B, dtype=int)
        C = rng.standard_normal((B, S, net.n_out)).astype(np.float32)
    al = None
    if with_alpha:
        al = [rng.random((B, C.shape[1], net.nodes[i].size)).astype(np.float32) for i in net.relu_ids()]
    return Workload(cfg=0, name="small_mlp_" + "_".join(map(str, widths)), net=net, x0=x0,
                    eps=np.full((B,), eps, dtype=np.float32), C=C, labels=labels, alpha=al,
                    intermediate="crown", eps_set=(eps,))


def sample_points(cfg: int, lo: np.ndarray, hi: np.ndarray, n_uniform: int, n_corner: int) -> np.ndarray:
    """Seeded probe points inside the box [lo, hi] of ONE property:
    n_uniform uniform points, n_corner random corners, and the centre. float64 [n, n0]."""
    rng = rng_for(cfg, 3)
    lo = lo.astype(np.float64)
    hi = hi.astype(np.float64)
    u = lo[None, :] + rng.random((n_uniform, lo.size)) * (hi - lo)[None, :]
    c = np.where(rng.random((n_corner, lo.size)) < 0.5, lo[None, :], hi[None, :])
    return np.concatenate([u, c, 0.5 * (lo + hi)[None, :]], axis=0)
