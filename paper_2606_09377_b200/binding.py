"""Thin ctypes binding of libcrownb200.so (include/crownb200.h).  Argument marshalling only: every
step of the path runs in the library's CUDA kernels.  PyTorch is used for device memory and streams.
There is no CPU fallback: loading fails loudly when the library is missing, and every compute call
needs a CUDA device.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Dict, List, Optional, Sequence

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libcrownb200.so")

OP_CODES = {"linear": 1, "conv": 2, "relu": 3, "add": 4, "flatten": 5}
K_CLASSES = ["ibp", "coeff", "relax", "gemm_tc", "gemm_ffma", "concretize", "conv", "misc"]

EXPORTS = ["crown_h2d_bytes", "crown_workspace_bytes", "crown_init", "ibp_forward", "crown_backward", "concretize", "crown_verdict", "crown_run",
           "crown_run_host", "crown_alpha_scratch_bytes", "crown_alpha_grad", "crown_alpha_ascent", "crown_backward_split", "crown_beta_grad", "crown_beta_ascent", "crown_gemm", "crown_split_tf32", "crown_peak_bytes", "crown_row_chunk", "crown_launch_count", "crown_graph_replays",
           "crown_gemm_flops", "crown_timing", "crown_timing_read", "crown_last_error", "crown_destroy",
           "crown_version", "crown_gemm_noalloc", "crown_gemm_noalloc_max_elems", "crown_gemm_noalloc_error"]


class CrownNode(C.Structure):
    _fields_ = [("op", C.c_int32), ("in0", C.c_int32), ("in1", C.c_int32), ("n_out", C.c_int32),
                ("n_in", C.c_int32), ("c_out", C.c_int32), ("c_in", C.c_int32), ("kh", C.c_int32),
                ("kw", C.c_int32), ("stride", C.c_int32), ("pad", C.c_int32), ("h_in", C.c_int32),
                ("w_in", C.c_int32), ("W_dev", C.c_void_p), ("b_dev", C.c_void_p), ("W_host", C.c_void_p)]


class CrownOpts(C.Structure):
    _fields_ = [("mem_cap_bytes", C.c_uint64), ("stream_weights", C.c_int32), ("mma_scheme", C.c_int32),
                ("slope_rule", C.c_int32), ("k_drain", C.c_int32), ("stream_min_elems", C.c_uint64),
                ("stream_stage_bytes", C.c_uint64), ("disable_epi_fusion", C.c_int32),
                ("disable_conc_fusion", C.c_int32), ("disable_graph", C.c_int32), ("disable_conv_tc", C.c_int32)]


class CrownError(RuntimeError):
    pass


_lib = None


def load_library() -> C.CDLL:
    """Loads the C-ABI library; raises if it was not built (python -m paper_2606_09377_b200.build)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise CrownError(f"{LIB_PATH} is missing: build it with `python -m paper_2606_09377_b200.build` "
                         "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    for name in EXPORTS:
        getattr(lib, name)   # AttributeError if a declared symbol is not exported
    lib.crown_last_error.restype = C.c_char_p
    lib.crown_last_error.argtypes = [C.c_void_p]
    lib.crown_version.restype = C.c_char_p
    vp, i32 = C.c_void_p, C.c_int
    lib.crown_workspace_bytes.argtypes = [C.POINTER(CrownNode), i32, i32, i32, i32, i32, i32,
                                          C.POINTER(CrownOpts), C.POINTER(C.c_size_t)]
    lib.crown_init.argtypes = [C.POINTER(vp), C.POINTER(CrownNode), i32, i32, i32, i32, i32, i32, vp, C.c_size_t,
                               C.POINTER(CrownOpts), vp]
    lib.ibp_forward.argtypes = [vp, i32, vp, vp, C.POINTER(vp), C.POINTER(vp), vp, i32, vp, vp]
    lib.crown_backward.argtypes = [vp, i32, i32, i32, i32, vp, C.POINTER(vp), C.POINTER(vp), C.POINTER(vp),
                                   C.POINTER(vp), vp, vp, vp, vp, vp, vp]
    lib.concretize.argtypes = [vp, i32, i32, vp, vp, vp, vp, vp, vp, i32]
    lib.crown_verdict.argtypes = [vp, i32, i32, vp, vp]
    lib.crown_run.argtypes = [vp, i32, vp, vp, vp, i32, C.POINTER(vp), i32, C.POINTER(vp), C.POINTER(vp), vp, vp, vp]
    lib.crown_run_host.argtypes = [vp, i32, vp, vp, vp, i32, C.POINTER(vp), i32, vp, vp, vp]
    lib.crown_alpha_scratch_bytes.argtypes = [vp, i32, i32, C.POINTER(C.c_size_t)]
    lib.crown_alpha_grad.argtypes = [vp, i32, vp, i32, C.POINTER(vp), C.POINTER(vp), C.POINTER(vp), C.POINTER(vp), vp, vp,
                                     C.POINTER(vp), C.POINTER(vp), vp, vp, vp, C.c_size_t]
    lib.crown_alpha_ascent.argtypes = [vp, i32, vp, i32, C.POINTER(vp), C.POINTER(vp), C.POINTER(vp), C.POINTER(vp), vp, vp,
                                       C.c_float, C.c_float, i32, i32, vp, vp, vp, vp, vp, vp, C.c_size_t]
    pp = C.POINTER(vp)
    lib.crown_backward_split.argtypes = [vp, i32, i32, i32, i32, vp, pp, pp, pp, pp, pp, pp, pp, vp, vp, vp, vp, vp, vp]
    lib.crown_beta_grad.argtypes = [vp, i32, vp, i32, pp, pp, pp, pp, pp, pp, pp, vp, vp, pp, pp, pp, pp, vp, vp, vp, C.c_size_t]
    lib.crown_beta_ascent.argtypes = [vp, i32, vp, i32, pp, pp, pp, pp, pp, pp, pp, vp, vp, C.c_float, C.c_float, C.c_float,
                                      i32, i32, vp, vp, vp, vp, vp, vp, C.c_size_t]
    lib.crown_gemm.argtypes = [vp, i32, i32, i32, i32, vp, vp, vp, vp, vp]
    lib.crown_split_tf32.argtypes = [vp, vp, i32, i32, i32, vp, vp]
    lib.crown_peak_bytes.argtypes = [vp, C.POINTER(C.c_size_t)]
    lib.crown_row_chunk.argtypes = [vp, C.POINTER(C.c_int)]
    lib.crown_launch_count.argtypes = [vp, C.POINTER(C.c_uint64)]
    lib.crown_graph_replays.argtypes = [vp, C.POINTER(C.c_uint64)]
    lib.crown_gemm_flops.argtypes = [vp, C.POINTER(C.c_double)]
    lib.crown_h2d_bytes.argtypes = [vp, C.POINTER(C.c_double)]
    lib.crown_timing.argtypes = [vp, i32]
    lib.crown_timing_read.argtypes = [vp, i32, C.POINTER(C.c_double), C.POINTER(C.c_uint64),
                                      C.POINTER(C.c_double), C.POINTER(C.c_double)]
    lib.crown_destroy.argtypes = [vp]
    lib.crown_gemm_noalloc.argtypes = [i32, i32, i32, vp, vp, vp, vp]
    lib.crown_gemm_noalloc_max_elems.argtypes = []
    lib.crown_gemm_noalloc_error.restype = C.c_char_p
    lib.crown_gemm_noalloc_error.argtypes = []
    _lib = lib
    return lib


def gemm_noalloc(A: torch.Tensor, W: torch.Tensor, out: Optional[torch.Tensor] = None) -> torch.Tensor:
    """D[M,N] = A[M,K] . W[K,N] through crown_gemm_noalloc: the 3xTF32 tcgen05 contraction with its operand limbs in the
    library's static device scratch (no context, no device allocation inside the call; `out` lets the caller bring D
    too).  Queued on torch's current stream of A's device.  Calls that overlap on the GPU race on the scratch."""
    lib = load_library()
    if not (A.is_cuda and W.is_cuda and A.dtype == torch.float32 and W.dtype == torch.float32
            and A.is_contiguous() and W.is_contiguous() and A.dim() == 2 and W.dim() == 2 and A.shape[1] == W.shape[0]):
        raise CrownError("gemm_noalloc: A [M,K] and W [K,N] must be contiguous float32 CUDA tensors")
    M, K = A.shape
    N = W.shape[1]
    if out is None:
        out = torch.empty(M, N, device=A.device)
    elif not (out.is_cuda and out.dtype == torch.float32 and out.is_contiguous() and tuple(out.shape) == (M, N)):
        raise CrownError("gemm_noalloc: out must be a contiguous float32 CUDA tensor [M,N]")
    with torch.cuda.device(A.device):
        rc = lib.crown_gemm_noalloc(M, N, K, A.data_ptr(), W.data_ptr(), out.data_ptr(),
                                    torch.cuda.current_stream().cuda_stream)
        if rc != 0:
            raise CrownError(f"[{rc}] " + lib.crown_gemm_noalloc_error().decode())
    return out


def _ptr(t: Optional[torch.Tensor]) -> Optional[int]:
    return None if t is None else t.data_ptr()


class CrownContext:
    """crown_init / ibp_forward / crown_backward / concretize / crown_run over torch device tensors.

    net: any object with .in_shape and .nodes, each node having op ('linear'|'conv'|'relu'|'add'|'flatten'),
    in0, in1, W, b (numpy float32), stride, pad, shape (output shape)."""

    def __init__(self, net, B_max: int, S_max: int, device: str = "cuda:0", mem_cap_bytes: int = 0,
                 mma_scheme: int = 0, slope_rule: int = 0, k_drain: int = 0, stream_weights: int = 0,
                 stream_min_elems: int = 0, stream_stage_bytes: int = 0, disable_epi_fusion: int = 0,
                 disable_conc_fusion: int = 0, disable_graph: int = 0, disable_conv_tc: int = 0):
        if not torch.cuda.is_available():
            raise CrownError("no CUDA device: the crownb200 hot path has no CPU fallback")
        self.lib = load_library()
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.net = net
        self.n_nodes = len(net.nodes)
        in_shape = tuple(net.in_shape)
        self.in_chw = in_shape if len(in_shape) == 3 else (int(np.prod(in_shape)), 1, 1)
        self.n0 = int(np.prod(in_shape))
        self.sizes = [int(np.prod(n.shape)) for n in net.nodes]
        self.relu_ids = [i for i, n in enumerate(net.nodes) if n.op == "relu"]
        self.B_max, self.S_max = int(B_max), int(S_max)
        self._keep: List[torch.Tensor] = []
        self.streamed_ids: List[int] = []
        arr = (CrownNode * self.n_nodes)()
        for i, n in enumerate(net.nodes):
            cn = arr[i]
            cn.op, cn.in0, cn.in1 = OP_CODES[n.op], n.in0, (n.in1 if n.op == "add" else -1)
            if n.op == "linear":
                cn.n_out, cn.n_in = n.W.shape
            elif n.op == "conv":
                src = in_shape if n.in0 < 0 else net.nodes[n.in0].shape
                cn.c_out, cn.c_in, cn.kh, cn.kw = n.W.shape
                cn.stride, cn.pad, cn.h_in, cn.w_in = n.stride, n.pad, src[1], src[2]
            if n.op in ("linear", "conv"):
                bd = torch.from_numpy(np.ascontiguousarray(n.b, dtype=np.float32)).to(self.device)
                self._keep.append(bd)
                cn.b_dev = bd.data_ptr()
                min_elems = stream_min_elems or (1 << 28)
                if stream_weights and n.op == "linear" and n.W.size >= min_elems:
                    # streamed layer: no resident copy, only a pinned host buffer the library copies from
                    Wh = torch.from_numpy(np.ascontiguousarray(n.W, dtype=np.float32)).pin_memory()
                    self._keep.append(Wh)
                    cn.W_dev, cn.W_host = None, Wh.data_ptr()
                    self.streamed_ids.append(i)
                else:
                    Wd = torch.from_numpy(np.ascontiguousarray(n.W, dtype=np.float32)).to(self.device)
                    self._keep.append(Wd)
                    cn.W_dev = Wd.data_ptr()
        self._nodes = arr
        self.opts = CrownOpts(mem_cap_bytes, stream_weights, mma_scheme, slope_rule, k_drain, stream_min_elems,
                              stream_stage_bytes, disable_epi_fusion, disable_conc_fusion, disable_graph, disable_conv_tc)
        need = C.c_size_t(0)
        self._check(self.lib.crown_workspace_bytes(arr, self.n_nodes, *self.in_chw, self.B_max, self.S_max,
                                                   C.byref(self.opts), C.byref(need)), None)
        self.workspace_bytes = need.value
        self.workspace = torch.empty(need.value, dtype=torch.uint8, device=self.device)
        self.stream = torch.cuda.current_stream(self.device)
        h = C.c_void_p()
        rc = self.lib.crown_init(C.byref(h), arr, self.n_nodes, *self.in_chw, self.B_max, self.S_max,
                                 self.workspace.data_ptr(), need.value, C.byref(self.opts),
                                 C.c_void_p(self.stream.cuda_stream))
        if rc != 0 or not h.value:
            raise CrownError(f"crown_init failed with status {rc}")
        self.h = h

    # ---- helpers -----------------------------------------------------------------------------
    def _check(self, rc: int, h):
        if rc != 0:
            msg = self.lib.crown_last_error(h).decode() if h is not None else ""
            raise CrownError(f"crownb200 status {rc}: {msg}")

    def _dev(self, x, dtype=torch.float32) -> torch.Tensor:
        if isinstance(x, torch.Tensor):
            return x.to(device=self.device, dtype=dtype).contiguous()
        return torch.from_numpy(np.ascontiguousarray(x)).to(device=self.device, dtype=dtype)

    def _ptr_array(self, tensors: Optional[Dict[int, torch.Tensor]]):
        arr = (C.c_void_p * self.n_nodes)()
        if tensors:
            for i, t in tensors.items():
                arr[i] = None if t is None else t.data_ptr()
        return arr

    def close(self):
        if getattr(self, "h", None) is not None and self.h.value:
            self.lib.crown_destroy(self.h)
            self.h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- the four calls of the boundary --------------------------------------------------------
    def ibp_forward(self, x_lo, x_hi, Cmat=None, nodes: Optional[Sequence[int]] = None):
        """O1.  Returns ({node id: (l, u)} for `nodes` (default: all), (lb, ub) or None)."""
        x_lo, x_hi = self._dev(x_lo), self._dev(x_hi)
        B = x_lo.shape[0]
        want = range(self.n_nodes) if nodes is None else nodes
        L = {i: torch.empty(B, self.sizes[i], device=self.device) for i in want}
        U = {i: torch.empty(B, self.sizes[i], device=self.device) for i in want}
        lb = ub = None
        S = 0
        if Cmat is not None:
            Cmat = self._dev(Cmat)
            S = Cmat.shape[1]
            lb = torch.empty(B, S, device=self.device)
            ub = torch.empty(B, S, device=self.device)
        self._check(self.lib.ibp_forward(self.h, B, x_lo.data_ptr(), x_hi.data_ptr(), self._ptr_array(L),
                                         self._ptr_array(U), _ptr(Cmat), S, _ptr(lb), _ptr(ub)), self.h)
        return {i: (L[i], U[i]) for i in want}, (None if Cmat is None else (lb, ub))

    def crown_backward(self, B: int, start: int, pre: Dict[int, tuple], Cmat=None, row0: int = 0,
                       rows: Optional[int] = None, alpha_lo: Optional[Dict[int, torch.Tensor]] = None,
                       alpha_up: Optional[Dict[int, torch.Tensor]] = None, box=None, want_A: bool = True):
        """O3.  pre: {relu id: (l, u)} device tensors [B, n].  Returns dict with A [2,B,R,n0], d [2,B,R] and,
        if box=(x_lo, x_hi) is given, lb/ub [B,R]."""
        if Cmat is not None:
            Cmat = self._dev(Cmat)
            rows = Cmat.shape[1]
        assert rows is not None
        l = {i: self._dev(v[0]) for i, v in pre.items()}
        u = {i: self._dev(v[1]) for i, v in pre.items()}
        al = None if alpha_lo is None else {i: self._dev(v) for i, v in alpha_lo.items()}
        au = al if alpha_up is alpha_lo else (None if alpha_up is None else {i: self._dev(v) for i, v in alpha_up.items()})
        A = torch.empty(2, B, rows, self.n0, device=self.device) if want_A else None
        d = torch.empty(2, B, rows, device=self.device)
        x_lo = x_hi = lb = ub = None
        if box is not None:
            x_lo, x_hi = self._dev(box[0]), self._dev(box[1])
            lb = torch.empty(B, rows, device=self.device)
            ub = torch.empty(B, rows, device=self.device)
        self._check(self.lib.crown_backward(self.h, B, start, row0, rows, _ptr(Cmat), self._ptr_array(l),
                                            self._ptr_array(u), self._ptr_array(al) if al else None,
                                            self._ptr_array(au) if au else None, _ptr(A), _ptr(d), _ptr(x_lo),
                                            _ptr(x_hi), _ptr(lb), _ptr(ub)), self.h)
        return {"A": A, "d": d, "lb": lb, "ub": ub}

    def concretize(self, A: torch.Tensor, d: torch.Tensor, x_lo, x_hi):
        x_lo, x_hi = self._dev(x_lo), self._dev(x_hi)
        _, B, R, _ = A.shape
        lb = torch.empty(B, R, device=self.device)
        ub = torch.empty(B, R, device=self.device)
        self._check(self.lib.concretize(self.h, B, R, A.data_ptr(), d.data_ptr(), x_lo.data_ptr(), x_hi.data_ptr(),
                                        lb.data_ptr(), ub.data_ptr(), R), self.h)
        return lb, ub

    def verdict(self, lb: torch.Tensor) -> torch.Tensor:
        """a9: verified[b] = 1 iff every lb[b, s] > 0 (device kernel)."""
        B, S = lb.shape
        v = torch.empty(B, dtype=torch.uint8, device=self.device)
        self._check(self.lib.crown_verdict(self.h, B, S, lb.data_ptr(), v.data_ptr()), self.h)
        return v

    # ---- whole path ----------------------------------------------------------------------------
    def alloc_io(self, B: int, S: int):
        """Device outputs of crown_run for batch B: per-ReLU (l, u), lb, ub, verified."""
        l = {i: torch.empty(B, self.sizes[i], device=self.device) for i in self.relu_ids}
        u = {i: torch.empty(B, self.sizes[i], device=self.device) for i in self.relu_ids}
        lb = torch.empty(B, S, device=self.device)
        ub = torch.empty(B, S, device=self.device)
        ver = torch.empty(B, dtype=torch.uint8, device=self.device)
        return {"l": l, "u": u, "lb": lb, "ub": ub, "verified": ver}

    def run_device(self, x_lo: torch.Tensor, x_hi: torch.Tensor, Cmat: torch.Tensor,
                   alpha: Optional[Dict[int, torch.Tensor]], intermediate: int, io) -> None:
        """crown_run on tensors already resident in HBM; asynchronous on the context's stream."""
        B, S = Cmat.shape[0], Cmat.shape[1]
        self._check(self.lib.crown_run(self.h, B, x_lo.data_ptr(), x_hi.data_ptr(), Cmat.data_ptr(), S,
                                       self._ptr_array(alpha) if alpha else None, intermediate,
                                       self._ptr_array(io["l"]), self._ptr_array(io["u"]), io["lb"].data_ptr(),
                                       io["ub"].data_ptr(), io["verified"].data_ptr()), self.h)

    def run(self, x_lo, x_hi, Cmat, alpha: Optional[Sequence] = None, intermediate: str = "crown"):
        """O4 + O5 + verdict.  alpha: per ReLU (topological order) [B,S,n_k] or None.  Returns dict of device
        tensors: pre {relu id: (l,u)}, lb, ub, verified."""
        x_lo, x_hi, Cmat = self._dev(x_lo), self._dev(x_hi), self._dev(Cmat)
        al = None
        if alpha is not None:
            al = {i: self._dev(a) for i, a in zip(self.relu_ids, alpha)}
        io = self.alloc_io(Cmat.shape[0], Cmat.shape[1])
        self.run_device(x_lo, x_hi, Cmat, al, 1 if intermediate == "ibp" else 0, io)
        self.stream.synchronize()
        return {"pre": {i: (io["l"][i], io["u"][i]) for i in self.relu_ids}, "lb": io["lb"], "ub": io["ub"],
                "verified": io["verified"]}

    def run_host(self, x_lo: np.ndarray, x_hi: np.ndarray, Cmat: np.ndarray, alpha: Optional[Sequence[np.ndarray]],
                 intermediate: str, lb: np.ndarray, ub: np.ndarray, verified: np.ndarray) -> None:
        """crown_run_host: HOST (ideally pinned) numpy buffers in and out; H2D/D2H copies inside the call."""
        B, S = Cmat.shape[0], Cmat.shape[1]
        arr = None
        if alpha is not None:
            arr = (C.c_void_p * self.n_nodes)()
            for i, a in zip(self.relu_ids, alpha):
                arr[i] = a.ctypes.data
        self._check(self.lib.crown_run_host(self.h, B, x_lo.ctypes.data, x_hi.ctypes.data, Cmat.ctypes.data, S, arr,
                                            1 if intermediate == "ibp" else 0, lb.ctypes.data, ub.ctypes.data,
                                            verified.ctypes.data), self.h)

    # ---- NEXT-1: alpha optimisation ---------------------------------------------------
    def _alpha_scratch(self, B: int, S: int) -> torch.Tensor:
        need = C.c_size_t(0)
        self._check(self.lib.crown_alpha_scratch_bytes(self.h, B, S, C.byref(need)), self.h)
        cur = getattr(self, "_alpha_scr", None)
        if cur is None or cur.numel() < need.value:
            self._alpha_scr = torch.empty(need.value, dtype=torch.uint8, device=self.device)
        return self._alpha_scr

    def alpha_grad(self, pre: Dict[int, tuple], Cmat, alpha_lo: Dict[int, torch.Tensor], alpha_up: Dict[int, torch.Tensor], box):
        """Bounds of the final pass at (alpha_lo, alpha_up) and their derivatives w.r.t. the slopes.
        Returns dict lb, ub [B,S], g_lo, g_up {relu id: [B,S,n]}."""
        Cmat = self._dev(Cmat)
        B, S = Cmat.shape[0], Cmat.shape[1]
        l = {i: self._dev(v[0]) for i, v in pre.items()}
        u = {i: self._dev(v[1]) for i, v in pre.items()}
        al = {i: self._dev(v) for i, v in alpha_lo.items()}
        au = al if alpha_up is alpha_lo else {i: self._dev(v) for i, v in alpha_up.items()}
        x_lo, x_hi = self._dev(box[0]), self._dev(box[1])
        g_lo = {i: torch.empty(B, S, self.sizes[i], device=self.device) for i in self.relu_ids}
        g_up = {i: torch.empty(B, S, self.sizes[i], device=self.device) for i in self.relu_ids}
        lb = torch.empty(B, S, device=self.device)
        ub = torch.empty(B, S, device=self.device)
        scr = self._alpha_scratch(B, S)
        self._check(self.lib.crown_alpha_grad(self.h, B, Cmat.data_ptr(), S, self._ptr_array(l), self._ptr_array(u),
                                              self._ptr_array(al), self._ptr_array(au), x_lo.data_ptr(), x_hi.data_ptr(),
                                              self._ptr_array(g_lo), self._ptr_array(g_up), lb.data_ptr(), ub.data_ptr(),
                                              scr.data_ptr(), scr.numel()), self.h)
        self.stream.synchronize()
        return {"lb": lb, "ub": ub, "g_lo": g_lo, "g_up": g_up}

    def alpha_ascent_device(self, l, u, Cmat, alpha_lo, alpha_up, x_lo, x_hi, eta, decay, iters, mode, out) -> None:
        """crown_alpha_ascent on device tensors (asynchronous); alpha_lo / alpha_up are updated in place."""
        B, S = Cmat.shape[0], Cmat.shape[1]
        scr = self._alpha_scratch(B, S)
        self._check(self.lib.crown_alpha_ascent(self.h, B, Cmat.data_ptr(), S, self._ptr_array(l), self._ptr_array(u),
                                                self._ptr_array(alpha_lo), self._ptr_array(alpha_up), x_lo.data_ptr(),
                                                x_hi.data_ptr(), float(eta), float(decay), int(iters), int(mode),
                                                out["lb_best"].data_ptr(), out["ub_best"].data_ptr(),
                                                out["lb_last"].data_ptr(), out["ub_last"].data_ptr(),
                                                out["verified"].data_ptr(), scr.data_ptr(), scr.numel()), self.h)

    def alpha_ascent(self, pre: Dict[int, tuple], Cmat, alpha_lo: Dict[int, torch.Tensor], alpha_up: Dict[int, torch.Tensor],
                     box, eta: float, iters: int, mode: str = "sign", decay: float = 1.0):
        """Projected gradient ascent on alpha_lo (lb) / descent on alpha_up (ub) with fixed intermediate bounds.
        Returns dict alpha_lo, alpha_up (optimised copies), lb_best, ub_best, lb_last, ub_last [B,S], verified [B]."""
        Cmat = self._dev(Cmat)
        B, S = Cmat.shape[0], Cmat.shape[1]
        l = {i: self._dev(v[0]) for i, v in pre.items()}
        u = {i: self._dev(v[1]) for i, v in pre.items()}
        al = {i: self._dev(v).clone() for i, v in alpha_lo.items()}
        au = {i: self._dev(v).clone() for i, v in alpha_up.items()}
        x_lo, x_hi = self._dev(box[0]), self._dev(box[1])
        out = {k: torch.empty(B, S, device=self.device) for k in ("lb_best", "ub_best", "lb_last", "ub_last")}
        out["verified"] = torch.empty(B, dtype=torch.uint8, device=self.device)
        self.alpha_ascent_device(l, u, Cmat, al, au, x_lo, x_hi, eta, decay, iters, {"plain": 0, "sign": 1}[mode], out)
        self.stream.synchronize()
        out["alpha_lo"], out["alpha_up"] = al, au
        return out

    # ---- NEXT-2: beta-CROWN bounds of BaB sub-domains -------------------------------------
    def _split_dev(self, split):
        return None if split is None else {i: self._dev(v, torch.int8) for i, v in split.items()}

    def backward_split(self, B: int, start: int, pre: Dict[int, tuple], split, Cmat=None, row0: int = 0,
                       rows: Optional[int] = None, alpha_lo=None, alpha_up=None, beta_lo=None, beta_up=None, box=None,
                       want_A: bool = True):
        """crown_backward_split: O3 for a batch of sub-domains.  split {relu id: int8 [B, n]}; beta {relu id: [B,R,n]}."""
        if Cmat is not None:
            Cmat = self._dev(Cmat)
            rows = Cmat.shape[1]
        l = {i: self._dev(v[0]) for i, v in pre.items()}
        u = {i: self._dev(v[1]) for i, v in pre.items()}
        dev = lambda d: None if d is None else {i: self._dev(v) for i, v in d.items()}
        al, au, bl, bu, sp = dev(alpha_lo), dev(alpha_up), dev(beta_lo), dev(beta_up), self._split_dev(split)
        A = torch.empty(2, B, rows, self.n0, device=self.device) if want_A else None
        d = torch.empty(2, B, rows, device=self.device)
        x_lo = x_hi = lb = ub = None
        if box is not None:
            x_lo, x_hi = self._dev(box[0]), self._dev(box[1])
            lb = torch.empty(B, rows, device=self.device)
            ub = torch.empty(B, rows, device=self.device)
        arr = lambda d_: self._ptr_array(d_) if d_ else None
        self._check(self.lib.crown_backward_split(self.h, B, start, row0, rows, _ptr(Cmat), self._ptr_array(l),
                                                  self._ptr_array(u), arr(sp), arr(al), arr(au), arr(bl), arr(bu),
                                                  _ptr(A), _ptr(d), _ptr(x_lo), _ptr(x_hi), _ptr(lb), _ptr(ub)), self.h)
        self.stream.synchronize()
        return {"A": A, "d": d, "lb": lb, "ub": ub}

    def beta_grad(self, pre, split, Cmat, alpha_lo, alpha_up, beta_lo, beta_up, box):
        """crown_beta_grad: bounds and their derivatives w.r.t. alpha and beta for a batch of sub-domains."""
        Cmat = self._dev(Cmat)
        B, S = Cmat.shape[0], Cmat.shape[1]
        l = {i: self._dev(v[0]) for i, v in pre.items()}
        u = {i: self._dev(v[1]) for i, v in pre.items()}
        dev = lambda d: {i: self._dev(v) for i, v in d.items()}
        al, au, bl, bu, sp = dev(alpha_lo), dev(alpha_up), dev(beta_lo), dev(beta_up), self._split_dev(split)
        x_lo, x_hi = self._dev(box[0]), self._dev(box[1])
        mk = lambda: {i: torch.zeros(B, S, self.sizes[i], device=self.device) for i in self.relu_ids}
        g_lo, g_up, gb_lo, gb_up = mk(), mk(), mk(), mk()
        lb = torch.empty(B, S, device=self.device)
        ub = torch.empty(B, S, device=self.device)
        scr = self._alpha_scratch(B, S)
        self._check(self.lib.crown_beta_grad(self.h, B, Cmat.data_ptr(), S, self._ptr_array(l), self._ptr_array(u),
                                             self._ptr_array(sp), self._ptr_array(al), self._ptr_array(au),
                                             self._ptr_array(bl), self._ptr_array(bu), x_lo.data_ptr(), x_hi.data_ptr(),
                                             self._ptr_array(g_lo), self._ptr_array(g_up), self._ptr_array(gb_lo),
                                             self._ptr_array(gb_up), lb.data_ptr(), ub.data_ptr(), scr.data_ptr(),
                                             scr.numel()), self.h)
        self.stream.synchronize()
        return {"lb": lb, "ub": ub, "g_lo": g_lo, "g_up": g_up, "gb_lo": gb_lo, "gb_up": gb_up}

    def beta_ascent_device(self, l, u, split, Cmat, alpha_lo, alpha_up, beta_lo, beta_up, x_lo, x_hi, eta_alpha, eta_beta,
                           decay, iters, mode, out) -> None:
        """crown_beta_ascent on device tensors (asynchronous); alpha / beta are updated in place."""
        B, S = Cmat.shape[0], Cmat.shape[1]
        scr = self._alpha_scratch(B, S)
        self._check(self.lib.crown_beta_ascent(self.h, B, Cmat.data_ptr(), S, self._ptr_array(l), self._ptr_array(u),
                                               self._ptr_array(split), self._ptr_array(alpha_lo), self._ptr_array(alpha_up),
                                               self._ptr_array(beta_lo), self._ptr_array(beta_up), x_lo.data_ptr(),
                                               x_hi.data_ptr(), float(eta_alpha), float(eta_beta), float(decay), int(iters),
                                               int(mode), out["lb_best"].data_ptr(), out["ub_best"].data_ptr(),
                                               out["lb_last"].data_ptr(), out["ub_last"].data_ptr(),
                                               out["verified"].data_ptr(), scr.data_ptr(), scr.numel()), self.h)

    def beta_ascent(self, pre, split, Cmat, alpha_lo, alpha_up, beta_lo, beta_up, box, eta_alpha: float, eta_beta: float,
                    iters: int, mode: str = "sign", decay: float = 1.0):
        """Joint projected ascent on (alpha, beta) for a batch of sub-domains; returns optimised copies and bounds."""
        Cmat = self._dev(Cmat)
        B, S = Cmat.shape[0], Cmat.shape[1]
        l = {i: self._dev(v[0]) for i, v in pre.items()}
        u = {i: self._dev(v[1]) for i, v in pre.items()}
        cl = lambda d: {i: self._dev(v).clone() for i, v in d.items()}
        al, au, bl, bu, sp = cl(alpha_lo), cl(alpha_up), cl(beta_lo), cl(beta_up), self._split_dev(split)
        x_lo, x_hi = self._dev(box[0]), self._dev(box[1])
        out = {k: torch.empty(B, S, device=self.device) for k in ("lb_best", "ub_best", "lb_last", "ub_last")}
        out["verified"] = torch.empty(B, dtype=torch.uint8, device=self.device)
        self.beta_ascent_device(l, u, sp, Cmat, al, au, bl, bu, x_lo, x_hi, eta_alpha, eta_beta, decay, iters,
                                {"plain": 0, "sign": 1}[mode], out)
        self.stream.synchronize()
        out.update(alpha_lo=al, alpha_up=au, beta_lo=bl, beta_up=bu)
        return out

    # ---- kernel 1 on its own ---------------------------------------------------------------------
    def split_tf32(self, X: torch.Tensor, transpose: bool = False):
        rows, cols = X.shape
        shape = (cols, rows) if transpose else (rows, cols)
        hi = torch.empty(shape, device=self.device)
        lo = torch.empty(shape, device=self.device)
        self._check(self.lib.crown_split_tf32(self.h, X.data_ptr(), rows, cols, int(transpose), hi.data_ptr(),
                                              lo.data_ptr()), self.h)
        return hi, lo

    def gemm_prepared(self, A_hi, A_lo, Wt_hi, Wt_lo, D, scheme: int = 0):
        M, K = A_hi.shape
        N = D.shape[1]
        self._check(self.lib.crown_gemm(self.h, scheme, M, N, K, A_hi.data_ptr(), _ptr(A_lo), Wt_hi.data_ptr(),
                                        _ptr(Wt_lo), D.data_ptr()), self.h)

    def gemm(self, A: torch.Tensor, W: torch.Tensor, scheme: int = 0) -> torch.Tensor:
        """D[M,N] = A[M,K] . W[K,N] through the contraction kernel (scheme 0 = 3xTF32 tcgen05 CTA-pair tiles, 2 = FFMA)."""
        A, W = self._dev(A), self._dev(W)
        D = torch.empty(A.shape[0], W.shape[1], device=self.device)
        if scheme == 0:
            A_hi, A_lo = self.split_tf32(A, False)
            Wt_hi, Wt_lo = self.split_tf32(W, True)
            self.gemm_prepared(A_hi, A_lo, Wt_hi, Wt_lo, D, 0)
        else:
            self.gemm_prepared(A, None, W, None, D, 2)
        return D

    # ---- introspection ---------------------------------------------------------------------------
    def peak_bytes(self) -> int:
        v = C.c_size_t(0)
        self._check(self.lib.crown_peak_bytes(self.h, C.byref(v)), self.h)
        return v.value

    def row_chunk(self) -> int:
        """Rows per chunk of an identity-start pass under mem_cap_bytes (chunks start at multiples of it)."""
        v = C.c_int(0)
        self._check(self.lib.crown_row_chunk(self.h, C.byref(v)), self.h)
        return v.value

    def graph_replays(self) -> int:
        v = C.c_uint64(0)
        self._check(self.lib.crown_graph_replays(self.h, C.byref(v)), self.h)
        return v.value

    def graph_active(self) -> bool:
        """True once crown_run has been served from a captured CUDA graph."""
        return self.graph_replays() > 0

    def launch_count(self) -> int:
        v = C.c_uint64(0)
        self._check(self.lib.crown_launch_count(self.h, C.byref(v)), self.h)
        return v.value

    def gemm_flops(self) -> float:
        v = C.c_double(0)
        self._check(self.lib.crown_gemm_flops(self.h, C.byref(v)), self.h)
        return v.value

    def h2d_bytes(self) -> float:
        """Bytes of weights streamed host->device so far (0 unless stream_weights)."""
        v = C.c_double(0)
        self._check(self.lib.crown_h2d_bytes(self.h, C.byref(v)), self.h)
        return v.value

    def timing(self, enable: bool) -> None:
        self._check(self.lib.crown_timing(self.h, int(enable)), self.h)

    def timing_read(self) -> Dict[str, dict]:
        out = {}
        for k, name in enumerate(K_CLASSES):
            ms, n, by, fl = C.c_double(0), C.c_uint64(0), C.c_double(0), C.c_double(0)
            self._check(self.lib.crown_timing_read(self.h, k, C.byref(ms), C.byref(n), C.byref(by), C.byref(fl)), self.h)
            out[name] = {"ms": ms.value, "launches": n.value, "bytes": by.value, "flops": fl.value}
        return out
