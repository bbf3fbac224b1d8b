"""paper_2606_11402_b200 — thin Python binding over libgraphgp.so (include/graphgp.h).

Argument marshalling only: every step of the Vecchia conditioning path runs in the CUDA kernels of
csrc/.  PyTorch supplies device memory and streams.  There is no CPU fallback: if the extension is
missing or there is no CUDA device the calls raise.

Names follow the C ABI: gp_forward, gp_inverse, gp_logdet, gp_vjp, gp_graph_build.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass, field

import numpy as np

from .build import LIB, build_library

GP_OK, GP_ERR_INVALID_ARG, GP_ERR_UNSUPPORTED, GP_ERR_NOT_PD, GP_ERR_CUDA, GP_ERR_WORKSPACE, GP_ERR_TOO_LARGE = range(7)
GP_F32, GP_F64 = 0, 1
GP_OP_FORWARD, GP_OP_INVERSE, GP_OP_LOGDET, GP_OP_VJP, GP_OP_BUILD, GP_OP_FORWARD_MULTI, GP_OP_INVERSE_MULTI = range(7)
GP_FLAG_PER_BATCH_LAUNCH, GP_FLAG_GENERIC_KERNEL, GP_FLAG_FLOW_CARRY, GP_FLAG_FLOW_WEIGHTS = 1, 2, 4, 8
GP_BUILD_SPATIAL_BATCHES, GP_BUILD_RADIUS_CLASSES, GP_BUILD_PLAIN_KNN, GP_BUILD_PLAIN_ORDER = 1, 2, 4, 8
KIND_ID = {"se": 0, "matern32": 1, "exp": 2}

EXPORTS = ["gp_workspace_bytes", "gp_forward", "gp_inverse", "gp_logdet", "gp_vjp", "gp_forward_host",
           "gp_inverse_host", "gp_logdet_host", "gp_vjp_host", "gp_graph_build", "gp_graph_build_workspace_bytes", "gp_graph_build_times",
           "gp_check_errors", "gp_status_string", "gp_has_specialised", "gp_launch_count", "gp_kernel_time_enable",
           "gp_kernel_time_last", "gp_measure_alu_peak", "gp_workspace_bytes_multi", "gp_forward_multi", "gp_inverse_multi", "gp_jvp", "gp_inverse_vjp",
           "gp_logdet_noalloc", "gp_logdet_noalloc_scratch_bytes"]


class GraphGPError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__(f"{where}: {status_string(status)} (gp_status {status})")


class _Kernel(C.Structure):
    _fields_ = [("kind", C.c_int32), ("sigma", C.c_double), ("ell", C.c_double), ("jitter", C.c_double)]


class _Graph(C.Structure):
    _fields_ = [("n", C.c_int64), ("n0", C.c_int64), ("d", C.c_int32), ("k", C.c_int32),
                ("n_batches", C.c_int32), ("dtype", C.c_int32), ("flags", C.c_int32), ("reserved", C.c_int32),
                ("x", C.c_void_p), ("nbr", C.c_void_p), ("batch_off", C.c_void_p)]


_lib = None


def lib():
    """Load libgraphgp.so (fails loudly if it has not been built: run `python -m paper_2606_11402_b200.build`)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB):
            raise ImportError(f"{LIB} is missing: build it with `python -m paper_2606_11402_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(LIB)
        L.gp_workspace_bytes.restype = C.c_size_t
        L.gp_workspace_bytes.argtypes = [C.POINTER(_Graph), C.c_int32]
        L.gp_graph_build_workspace_bytes.restype = C.c_size_t
        L.gp_graph_build_workspace_bytes.argtypes = [C.c_int64, C.c_int32, C.c_int32, C.c_int32]
        L.gp_status_string.restype = C.c_char_p
        L.gp_status_string.argtypes = [C.c_int]
        L.gp_launch_count.restype = C.c_int64
        L.gp_kernel_time_enable.restype = None
        L.gp_kernel_time_enable.argtypes = [C.c_int32]
        L.gp_kernel_time_last.restype = C.c_int
        L.gp_kernel_time_last.argtypes = [C.POINTER(C.c_double)]
        L.gp_has_specialised.restype = C.c_int32
        L.gp_has_specialised.argtypes = [C.c_int32] * 4
        vp, sz = C.c_void_p, C.c_size_t
        gk = [C.POINTER(_Graph), C.POINTER(_Kernel)]
        L.gp_forward.argtypes = gk + [vp, vp, vp, sz, vp]
        L.gp_inverse.argtypes = gk + [vp, vp, vp, sz, vp]
        L.gp_logdet.argtypes = gk + [vp, vp, vp, sz, vp]
        L.gp_vjp.argtypes = gk + [vp, vp, vp, vp, vp, vp, sz, vp]
        L.gp_forward_host.argtypes = gk + [vp, vp, vp, vp, vp, sz, vp]
        L.gp_inverse_host.argtypes = gk + [vp, vp, vp, vp, vp, sz, vp]
        L.gp_vjp_host.argtypes = gk + [vp] * 11 + [sz, vp]
        L.gp_logdet_host.argtypes = gk + [vp, vp, vp, vp, vp, sz, vp]
        L.gp_graph_build.argtypes = [vp, C.c_int64, C.c_int32, C.c_int32, C.c_int64, C.c_int32, C.c_int32, vp, vp,
                                     vp, vp, vp, C.c_int32, C.POINTER(C.c_int32), vp, sz, vp]
        L.gp_graph_build_times.argtypes = [vp, vp]
        L.gp_check_errors.argtypes = [vp, C.POINTER(C.c_int64)]
        L.gp_jvp.argtypes = gk + [vp, vp, vp, C.c_double, C.c_double, vp, vp, sz, vp]
        L.gp_inverse_vjp.argtypes = gk + [vp, vp, vp, vp, vp, vp, sz, vp]
        L.gp_jvp.restype = C.c_int
        L.gp_inverse_vjp.restype = C.c_int
        L.gp_workspace_bytes_multi.restype = C.c_size_t
        L.gp_workspace_bytes_multi.argtypes = [C.POINTER(_Graph), C.c_int32, C.c_int32]
        L.gp_forward_multi.argtypes = gk + [C.c_int32, vp, vp, vp, sz, vp]
        L.gp_inverse_multi.argtypes = gk + [C.c_int32, vp, vp, vp, sz, vp]
        L.gp_forward_multi.restype = C.c_int
        L.gp_inverse_multi.restype = C.c_int
        L.gp_measure_alu_peak.argtypes = [vp, C.c_int32, vp, sz, vp]
        L.gp_logdet_noalloc.argtypes = gk + [vp, vp]
        L.gp_logdet_noalloc_scratch_bytes.argtypes = []
        L.gp_logdet_noalloc_scratch_bytes.restype = C.c_size_t
        L.gp_logdet_noalloc.restype = C.c_int
        L.gp_measure_alu_peak.restype = C.c_int
        for name in ("gp_forward", "gp_inverse", "gp_logdet", "gp_vjp", "gp_forward_host", "gp_inverse_host",
                     "gp_vjp_host", "gp_logdet_host", "gp_graph_build", "gp_graph_build_times", "gp_check_errors"):
            getattr(L, name).restype = C.c_int
        _lib = L
    return _lib


def status_string(status: int) -> str:
    return lib().gp_status_string(int(status)).decode()


def launch_count() -> int:
    return int(lib().gp_launch_count())


def kernel_time_enable(on: bool) -> None:
    """Bracket each op's dominant kernel(s) with CUDA events on the launching stream (bench.py's roofline)."""
    lib().gp_kernel_time_enable(1 if on else 0)


def kernel_time_last() -> float:
    """Device milliseconds of the dominant kernel(s) of the most recent op (synchronises on its closing event)."""
    ms = C.c_double(0.0)
    _check(lib().gp_kernel_time_last(C.byref(ms)), "gp_kernel_time_last")
    return float(ms.value)


PEAK_NAMES = ("ffma", "ffma_imm", "ffma2", "ffma2_bcast", "dfma", "mufu", "ffma2_dfma", "ffma2_mufu")


def measure_alu_peak(stream=None) -> dict:
    """Non-tensor ALU rates of the current device from register-resident loops (gp_measure_alu_peak), TFLOP/s."""
    torch = _torch()
    out = np.zeros(len(PEAK_NAMES), dtype=np.float64)
    ws = torch.empty(256, dtype=torch.uint8, device="cuda")
    _check(lib().gp_measure_alu_peak(out.ctypes.data, len(PEAK_NAMES), ws.data_ptr(), ws.numel(), _stream_ptr(stream)),
           "gp_measure_alu_peak")
    return {k: float(v) for k, v in zip(PEAK_NAMES, out)}


def has_specialised(dtype: str, k: int, d: int, kind: str) -> bool:
    return bool(lib().gp_has_specialised(GP_F64 if dtype == "f64" else GP_F32, k, d, KIND_ID[kind]))


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("paper_2606_11402_b200 needs a CUDA device (no CPU fallback)")
    return torch


@dataclass
class Kernel:
    kind: str
    sigma: float
    ell: float
    jitter: float

    def c(self) -> _Kernel:
        return _Kernel(KIND_ID[self.kind], float(self.sigma), float(self.ell), float(self.jitter))


@dataclass
class Graph:
    """Device-resident generation graph in GRAPH order (Alg. 1 `Require`)."""
    x: "object"              # torch [n, d] float32/float64, cuda
    nbr: "object"            # torch [n - n0, k] int32, cuda
    batch_off: np.ndarray    # host int64 [L + 1]
    n0: int
    flags: int = 0
    perm: "object" = None    # torch [n] int64 graph position -> user id (builder output)
    depth: "object" = None
    _ws: dict = field(default_factory=dict, repr=False)

    @property
    def n(self) -> int:
        return int(self.x.shape[0])

    @property
    def d(self) -> int:
        return int(self.x.shape[1])

    @property
    def k(self) -> int:
        return int(self.nbr.shape[1])

    @property
    def dtype_id(self) -> int:
        torch = _torch()
        return GP_F64 if self.x.dtype == torch.float64 else GP_F32

    def c(self) -> _Graph:
        torch = _torch()
        if self.x.device.type != "cuda" or not self.x.is_contiguous() or self.x.dim() != 2:
            raise ValueError("Graph.x must be a contiguous [n, d] CUDA tensor")
        if self.nbr.dtype != torch.int32 or not self.nbr.is_contiguous() or self.nbr.device != self.x.device:
            raise ValueError("Graph.nbr must be a contiguous int32 tensor on the device of Graph.x")
        self.batch_off = np.ascontiguousarray(self.batch_off, dtype=np.int64)
        nb = max(self.batch_off.size - 1, 0)
        return _Graph(self.n, int(self.n0), self.d, self.k, nb, self.dtype_id, int(self.flags), 0,
                      self.x.data_ptr(), self.nbr.data_ptr() if self.nbr.numel() else None,
                      self.batch_off.ctypes.data if self.batch_off.size else None)

    def workspace(self, op: int):
        """A cached, caller-side workspace tensor for `op` (the library itself never allocates)."""
        torch = _torch()
        g = self.c()
        need = int(lib().gp_workspace_bytes(C.byref(g), op))
        if need == 0:
            raise GraphGPError(GP_ERR_INVALID_ARG, "gp_workspace_bytes")
        ws = self._ws.get(op)
        if ws is None or ws.numel() < need:
            ws = torch.empty(need, dtype=torch.uint8, device=self.x.device)
            self._ws[op] = ws
        return ws


def graph_from_arrays(x, nbr, batch_off, n0, dtype="f32", device="cuda", flags=0) -> Graph:
    """Upload host arrays (e.g. a graph made elsewhere) as a device-resident Graph."""
    torch = _torch()
    tdt = torch.float64 if dtype == "f64" else torch.float32
    xt = torch.as_tensor(np.ascontiguousarray(x), device=device).to(tdt).contiguous()
    k = nbr.shape[1]
    nt = torch.as_tensor(np.ascontiguousarray(nbr, dtype=np.int32), device=device).contiguous().reshape(-1, k)
    return Graph(x=xt, nbr=nt, batch_off=np.ascontiguousarray(batch_off, dtype=np.int64), n0=int(n0), flags=flags)


def _stream_ptr(stream):
    torch = _torch()
    s = stream if stream is not None else torch.cuda.current_stream()
    return C.c_void_p(s.cuda_stream)


def _check(status: int, where: str):
    if status != GP_OK:
        raise GraphGPError(status, where)


def _vec(graph: "Graph", t, name: str, host: bool = False):
    """Marshalling check: a [n] vector of the graph's dtype, contiguous, on the graph's device (or pinned/host)."""
    torch = _torch()
    want = torch.float64 if graph.dtype_id == GP_F64 else torch.float32
    if not isinstance(t, torch.Tensor):
        raise TypeError(f"{name}: expected a torch tensor")
    if t.dtype != want:
        raise TypeError(f"{name}: dtype {t.dtype} does not match the graph's {want}")
    if t.numel() != graph.n or not t.is_contiguous():
        raise ValueError(f"{name}: expected a contiguous vector of {graph.n} elements")
    if host:
        if t.device.type != "cpu":
            raise ValueError(f"{name}: expected a host tensor")
    elif t.device != graph.x.device:
        raise ValueError(f"{name}: on {t.device}, the graph is on {graph.x.device}")
    return t


def _f64(t, count: int, name: str, device=None):
    torch = _torch()
    if t.dtype != torch.float64 or t.numel() != count or not t.is_contiguous():
        raise TypeError(f"{name}: expected a contiguous float64 tensor of {count} elements")
    if device is None:
        if t.device.type != "cpu":
            raise ValueError(f"{name}: expected a host tensor")
    elif t.device != device:
        raise ValueError(f"{name}: on {t.device}, expected {device}")
    return t


def check_errors(ws) -> int:
    """Synchronise, then return the number of points whose conditional was not positive definite."""
    torch = _torch()
    torch.cuda.synchronize()
    nbad = C.c_int64(0)
    st = lib().gp_check_errors(C.c_void_p(ws.data_ptr()), C.byref(nbad))
    if st not in (GP_OK, GP_ERR_NOT_PD):
        raise GraphGPError(st, "gp_check_errors")
    return int(nbad.value)


def gp_forward(graph: Graph, kern: Kernel, xi, out=None, stream=None):
    """v = forward(xi): Alg. 1.  xi, v: device [n] in graph order."""
    torch = _torch()
    _vec(graph, xi, "xi")
    v = torch.empty_like(xi) if out is None else _vec(graph, out, "out")
    ws = graph.workspace(GP_OP_FORWARD)
    g, k = graph.c(), kern.c()
    _check(lib().gp_forward(C.byref(g), C.byref(k), xi.data_ptr(), v.data_ptr(), ws.data_ptr(), ws.numel(),
                            _stream_ptr(stream)), "gp_forward")
    return v


def gp_inverse(graph: Graph, kern: Kernel, v, out=None, stream=None):
    """xi = inverse(v)."""
    torch = _torch()
    _vec(graph, v, "v")
    xi = torch.empty_like(v) if out is None else _vec(graph, out, "out")
    ws = graph.workspace(GP_OP_INVERSE)
    g, k = graph.c(), kern.c()
    _check(lib().gp_inverse(C.byref(g), C.byref(k), v.data_ptr(), xi.data_ptr(), ws.data_ptr(), ws.numel(),
                            _stream_ptr(stream)), "gp_inverse")
    return xi


def gp_logdet(graph: Graph, kern: Kernel, grad: bool = False, stream=None):
    """log det of the Vecchia covariance (device double[1]); with grad=True also d/d(sigma, ell) (double[2])."""
    torch = _torch()
    out = torch.empty(1, dtype=torch.float64, device=graph.x.device)
    gout = torch.empty(2, dtype=torch.float64, device=graph.x.device) if grad else None
    ws = graph.workspace(GP_OP_VJP if grad else GP_OP_LOGDET)
    g, k = graph.c(), kern.c()
    _check(lib().gp_logdet(C.byref(g), C.byref(k), out.data_ptr(), gout.data_ptr() if grad else None,
                           ws.data_ptr(), ws.numel(), _stream_ptr(stream)), "gp_logdet")
    return (out, gout) if grad else out


def gp_logdet_noalloc(graph: Graph, kern: Kernel, out, stream=None):
    """gp_logdet without a workspace (fixed scratch array inside the library; n0 <= 1024, k <= 64, else GraphGPError with
    GP_ERR_TOO_LARGE).  out: caller's device float64[1].  Calls that overlap on the GPU race on the scratch."""
    torch = _torch()
    if not isinstance(out, torch.Tensor) or out.dtype != torch.float64 or out.numel() < 1 or out.device != graph.x.device:
        raise TypeError("gp_logdet_noalloc: out must be a float64 tensor with >= 1 element on the graph's device")
    g, k = graph.c(), kern.c()
    _check(lib().gp_logdet_noalloc(C.byref(g), C.byref(k), out.data_ptr(), _stream_ptr(stream)), "gp_logdet_noalloc")
    return out


def logdet_noalloc_scratch_bytes() -> int:
    return int(lib().gp_logdet_noalloc_scratch_bytes())


def gp_vjp(graph: Graph, kern: Kernel, xi, v, v_bar, stream=None):
    """VJP of gp_forward: returns (xi_bar [n], theta_bar double[2] = d/dsigma, d/dell)."""
    torch = _torch()
    _vec(graph, xi, "xi"), _vec(graph, v, "v"), _vec(graph, v_bar, "v_bar")
    xi_bar = torch.empty_like(xi)
    tb = torch.empty(2, dtype=torch.float64, device=graph.x.device)
    ws = graph.workspace(GP_OP_VJP)
    g, k = graph.c(), kern.c()
    _check(lib().gp_vjp(C.byref(g), C.byref(k), xi.data_ptr(), v.data_ptr(), v_bar.data_ptr(), xi_bar.data_ptr(),
                        tb.data_ptr(), ws.data_ptr(), ws.numel(), _stream_ptr(stream)), "gp_vjp")
    return xi_bar, tb


def gp_jvp(graph: Graph, kern: Kernel, xi, v, xi_dot, sigma_dot: float, ell_dot: float, stream=None):
    """Forward-mode derivative of gp_forward: v_dot [n] along (xi_dot, sigma_dot, ell_dot) at (xi, v)."""
    torch = _torch()
    _vec(graph, xi, "xi"), _vec(graph, v, "v"), _vec(graph, xi_dot, "xi_dot")
    v_dot = torch.empty_like(xi)
    ws = graph.workspace(GP_OP_VJP)
    g, k = graph.c(), kern.c()
    _check(lib().gp_jvp(C.byref(g), C.byref(k), xi.data_ptr(), v.data_ptr(), xi_dot.data_ptr(), float(sigma_dot),
                        float(ell_dot), v_dot.data_ptr(), ws.data_ptr(), ws.numel(), _stream_ptr(stream)), "gp_jvp")
    return v_dot


def gp_inverse_vjp(graph: Graph, kern: Kernel, v, xi, xi_bar, stream=None):
    """VJP of gp_inverse: (v_bar [n], theta_bar double[2]) for a cotangent xi_bar at (v, xi = inverse(v))."""
    torch = _torch()
    _vec(graph, v, "v"), _vec(graph, xi, "xi"), _vec(graph, xi_bar, "xi_bar")
    v_bar = torch.empty_like(v)
    tb = torch.empty(2, dtype=torch.float64, device=graph.x.device)
    ws = graph.workspace(GP_OP_VJP)
    g, k = graph.c(), kern.c()
    _check(lib().gp_inverse_vjp(C.byref(g), C.byref(k), v.data_ptr(), xi.data_ptr(), xi_bar.data_ptr(), v_bar.data_ptr(),
                                tb.data_ptr(), ws.data_ptr(), ws.numel(), _stream_ptr(stream)), "gp_inverse_vjp")
    return v_bar, tb


def _multi(graph: Graph, kern: Kernel, op: int, name: str, src, out, stream):
    torch = _torch()
    want = torch.float64 if graph.dtype_id == GP_F64 else torch.float32
    if src.dim() != 2 or src.shape[0] != graph.n or src.dtype != want or not src.is_contiguous() or src.device != graph.x.device:
        raise ValueError(f"{name}: expected a contiguous [n, S] tensor of the graph's dtype on the graph's device")
    S = int(src.shape[1])
    if out is None:
        out = torch.empty_like(src)
    elif out.shape != src.shape or out.dtype != src.dtype or not out.is_contiguous() or out.device != src.device:
        raise ValueError(f"{name}: out must match the input")
    g, k = graph.c(), kern.c()
    need = int(lib().gp_workspace_bytes_multi(C.byref(g), op, S))
    key = (op, S)
    ws = graph._ws.get(key)
    if ws is None or ws.numel() < need:
        ws = torch.empty(max(need, 256), dtype=torch.uint8, device=graph.x.device)
        graph._ws[key] = ws
    fn = lib().gp_forward_multi if op == GP_OP_FORWARD_MULTI else lib().gp_inverse_multi
    _check(fn(C.byref(g), C.byref(k), S, src.data_ptr(), out.data_ptr(), ws.data_ptr(), ws.numel(), _stream_ptr(stream)), name)
    return out


def gp_forward_multi(graph: Graph, kern: Kernel, xi, out=None, stream=None):
    """S samples at once: xi, v device [n, S]; column s equals gp_forward on xi[:, s]."""
    return _multi(graph, kern, GP_OP_FORWARD_MULTI, "gp_forward_multi", xi, out, stream)


def gp_inverse_multi(graph: Graph, kern: Kernel, v, out=None, stream=None):
    """S samples at once: v, xi device [n, S]; column s equals gp_inverse on v[:, s]."""
    return _multi(graph, kern, GP_OP_INVERSE_MULTI, "gp_inverse_multi", v, out, stream)


def gp_forward_host(graph: Graph, kern: Kernel, xi_host, v_host, in_dev, out_dev, stream=None):
    """End-to-end forward with HOST (pinned) xi / v: H2D copy, forward, D2H copy on one stream."""
    _vec(graph, xi_host, "xi_host", host=True), _vec(graph, v_host, "v_host", host=True)
    _vec(graph, in_dev, "in_dev"), _vec(graph, out_dev, "out_dev")
    ws = graph.workspace(GP_OP_FORWARD)
    g, k = graph.c(), kern.c()
    _check(lib().gp_forward_host(C.byref(g), C.byref(k), xi_host.data_ptr(), v_host.data_ptr(), in_dev.data_ptr(),
                                 out_dev.data_ptr(), ws.data_ptr(), ws.numel(), _stream_ptr(stream)),
           "gp_forward_host")
    return v_host


def gp_inverse_host(graph: Graph, kern: Kernel, v_host, xi_host, in_dev, out_dev, stream=None):
    _vec(graph, xi_host, "xi_host", host=True), _vec(graph, v_host, "v_host", host=True)
    _vec(graph, in_dev, "in_dev"), _vec(graph, out_dev, "out_dev")
    ws = graph.workspace(GP_OP_INVERSE)
    g, k = graph.c(), kern.c()
    _check(lib().gp_inverse_host(C.byref(g), C.byref(k), v_host.data_ptr(), xi_host.data_ptr(), in_dev.data_ptr(),
                                 out_dev.data_ptr(), ws.data_ptr(), ws.numel(), _stream_ptr(stream)),
           "gp_inverse_host")
    return xi_host


def gp_logdet_host(graph: Graph, kern: Kernel, logdet_host, logdet_dev, grad_host=None, grad_dev=None, stream=None):
    """End-to-end logdet: the op, then the device double(s) copied into HOST (pinned) tensors on one stream."""
    grad = grad_host is not None
    _f64(logdet_host, 1, "logdet_host"), _f64(logdet_dev, 1, "logdet_dev", graph.x.device)
    if grad:
        _f64(grad_host, 2, "grad_host"), _f64(grad_dev, 2, "grad_dev", graph.x.device)
    ws = graph.workspace(GP_OP_VJP if grad else GP_OP_LOGDET)
    g, k = graph.c(), kern.c()
    _check(lib().gp_logdet_host(C.byref(g), C.byref(k), logdet_host.data_ptr(), grad_host.data_ptr() if grad else None,
                                logdet_dev.data_ptr(), grad_dev.data_ptr() if grad else None, ws.data_ptr(), ws.numel(),
                                _stream_ptr(stream)), "gp_logdet_host")
    return (logdet_host, grad_host) if grad else logdet_host


def gp_vjp_host(graph: Graph, kern: Kernel, xi_host, v_host, vbar_host, xibar_host, theta_bar_host, staging,
                stream=None):
    """End-to-end VJP with HOST (pinned) xi, v, v_bar -> xi_bar, theta_bar.  staging = (xi_dev, v_dev, v_bar_dev,
    xi_bar_dev, theta_bar_dev): caller-owned device buffers.  Synchronise the stream before reading the results."""
    ws = graph.workspace(GP_OP_VJP)
    g, k = graph.c(), kern.c()
    xd, vd, vbd, xbd, tbd = staging
    for t, nm in ((xi_host, "xi_host"), (v_host, "v_host"), (vbar_host, "vbar_host"), (xibar_host, "xibar_host")):
        _vec(graph, t, nm, host=True)
    for t, nm in ((xd, "xi_dev"), (vd, "v_dev"), (vbd, "v_bar_dev"), (xbd, "xi_bar_dev")):
        _vec(graph, t, nm)
    _f64(theta_bar_host, 2, "theta_bar_host"), _f64(tbd, 2, "theta_bar_dev", graph.x.device)
    _check(lib().gp_vjp_host(C.byref(g), C.byref(k), xi_host.data_ptr(), v_host.data_ptr(), vbar_host.data_ptr(),
                             xibar_host.data_ptr(), theta_bar_host.data_ptr(), xd.data_ptr(), vd.data_ptr(),
                             vbd.data_ptr(), xbd.data_ptr(), tbd.data_ptr(), ws.data_ptr(), ws.numel(),
                             _stream_ptr(stream)), "gp_vjp_host")
    return xibar_host, theta_bar_host


def gp_graph_build(x_user, k: int, n0: int, build_flags: int = GP_BUILD_SPATIAL_BATCHES, max_batches: int = 1 << 16,
                   stream=None) -> Graph:
    """Build order, preceding-kNN graph, depths and batches on the GPU.  x_user: device [n, d]."""
    torch = _torch()
    if x_user.device.type != "cuda" or x_user.dim() != 2 or x_user.dtype not in (torch.float32, torch.float64):
        raise TypeError("gp_graph_build: x_user must be a [n, d] float32/float64 CUDA tensor")
    x_user = x_user.contiguous()
    n, d = int(x_user.shape[0]), int(x_user.shape[1])
    dt = GP_F64 if x_user.dtype == torch.float64 else GP_F32
    dev = x_user.device
    perm = torch.empty(n, dtype=torch.int64, device=dev)
    xg = torch.empty_like(x_user)
    nbr = torch.empty((max(n - n0, 0), k), dtype=torch.int32, device=dev)
    depth = torch.empty(n, dtype=torch.int32, device=dev)
    boff = np.zeros(max_batches + 1, dtype=np.int64)
    nb = C.c_int32(0)
    need = int(lib().gp_graph_build_workspace_bytes(n, d, k, dt))
    ws = torch.empty(max(need, 256), dtype=torch.uint8, device=dev)
    _check(lib().gp_graph_build(x_user.data_ptr(), n, d, k, n0, dt, build_flags, perm.data_ptr(), xg.data_ptr(),
                                nbr.data_ptr() if nbr.numel() else None, depth.data_ptr(), boff.ctypes.data,
                                max_batches, C.byref(nb), ws.data_ptr(), ws.numel(), _stream_ptr(stream)),
           "gp_graph_build")
    times = np.zeros(4, dtype=np.float64)
    lib().gp_graph_build_times(ws.data_ptr(), times.ctypes.data)
    g = Graph(x=xg, nbr=nbr, batch_off=boff[: nb.value + 1].copy(), n0=int(n0), perm=perm, depth=depth)
    g.build_ms = times
    return g
