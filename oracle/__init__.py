"""GraphGP oracle — TEST INFRASTRUCTURE ONLY (see graphgp_oracle.cpp for the header).

Thin ctypes/numpy glue around `libgraphgp_oracle.so`.  Only tests/, `__graft_entry__.smoke()`
and bench.py's `cpu_baseline` / `--impl reference` legs may import this package; the product
path (`paper_2606_11402_b200/`) never does, and this package never imports the product.

All arrays are fp64 on the host.  For fp32-mode comparisons the caller passes the fp32 inputs
promoted exactly to double (O-1).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "graphgp_oracle.cpp")
_LIB = os.path.join(_HERE, "libgraphgp_oracle.so")
_lib = None

KIND_ID = {"se": 0, "matern32": 1, "exp": 2}


def build(force: bool = False) -> str:
    """Compile the oracle (g++ -O2 -fopenmp -ffp-contract=off).  Building the checker is not using it."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["g++", "-O2", "-fopenmp", "-ffp-contract=off", "-shared", "-fPIC", "-std=c++17",
               "-o", _LIB, _SRC]
        subprocess.run(cmd, check=True)
    return _LIB


class _Kernel(C.Structure):
    _fields_ = [("kind", C.c_int32), ("sigma", C.c_double), ("ell", C.c_double), ("jitter", C.c_double)]


@dataclass(frozen=True)
class Kernel:
    kind: str
    sigma: float
    ell: float
    jitter: float

    def c(self) -> _Kernel:
        return _Kernel(KIND_ID[self.kind], self.sigma, self.ell, self.jitter)


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_LIB)
        _lib.orc_rho.restype = C.c_double
        _lib.orc_rho.argtypes = [C.c_int32, C.c_double, C.c_double]
        _lib.orc_drho_dell.restype = C.c_double
        _lib.orc_drho_dell.argtypes = [C.c_int32, C.c_double, C.c_double]
        _lib.orc_d2.restype = C.c_double
        _lib.orc_depth_fixed_point.restype = C.c_int64
    return _lib


def num_threads() -> int:
    return int(lib().orc_num_threads())


def _p(a, ctype):
    return None if a is None else a.ctypes.data_as(C.POINTER(ctype))


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


# ---------------------------------------------------------------------------------------------
# graph construction (O-2 .. O-4)
# ---------------------------------------------------------------------------------------------
def order(x: np.ndarray) -> np.ndarray:
    """O-2: perm_tree[node] = user id, bit-reversed left-balanced k-d tree order."""
    x = _f64(x)
    n, d = x.shape
    perm = np.empty(n, dtype=np.int64)
    lib().orc_order(_p(x, C.c_double), C.c_int64(n), C.c_int32(d), _p(perm, C.c_int64))
    return perm


def subtree_sizes(n: int) -> np.ndarray:
    sz = np.ones(n, dtype=np.int64)
    lib().orc_subtree_sizes(C.c_int64(n), _p(sz, C.c_int64))
    return sz


def knn_rows(x_tree: np.ndarray, k: int, rows: np.ndarray) -> np.ndarray:
    """O-3 for the listed rows: k nearest PRECEDING points by brute force, nearest first."""
    x = _f64(x_tree)
    n, d = x.shape
    rows = np.ascontiguousarray(rows, dtype=np.int64)
    out = np.empty((rows.size, k), dtype=np.int32)
    lib().orc_knn_rows(_p(x, C.c_double), C.c_int64(n), C.c_int32(d), C.c_int32(k),
                       _p(rows, C.c_int64), C.c_int64(rows.size), _p(out, C.c_int32))
    return out


def knn(x_tree: np.ndarray, k: int, n0: int) -> np.ndarray:
    """O-3 for every row n0..n-1 (O(N^2): use for N <= 2^17)."""
    n = x_tree.shape[0]
    return knn_rows(x_tree, k, np.arange(n0, n, dtype=np.int64))


def depth(nbr: np.ndarray, n: int, n0: int) -> np.ndarray:
    """O-4: sequential depth pass."""
    nbr = np.ascontiguousarray(nbr, dtype=np.int32)
    k = nbr.shape[1]
    out = np.empty(n, dtype=np.int32)
    lib().orc_depth(_p(nbr, C.c_int32), C.c_int64(n), C.c_int64(n0), C.c_int32(k), _p(out, C.c_int32))
    return out


def depth_fixed_point(nbr: np.ndarray, n: int, n0: int):
    """The parallel fixed point of PAPER.md:59 (Jacobi sweeps).  Returns (depth, sweeps)."""
    nbr = np.ascontiguousarray(nbr, dtype=np.int32)
    k = nbr.shape[1]
    out = np.empty(n, dtype=np.int32)
    sweeps = lib().orc_depth_fixed_point(_p(nbr, C.c_int32), C.c_int64(n), C.c_int64(n0), C.c_int32(k),
                                         _p(out, C.c_int32))
    return out, int(sweeps)


@dataclass
class GraphData:
    """A generation graph in GRAPH order (tree order stably sorted by depth, O-4)."""
    x: np.ndarray          # [n, d] float64, graph order
    nbr: np.ndarray        # [n - n0, k] int32, graph positions, every entry < its row's position
    batch_off: np.ndarray  # [L + 1] int64, batch_off[0] = n0, batch_off[L] = n
    perm: np.ndarray       # [n] int64: graph position -> user id
    n0: int
    k: int
    depth: np.ndarray      # [n] int32 in graph order

    @property
    def n(self):
        return self.x.shape[0]


def depth_sort(x_tree, nbr_tree, depth_tree, perm_tree, n0) -> GraphData:
    """O-4: graph order = stable sort of tree indices by depth; neighbour indices remapped."""
    n = x_tree.shape[0]
    k = nbr_tree.shape[1]
    pos2tree = np.argsort(depth_tree, kind="stable")          # head (depth 0) stays first, unchanged
    tree2pos = np.empty(n, dtype=np.int64)
    tree2pos[pos2tree] = np.arange(n, dtype=np.int64)
    d_sorted = depth_tree[pos2tree]
    nb = int(d_sorted[-1]) if n > n0 else 0
    batch_off = np.searchsorted(d_sorted, np.arange(1, nb + 2), side="left").astype(np.int64)
    nbr_g = tree2pos[nbr_tree[pos2tree[n0:] - n0].astype(np.int64)].astype(np.int32)
    return GraphData(x=_f64(x_tree)[pos2tree], nbr=np.ascontiguousarray(nbr_g), batch_off=batch_off,
                     perm=np.asarray(perm_tree)[pos2tree], n0=int(n0), k=int(k), depth=d_sorted.astype(np.int32))


def build_graph(x_user: np.ndarray, k: int, n0: int) -> GraphData:
    """O-2..O-4 end to end (brute-force kNN: N <= 2^17)."""
    x_user = _f64(x_user)
    perm_tree = order(x_user)
    x_tree = x_user[perm_tree]
    nbr = knn(x_tree, k, n0)
    dep = depth(nbr, x_tree.shape[0], n0)
    return depth_sort(x_tree, nbr, dep, perm_tree, n0)


# ---------------------------------------------------------------------------------------------
# conditioning (O-5 .. O-7)
# ---------------------------------------------------------------------------------------------
def rho(kind: str, r: float, ell: float) -> float:
    return float(lib().orc_rho(KIND_ID[kind], float(r), float(ell)))


def drho_dell(kind: str, r: float, ell: float) -> float:
    return float(lib().orc_drho_dell(KIND_ID[kind], float(r), float(ell)))


def d2(a: np.ndarray, b: np.ndarray) -> float:
    a = _f64(a)
    b = _f64(b)
    return float(lib().orc_d2(_p(a, C.c_double), _p(b, C.c_double), C.c_int32(a.size)))


def condition(x, kern: Kernel, i: int, c):
    """Eq. 2 for one point: returns (w, s2)."""
    x = _f64(x)
    c = np.ascontiguousarray(c, dtype=np.int32)
    w = np.empty(c.size, dtype=np.float64)
    s2 = C.c_double(0.0)
    kc = kern.c()
    rc = lib().orc_condition(_p(x, C.c_double), C.c_int32(x.shape[1]), C.byref(kc), C.c_int64(i),
                             _p(c, C.c_int32), C.c_int32(c.size), _p(w, C.c_double), C.byref(s2))
    if rc:
        raise FloatingPointError("oracle: matrix not positive definite")
    return w, s2.value


class NotPositiveDefinite(FloatingPointError):
    pass


def _graph_args(x, n0, k, nbr, rowptr, col, batch_off):
    x = _f64(x)
    n, d = x.shape
    keep = [x]
    if rowptr is not None:
        rowptr = np.ascontiguousarray(rowptr, dtype=np.int64)
        col = np.ascontiguousarray(col, dtype=np.int32)
        keep += [rowptr, col]
        nbr_p, n0, k = None, 0, 0
    else:
        nbr = np.ascontiguousarray(nbr, dtype=np.int32)
        keep.append(nbr)
        nbr_p = _p(nbr, C.c_int32)
    if batch_off is not None:
        batch_off = np.ascontiguousarray(batch_off, dtype=np.int64)
        keep.append(batch_off)
        nb = batch_off.size - 1
    else:
        nb = 0
    args = [_p(x, C.c_double), C.c_int64(n), C.c_int32(d), C.c_int64(n0), C.c_int32(k), nbr_p,
            _p(rowptr, C.c_int64) if rowptr is not None else None,
            _p(col, C.c_int32) if rowptr is not None else None,
            _p(batch_off, C.c_int64) if batch_off is not None else None, C.c_int64(nb)]
    return args, keep, n


def _check(rc):
    if rc == 3:
        raise NotPositiveDefinite("oracle: a conditional variance or pivot was not positive")
    if rc:
        raise RuntimeError(f"oracle error {rc}")


def forward(x, kern: Kernel, xi, *, n0=0, k=0, nbr=None, rowptr=None, col=None, batch_off=None,
            long_double=False) -> np.ndarray:
    """O-6: v_i = w.v_c + s xi_i in generation order; dense head by Alg. 1 line 1 (regular graphs)."""
    args, keep, n = _graph_args(x, n0, k, nbr, rowptr, col, batch_off)
    xi = _f64(xi)
    v = np.empty(n, dtype=np.float64)
    kc = kern.c()
    _check(lib().orc_forward(*args, C.byref(kc), _p(xi, C.c_double), _p(v, C.c_double), C.c_int32(int(long_double))))
    return v


def inverse(x, kern: Kernel, v, *, n0=0, k=0, nbr=None, rowptr=None, col=None, long_double=False) -> np.ndarray:
    """O-6: xi_i = (v_i - w.v_c) / s."""
    args, keep, n = _graph_args(x, n0, k, nbr, rowptr, col, None)
    v = _f64(v)
    xi = np.empty(n, dtype=np.float64)
    kc = kern.c()
    _check(lib().orc_inverse(*args, C.byref(kc), _p(v, C.c_double), _p(xi, C.c_double), C.c_int32(int(long_double))))
    return xi


def logdet(x, kern: Kernel, *, n0=0, k=0, nbr=None, rowptr=None, col=None, grad=False, long_double=False):
    """O-6: sum_i log s_i^2 (+ dense head).  With grad=True also d/d(sigma, ell)."""
    args, keep, n = _graph_args(x, n0, k, nbr, rowptr, col, None)
    out = C.c_double(0.0)
    g = np.zeros(2, dtype=np.float64)
    kc = kern.c()
    _check(lib().orc_logdet(*args, C.byref(kc), C.byref(out), _p(g, C.c_double) if grad else None,
                            C.c_int32(int(long_double))))
    return (out.value, g) if grad else out.value


def vjp(x, kern: Kernel, xi, v, vbar, *, n0=0, k=0, nbr=None, rowptr=None, col=None, batch_off=None,
        long_double=False):
    """O-7: VJP of forward for cotangent vbar: returns (xi_bar [n], theta_bar [2] = d/dsigma, d/dell)."""
    args, keep, n = _graph_args(x, n0, k, nbr, rowptr, col, batch_off)
    xi, v, vbar = _f64(xi), _f64(v), _f64(vbar)
    xibar = np.empty(n, dtype=np.float64)
    tb = np.zeros(2, dtype=np.float64)
    kc = kern.c()
    _check(lib().orc_vjp(*args, C.byref(kc), _p(xi, C.c_double), _p(v, C.c_double), _p(vbar, C.c_double),
                         _p(xibar, C.c_double), _p(tb, C.c_double), C.c_int32(int(long_double))))
    return xibar, tb


def jvp(x, kern: Kernel, xi, v, dxi, dsigma, dell, *, n0=0, k=0, nbr=None, rowptr=None, col=None, batch_off=None) -> np.ndarray:
    """JVP of forward along (dxi, dsigma, dell) at (xi, v = forward(xi)): returns dv [n]."""
    args, keep, n = _graph_args(x, n0, k, nbr, rowptr, col, batch_off)
    xi, v, dxi = _f64(xi), _f64(v), _f64(dxi)
    dv = np.empty(n, dtype=np.float64)
    kc = kern.c()
    _check(lib().orc_jvp(*args, C.byref(kc), _p(xi, C.c_double), _p(v, C.c_double), _p(dxi, C.c_double),
                         C.c_double(dsigma), C.c_double(dell), _p(dv, C.c_double)))
    return dv


def inverse_vjp(x, kern: Kernel, v, xi, h, *, n0=0, k=0, nbr=None, rowptr=None, col=None):
    """VJP of inverse for a cotangent h on xi at (v, xi = inverse(v)): returns (v_bar [n], theta_bar [2])."""
    args, keep, n = _graph_args(x, n0, k, nbr, rowptr, col, None)
    v, xi, h = _f64(v), _f64(xi), _f64(h)
    vbar = np.empty(n, dtype=np.float64)
    tb = np.zeros(2, dtype=np.float64)
    kc = kern.c()
    _check(lib().orc_inverse_vjp(*args, C.byref(kc), _p(v, C.c_double), _p(xi, C.c_double), _p(h, C.c_double),
                                 _p(vbar, C.c_double), _p(tb, C.c_double)))
    return vbar, tb


def cond_std(x, kern: Kernel, *, n0=0, k=0, nbr=None, rowptr=None, col=None) -> np.ndarray:
    """s_i of Eq. 2 for every point (head: diagonal of the dense factor): dv_i / dxi_i."""
    args, keep, n = _graph_args(x, n0, k, nbr, rowptr, col, None)
    s = np.empty(n, dtype=np.float64)
    kc = kern.c()
    _check(lib().orc_cond_std(*args[:8], C.byref(kc), _p(s, C.c_double)))
    return s


def all_preceding_csr(n: int):
    """c(i) = {0..i-1} for every i (the exact case)."""
    rowptr = np.zeros(n + 1, dtype=np.int64)
    rowptr[1:] = np.cumsum(np.arange(n, dtype=np.int64))
    col = np.concatenate([np.arange(i, dtype=np.int32) for i in range(n)]) if n > 1 else np.zeros(0, np.int32)
    return rowptr, col
