"""Host-side checks that need no GPU: the C-ABI library builds, loads and exports every symbol that
include/graphgp.h declares; workspace sizing and argument validation (host logic) behave as the header says;
compute entry points refuse to run without a CUDA device (there is no CPU fallback)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def gp():
    from paper_2606_11402_b200.build import build_library
    build_library()
    import paper_2606_11402_b200 as gp
    gp.lib()
    return gp


def declared_functions():
    src = open(os.path.join(ROOT, "include", "graphgp.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(gp_[a-z_0-9]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(gp):
    names = declared_functions()
    assert {"gp_forward", "gp_inverse", "gp_logdet", "gp_vjp", "gp_graph_build", "gp_workspace_bytes"} <= set(names)
    lib = C.CDLL(gp.LIB)
    missing = [n for n in names if not hasattr(lib, n)]
    assert not missing, missing
    assert sorted(gp.EXPORTS) == names


def test_binding_does_not_import_the_oracle(gp):
    import sys
    src = open(os.path.join(ROOT, "paper_2606_11402_b200", "__init__.py")).read()
    assert "oracle" not in src.replace("the oracle", "")
    for f in os.listdir(os.path.join(ROOT, "paper_2606_11402_b200", "csrc")):
        assert "oracle/" not in open(os.path.join(ROOT, "paper_2606_11402_b200", "csrc", f)).read().replace(
            "shared with oracle/", "")


def _graph(gp, n=5000, n0=64, k=8, d=3, dtype=0, nb=3):
    boff = np.array([n0, 1000, 3000, n][: nb + 1], dtype=np.int64)
    g = gp._Graph(n, n0, d, k, nb, dtype, 0, 0, 0x1000, 0x2000, boff.ctypes.data)
    return g, boff


def test_workspace_bytes_host_logic(gp):
    L = gp.lib()
    g, _keep = _graph(gp)
    sizes = [L.gp_workspace_bytes(C.byref(g), op) for op in range(4)]
    assert all(s > 0 and s % 256 == 0 for s in sizes)
    # forward: control + batch offsets + n0 x n0 fp64 head + packed records
    assert sizes[0] >= 64 * 64 * 8 + 5000 * 16
    assert sizes[1] >= 64 * 65 * 8 + 5000 * 16   # inverse carries one extra head row (forward adds its group table)
    assert sizes[3] >= sizes[0] + 2 * 64 * 64 * 8 + 5000 * 4   # VJP: two carried blocks + the running cotangent
    assert L.gp_workspace_bytes(C.byref(g), 7) == 0
    assert L.gp_workspace_bytes(None, 0) == 0
    assert L.gp_graph_build_workspace_bytes(1 << 20, 3, 16, 0) > (1 << 20) * 16 * 4
    assert L.gp_graph_build_workspace_bytes(0, 3, 16, 0) == 0
    assert L.gp_graph_build_workspace_bytes(100, 9, 16, 0) == 0


def test_argument_validation_is_synchronous_and_needs_no_gpu(gp):
    L = gp.lib()
    g, _keep = _graph(gp)
    kern = gp.Kernel("se", 1.0, 0.1, 1e-6).c()
    ws = C.c_void_p(0x10000)
    big = C.c_size_t(1 << 40)
    assert L.gp_forward(None, C.byref(kern), 1, 1, ws, big, None) == gp.GP_ERR_INVALID_ARG
    bad = gp.Kernel("se", 1.0, -0.1, 0.0).c()
    assert L.gp_forward(C.byref(g), C.byref(bad), 1, 1, ws, big, None) == gp.GP_ERR_INVALID_ARG
    g2, _k2 = _graph(gp, k=200)
    assert L.gp_forward(C.byref(g2), C.byref(kern), 1, 1, ws, big, None) == gp.GP_ERR_UNSUPPORTED
    g3, _k3 = _graph(gp, n0=4)                                  # n0 < k
    assert L.gp_inverse(C.byref(g3), C.byref(kern), 1, 1, ws, big, None) == gp.GP_ERR_INVALID_ARG
    assert L.gp_forward(C.byref(g), C.byref(kern), 1, 1, None, 0, None) == gp.GP_ERR_WORKSPACE
    assert L.gp_forward(C.byref(g), C.byref(kern), 1, 1, ws, 16, None) == gp.GP_ERR_WORKSPACE
    boff = np.array([64, 3000, 1000, 5000], dtype=np.int64)      # not increasing
    g4 = gp._Graph(5000, 64, 3, 8, 3, 0, 0, 0, 0x1000, 0x2000, boff.ctypes.data)
    assert L.gp_logdet(C.byref(g4), C.byref(kern), 1, None, ws, big, None) == gp.GP_ERR_INVALID_ARG
    assert gp.status_string(gp.GP_ERR_NOT_PD).startswith("a conditional covariance")


def test_no_cpu_fallback(gp):
    """Without a CUDA device the compute calls return GP_ERR_CUDA and the Python layer raises."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    L = gp.lib()
    g, _keep = _graph(gp)
    kern = gp.Kernel("se", 1.0, 0.1, 1e-6).c()
    ws = C.c_void_p(0x10000)
    assert L.gp_forward(C.byref(g), C.byref(kern), 1, 1, ws, C.c_size_t(1 << 40), None) == gp.GP_ERR_CUDA
    with pytest.raises(RuntimeError):
        gp.gp_graph_build(torch.zeros(10, 3), 2, 4)


def test_specialisation_table(gp):
    assert gp.has_specialised("f32", 16, 3, "matern32")
    assert gp.has_specialised("f64", 8, 3, "se")
    assert not gp.has_specialised("f32", 5, 3, "se")
